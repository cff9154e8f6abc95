// tcw_tables.cuh -- per-search tables of the tCW track sum (sm_100a).
//
//   D[s][j]    = 1 + ((vx*nx + vy*ny) + vz*nz)/c                       eq. (2)
//   g[a][b][j] = RN( ((t_j - T0)/tau_a + 1)^(1/(1 - n_b)) )            eq. (1)
//
// Both are evaluated once per search and shared by every template of a group, so the only
// transcendental of the path (the power) costs n_tau*n_brk*n_sft evaluations instead of one
// per lookup.  D is a chain of single IEEE-754 binary64 operations (the *_rn intrinsics are
// never contracted into FMAs).  g must be the correctly rounded power (reading Q9);
// CUDA's pow() is documented at 2 ulp, so the power is evaluated here in double-double
// arithmetic (two binary64 words, ~2^-100 relative error) as exp(e*log(b)) and rounded once.
// The double-double kernels below restate the classical error-free transformations
// (Knuth two-sum, FMA two-product) and the exp/log scheme of Hida, Li and Bailey's
// "Library for double-double and quad-double arithmetic" in this file's own code.
#pragma once
#include <cuda_runtime.h>

namespace tcw {

struct dd {
    double hi, lo;
};

__device__ __forceinline__ dd two_sum(double a, double b)
{
    double s = __dadd_rn(a, b);
    double bb = __dsub_rn(s, a);
    double e = __dadd_rn(__dsub_rn(a, __dsub_rn(s, bb)), __dsub_rn(b, bb));
    return {s, e};
}

// requires |a| >= |b|
__device__ __forceinline__ dd quick_two_sum(double a, double b)
{
    double s = __dadd_rn(a, b);
    double e = __dsub_rn(b, __dsub_rn(s, a));
    return {s, e};
}

__device__ __forceinline__ dd two_prod(double a, double b)
{
    double p = __dmul_rn(a, b);
    double e = __fma_rn(a, b, -p);
    return {p, e};
}

__device__ __forceinline__ dd dd_add(dd a, dd b)
{
    dd s = two_sum(a.hi, b.hi);
    dd t = two_sum(a.lo, b.lo);
    s.lo = __dadd_rn(s.lo, t.hi);
    s = quick_two_sum(s.hi, s.lo);
    s.lo = __dadd_rn(s.lo, t.lo);
    return quick_two_sum(s.hi, s.lo);
}

__device__ __forceinline__ dd dd_add_d(dd a, double b)
{
    dd s = two_sum(a.hi, b);
    s.lo = __dadd_rn(s.lo, a.lo);
    return quick_two_sum(s.hi, s.lo);
}

__device__ __forceinline__ dd dd_mul(dd a, dd b)
{
    dd p = two_prod(a.hi, b.hi);
    p.lo = __dadd_rn(p.lo, __dadd_rn(__dmul_rn(a.hi, b.lo), __dmul_rn(a.lo, b.hi)));
    return quick_two_sum(p.hi, p.lo);
}

__device__ __forceinline__ dd dd_mul_d(dd a, double b)
{
    dd p = two_prod(a.hi, b);
    p.lo = __dadd_rn(p.lo, __dmul_rn(a.lo, b));
    return quick_two_sum(p.hi, p.lo);
}

__device__ __forceinline__ dd dd_neg(dd a) { return {-a.hi, -a.lo}; }

// exp of a double-double, |a| < 64.  a = k*ln2 + 512*r; exp(r) - 1 by its Taylor series
// (|r| < 6.8e-4, nine terms reach 1e-34); nine squarings (1+s)^2 - 1 = 2s + s^2; scale by 2^k.
__device__ dd dd_exp(dd a)
{
    const dd LN2 = {0.6931471805599453, 2.3190468138462996e-17};
    const dd INV_FACT[9] = {
        {0.16666666666666666, 9.25185853854297e-18},     // 1/3!
        {0.041666666666666664, 2.3129646346357427e-18},  // 1/4!
        {0.008333333333333333, 1.1564823173178714e-19},  // 1/5!
        {0.001388888888888889, -5.300543954373577e-20},  // 1/6!
        {0.0001984126984126984, 1.7209558293420705e-22}, // 1/7!
        {2.48015873015873e-05, 2.1511947866775882e-23},  // 1/8!
        {2.7557319223985893e-06, -1.858393274046472e-22},// 1/9!
        {2.755731922398589e-07, 2.3767714622250297e-23}, // 1/10!
        {2.505210838544172e-08, -1.448814070935912e-24}, // 1/11!
    };
    double kd = rint(__dmul_rn(a.hi, 1.4426950408889634));
    dd r = dd_add(a, dd_neg(dd_mul_d(LN2, kd)));
    r.hi = __dmul_rn(r.hi, 0.001953125);  // exact: 1/512
    r.lo = __dmul_rn(r.lo, 0.001953125);

    dd p = dd_mul(r, r);                       // r^2
    dd s = dd_add(r, {__dmul_rn(p.hi, 0.5), __dmul_rn(p.lo, 0.5)});
    p = dd_mul(p, r);                          // r^3
    dd t = dd_mul(p, INV_FACT[0]);
#pragma unroll 1
    for (int i = 1; i < 9; ++i) {
        s = dd_add(s, t);
        p = dd_mul(p, r);
        t = dd_mul(p, INV_FACT[i]);
    }
    s = dd_add(s, t);
#pragma unroll 1
    for (int i = 0; i < 9; ++i) {
        dd s2 = dd_mul(s, s);
        s = dd_add({__dmul_rn(s.hi, 2.0), __dmul_rn(s.lo, 2.0)}, s2);
    }
    s = dd_add_d(s, 1.0);
    int k = (int)kd;
    return {ldexp(s.hi, k), ldexp(s.lo, k)};
}

// log of a positive double b: y0 = log(b) in binary64, then one Newton step on exp(y) = b in
// double-double, y1 = y0 + b*exp(-y0) - 1, which squares the error of y0.
__device__ dd dd_log_d(double b)
{
    double y0 = log(b);
    dd em = dd_exp({-y0, 0.0});
    dd c = dd_add_d(dd_mul_d(em, b), -1.0);
    return dd_add_d(c, y0);
}

// RN(b^e) for b >= 1 (the base of eq. (1) for t >= T0) and finite e.
__device__ double pow_rn(double b, double e)
{
    dd l = dd_log_d(b);
    dd r = dd_exp(dd_mul_d(l, e));
    return r.hi;  // normalised: |lo| <= ulp(hi)/2, so hi is the nearest double of hi + lo
}

// g[a][b][j], one thread per entry.  Entries with t_j < T0 are 0 (outside the span, reading Q2).
__global__ void __launch_bounds__(128)
spindown_table_kernel(const double *__restrict__ ts, int n_sft, double T0,
                      const double *__restrict__ tau, int n_tau,
                      const double *__restrict__ brk, int n_brk, double *__restrict__ g_out)
{
    long q = (long)blockIdx.x * blockDim.x + threadIdx.x;
    long total = (long)n_tau * n_brk * n_sft;
    if (q >= total) return;
    int j = (int)(q % n_sft);
    int b = (int)((q / n_sft) % n_brk);
    int a = (int)(q / ((long)n_sft * n_brk));
    double t = ts[j];
    if (t < T0) {
        g_out[q] = 0.0;
        return;
    }
    double base = __dadd_rn(__ddiv_rn(__dsub_rn(t, T0), tau[a]), 1.0);
    double e = __ddiv_rn(1.0, __dsub_rn(1.0, brk[b]));
    g_out[q] = pow_rn(base, e);
}

// D = 1 + ((vx*nx + vy*ny) + vz*nz)/c, eq. (2): five single binary64 operations, never fused.
__device__ __forceinline__ double doppler_factor(const double *__restrict__ v, const double *__restrict__ n)
{
    double dot = __dadd_rn(__dadd_rn(__dmul_rn(v[0], n[0]), __dmul_rn(v[1], n[1])), __dmul_rn(v[2], n[2]));
    return __dadd_rn(1.0, __ddiv_rn(dot, 299792458.0));
}

// D[s][j], one thread per entry.
__global__ void __launch_bounds__(256)
doppler_table_kernel(const double *__restrict__ vel, int n_sft, const double *__restrict__ sky,
                     int n_sky, double *__restrict__ d_out)
{
    long q = (long)blockIdx.x * blockDim.x + threadIdx.x;
    long total = (long)n_sky * n_sft;
    if (q >= total) return;
    int j = (int)(q % n_sft);
    int s = (int)(q / n_sft);
    d_out[q] = doppler_factor(vel + 3 * (long)j, sky + 3 * (long)s);
}

}  // namespace tcw
