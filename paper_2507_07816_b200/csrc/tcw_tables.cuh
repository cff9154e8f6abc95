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

#include "tcw_exp_tables.inc"

// exp of a double-double.  a = k*ln2 + i1/64 + i2/4096 + r with |r| <= 2^-13:
// exp(a) = 2^k * T1[i1] * T2[i2] * (1 + s), s = exp(r) - 1 = r + r^2/2 + r^3/6 + tail.  The three
// leading terms are formed in double-double; the tail r^4/24 + ... + r^7/5040 is below 1e-17 and
// plain binary64 carries it to 1e-33.  Tables: exp(i/64), exp(i/4096), i = -32..32, as hi + lo
// (tcw_exp_tables.inc, written by gen_exp_tables.py).  Relative error about 2^-100.
__device__ dd dd_exp(dd a)
{
    const double kd = rint(__dmul_rn(a.hi, 1.4426950408889634));
    dd r = dd_add(a, dd_neg(dd_mul_d(DD_LN2, kd)));          // |r| <= 0.347
    const double i1 = rint(__dmul_rn(r.hi, 64.0));
    r = dd_add_d(r, -__dmul_rn(i1, 0.015625));                // exact products: i/64, i/4096
    const double i2 = rint(__dmul_rn(r.hi, 4096.0));
    r = dd_add_d(r, -__dmul_rn(i2, 0.000244140625));
    const dd r2 = dd_mul(r, r);
    const dd r3 = dd_mul(r2, r);
    const double x = r.hi;
    // r^4/24 (1 + r/5 (1 + r/6 (1 + r/7))) with fused multiply-adds: accuracy, not a defined rounding, matters here
    double tail = __fma_rn(x, 1.0 / 7.0, 1.0);
    tail = __fma_rn(__dmul_rn(x, 1.0 / 6.0), tail, 1.0);
    tail = __fma_rn(__dmul_rn(x, 0.2), tail, 1.0);
    tail = __dmul_rn(__dmul_rn(__dmul_rn(r2.hi, r2.hi), 1.0 / 24.0), tail);
    dd s = dd_add(r, {__dmul_rn(r2.hi, 0.5), __dmul_rn(r2.lo, 0.5)});
    s = dd_add(s, dd_add_d(dd_mul(r3, DD_SIXTH), tail));
    const dd m = dd_mul(EXP_T1[(int)i1 + 32], EXP_T2[(int)i2 + 32]);
    const dd v = dd_add(m, dd_mul(m, s));
    const int k = (int)kd;
    return {ldexp(v.hi, k), ldexp(v.lo, k)};
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

// g[a][b][j] = RN(base^e): one thread per (tau_a, SFT j) evaluates log(base) once in double-double
// and one exp per braking index.  exp returns a normalised pair (|lo| <= ulp(hi)/2), so hi is the
// nearest double of hi + lo.  Entries with t_j < T0 are 0 (outside the span, reading Q2).
__global__ void __launch_bounds__(128)
spindown_table_kernel(const double *__restrict__ ts, int n_sft, double T0,
                      const double *__restrict__ tau, int n_tau,
                      const double *__restrict__ brk, int n_brk, double *__restrict__ g_out)
{
    long q = (long)blockIdx.x * blockDim.x + threadIdx.x;
    long total = (long)n_tau * n_sft;
    if (q >= total) return;
    const int j = (int)(q % n_sft);
    const int a = (int)(q / n_sft);
    double *out = g_out + (long)a * n_brk * n_sft + j;
    const double t = ts[j];
    if (t < T0) {
        for (int b = 0; b < n_brk; ++b) out[(long)b * n_sft] = 0.0;
        return;
    }
    const double base = __dadd_rn(__ddiv_rn(__dsub_rn(t, T0), tau[a]), 1.0);
    const dd l = dd_log_d(base);
    for (int b = 0; b < n_brk; ++b) {
        const double e = __ddiv_rn(1.0, __dsub_rn(1.0, brk[b]));
        out[(long)b * n_sft] = dd_exp(dd_mul_d(l, e)).hi;
    }
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
