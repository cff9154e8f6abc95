// tcw_bank.cuh -- track sum over a random template bank (sm_100a).
//
// "(ii) the uniform random template bank that samples templates from a uniform prior over the
// parameter space".  Every template carries its own (f0, tau, n) and optionally its own
// n-hat, so nothing of eq. (1) can be shared between templates: there is one power per (template,
// SFT) and the templates' tracks have no common window to stage.  One thread owns one template and
// walks the SFTs in order; all threads of the grid are at about the same SFT at the same time, so
// the spectrogram row in use is served from L1/L2.
//
// The bin index must equal the oracle's, which is defined through the correctly rounded power
// (reading Q9).  A correctly rounded power per lookup would cost several hundred FP64
// operations, so the kernel decides the bin in two steps:
//   1. fast:  x~ = (f0*T) * exp2(e * log2(1 + (t_j - T0)/tau)) * D  in plain binary64, with a
//      table-driven log2 and exp2 (bank_pow below, about 20 FP64 operations).  Its relative distance
//      from the oracle's x is below 2^-45 (error budget in DESIGN.md section 7; it needs
//      |e| <= 4, base < 2^40 and |e*log2 base| <= 64, which are checked once per template).
//   2. if x~ lies within x~ * 2^-40 of a half-integer (about 1.5e-8 of all lookups at 1 kHz), or
//      the checks of step 1 fail, the bin is recomputed by the defining chain: base and exponent
//      in single IEEE operations, the double-double power of tcw_tables.cuh rounded once, then
//      ((f0*g)*D)*T with the magic-add rounding -- the same device function the table kernel uses.
// Otherwise rint(x~) = rint(x): the two values are on the same side of every rounding boundary.
#pragma once
#include "tcw_sum.cuh"
#include "tcw_tables.cuh"

namespace tcw {

struct BankParams {
    const unsigned char *spec;   // bin 0 of row 0 of the library's copy
    long pitch;
    int n_sft, n_bins, k_min, j_begin;
    double T, T0;
    const double *ts;            // [n_sft]
    const double *vel;           // [n_sft][3]
    const double *dshared;       // [n_sft] exact Doppler factor of the shared sky point (sky_shared), else NULL
    long n_tpl;
    const double *f0, *tau, *brk;   // [n_tpl]
    const double *sky;           // [n_tpl][3] (ignored when dshared is set)
    double dmax;                 // upper bound of D over every sky point and SFT
    void *out_stat;              // float32 / int32 [n_tpl]
    int *out_inband;             // [n_tpl] or NULL
    int *out_k;                  // [n_tpl][n_sft] or NULL (inspection)
    unsigned long long *n_exact; // lookups decided by the defining chain
};

constexpr int BANK_THREADS = 128;

#include "tcw_pow_tables.inc"
// polynomial coefficients as constant-bank operands of the FMAs (no per-iteration materialisation)
__constant__ double BANK_LC[6] = {POW_LC0, POW_LC1, POW_LC2, POW_LC3, POW_LC4, POW_LC5};
__constant__ double BANK_EC[6] = {POW_EC0, POW_EC1, POW_EC2, POW_EC3, POW_EC4, POW_EC5};
constexpr int BANK_CH = 256;   // SFTs whose per-SFT data (t_j - T0, Doppler factor or velocity) are staged in shared memory at a time

// 2^y and y = e*log2(b) for 1 <= b < 2^40, in plain binary64 (a few ulp; no defined rounding).
//   log2: b = 2^E * m, interval i = top 7 mantissa bits, u = m*r_i - 1 (one FMA, |u| <= 2^-8),
//         log2 b = E + L_i + u*P(u), P = degree-5 Taylor polynomial of log2(1+u)/u.
//   exp2: y = (64 q + j)/64 + r with |r| <= 2^-7 (magic-add rounding; r is exact),
//         2^y = 2^q * T_j * (1 + r*Q(r)), Q = degree-5 Taylor polynomial of (2^r - 1)/r.
// logt/expt are the shared-memory copies of POW_LOGT / POW_EXPT.
__device__ __forceinline__ double bank_pow(double b, double e, const double2 *logt, const double *expt, double &y_out)
{
    const int hi = __double2hiint(b);
    const int E = (hi >> 20) - 1023;
    const double m = __hiloint2double((hi & 0x000fffff) | 0x3ff00000, __double2loint(b));
    const double2 rl = logt[(hi >> 13) & 127];
    const double u = fma(m, rl.x, -1.0);
    double P = fma(u, BANK_LC[5], BANK_LC[4]);
    P = fma(u, P, BANK_LC[3]);
    P = fma(u, P, BANK_LC[2]);
    P = fma(u, P, BANK_LC[1]);
    P = fma(u, P, BANK_LC[0]);
    // (double)E without a conversion instruction: 2^52 + 2^51 + E, minus the magic
    const double Ed = __hiloint2double(0x43380000, E) - TCW_MAGIC;
    const double l2 = fma(u, P, rl.y + Ed);
    const double y = e * l2;
    y_out = y;
    const double t = fma(y, 64.0, TCW_MAGIC);
    const int n = __double2loint(t);
    const double r = fma(t - TCW_MAGIC, -0.015625, y);
    double Q = fma(r, BANK_EC[5], BANK_EC[4]);
    Q = fma(r, Q, BANK_EC[3]);
    Q = fma(r, Q, BANK_EC[2]);
    Q = fma(r, Q, BANK_EC[1]);
    Q = fma(r, Q, BANK_EC[0]);
    const double T = expt[n & 63];
    const double v = fma(T, r * Q, T);
    return __hiloint2double(__double2hiint(v) + (n >> 6) * 1048576, __double2loint(v));
}

// The defining chain of SURVEY.md section 8(c), steps 1-9, for one lookup.
template <bool TPOW2>
__device__ __noinline__ int bank_exact_bin(double t, double T0, double tau, double brk, double f0, double D, double T)
{
    const double base = __dadd_rn(__ddiv_rn(__dsub_rn(t, T0), tau), 1.0);
    const double e = __ddiv_rn(1.0, __dsub_rn(1.0, brk));
    const double g = dd_exp(dd_mul_d(dd_log_d(base), e)).hi;
    const double Dp = TPOW2 ? __dmul_rn(D, T) : D;
    return bin_lo<TPOW2>(f0, g, Dp, T);
}

template <int FMT, bool TPOW2>
__global__ void __launch_bounds__(BANK_THREADS)
sum_bank_kernel(const BankParams p)
{
    typedef typename Acc<FMT>::type V;
    __shared__ double2 logt[128];
    __shared__ double expt[64];
    if (threadIdx.x < 128) logt[threadIdx.x] = make_double2(POW_LOGT[2 * threadIdx.x], POW_LOGT[2 * threadIdx.x + 1]);
    if (threadIdx.x < 64) expt[threadIdx.x] = POW_EXPT[threadIdx.x];
    __syncthreads();
    const long q = (long)blockIdx.x * BANK_THREADS + threadIdx.x;
    const bool valid = q < p.n_tpl;
    const long qq = valid ? q : p.n_tpl - 1;
    const double f0 = p.f0[qq], tau = p.tau[qq], brk = p.brk[qq];
    double nx = 0, ny = 0, nz = 0;
    if (!p.dshared) { nx = p.sky[3 * qq]; ny = p.sky[3 * qq + 1]; nz = p.sky[3 * qq + 2]; }
    const double inv_tau = 1.0 / tau;
    const double e = __ddiv_rn(1.0, __dsub_rn(1.0, brk));
    const double f0T = f0 * p.T;
    // preconditions of the fast evaluation, checked once per template: the base grows with t, so its
    // largest value (last SFT) bounds both the base and |e*log2(base)| of every lookup
    const double b_last = fma(__dsub_rn(__ldg(p.ts + p.n_sft - 1), p.T0), inv_tau, 1.0);
    const bool fast_ok = fabs(e) <= 4.0 && b_last < 1.0e12 && fabs(e) * log2(fmax(b_last, 1.0)) <= 63.0;
    const double below = (double)p.k_min - 1.0;
    constexpr double INV_C = 1.0 / 299792458.0;
    constexpr double GUARD = 9.094947017729282e-13;   // 2^-40

    V acc = 0, pend = 0, pend2 = 0;   // gathered elements in flight (even / odd SFTs of a chunk): added two SFTs later, so
                                      // the load latency overlaps the next bins; the order of the additions stays fixed
    int inband = 0;
    unsigned int n_exact = 0;
    int *kq = p.out_k && valid ? p.out_k + q * p.n_sft : nullptr;
    if (kq)
        for (int j = 0; j < p.j_begin; ++j) kq[j] = INT32_MIN;
    // per-SFT data of the current chunk: {t_j - T0, D_j, -, -} (shared sky) or {t_j - T0, vx, vy, vz}
    __shared__ double4 sft[BANK_CH];
    bool done = !valid;
    for (int j0 = p.j_begin; j0 < p.n_sft; j0 += BANK_CH) {
        const int nj = min(BANK_CH, p.n_sft - j0);
        __syncthreads();      // the previous chunk has been consumed
        for (int t = threadIdx.x; t < nj; t += BANK_THREADS) {
            const int j = j0 + t;
            double4 c;
            c.x = __dsub_rn(__ldg(p.ts + j), p.T0);
            if (p.dshared) { c.y = __ldg(p.dshared + j); c.z = c.w = 0.0; }
            else { c.y = __ldg(p.vel + 3 * (long)j); c.z = __ldg(p.vel + 3 * (long)j + 1); c.w = __ldg(p.vel + 3 * (long)j + 2); }
            sft[t] = c;
        }
        if (__syncthreads_and(done)) break;   // barrier after the fill; leave when every template of the CTA has left the band
        if (done) continue;
        const unsigned char *row = p.spec + (long)j0 * p.pitch;
        // one SFT of one template; the gathered element lands in `pd` and is added when the same slot
        // is used again, two SFTs later (even and odd SFTs keep separate slots)
        auto step = [&](int t, const unsigned char *rw, V &pd) -> bool {
            const double4 c = sft[t];
            const double D = p.dshared ? c.y : fma(fma(c.w, nz, fma(c.z, ny, c.y * nx)), INV_C, 1.0);
            const double b = fma(c.x, inv_tau, 1.0);
            double E;
            const double g = bank_pow(fast_ok ? b : 1.0, e, logt, expt, E);
            const double fg = f0T * g;
            // the track only moves down (g decreases with t): once it is a whole bin below the band for
            // the largest Doppler factor, it stays there
            if (!kq && fg * p.dmax < below) return false;
            const double x = fg * D;
            const double y = x + TCW_MAGIC;
            int lo = __double2loint(y);
            const double d = x - (y - TCW_MAGIC);
            if (!(fabs(d) < 0.5 - x * GUARD) || !fast_ok) {
                const int j = j0 + t;
                double De = D;
                if (!p.dshared) {
                    const double nv[3] = {nx, ny, nz};
                    De = doppler_factor(p.vel + 3 * (long)j, nv);
                }
                lo = bank_exact_bin<TPOW2>(__ldg(p.ts + j), p.T0, tau, brk, f0, De, p.T);
                ++n_exact;
            }
            const int k = lo - p.k_min;
            if (kq) kq[j0 + t] = k;
            if ((unsigned)k < (unsigned)p.n_bins) {
                acc += pd;
                if (FMT == FMT_F32) pd = __ldg((const float *)rw + k);
                else pd = (V)__ldg(rw + k);
                ++inband;
            }
            return true;
        };
        int t = 0;
        for (; t + 1 < nj; t += 2, row += 2 * p.pitch) {
            if (!step(t, row, pend)) { done = true; break; }
            if (!step(t + 1, row + p.pitch, pend2)) { done = true; break; }
        }
        if (!done && t < nj && !step(t, row, pend)) done = true;
    }
    acc += pend;
    acc += pend2;
    if (valid) {
        ((V *)p.out_stat)[q] = acc;
        if (p.out_inband) p.out_inband[q] = inband;
        if (n_exact) atomicAdd(p.n_exact, (unsigned long long)n_exact);
    }
}

}  // namespace tcw
