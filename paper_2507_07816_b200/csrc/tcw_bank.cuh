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
//   1. fast:  x~ = (f0*T) * exp2(e * log2(1 + (t_j - T0)/tau)) * D  in plain binary64.  Its relative
//      distance from the oracle's x is below 2^-43.9 (error budget in DESIGN.md section 7: CUDA's
//      log2 and exp2 are 1-ulp functions; |e| <= 2^10 and |e*log2 b| <= 2^8 are checked).
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
    const long q = (long)blockIdx.x * BANK_THREADS + threadIdx.x;
    const bool valid = q < p.n_tpl;
    const long qq = valid ? q : p.n_tpl - 1;
    const double f0 = p.f0[qq], tau = p.tau[qq], brk = p.brk[qq];
    double nx = 0, ny = 0, nz = 0;
    if (!p.dshared) { nx = p.sky[3 * qq]; ny = p.sky[3 * qq + 1]; nz = p.sky[3 * qq + 2]; }
    const double inv_tau = 1.0 / tau;
    const double e = __ddiv_rn(1.0, __dsub_rn(1.0, brk));
    const double f0T = f0 * p.T;
    const bool fast_ok = fabs(e) <= 1024.0;
    const double below = (double)p.k_min - 1.0;
    constexpr double INV_C = 1.0 / 299792458.0;
    constexpr double GUARD = 9.094947017729282e-13;   // 2^-40

    V acc = 0;
    int inband = 0;
    unsigned int n_exact = 0;
    int *kq = p.out_k && valid ? p.out_k + q * p.n_sft : nullptr;
    if (kq)
        for (int j = 0; j < p.j_begin; ++j) kq[j] = INT32_MIN;
    for (int j = p.j_begin; j < p.n_sft; ++j) {
        const double dt = __dsub_rn(__ldg(p.ts + j), p.T0);
        double D;
        if (p.dshared) D = __ldg(p.dshared + j);
        else {
            const double *v = p.vel + 3 * (long)j;
            D = fma(fma(__ldg(v + 2), nz, fma(__ldg(v + 1), ny, __ldg(v) * nx)), INV_C, 1.0);
        }
        const double b = fma(dt, inv_tau, 1.0);
        const double E = e * log2(b);
        const double g = exp2(E);
        const double x = f0T * g * D;
        // the track only moves down (g decreases with t): once it is a whole bin below the band for
        // the largest Doppler factor, it stays there
        if (!kq && f0T * g * p.dmax < below) break;
        const double y = x + TCW_MAGIC;
        int lo = __double2loint(y);
        const double d = x - (y - TCW_MAGIC);
        if (!(fabs(d) < 0.5 - x * GUARD) || !fast_ok || !(fabs(E) <= 256.0)) {
            double De = D;
            if (!p.dshared) {
                const double nv[3] = {nx, ny, nz};
                De = doppler_factor(p.vel + 3 * (long)j, nv);
            }
            lo = bank_exact_bin<TPOW2>(__ldg(p.ts + j), p.T0, tau, brk, f0, De, p.T);
            ++n_exact;
        }
        const int k = lo - p.k_min;
        if (kq) kq[j] = k;
        if ((unsigned)k < (unsigned)p.n_bins) {
            const unsigned char *row = p.spec + (long)j * p.pitch;
            if (FMT == FMT_F32) acc += __ldg((const float *)row + k);
            else acc += (V)__ldg(row + k);
            ++inband;
        }
    }
    if (valid) {
        ((V *)p.out_stat)[q] = acc;
        if (p.out_inband) p.out_inband[q] = inband;
        if (n_exact) atomicAdd(p.n_exact, (unsigned long long)n_exact);
    }
}

}  // namespace tcw
