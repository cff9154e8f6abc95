/* oracle/tcw_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow CPU definition of the tCW track sum of arxiv 2507.07816 (Merou, Tenorio,
 * Sintes), written from the paper and sharing no code, header, table or constant with the
 * CUDA path under paper_2507_07816_b200/.  Only tests/, __graft_entry__.smoke() and the
 * cpu_baseline / --impl reference legs of bench.py may load it.
 *
 * What it computes, per template (f0, tau, n, n-hat) and per SFT j with t_j >= T0
 * (section 1 eq. (1), eq. (2); section 2 "summed across the data bins selected by
 * the track"; readings Q1-Q19 in DESIGN.md section 3):
 *
 *   1  b    = (t_j - T0) / tau + 1.0                  eq. (1) base
 *   2  e    = 1.0 / (1.0 - n)                         eq. (1) exponent
 *   3  g    = RN(b ^ e)                               correctly rounded power of the doubles b, e
 *   4  fgw  = f0 * g                                  eq. (1)
 *   5  beta = ((vx*nx + vy*ny) + vz*nz) / c           eq. (2)
 *   6  D    = 1.0 + beta                              eq. (2)
 *   7  fhat = fgw * D                                 eq. (2)
 *   8  x    = fhat * T_sft
 *   9  k    = rint(x) - k_min                         round half to even; k_min = rint(f_min*T_sft)
 *  10  if 0 <= k < n_bins:  s += rho[j][k]  (or nu[j][k])   out-of-band bins are skipped
 *
 * Every line is one IEEE-754 binary64 operation (compile with -ffp-contract=off, no
 * -ffast-math).  Power sums accumulate in float64 in ascending j, counts in int64.
 * Step 3 uses libquadmath powq (113-bit) rounded once to double; it can differ from the
 * correctly rounded value only if b^e lies within ~2^-112 (relative) of the midpoint of two
 * doubles.  tcwo_spindown_table reports how close each entry comes (`hard` flag at 2^-90).
 *
 * Mode `literal` = 1 evaluates steps 1-3 inside the (template, SFT) loop exactly as listed.
 * Mode 0 evaluates the same function tcwo_spindown once per (tau, n, j) and reuses the value
 * across f0 and sky; tests/test_oracle_pins.py checks the two modes agree bit for bit.
 * Parity status: pinned (see tests/test_oracle_pins.py and tests/golden/).
 */
#include <math.h>
#include <quadmath.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define TCWO_C_LIGHT 299792458.0 /* m/s, exact by definition of the metre */

enum { TCWO_F32_POWER = 0, TCWO_U8_COUNT = 1, TCWO_BIT_COUNT = 2 };

/* steps 1-3: spin-down factor g of eq. (1) */
double tcwo_spindown(double t, double T0, double tau, double n)
{
    double b = (t - T0) / tau + 1.0;
    double e = 1.0 / (1.0 - n);
    __float128 gq = powq((__float128)b, (__float128)e);
    return (double)gq;
}

/* steps 5-6: Doppler factor of eq. (2) */
double tcwo_doppler(const double *v, const double *nhat)
{
    double beta = ((v[0] * nhat[0] + v[1] * nhat[1]) + v[2] * nhat[2]) / TCWO_C_LIGHT;
    return 1.0 + beta;
}

/* steps 4, 7, 8: x = ((f0*g)*D)*T_sft, in bins */
double tcwo_track_x(double f0, double g, double D, double T_sft)
{
    double fgw = f0 * g;
    double fhat = fgw * D;
    return fhat * T_sft;
}

/* step 9 */
long tcwo_bin(double x, long k_min)
{
    return (long)rint(x) - k_min; /* default rounding mode: half to even */
}

long tcwo_kmin(double f_min, double T_sft)
{
    return (long)rint(f_min * T_sft);
}

/* OpenMP thread count of the following calls (bench.py times the oracle with all cores and with one) */
void tcwo_set_num_threads(int n)
{
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

int tcwo_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* g[a][b][j] for the whole grid, by the same function as above.  hard[...] (optional) is set
 * where the 113-bit value lies within 2^-90 (relative) of a double rounding boundary, i.e.
 * where "correctly rounded" is not certain at quad precision.  Entries with t_j < T0 are 0. */
void tcwo_spindown_table(int n_sft, const double *ts, double T0, int n_tau, const double *tau,
                         int n_brk, const double *brk, double *g_out, unsigned char *hard)
{
    long total = (long)n_tau * n_brk * n_sft;
#pragma omp parallel for schedule(static)
    for (long q = 0; q < total; ++q) {
        int j = (int)(q % n_sft);
        int b = (int)((q / n_sft) % n_brk);
        int a = (int)(q / ((long)n_sft * n_brk));
        if (ts[j] < T0) {
            g_out[q] = 0.0;
            if (hard) hard[q] = 0;
            continue;
        }
        double g = tcwo_spindown(ts[j], T0, tau[a], brk[b]);
        g_out[q] = g;
        if (hard) {
            double base = (ts[j] - T0) / tau[a] + 1.0;
            double e = 1.0 / (1.0 - brk[b]);
            __float128 gq = powq((__float128)base, (__float128)e);
            /* distance of gq from the nearer of the two midpoints next to g */
            double up = nextafter(g, INFINITY), dn = nextafter(g, -INFINITY);
            __float128 m1 = ((__float128)g + (__float128)up) / 2, m0 = ((__float128)g + (__float128)dn) / 2;
            __float128 d1 = fabsq(gq - m1), d0 = fabsq(gq - m0);
            __float128 d = d1 < d0 ? d1 : d0;
            hard[q] = (d < fabsq(gq) * 0x1p-90Q) ? 1 : 0;
        }
    }
}

void tcwo_doppler_table(int n_sft, const double *vel, int n_sky, const double *sky, double *d_out)
{
    long total = (long)n_sky * n_sft;
#pragma omp parallel for schedule(static)
    for (long q = 0; q < total; ++q) {
        int j = (int)(q % n_sft);
        int s = (int)(q / n_sft);
        d_out[q] = tcwo_doppler(vel + 3 * (long)j, sky + 3 * (long)s);
    }
}

static inline double spec_value(const unsigned char *spec, int format, long pitch, int j, long k)
{
    const unsigned char *row = spec + (long)j * pitch;
    if (format == TCWO_F32_POWER) return (double)((const float *)row)[k];
    if (format == TCWO_U8_COUNT) return (double)row[k];
    return (double)((((const uint32_t *)row)[k >> 5] >> (k & 31)) & 1u);
}

/* The track sum.  Template linear index = ((s*n_tau + a)*n_brk + b)*n_f0 + i (f0 fastest).
 * sel == NULL evaluates templates [0, n_sel) in order; otherwise the listed indices.
 * Outputs (any may be NULL): stat_f64 [n_sel] (power formats: float64 sum; count formats: the
 * exact count as a double), stat_i64 [n_sel] (count formats only), k_out [n_sel][n_sft] with
 * INT32_MIN where t_j < T0, n_inband [n_sel], n_ambig [n_sel] = lookups whose x lies within
 * 1e-9 bin of a half-integer (reading Q10).  Returns 0, or -1 on bad arguments. */
int tcwo_eval(const void *spectrogram, int format, long pitch_bytes, int n_sft, int n_bins,
              double f_min, double T_sft, const double *ts, const double *vel, double T0,
              int n_f0, const double *f0, int n_tau, const double *tau, int n_brk,
              const double *brk, int n_sky, const double *sky, long n_sel, const long *sel,
              double *stat_f64, long long *stat_i64, int32_t *k_out, int32_t *n_inband,
              int32_t *n_ambig, int literal)
{
    if (!spectrogram || !ts || !vel || !f0 || !tau || !brk || !sky) return -1;
    if (format < 0 || format > 2 || n_sft <= 0 || n_bins <= 0) return -1;
    const unsigned char *spec = (const unsigned char *)spectrogram;
    const long k_min = tcwo_kmin(f_min, T_sft);
    const long n_templates = (long)n_sky * n_tau * n_brk * n_f0;

    double *gtab = NULL;
    if (!literal) {
        gtab = (double *)malloc(sizeof(double) * (size_t)n_tau * n_brk * n_sft);
        if (!gtab) return -1;
        tcwo_spindown_table(n_sft, ts, T0, n_tau, tau, n_brk, brk, gtab, NULL);
    }

    int bad = 0;
#pragma omp parallel for schedule(dynamic, 16)
    for (long q = 0; q < n_sel; ++q) {
        long lin = sel ? sel[q] : q;
        if (lin < 0 || lin >= n_templates) {
#pragma omp atomic write
            bad = 1;
            continue;
        }
        int i = (int)(lin % n_f0);
        long grp = lin / n_f0;
        int b = (int)(grp % n_brk);
        int a = (int)((grp / n_brk) % n_tau);
        int s = (int)(grp / ((long)n_brk * n_tau));

        double sum = 0.0;
        long long cnt = 0;
        int32_t inband = 0, ambig = 0;
        for (int j = 0; j < n_sft; ++j) {
            if (ts[j] < T0) { /* before the signal starts: outside the span (Q2) */
                if (k_out) k_out[q * n_sft + j] = INT32_MIN;
                continue;
            }
            double g = literal ? tcwo_spindown(ts[j], T0, tau[a], brk[b])
                               : gtab[((long)a * n_brk + b) * n_sft + j];
            double D = tcwo_doppler(vel + 3 * (long)j, sky + 3 * (long)s);
            double x = tcwo_track_x(f0[i], g, D, T_sft);
            long k = tcwo_bin(x, k_min);
            if (k_out) k_out[q * n_sft + j] = (int32_t)k;
            double fr = x - floor(x);
            if (fabs(fr - 0.5) < 1e-9) ambig++;
            if (k >= 0 && k < n_bins) {
                inband++;
                if (format == TCWO_F32_POWER)
                    sum += spec_value(spec, format, pitch_bytes, j, k);
                else
                    cnt += (long long)spec_value(spec, format, pitch_bytes, j, k);
            }
        }
        if (format != TCWO_F32_POWER) sum = (double)cnt;
        if (stat_f64) stat_f64[q] = sum;
        if (stat_i64) stat_i64[q] = cnt;
        if (n_inband) n_inband[q] = inband;
        if (n_ambig) n_ambig[q] = ambig;
    }
    free(gtab);
    return bad ? -1 : 0;
}

/* ---- NEXT-1: weighted statistic and critical ratio ------------------
 *
 * "The power and number count statistics are weighed taking into account the antenna patterns
 * and changing noise floors ... summed across the data bins selected by the track"
 * and the critical ratio of eq. (4):  Psi_s = (s - <s>) / sigma_s.
 * The weight formula is in the paper's ref. [14], which is not available: weights are an INPUT,
 * w[s][j] >= 0 per (sky point, SFT) (reading Q21).  Per template, over the SFTs j
 * with t_j >= T0 whose bin k_j (steps 1-9 above) is in band:
 *
 *  11  s   += (double) w[s][j] * (double) spectrogram[j][k_j]
 *  12  W1  += (double) w[s][j]
 *  13  W2  += (double) w[s][j] * (double) w[s][j]
 *  14  <s>      = mean1 * W1          mean of a weighted sum of independent bins of mean mean1
 *  15  sigma_s  = sqrt(var1 * W2)     its standard deviation (reading Q14: sigma_s is the
 *                                     standard deviation), bins of variance var1
 *  16  Psi      = (s - <s>) / sigma_s,  0 when W2 == 0 (no in-band SFT carries weight)
 *
 * (mean1, var1) are the per-bin noise moments of the spectrogram: (1, 1) for normalised power
 * rho ~ Exp(1); (p, p(1-p)) with p = exp(-threshold) for the number count nu.  weights == NULL
 * means w = 1.  Outputs (any may be NULL): s_out, w1_out, w2_out, psi_out, each [n_sel].
 * `literal` as in tcwo_eval.
 * Parity status: pinned (tests/test_oracle_pins.py, section "weighted"). */
int tcwo_eval_weighted(const void *spectrogram, int format, long pitch_bytes, int n_sft, int n_bins,
                       double f_min, double T_sft, const double *ts, const double *vel, double T0,
                       int n_f0, const double *f0, int n_tau, const double *tau, int n_brk,
                       const double *brk, int n_sky, const double *sky, const float *weights,
                       double mean1, double var1, long n_sel, const long *sel, double *s_out,
                       double *w1_out, double *w2_out, double *psi_out, int literal)
{
    if (!spectrogram || !ts || !vel || !f0 || !tau || !brk || !sky) return -1;
    if (format < 0 || format > 2 || n_sft <= 0 || n_bins <= 0) return -1;
    const unsigned char *spec = (const unsigned char *)spectrogram;
    const long k_min = tcwo_kmin(f_min, T_sft);
    const long n_templates = (long)n_sky * n_tau * n_brk * n_f0;
    double *gtab = NULL;
    if (!literal) { /* as in tcwo_eval: the same tcwo_spindown, evaluated once per (tau, n, j) */
        gtab = (double *)malloc(sizeof(double) * (size_t)n_tau * n_brk * n_sft);
        if (!gtab) return -1;
        tcwo_spindown_table(n_sft, ts, T0, n_tau, tau, n_brk, brk, gtab, NULL);
    }
    int bad = 0;
#pragma omp parallel for schedule(dynamic, 16)
    for (long q = 0; q < n_sel; ++q) {
        long lin = sel ? sel[q] : q;
        if (lin < 0 || lin >= n_templates) {
#pragma omp atomic write
            bad = 1;
            continue;
        }
        int i = (int)(lin % n_f0);
        long grp = lin / n_f0;
        int b = (int)(grp % n_brk);
        int a = (int)((grp / n_brk) % n_tau);
        int s = (int)(grp / ((long)n_brk * n_tau));
        double sum = 0.0, W1 = 0.0, W2 = 0.0;
        for (int j = 0; j < n_sft; ++j) {
            if (ts[j] < T0) continue;
            double g = literal ? tcwo_spindown(ts[j], T0, tau[a], brk[b])
                               : gtab[((long)a * n_brk + b) * n_sft + j];
            double D = tcwo_doppler(vel + 3 * (long)j, sky + 3 * (long)s);
            double x = tcwo_track_x(f0[i], g, D, T_sft);
            long k = tcwo_bin(x, k_min);
            if (k >= 0 && k < n_bins) {
                double w = weights ? (double)weights[(long)s * n_sft + j] : 1.0;
                sum += w * spec_value(spec, format, pitch_bytes, j, k);
                W1 += w;
                W2 += w * w;
            }
        }
        double mean = mean1 * W1;
        double sigma = sqrt(var1 * W2);
        if (s_out) s_out[q] = sum;
        if (w1_out) w1_out[q] = W1;
        if (w2_out) w2_out[q] = W2;
        if (psi_out) psi_out[q] = W2 > 0.0 ? (sum - mean) / sigma : 0.0;
    }
    free(gtab);
    return bad ? -1 : 0;
}

/* ---- NEXT-2: uniform random template bank --------------------------
 *
 * "(ii) the uniform random template bank that samples templates from a uniform prior over the
 * parameter space".  Every template q carries its own (f0, tau, n) and, unless
 * sky_shared, its own n-hat; with sky_shared all templates use sky[0..2] ("each template used the
 * T0, and sky position values of the injection being searched for").  The statistic
 * is the same ten steps as tcwo_eval, evaluated literally per (template, SFT): nothing is hoisted,
 * g is the correctly rounded power evaluated for every lookup.
 * Outputs as in tcwo_eval (any may be NULL).  Parity status: pinned (tests/test_oracle_bank_pins.py). */
int tcwo_eval_bank(const void *spectrogram, int format, long pitch_bytes, int n_sft, int n_bins,
                   double f_min, double T_sft, const double *ts, const double *vel, double T0,
                   long n_tpl, const double *f0, const double *tau, const double *brk,
                   const double *sky, int sky_shared, double *stat_f64, long long *stat_i64,
                   int32_t *k_out, int32_t *n_inband, int32_t *n_ambig)
{
    if (!spectrogram || !ts || !vel || !f0 || !tau || !brk || !sky) return -1;
    if (format < 0 || format > 2 || n_sft <= 0 || n_bins <= 0 || n_tpl < 0) return -1;
    const unsigned char *spec = (const unsigned char *)spectrogram;
    const long k_min = tcwo_kmin(f_min, T_sft);
#pragma omp parallel for schedule(dynamic, 16)
    for (long q = 0; q < n_tpl; ++q) {
        const double *nhat = sky + (sky_shared ? 0 : 3 * q);
        double sum = 0.0;
        long long cnt = 0;
        int32_t inband = 0, ambig = 0;
        for (int j = 0; j < n_sft; ++j) {
            if (ts[j] < T0) {
                if (k_out) k_out[q * n_sft + j] = INT32_MIN;
                continue;
            }
            double g = tcwo_spindown(ts[j], T0, tau[q], brk[q]);
            double D = tcwo_doppler(vel + 3 * (long)j, nhat);
            double x = tcwo_track_x(f0[q], g, D, T_sft);
            long k = tcwo_bin(x, k_min);
            if (k_out) k_out[q * n_sft + j] = (int32_t)k;
            double fr = x - floor(x);
            if (fabs(fr - 0.5) < 1e-9) ambig++;
            if (k >= 0 && k < n_bins) {
                inband++;
                if (format == TCWO_F32_POWER)
                    sum += spec_value(spec, format, pitch_bytes, j, k);
                else
                    cnt += (long long)spec_value(spec, format, pitch_bytes, j, k);
            }
        }
        if (format != TCWO_F32_POWER) sum = (double)cnt;
        if (stat_f64) stat_f64[q] = sum;
        if (stat_i64) stat_i64[q] = cnt;
        if (n_inband) n_inband[q] = inband;
        if (n_ambig) n_ambig[q] = ambig;
    }
    return 0;
}

/* Candidate reduction (north_star (d)): per group of n_f0 consecutive entries,
 * the maximum and the lowest f0 index attaining it. */
void tcwo_best_f64(const double *stat, long n_groups, int n_f0, double *best_val, int32_t *best_idx)
{
    for (long gq = 0; gq < n_groups; ++gq) {
        const double *p = stat + gq * n_f0;
        double m = p[0];
        int32_t mi = 0;
        for (int i = 1; i < n_f0; ++i)
            if (p[i] > m) { m = p[i]; mi = i; }
        best_val[gq] = m;
        best_idx[gq] = mi;
    }
}

void tcwo_best_i64(const long long *stat, long n_groups, int n_f0, long long *best_val, int32_t *best_idx)
{
    for (long gq = 0; gq < n_groups; ++gq) {
        const long long *p = stat + gq * n_f0;
        long long m = p[0];
        int32_t mi = 0;
        for (int i = 1; i < n_f0; ++i)
            if (p[i] > m) { m = p[i]; mi = i; }
        best_val[gq] = m;
        best_idx[gq] = mi;
    }
}
