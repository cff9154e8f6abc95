/* tcw.h -- C ABI of the B200-native tCW track-sum library (libtcw.so).
 *
 * The operation is the search statistic of arxiv 2507.07816 (Merou, Tenorio, Sintes):
 * "templates ... describe the corresponding time-frequency evolution track of potential signals
 *  in data ... The statistics are then summed across the data bins selected by the track"
 * (section 2).  For a template (f0, tau, n, n-hat) and every SFT j with t_j >= T0
 *
 *     f_gw(t_j)  = f0 * ((t_j - T0)/tau + 1)^(1/(1-n))                  eq. (1)
 *     f_hat(t_j) = f_gw(t_j) * (1 + v(t_j).n-hat / c)                   eq. (2)
 *     k_j        = rint(f_hat(t_j) * T_sft) - k_min,  k_min = rint(f_min * T_sft)
 *     stat       = sum over j with 0 <= k_j < n_bins of spectrogram[j][k_j]
 *
 * where spectrogram[j][k] is the normalised power rho_j[k] or the number count nu_j[k] of
 * SFT j.  Every floating-point step of k_j is one IEEE-754 binary64 operation
 * in the order ((f0*g)*D)*T_sft with g the correctly rounded power and D = 1 + beta,
 * beta = ((vx*nx + vy*ny) + vz*nz)/c, c = 299792458 m/s (readings
 * Q1-Q19).  rint is round-half-to-even.  Out-of-band bins are skipped.  The candidate
 * reduction is the per-(sky, tau, n) maximum over f0 with the lowest f0 index attaining it
 * (PAPER.md:79 compares the best template near a signal with a threshold).
 *
 * Template linear index = ((s*n_tau + a)*n_brk + b)*n_f0 + i   (f0 fastest, sky slowest);
 * a "group" is the n_f0 templates sharing one (s, a, b); group index = (s*n_tau + a)*n_brk + b.
 *
 * All work runs in CUDA kernels for sm_100a on the device that is current at tcw_create.
 * There is no CPU fallback: without a usable CUDA device tcw_create returns TCW_ECUDA.
 *
 * Error behaviour: every function returns an int code (below); nothing is thrown across the
 * ABI; on error no output buffer is written.  tcw_last_error() gives a thread-local message.
 * Argument validation happens before the first CUDA call, so TCW_EINVAL is returned for bad
 * arguments even on a machine with no GPU.
 */
#ifndef TCW_H_
#define TCW_H_

#ifdef __cplusplus
extern "C" {
#endif

typedef struct tcw_handle tcw_handle; /* opaque, owned by the library */

enum {
    TCW_OK = 0,
    TCW_EINVAL = -1,       /* bad argument (NULL, size, ordering, range) */
    TCW_ENOMEM = -2,       /* host or device allocation failed */
    TCW_ECUDA = -3,        /* a CUDA runtime call failed (message in tcw_last_error) */
    TCW_EUNSUPPORTED = -4, /* valid request the library cannot serve */
    TCW_EINTERNAL = -5     /* a kernel found a staged window larger than the bound the host planned and
                              skipped rows: the results of that search are NOT valid (never expected;
                              reported by tcw_search_host, tcw_check, tcw_get_timing, tcw_get_info) */
};

/* Spectrogram element formats (normalised power rho or number count nu). */
enum {
    TCW_F32_POWER = 0, /* float32 [n_sft][n_bins]                                            */
    TCW_U8_COUNT = 1,  /* uint8   [n_sft][n_bins], value added as an integer (0/1 for nu)     */
    TCW_BIT_COUNT = 2  /* uint32 words, bit k of row j = (word[k >> 5] >> (k & 31)) & 1       */
};

/* tcw_create -- bind a spectrogram and its per-SFT metadata to a handle.
 *
 *  out             receives the handle.
 *  spectrogram     SFT-major rows, row j at byte offset j*row_pitch_bytes.  DEVICE pointer, or
 *                  HOST pointer (pageable or pinned): the library copies it with
 *                  cudaMemcpyDefault into its own layout (16-byte-aligned rows with zero bins on
 *                  both sides; bit-packed counts expanded to one byte per bin), so the caller
 *                  may free or overwrite it as soon as tcw_create returns.
 *  format          one of TCW_F32_POWER / TCW_U8_COUNT / TCW_BIT_COUNT.
 *  row_pitch_bytes >= the bytes of one row (4*n_bins, n_bins, 4*ceil(n_bins/32)).
 *  n_sft, n_bins   > 0.  SFTs that are missing are simply absent from the list (reading Q16).
 *  f_min, T_sft    band start (Hz) and SFT length (s); bin k is centred on (k_min + k)/T_sft.
 *                  TCW_EINVAL if |f_min*T_sft - rint(f_min*T_sft)| > 1e-9.
 *  timestamps      HOST, [n_sft], strictly increasing; timestamps[j] IS the time t_j at which
 *                  eq. (1)-(2) are evaluated for SFT j (callers pass mid-SFT times, reading Q1).
 *  velocities      HOST, [n_sft][3], detector velocity wrt the SSB in m/s, equatorial frame.
 *  stream          cudaStream_t (NULL = default stream).  The stream is synchronised before
 *                  tcw_create returns.
 *
 * Device memory of the library (the spectrogram copy, tables, scratch) comes from a library-owned
 * CUDA memory pool per device (stream-ordered allocation on the call's stream); the pool keeps up
 * to 8 GiB of freed blocks for reuse by the next handle, so a create / search / destroy cycle
 * does not pay cudaMalloc / cudaFree.  A contiguous HOST spectrogram is sent in one copy and
 * re-laid on the device.  If a later call on the same handle uses a different stream, the library
 * first waits for the handle's previous stream.
 */
int tcw_create(tcw_handle **out, const void *spectrogram, int format, long row_pitch_bytes,
               int n_sft, int n_bins, double f_min, double T_sft, const double *timestamps,
               const double *velocities, void *stream);

/* tcw_create_async -- tcw_create for a contiguous HOST spectrogram (row_pitch_bytes = bytes of one
 * row; float32 or uint8) that lets the transfer overlap the first search: the rows are sent in
 * pieces on a copy stream owned by the handle, the call returns without waiting for them, and the
 * first search on the handle launches SFT chunk by SFT chunk, each behind the piece that completes
 * its rows.  The caller must keep the host spectrogram valid and unchanged until that first search
 * has completed on its stream, or until tcw_upload_wait returns.  Pinned host memory is needed for
 * the overlap (a pageable array is staged synchronously by the driver).  For any other input
 * (device pointer, padded rows, bit-packed counts) it behaves exactly like tcw_create.  Results are
 * identical to those of a handle made by tcw_create. */
int tcw_create_async(tcw_handle **out, const void *spectrogram, int format, long row_pitch_bytes,
                     int n_sft, int n_bins, double f_min, double T_sft, const double *timestamps,
                     const double *velocities, void *stream);

/* tcw_upload_wait -- block until every piece of a tcw_create_async upload has arrived (a no-op for
 * other handles). */
int tcw_upload_wait(tcw_handle *h);

/* The cubic-lattice template bank: explicit axes, HOST pointers, copied during
 * the call.  Spacing is the caller's business; only f0 must be ascending. */
typedef struct {
    double T0;          /* signal start time, same clock as timestamps; SFTs with t_j < T0 are skipped */
    int n_f0;
    const double *f0;   /* [n_f0] Hz, > 0, strictly ascending                     */
    int n_tau;
    const double *tau;  /* [n_tau] s, > 0                                          */
    int n_brk;
    const double *brk;  /* [n_brk] braking index n, > 1                            */
    int n_sky;
    const double *sky;  /* [n_sky][3] unit vectors n-hat towards the source, equatorial */
} tcw_grid;

/* Candidate record per group.  Power format: stat is float32.  Count formats: the same 8 bytes
 * hold { int32 stat; int32 f0_index }. */
typedef struct {
    float stat;
    int f0_index;
} tcw_best_f32;
typedef struct {
    int stat;
    int f0_index;
} tcw_best_i32;

/* tcw_search -- track sums for the whole grid, and the per-group best template.
 *
 *  out_stat  DEVICE, [n_sky][n_tau][n_brk][n_f0], float32 (power) or int32 (counts); may be NULL.
 *  out_best  DEVICE, [n_sky*n_tau*n_brk] tcw_best_f32 / tcw_best_i32; may be NULL (not both).
 *            Ties go to the lowest f0 index.  A template with no in-band SFT has stat 0 and
 *            still takes part in the maximum.
 *  stream    cudaStream_t.  The call enqueues its kernels and returns; outputs are valid once
 *            the stream has been synchronised.  The grid arrays are copied before returning.
 *            One search at a time per handle.
 *
 * Power sums are accumulated in float32 in a fixed order (run-to-run bit-identical); counts in
 * int32, exact.  TCW_EINVAL for NULL / non-positive sizes, tau <= 0, n <= 1, f0 <= 0 or not
 * ascending, | |n-hat| - 1 | > 1e-6, or f0_max*T_sft >= 2^31 - 2^20.
 */
int tcw_search(tcw_handle *h, const tcw_grid *grid, void *out_stat, void *out_best, void *stream);

/* tcw_search_groups -- tcw_search restricted to the groups [group_begin, group_end) of the grid's
 * flattened group index (s*n_tau + a)*n_brk + b: the unit of the multi-GPU partition (SURVEY.md
 * section 8(e): whole (tau, n, sky) groups per GPU, spectrogram replicated, no collective).
 *  out_stat  DEVICE, [(group_end - group_begin)][n_f0], the range's slice of tcw_search's out_stat; may be NULL.
 *  out_best  DEVICE, [(group_end - group_begin)] candidate records; may be NULL (not both).
 * The range is served as at most seven sub-grid searches (whole sky points, whole tau rows, part of a
 * tau row), enqueued on `stream`; every template is evaluated exactly as by tcw_search -- the
 * SFT-chunk plan, which fixes the float32 summation order, is decided on the WHOLE grid's size for
 * every sub-grid -- so the outputs equal the corresponding slices of a whole-grid search bit for bit.
 * Asynchronous.  TCW_EINVAL for an empty range or one outside 0..n_groups (the Python binding
 * turns an empty in-range interval, a rank with no groups, into a no-op). */
int tcw_search_groups(tcw_handle *h, const tcw_grid *grid, long group_begin, long group_end,
                      void *out_stat, void *out_best, void *stream);

/* tcw_split_groups -- the decomposition tcw_search_groups uses, as a host-only call (no CUDA): the
 * range [group_begin, group_end) of the flattened group index as *n_rects <= 7 sub-grids in
 * ascending group order, rects[i] = { sky_begin, sky_end, tau_begin, tau_end, brk_begin, brk_end }
 * (half-open index ranges).  Each sub-grid's own [sky][tau][brk] order is a contiguous run of the
 * flattened index.  An empty range gives *n_rects = 0.  TCW_EINVAL for non-positive sizes. */
int tcw_split_groups(int n_tau, int n_brk, long group_begin, long group_end, int rects[7][6], int *n_rects);

/* tcw_check -- synchronise the handle's last stream and report whether the last search on it was
 * valid: TCW_OK, or TCW_EINTERNAL if a kernel set the device status word (see TCW_EINTERNAL).
 * tcw_search, tcw_search_weighted, tcw_search_groups and tcw_search_bank are asynchronous and cannot
 * report this themselves: a caller that does not use tcw_search_host should call tcw_check (or
 * tcw_get_info) once the outputs are needed.  Every search clears the status word when it starts. */
int tcw_check(tcw_handle *h);

/* tcw_search_host -- the same search with HOST output buffers (either may be NULL, not both):
 * runs tcw_search into library scratch, copies the results to the host and synchronises the
 * stream before returning.  For an out_stat of 64 MiB or more the search issues its CTAs tau range by
 * tau range, every CTA counts itself done in a per-range device counter, and a second stream waits for
 * each counter (cuStreamWaitValue32) and copies that range while the later ranges are still being
 * searched (pinned host buffers are needed for the overlap).  It is one search, not several: the
 * values are those of tcw_search, bit for bit.  Returns TCW_EINTERNAL if a kernel set the device
 * status word (see above). */
int tcw_search_host(tcw_handle *h, const tcw_grid *grid, void *out_stat_host, void *out_best_host,
                    void *stream);

/* ---- weighted statistic and critical ratio -------------------
 *
 * "The power and number count statistics are weighed taking into account the antenna patterns
 *  and changing noise floors that modulate the signal amplitude.  The statistics are then summed
 *  across the data bins selected by the track. ... we compute the critical ratio
 *  Psi_s = (s - <s>)/sigma_s"  (eq. (4)).
 * The weight formula is in the paper's ref. [14] and is not restated there, so weights are an
 * input (reading Q21).  Over the SFTs j with t_j >= T0 whose bin k_j is in band:
 *
 *     s   = sum_j w[s][j] * spectrogram[j][k_j]        W1 = sum_j w[s][j]      W2 = sum_j w[s][j]^2
 *     <s> = mean1 * W1      sigma_s = sqrt(var1 * W2)      Psi = (s - <s>)/sigma_s,  0 if W2 == 0
 *
 * (the mean and the standard deviation of a weighted sum of independent bins of mean mean1 and
 * variance var1; reading Q14: sigma_s is the standard deviation).
 *
 *  weights   [n_sky][n_sft] float32, row s for sky point s of the grid; HOST or DEVICE pointer
 *            (copied with cudaMemcpyDefault on `stream`: a pageable host array may be freed when
 *            the call returns, a pinned or device array once the stream has passed the call).
 *            NULL = all ones.  Values are not checked: negative or non-finite weights propagate.
 *  mean1     per-bin noise mean of the spectrogram elements: 1 for normalised power rho ~ Exp(1),
 *            p = exp(-threshold) for number counts nu = (rho > threshold).
 *  var1      per-bin noise variance: 1 for rho, p(1-p) for nu.  TCW_EINVAL unless finite and > 0.
 */
typedef struct {
    const float *weights;
    double mean1, var1;
} tcw_weighting;

/* tcw_search_weighted -- weighted statistic, critical ratio and the per-group best critical ratio.
 *
 *  out_psi   DEVICE, float32 [n_sky][n_tau][n_brk][n_f0], Psi per template; may be NULL.
 *  out_stat  DEVICE, float32 (for every spectrogram format), the weighted statistic s; may be NULL.
 *  out_best  DEVICE, [n_sky*n_tau*n_brk] tcw_best_f32 = { max over f0 of Psi, lowest f0 index
 *            attaining it }; may be NULL (not all three NULL).
 *  stream    as for tcw_search (asynchronous).
 *
 * s accumulates in float32 (fused multiply-add of weight and element) in a fixed order; W1 and W2 in
 * float64 (per-chunk partial sums of a chunked search included), except over the SFTs in which a
 * 32*R-template tile straddles a band edge, where they are counted per template in float32.  Runs on the TMA-staged or the
 * gather kernel (one sky point at a time: weights differ between sky points, so the sky-block
 * kernel does not apply; forcing that kernel through tcw_set_option gives TCW_EUNSUPPORTED). */
int tcw_search_weighted(tcw_handle *h, const tcw_grid *grid, const tcw_weighting *weighting,
                        float *out_psi, float *out_stat, tcw_best_f32 *out_best, void *stream);

/* ---- uniform random template bank ---------------------------
 *
 * "(ii) the uniform random template bank that samples templates from a uniform prior over the
 *  parameter space"; "Each template used the T0, and sky position values of the
 *  injection being searched for".  Template q has its own (f0[q], tau[q], brk[q])
 * and either its own unit vector sky[3q..3q+2] or, with sky_shared != 0, the one vector sky[0..2].
 * The statistic of a template is the one tcw_search computes (same bin indices: the kernel decides
 * each bin with a fast binary64 evaluation of eq. (1)-(2) and falls back to the defining chain
 * with the correctly rounded power wherever the fast value lies within x*2^-40 of a rounding
 * boundary).
 * All pointers are HOST arrays, validated and copied with cudaMemcpyAsync during the call
 * (pageable arrays may be freed on return; pinned arrays once the stream has passed the call). */
typedef struct {
    double T0;          /* signal start time; SFTs with t_j < T0 are skipped                  */
    long n;             /* number of templates, > 0                                           */
    const double *f0;   /* [n] Hz, > 0 (any order)                                            */
    const double *tau;  /* [n] s, > 0                                                         */
    const double *brk;  /* [n] braking index, > 1                                             */
    const double *sky;  /* [n][3] unit vectors, or [3] when sky_shared != 0                   */
    int sky_shared;
} tcw_bank;

/* tcw_search_bank -- track sums of a template bank.
 *  out_stat    DEVICE, [n] float32 (power) or int32 (counts); required.
 *  out_inband  DEVICE, [n] int32 number of in-band SFTs of each template (the N of the noise
 *              moments: for unit weights Psi = (s - mean1*N)/sqrt(var1*N)); may be NULL.
 *  out_k       DEVICE, int32 [n][n_sft] bin indices (INT32_MIN where t_j < T0); inspection output
 *              for parity tests, may be NULL (and should be for large banks).
 * Power sums accumulate in float32 in a fixed order (ascending SFT order, except that the kernel keeps two
 * gathers in flight and may add the last two in-band elements in swapped order): deterministic, run-to-run
 * bit-identical; counts exactly.
 * Asynchronous like tcw_search. */
int tcw_search_bank(tcw_handle *h, const tcw_bank *bank, void *out_stat, int *out_inband, int *out_k,
                    void *stream);

/* tcw_get_counter -- diagnostic counters of the last search on this handle (synchronises its
 * stream).  which = 0: lookups of the last tcw_search_bank that were decided by the defining
 * chain (correctly rounded power) instead of the fast evaluation. */
int tcw_get_counter(tcw_handle *h, int which, long long *value);

/* ---- downstream selection ------------------------------------
 *
 * "a threshold was set on Psi based on the distribution of critical ratios on only noise using the
 *  same amount of templates (Psi_noise max).  That is, an injection was considered detected if a
 *  template close to the injection had Psi > Psi_noise max."
 * Both calls read a DEVICE array of n statistics -- dtype 0: float32 (Psi, power sums), 1: int32
 * (counts) -- e.g. an out_psi / out_stat of a search, and are exact and deterministic.
 * NaN is never selected; -0.0 equals +0.0.  Asynchronous on `stream`; `h` supplies the scratch. */

/* tcw_topk -- the K largest values in descending order, equal values in ascending index order
 * (reading Q23).  K in 1..2048, n < 2^32.  K = 1 on a noise-only search is Psi_noise max.  Arrays of 2^22
 * values or more are read twice (zoomed histogram, then ordered compaction of the candidates and an exact
 * selection among them); smaller ones, and heavily tied ones, take five streaming passes.  Same results.
 *  out_val    DEVICE [K], same dtype as values;  out_idx  DEVICE [K] int64 indices into values;
 *  out_count  DEVICE int32 (may be NULL): entries written = min(K, selectable values). */
int tcw_topk(tcw_handle *h, const void *values, int dtype, long n, int K, void *out_val,
             long long *out_idx, int *out_count, void *stream);

/* tcw_select_above -- the indices i with values[i] > threshold, ascending.
 *  out_idx    DEVICE [capacity] int64 (may be NULL when capacity == 0): the first `capacity` hits;
 *  out_count  DEVICE int64: the total number of hits (may exceed capacity). */
int tcw_select_above(tcw_handle *h, const void *values, int dtype, long n, double threshold,
                     long capacity, long long *out_idx, long long *out_count, void *stream);

/* tcw_select_above_static -- tcw_select_above for callers that must not allocate device memory.
 *
 * Who that is: a search job that sized its spectrograms and result arrays to fill the GPU and has
 * nothing left for a library to take; a host program whose own caching allocator owns the device
 * memory, so that a cudaMalloc from inside a library can fail even though "free" memory exists; and a
 * follow-up loop that runs beside searches on other streams, where cudaMalloc / cudaFree would
 * synchronise the whole device and stall them.  The other selection calls take their scratch from
 * the handle's grow-only pool block, and making a handle allocates; this call needs no handle.
 *
 * Same selection, same kernels, same results as tcw_select_above (the templates with
 * Psi > Psi_noise max): the indices i with values[i] > threshold, ascending; NaN never selected.
 * The scratch (per-CTA counts and offsets, one byte per row of 128 values) lives in ONE array that
 * is part of the library image: about 2.1 MB on every GPU that loads libtcw.so, held until the
 * process exits.  The call makes no cudaMalloc, cudaFree, pool or library allocation; the caller
 * supplies inputs and outputs.
 *  values     DEVICE [n], dtype 0: float32, 1: int32;  1 <= n <= TCW_SELECT_STATIC_MAX_N.
 *             A larger n returns TCW_EUNSUPPORTED and touches nothing (use tcw_select_above).
 *  out_idx    DEVICE [capacity] int64 (may be NULL when capacity == 0): the first `capacity` hits;
 *  out_count  DEVICE int64: the total number of hits (may exceed capacity).
 * Works on the CURRENT device (cudaSetDevice before calling); asynchronous on `stream`.
 * First call on each device: looks up the device address of the array (cudaGetSymbolAddress) and
 * keeps it.  Make that first call during set-up, before any stream capture is begun.
 * Sharing: every call on a device uses the same array, and the array keeps what the previous call
 * left in it.  The call itself clears the part that must start at zero (the per-row counts of the
 * rows it covers), so back-to-back calls on one stream are independent.  Two calls that may run
 * at the same time on one GPU (different streams, or different threads) RACE on the array and give
 * wrong results: order them on one stream or with events. */
#define TCW_SELECT_STATIC_MAX_N (1L << 28)
int tcw_select_above_static(const void *values, int dtype, long n, double threshold, long capacity,
                            long long *out_idx, long long *out_count, void *stream);

/* ---- data preparation ----------------------------------------
 *
 * "The data used in this study are 8-second Han-windowed Short Fourier Transforms (SFTs), which
 *  are processed into either normalized power rho_j or number count nu_j as described by Oliver
 *  et al. [14]".  Ref. [14] is not available; reading Q24:
 *    segment j = samples [j*N, (j+1)*N), N = fs*T_sft (no overlap, a trailing partial segment is dropped)
 *    X_j = DFT of w[t]*x_j[t], w[t] = 0.5 - 0.5 cos(2 pi t/N);   P_j[k] = |X_j[k]|^2
 *    m_j[k] = median of P_j[k-h .. k+h], h = (median_bins - 1)/2
 *    rho_j[k] = P_j[k]*ln 2/m_j[k]   (mean 1 in Gaussian noise);   nu_j[k] = rho_j[k] > threshold
 * for the band bins k_min .. k_min + n_bins - 1, k_min = rint(f_min*T_sft).  float32 arithmetic;
 * the DFT is cuFFT's batched real-to-complex transform. */
typedef struct {
    double fs;          /* sampling rate, Hz                                                      */
    double T_sft;       /* SFT length, s; fs*T_sft must be an even integer                        */
    double f_min;       /* band start, Hz; f_min*T_sft must be an integer                         */
    int n_bins;         /* band bins; the band plus h bins on both sides must lie in 0..N/2       */
    int median_bins;    /* running-median window W, odd, 1..1025                                  */
    double threshold;   /* number-count threshold on rho (1.6 in BASELINE.json's configs)         */
} tcw_prep;

/* tcw_prepare -- strain to spectrogram, written in the layout tcw_create reads.
 *  strain           HOST or DEVICE, float32 [n_samples].
 *  format           TCW_F32_POWER (rho), TCW_U8_COUNT or TCW_BIT_COUNT (nu).
 *  out_spectrogram  DEVICE, n_sft rows of out_pitch_bytes (>= one row; a multiple of 4 except for
 *                   uint8), n_sft = n_samples / N rows are written.
 *  n_sft            HOST int, receives the number of SFTs.
 * Synchronises `stream` before returning (scratch is allocated and freed inside the call).
 * TCW_EINVAL for inconsistent sizes; TCW_EUNSUPPORTED if the band does not fit one CTA's shared
 * memory (about 45 000 bins). */
int tcw_prepare(const float *strain, long n_samples, const tcw_prep *prep, int format,
                void *out_spectrogram, long out_pitch_bytes, int *n_sft, void *stream);

/* tcw_destroy -- free the handle and everything it owns.  NULL is a no-op returning TCW_OK. */
int tcw_destroy(tcw_handle *h);

/* tcw_last_error -- thread-local description of the last error on this thread; never NULL. */
const char *tcw_last_error(void);

/* ---- inspection entry points (used by the parity tests and by bench.py) ------------------- */

/* tcw_track_indices -- the bin indices k_j themselves, for the listed templates.
 *  sel      HOST, [n_sel] template linear indices.
 *  out_k    DEVICE, int32 [n_sel][n_sft]; INT32_MIN where t_j < T0.  Computed by the same device
 *           function the search kernels use.  Asynchronous like tcw_search. */
int tcw_track_indices(tcw_handle *h, const tcw_grid *grid, long n_sel, const long *sel,
                      int *out_k, void *stream);

/* tcw_tables -- the two per-search tables of the last tcw_search / tcw_track_indices call:
 *  out_g  HOST, float64 [n_tau][n_brk][n_sft], g = RN(((t_j - T0)/tau + 1)^(1/(1-n))), 0 where t_j < T0
 *  out_d  HOST, float64 [n_sky][n_sft],        D = 1 + beta
 * Either may be NULL.  Synchronises `stream`. */
int tcw_tables(tcw_handle *h, double *out_g, double *out_d, void *stream);

/* tcw_measure_peaks -- microbenchmarks of the limits that bind the track-sum kernels on the current
 * device (SURVEY.md section 0 asks the builder to measure them): kernels that
 * only issue independent instructions of one kind, timed with CUDA events on `stream` (best of three
 * launches after a warm-up).  Whole-GPU rates per second:
 *  out[0] FP64 DFMA warp instructions/s   out[1] FP64 DMUL   out[2] FP64 DADD
 *  out[3] FP32 FFMA warp instructions/s (= the schedulers' issue limit, one per scheduler per cycle)
 *  out[4] LDS.32 warp instructions/s for the staged kernel's gather pattern (conflict-free, stride < 1 word)
 *  out[5] lookups/s of the bare lookup chain of sum_staged_kernel as it ships (two rows per block: DFMA, address,
 *         LDS.32, half a FADD2, half a VIMNMX3 per lookup; no staging, metadata or band edges): the speed of light
 *         of the instruction mix
 *  out[6] number of SMs   out[7] nominal maximum SM clock in Hz
 *  out[8] lookups/s of the count formats' chain with one byte per bin (the device layout: LDS.U8 + IADD)
 *  out[9] the same chain gathering from bit-packed windows (LDS.U8 of byte k >> 3, shift by k & 7, mask):
 *         the measurement behind keeping one byte per bin on the device
 *  out[10] bytes/s the staged kernel's per-warp ring draws from L2 into shared memory when it stages alone (no
 *          consumer) with four 1-D bulk copies per slot, out[11] the same with one tensor-map copy per slot
 *          (both only when n_out >= 12; 0 if the tensor maps cannot be encoded)
 * n_out must be >= 10.  Synchronous; takes about 0.2 s. */
int tcw_measure_peaks(double *out, int n_out, void *stream);

/* Options.  tcw_set_option returns TCW_EINVAL for an unknown key or value. */
enum {
    TCW_OPT_KERNEL = 0,     /* 0 auto (default), 1 force the global-memory gather kernel,
                               2 force the TMA-staged kernel (TCW_EUNSUPPORTED at search if the
                               f0 spacing makes a tile's window exceed the row padding),
                               3 force the sky-block kernel (count formats only; exact sharing
                               of lookups between neighbouring sky points, auto for >= 16 sky
                               points; TCW_EUNSUPPORTED for the power format)                 */
    TCW_OPT_TIMING = 1,     /* 1: record CUDA events around each stage of tcw_search           */
    TCW_OPT_F0_PER_LANE = 2,/* staged kernel: templates per lane, 4, 8 or 16 (tile = 32x that); 0 auto */
    TCW_OPT_STAGES = 3,     /* staged kernel: upper limit of the per-warp ring depth, 2..16; 0 auto  */
    TCW_OPT_SKY_BLOCK = 4,  /* sky-block kernel: sky points per block, 64, 128 or 256 (256 = the two-level
                               kernel: needs n_sft * (largest count in the spectrogram) <= 32767, else
                               TCW_EUNSUPPORTED at search); 0 auto (256 when that holds and the grid has
                               >= 128 sky points, else 64)                                           */
    TCW_OPT_CHUNK_ROWS = 5, /* staged kernel: SFT rows per chunk (rounded up to a multiple of 64).  A
                               chunked search runs every (group, f0 tile) over one chunk of SFTs
                               before any over the next, so the rows in use stay in L2; per-chunk
                               partial sums are then added in ascending chunk order (fixed order).
                               0 auto (chunk only spectrograms larger than L2), -1 never chunk    */
    TCW_OPT_EXACT_INDEX = 6,/* staged kernel: 1 = decide every bin by the defining chain of three binary64
                               operations instead of the one-FMA fast index with its guard band (same
                               bins either way; the tests compare the two); 0 default                  */
    TCW_OPT_GENERAL_F0 = 7, /* staged kernel: 1 = treat the f0 axis as arbitrary even when it is equally spaced (the
                               equally spaced instantiation derives the templates of a lane from one product
                               and a stride; same bins either way); 0 default                              */
    TCW_OPT_ROW_COPIES = 8, /* staged kernel: 1 = stage every SFT row by its own 1-D bulk copy; 0 default: a ring slot (four
                               consecutive SFT rows) travels by ONE tensor-map copy wherever its rows' windows fit one
                               box (same bins, same sums bit for bit; the tests compare the two)            */
    TCW_OPT_DEBUG_SHRINK_SLOT = 100, /* test hook: the kernels check their staged windows against the planned
                               bound minus this many bytes, which forces the device status word and
                               hence TCW_EINTERNAL; 0 default.  Not for production use.               */
    TCW_OPT_DEBUG_FAIL_WAIT = 101,  /* test hook: in tcw_search_host's progressive read-back, the stream wait of
                               part (value - 1) behaves as if the driver had refused it; the call must
                               then still deliver every value (plain copies after the search).  0 default */
    TCW_OPT_DEBUG_CHUNK_SCRATCH = 102 /* test hook: byte cap on the SFT-chunk scratch (default 16e9) so that the
                               'whole grid too large to chunk' plan can be reached on a small grid; 0 default */
};
int tcw_set_option(tcw_handle *h, int key, long value);

/* tcw_get_timing -- device time of the stages of tcw_search, in milliseconds, AVERAGED over the
 * searches enqueued on this handle since TCW_OPT_TIMING was set or tcw_get_timing was last
 * called (at most 4096 are kept; later ones are not recorded):
 *  ms[0] Doppler + spin-down tables, ms[1] gather-accumulate kernel, ms[2] candidate reduction,
 *  ms[3] whole call.  *n_searches (may be NULL) receives how many searches were averaged.
 * The events are recorded on the search's own stream without synchronising it; this call
 * waits for the last of them. */
int tcw_get_timing(tcw_handle *h, float ms[4], int *n_searches);

/* tcw_get_info -- facts about the last tcw_search: info[0] kernel used (1 gather, 2 staged, 3 sky-block,
 * 4 bank),
 * info[1] templates per CTA tile, info[2] CTAs launched, info[3] dynamic shared memory bytes,
 * info[4] device status word (0 = ok; nonzero = an internal window-bound check failed),
 * info[5] kernels launched by the call, info[6] ring depth per warp (slots of four SFT rows in the staged kernel), info[7] sky points per
 * block (sky-block kernel, else 0), info[8] SFT chunks of the staged kernel (1 = not chunked),
 * info[9] SFT rows per chunk, info[10] tau ranges of the progressive read-back of the last search (tcw_search_host
 * with a large out_stat; 0 = none), info[11] 1 when the staged kernel staged ring slots by tensor-map copies
 * (0: one 1-D bulk copy per row, see TCW_OPT_ROW_COPIES).
 * Synchronises the search's stream. */
int tcw_get_info(tcw_handle *h, long info[12]);

#ifdef __cplusplus
}
#endif
#endif /* TCW_H_ */
