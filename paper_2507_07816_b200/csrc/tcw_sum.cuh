// tcw_sum.cuh -- bin index, gather-accumulate and candidate reduction kernels (sm_100a).
//
// The statistic is "summed across the data bins selected by the track": for
// template i of group (s, a, b) and SFT j
//     x = ((f0_i * g[a][b][j]) * D[s][j]) * T_sft ,  k = rint(x) - k_min         (eq. (1)-(2))
//     stat_i += spectrogram[j][k]  if 0 <= k < n_bins .
// Two kernels compute it:
//   * sum_staged_kernel -- the product path.  One CTA owns (group, tile of 32*R consecutive f0).
//     Consecutive f0 of one group select a narrow contiguous bin window per SFT (g <= 1).  Every
//     warp owns ring slots of RB consecutive SFT rows (slots warp, warp + NW, ...) and runs its own
//     software pipeline: it computes the windows [k(f_first, j), k(f_last, j)] of the rows a few slots
//     ahead, one lane issues ONE TMA copy per slot -- a tensor-map box of {128 B, n segments, RB rows}
//     (cp.async.bulk.tensor.3d, mbarrier complete_tx) where the rows' windows fit one box, else one 1-D
//     bulk copy per row -- into the warp's private shared-memory ring, and all lanes gather the rows from
//     shared memory, each lane carrying R templates in registers.  The library's spectrogram copy carries
//     PAD_BINS zero bins on both sides of every row, so a window that is partly out of band is
//     still copied whole and no per-lookup bounds test is needed (out-of-band bins add 0).
//   * sum_gather_kernel -- one thread per template gathering from global memory.  It serves f0
//     axes so sparse that the window of a 128-template tile does not fit the row padding, and it
//     is the simple kernel the staged one is checked against.
// Device formats: float32 power or uint8 counts (a bit-packed input is expanded to uint8 by
// tcw_create: with the index arithmetic fixed at 3 FP64 operations per lookup the count paths are
// bound by instruction issue, and a byte load + add is cheaper than word load + shift + mask).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace tcw {

enum { FMT_F32 = 0, FMT_U8 = 1 };

// zero bins on each side of every spectrogram row in the library's copy
constexpr int PAD_BINS = 1056;

// 1.5 * 2^52: adding it rounds x to the nearest integer (ties to even) in the low mantissa bits,
// so the low word of the sum is rint(x) for |x| < 2^31.
#define TCW_MAGIC 6755399441055744.0

// rint(((f0*g)*D)*T) as an int.  When T is a power of two, Dp = D*T is exact and
// (f0*g)*(D*T) rounds exactly like ((f0*g)*D)*T, which saves one FP64 multiply per lookup.
template <bool TPOW2>
__device__ __forceinline__ int bin_lo(double f0, double g, double Dp, double T)
{
    double x = __dmul_rn(__dmul_rn(f0, g), Dp);
    if (!TPOW2) x = __dmul_rn(x, T);
    return __double2loint(__dadd_rn(x, TCW_MAGIC));
}

struct SumParams {
    const unsigned char *spec;  // bin 0 of row 0 of the library's copy (PAD_BINS zero bins before it)
    const unsigned char *spec_pad;  // first byte of row 0 of that copy, left padding included (16-byte aligned)
    long pad_bytes;             // bytes of the left padding (a multiple of 16)
    long pitch;                 // row pitch in bytes (multiple of 16), padding included
    int n_sft, n_bins, k_min;
    double T;
    const double *gtab;         // [n_tau*n_brk][n_sft]
    const double *dtab;         // [n_sky][n_sft]
    const double *f0;
    int n_f0, n_ab;             // n_ab = n_tau*n_brk
    int j_begin;                // first SFT with t_j >= T0
    double dmaxT;               // upper bound of D*T over every sky point and SFT
    void *out_stat;             // float32 / int32 [n_groups][n_f0] or NULL
    void *partial;              // {stat, f0_index} [n_groups][n_tiles]
    int n_tiles, tile;          // tiles per group, templates per tile
    int stages, slot_bytes;     // staged kernel: ring depth per warp (slots of RB rows), bytes per staged row
    int slot_limit;             // bytes a staged row may take (= slot_bytes; a test hook lowers it to force the status word)
    long n_groups;              // n_sky * n_tau * n_brk
    int chunk_rows, n_chunks;   // staged kernel: SFT rows per chunk, number of chunks (1 = whole span per CTA)
    int chunk0;                 // first chunk of this launch (a search over a spectrogram that is still being
                                // uploaded launches chunk by chunk; otherwise 0 and one launch covers every chunk)
    void *cpart;                // chunked: float32 / int32 [n_chunks][n_groups][n_f0] partial sums
    unsigned char *clive;       // chunked: [n_chunks][n_groups][n_tiles] 1 where the CTA wrote its partial sums
    int *status;                // device status word
    // staged kernel, one tensor-map copy per ring slot: tmaps + 128*n is the CUtensorMap whose box is
    // {128 bytes, n segments, RB rows} over the library's copy seen as [n_sft][pitch/128][128 bytes]
    // (n = 1 .. max_seg); NULL = every row travels by its own 1-D bulk copy
    const unsigned char *tmaps;
    int max_seg;
    // staged kernel, fast bin index (one fused multiply-add per lookup, see RowMeta below)
    double fix_add;             // 0.5 + thr, thr = thr2 / 2^33 bins
    double d32;                 // equally spaced f0 axis: 32 * spacing (Hz), else 0
    uint32_t thr2;              // a row whose smallest fraction word is <= thr2 is decided by the defining chain;
                                // 0xffffffff = always (fast index switched off)
    // progressive read-back (tcw_search_host with a large out_stat): the (tau, n) axis is cut into n_parts ranges
    // [part_ab0[r], part_ab0[r+1]); CTAs are issued range by range, and each CTA adds one to progress[r] once its
    // outputs are written, so a copy stream can wait for a range (cuStreamWaitValue32) and fetch it while later
    // ranges are still being searched.  progress == NULL: plain block order, no counters.
    unsigned int *progress;
    int n_parts;
    int part_ab0[17];
    // weighted search (tcw_search_weighted; eq. (4)): s = sum w_j * spectrogram[j][k_j]
    const float *wtab;          // [n_sky][n_sft] weights, or NULL (all ones)
    double mean1, var1;         // per-bin noise mean and variance of the spectrogram elements
    float *out_psi;             // critical ratio [n_groups][n_f0]
    double *cw1, *cw2;          // chunked: per-chunk sums of w and w^2 over the in-band SFTs, laid out like cpart
};

template <int FMT> struct Acc { typedef int type; };
template <> struct Acc<FMT_F32> { typedef float type; };
// accumulator of a search: weighted sums are float32 whatever the spectrogram format
template <int FMT, bool WGT> struct AccW { typedef typename Acc<FMT>::type type; };
template <int FMT> struct AccW<FMT, true> { typedef float type; };

// Psi = (s - <s>)/sigma_s with <s> = mean1*W1, sigma_s^2 = var1*W2 (eq. (4)); 0 when W2 = 0.
__device__ __forceinline__ float critical_ratio(float s, double W1, double W2, double mean1, double var1)
{
    if (!(W2 > 0.0)) return 0.0f;
    return (float)(((double)s - mean1 * W1) / sqrt(var1 * W2));
}

template <typename V> __device__ __forceinline__ V lowest();
template <> __device__ __forceinline__ float lowest<float>() { return -__int_as_float(0x7f800000); }
template <> __device__ __forceinline__ int lowest<int>() { return INT32_MIN; }

template <typename V> struct __align__(8) Best { V stat; int idx; };

template <typename V>
__device__ __forceinline__ void argmax_step(V &v, int &i, V ov, int oi)
{
    if (ov > v || (ov == v && oi < i)) { v = ov; i = oi; }
}

// Block-wide (max, lowest index) over the threads' (v, i); thread 0 stores it.
// red must hold blockDim.x/32 entries.
template <typename V>
__device__ __forceinline__ void block_best(V v, int i, Best<V> *red, Best<V> *dst)
{
#pragma unroll
    for (int o = 16; o; o >>= 1) {
        V ov = __shfl_xor_sync(0xffffffffu, v, o);
        int oi = __shfl_xor_sync(0xffffffffu, i, o);
        argmax_step(v, i, ov, oi);
    }
    int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, nw = (blockDim.x + 31) >> 5;
    if (lane == 0) red[warp] = {v, i};
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int w = 1; w < nw; ++w) argmax_step(v, i, red[w].stat, red[w].idx);
        if (i == INT32_MAX) i = 0;
        *dst = {v, i};
    }
}

// Block index -> (unit, (tau, n) index, raw tile index) where unit is a sky point or a sky block.
// Plain order: unit slowest, tile fastest.  With progress counters: range of the (tau, n) axis slowest.
__device__ __forceinline__ void block_map(const SumParams &p, long bq, int n_units, int &unit, int &ab, int &tile_raw, int &part)
{
    part = 0;
    if (p.progress) {
        for (;;) {
            const long cnt = (long)n_units * (p.part_ab0[part + 1] - p.part_ab0[part]) * p.n_tiles;
            if (bq < cnt || part == p.n_parts - 1) break;
            bq -= cnt;
            ++part;
        }
        const int nab = p.part_ab0[part + 1] - p.part_ab0[part];
        tile_raw = (int)(bq % p.n_tiles);
        bq /= p.n_tiles;
        ab = p.part_ab0[part] + (int)(bq % nab);
        unit = (int)(bq / nab);
    } else {
        tile_raw = (int)(bq % p.n_tiles);
        bq /= p.n_tiles;
        ab = (int)(bq % p.n_ab);
        unit = (int)(bq / p.n_ab);
    }
}
// Called by every thread of a CTA after its last output store: publishes the CTA's outputs and counts it.
__device__ __forceinline__ void block_done(const SumParams &p, int part)
{
    if (!p.progress) return;
    __syncthreads();
    if (threadIdx.x == 0) {
        __threadfence_system();
        atomicAdd(p.progress + part, 1u);
    }
}

// --------------------------------------------------------------------------- gather kernel
template <int FMT, bool TPOW2, bool WGT>
__global__ void __launch_bounds__(128)
sum_gather_kernel(const SumParams p)
{
    typedef typename AccW<FMT, WGT>::type V;
    __shared__ Best<V> red[4];
    int sky_i, ab_i, tile, part;
    block_map(p, blockIdx.x, (int)(p.n_groups / p.n_ab), sky_i, ab_i, tile, part);
    const long grp = (long)sky_i * p.n_ab + ab_i;
    const int i = tile * p.tile + threadIdx.x;
    const bool valid = i < p.n_f0;
    const double f0 = p.f0[valid ? i : p.n_f0 - 1];
    const double *g = p.gtab + (grp % p.n_ab) * (long)p.n_sft;
    const double *d = p.dtab + (grp / p.n_ab) * (long)p.n_sft;
    const float *wr = WGT && p.wtab ? p.wtab + (grp / p.n_ab) * (long)p.n_sft : nullptr;
    V acc = 0;
    double W1 = 0, W2 = 0;
    for (int j = p.j_begin; j < p.n_sft; ++j) {
        double Dp = TPOW2 ? __dmul_rn(d[j], p.T) : d[j];
        int k = bin_lo<TPOW2>(f0, g[j], Dp, p.T) - p.k_min;
        if ((unsigned)k < (unsigned)p.n_bins) {
            const unsigned char *row = p.spec + (long)j * p.pitch;
            if (WGT) {
                const float w = wr ? wr[j] : 1.0f;
                const float v = FMT == FMT_F32 ? ((const float *)row)[k] : (float)row[k];
                acc = __fmaf_rn(w, v, acc);
                W1 += (double)w;
                W2 += (double)w * (double)w;
            } else if (FMT == FMT_F32) acc += ((const float *)row)[k];
            else acc += (V)row[k];
        }
    }
    if (WGT) {
        const float psi = critical_ratio(acc, W1, W2, p.mean1, p.var1);
        if (valid && p.out_stat) ((float *)p.out_stat)[grp * p.n_f0 + i] = acc;
        if (valid && p.out_psi) p.out_psi[grp * p.n_f0 + i] = psi;
        acc = psi;
    } else if (valid && p.out_stat) ((V *)p.out_stat)[grp * p.n_f0 + i] = acc;
    block_best<V>(valid ? acc : lowest<V>(), valid ? i : INT32_MAX, red,
                  (Best<V> *)p.partial + grp * p.n_tiles + tile);
    block_done(p, part);
}

// --------------------------------------------------------------------------- PTX wrappers
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint32_t bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity)
{
    asm volatile(
        "{\n"
        ".reg .pred P1;\n"
        "LAB_WAIT:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n"
        "@P1 bra DONE;\n"
        "bra LAB_WAIT;\n"
        "DONE:\n"
        "}\n" ::"r"(bar), "r"(parity) : "memory");
}
// TMA 1-D bulk copy global -> shared, completion counted in bytes on an mbarrier.
// dst, src and bytes are multiples of 16.
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void *src, uint32_t bytes, uint32_t bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}
// TMA tiled copy of a {128 bytes, n segments, RB rows} box of the spectrogram (tensor map `map`, coordinates
// {0, segment, row}) into shared memory, completion counted in bytes on an mbarrier.  dst is 128-byte aligned.
__device__ __forceinline__ void tensor3_g2s(uint32_t dst, const void *map, int seg, int row, uint32_t bar)
{
    asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
                 ::"r"(dst), "l"(map), "r"(0), "r"(seg), "r"(row), "r"(bar) : "memory");
}
__device__ __forceinline__ float lds_f32(uint32_t a)
{
    float v;
    asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(a));
    return v;
}
// two float32 additions in one instruction (add.rn.f32x2, SASS FADD2): each half rounds exactly like a scalar
// __fadd_rn, so results are bit-identical to the scalar form; the kernel is bound by instruction issue
__device__ __forceinline__ void fadd2(float &o0, float &o1, float a0, float a1, float b0, float b1)
{
    unsigned long long a, b, r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(a) : "f"(a0), "f"(a1));
    asm("mov.b64 %0, {%1, %2};" : "=l"(b) : "f"(b0), "f"(b1));
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    asm("mov.b64 {%0, %1}, %2;" : "=f"(o0), "=f"(o1) : "l"(r));
}
// two float32 fused multiply-adds in one instruction (fma.rn.f32x2, SASS FFMA2): each half rounds exactly like a
// scalar __fmaf_rn
__device__ __forceinline__ void ffma2(float &o0, float &o1, float w, float b0, float b1, float c0, float c1)
{
    unsigned long long a, b, c, r;
    asm("mov.b64 %0, {%1, %1};" : "=l"(a) : "f"(w));
    asm("mov.b64 %0, {%1, %2};" : "=l"(b) : "f"(b0), "f"(b1));
    asm("mov.b64 %0, {%1, %2};" : "=l"(c) : "f"(c0), "f"(c1));
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c));
    asm("mov.b64 {%0, %1}, %2;" : "=f"(o0), "=f"(o1) : "l"(r));
}
__device__ __forceinline__ uint32_t lds_u8(uint32_t a)
{
    uint32_t v;
    asm volatile("ld.shared.u8 %0, [%1];" : "=r"(v) : "r"(a));
    return v;
}

// --------------------------------------------------------------------------- staged kernel
#ifndef TCW_NW
#define TCW_NW 4
#endif
#ifndef TCW_RB
#define TCW_RB 4
#endif
constexpr int NW = TCW_NW;      // warps per CTA; warp w owns the rows j = j0 + w + NW*n of the CTA's SFT chunk
constexpr int STAGED_THREADS = 32 * NW;
constexpr int RB = TCW_RB;      // SFT rows per ring slot (one mbarrier phase, one wait, one refill per RB rows)
static_assert(RB == 1 || RB == 2 || RB == 4 || RB == 8, "RB must divide the 32-row metadata batch");

// ---- fast bin index of the staged kernel ("one FMA per lookup") -----------
// The defining chain k = rint(RN(RN(f0*g)*D*T)) costs three FP64 instructions per lookup.  The
// staged kernel evaluates, per lookup, ONE fused multiply-add
//     y = fma(f0 - f_first, c, Q),   c = RN(g*D*T),   Q = RN(f_first*c) - rint(x_first) + 0.5 + thr + W + 1.5*2^20
// whose result lies in [2^20, 2^21), where a double's unit in the last place is 2^-32: the high
// word of y is FIX_HC + W + (k - k_first) -- with W the place of the tile's first bin in shared memory
// (an integer), the index of the selected element itself -- and the low word is
// frac(x~ + 0.5 + thr) * 2^32, x~ the fast value of x.
// |x~ - x| <= 3*x*2^-52 + 2^-32 =: B (error budget in DESIGN.md), thr >= B, so floor(x~ + 0.5 + thr)
// equals rint(x) unless the low word is <= 2*thr*2^32.  Lanes track the minimum low word of a row;
// where it is that small (about once in 1e7 lookups) the row's bins are recomputed by the defining
// chain (bin_lo).  Either way the bin is the oracle's: tests compare both paths bit for bit.
constexpr uint32_t FIX_HC = 0x41380000u;     // high word of 1.5 * 2^20
#define TCW_FIX_BASE 1572864.0               /* 1.5 * 2^20 */

// What a warp needs to stage a row and to turn the fast index into a shared-memory address of it.
struct __align__(16) RowMeta {
    double c, Q;      // the fused multiply-add operands above; Q also carries the row's place in shared memory:
                      // byte address of the selected element = BPB * (high word of y - FIX_HC)
    uint32_t flags;   // first row of a ring slot: bit q = row q of the slot is staged, bit 8 = no further rows
    int by16;         // bytes staged (> 0, a multiple of 16), 0 row with no in-band bin, -1 no further rows
    uint32_t src_lo, src_hi;   // first staged byte of the row's window, relative to SumParams::spec_pad
};
// weighted search: per row also the row's weight and the constant that turns the fast index into a band-relative
// bin for the edge rows, in a second ring of 8-byte entries (the 32-byte RowMeta ring keeps its pitch, so that the
// weighted instantiation still fits 128-byte granular slot rows at three CTAs per SM); RowMeta::flags bit 10 of
// the row says that every template of the tile is in band in this row (then the weight sums W1, W2 advance by
// the same amount for the whole tile: one warp-uniform add)
struct __align__(8) RowWgt {
    float w;
    uint32_t ktest;   // bin - k_min = HI + ktest
};
static_assert(sizeof(RowMeta) == 32 && sizeof(RowWgt) == 8, "RowMeta layout");

// rows of the per-warp metadata ring: one batch of 32 rows plus the rows still in flight
__host__ __device__ inline int staged_meta_rows(int stages) { return 32 + RB * stages; }

// dynamic shared memory: [mbarrier NW*D] [RowMeta NW*meta_rows] [weighted: RowWgt NW*meta_rows] [slot NW*D*RB*slot_bytes].  The slot
// region is reused for the cross-warp reduction (NW * 32*R accumulators) once every copy has
// completed; the mbarrier words are never reused as data (they are updated through the async proxy,
// and a generic store to the same bytes is not ordered against that without a proxy fence).
__host__ __device__ inline size_t staged_bar_bytes(int stages) { return ((size_t)NW * stages * 8 + 15) & ~(size_t)15; }
__host__ __device__ inline size_t staged_header_bytes(int stages, bool wgt)
{
    return (staged_bar_bytes(stages) + (size_t)NW * staged_meta_rows(stages) * (sizeof(RowMeta) + (wgt ? sizeof(RowWgt) : 0)) + 127) & ~(size_t)127;
}
__host__ __device__ inline size_t staged_smem_bytes(int stages, int slot_bytes, int tile, bool wgt)
{
    size_t ring = (size_t)NW * stages * RB * (size_t)slot_bytes;
    size_t red = (size_t)NW * tile * 4 * (wgt ? 3 : 1) + (size_t)NW * 16 + 128;
    return staged_header_bytes(stages, wgt) + (ring > red ? ring : red);
}

__device__ __forceinline__ bool elect_one()
{
    uint32_t p;
    asm volatile("{ .reg .pred P; elect.sync _|P, 0xffffffff; selp.u32 %0, 1, 0, P; }" : "=r"(p));
    return p != 0;
}
__device__ __forceinline__ void lds_v2(uint32_t a, uint32_t &x, uint32_t &y)
{
    asm volatile("ld.shared.v2.u32 {%0, %1}, [%2];" : "=r"(x), "=r"(y) : "r"(a));
}
__device__ __forceinline__ void lds_v4(uint32_t a, uint32_t &x, uint32_t &y, uint32_t &z, uint32_t &w)
{
    asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(x), "=r"(y), "=r"(z), "=r"(w) : "r"(a));
}
__device__ __forceinline__ void lds_v2f64(uint32_t a, double &x, double &y)
{
    asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(x), "=d"(y) : "r"(a));
}
__device__ __forceinline__ uint32_t lds_u32(uint32_t a)
{
    uint32_t v;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(a));
    return v;
}

template <int FMT, int R, bool TPOW2, bool WGT, bool UNI>
#ifndef TCW_MINB
#define TCW_MINB (12 / TCW_NW)
#endif
__global__ void __launch_bounds__(STAGED_THREADS, TCW_MINB)
sum_staged_kernel(const SumParams p)
{
#ifndef TCW_PAIR
#define TCW_PAIR 1
#endif
#ifndef TCW_FADD2
#define TCW_FADD2 1
#endif
#ifndef TCW_WGT_PAIR
#define TCW_WGT_PAIR 1
#endif
    constexpr bool PAIR = TCW_PAIR && RB % 2 == 0 && (!WGT || TCW_WGT_PAIR);     // live slots are consumed two rows at a time
    typedef typename AccW<FMT, WGT>::type V;
    typedef RowMeta Meta;
    constexpr int MB = (int)sizeof(Meta);
    constexpr int F = 32 * R;                      // templates per tile
    constexpr int BPB = FMT == FMT_F32 ? 4 : 1;    // bytes per bin
    constexpr int SH = FMT == FMT_F32 ? 2 : 0;
    extern __shared__ __align__(128) unsigned char smem[];
    const int D = p.stages;
    const int MR = staged_meta_rows(D);
    // the warp index through a warp reduction: the compiler then knows it is warp-uniform and keeps the
    // ring pointers derived from it in uniform registers (the copy operands need them there)
    const int warp = (int)__reduce_or_sync(0xffffffffu, threadIdx.x >> 5), lane = threadIdx.x & 31;
    uint64_t *bars = (uint64_t *)smem + warp * D;
    Meta *meta = (Meta *)(smem + staged_bar_bytes(D)) + warp * MR;
    unsigned char *slots = smem + staged_header_bytes(D, WGT);
    const uint32_t slot_stride = (uint32_t)(RB * p.slot_bytes);
    const uint32_t slots_s = smem_u32(slots) + (uint32_t)(warp * D) * slot_stride;
    const uint32_t slots_e = slots_s + (uint32_t)D * slot_stride;
    const uint32_t bars_s = smem_u32(bars);
    const uint32_t meta_s = smem_u32(meta), meta_e = meta_s + (uint32_t)(MR * MB);
    // weighted: the warp's ring of RowWgt entries, row for row beside its RowMeta ring
    RowWgt *wmeta = (RowWgt *)(smem + staged_bar_bytes(D) + (size_t)NW * MR * MB) + warp * MR;
    const uint32_t wmeta_s = smem_u32(wmeta);

    // block -> (SFT chunk, group, f0 tile).  Chunks are the slowest index: the CTAs in flight work
    // on the same few hundred SFT rows, which therefore stay in L2 while every group reads them.
    // Within a group heavy tiles (high f0 stays in band longest) are launched first.
    const long per_chunk = p.n_groups * p.n_tiles;
    const int chunk = p.chunk0 + (int)(blockIdx.x / per_chunk);
    int sky_i, ab_i, tile_raw, part;
    block_map(p, blockIdx.x % per_chunk, (int)(p.n_groups / p.n_ab), sky_i, ab_i, tile_raw, part);
    const int tile = p.n_tiles - 1 - tile_raw;
    const long grp = (long)sky_i * p.n_ab + ab_i;
    const int i0 = tile * F;
    const int i_last = min(i0 + F, p.n_f0) - 1;
    const int j0 = p.j_begin + chunk * p.chunk_rows;
    const int j1 = min(p.n_sft, j0 + p.chunk_rows);
    const double *g = p.gtab + (grp % p.n_ab) * (long)p.n_sft;
    const double *d = p.dtab + (grp / p.n_ab) * (long)p.n_sft;
    const float *wr = WGT && p.wtab ? p.wtab + (grp / p.n_ab) * (long)p.n_sft : nullptr;
    const double f_first = p.f0[i0], f_last = p.f0[i_last];
    const double below = (double)p.k_min - 1.0;

    if (p.n_chunks > 1) {
        // g decreases with j: a tile whose highest template is below the band at the chunk's first
        // row, for the largest possible Doppler factor, has nothing to add in this chunk
        const bool dead = f_last * __ldg(g + j0) * p.dmaxT < below;
        if (threadIdx.x == 0) p.clive[((long)chunk * p.n_groups + grp) * p.n_tiles + tile] = dead ? 0 : 1;
        if (dead) return;
    }

    if (lane == 0) {
        for (int s = 0; s < D; ++s) mbar_init(bars_s + 8u * s, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncwarp();

    V acc[R];
    double df[UNI ? 1 : R];      // f0 of the lane's templates minus the tile's first f0 (equally spaced f0: lane*delta instead)
    const double dlane = __dmul_rn((double)lane, p.d32 * 0.03125);
    // weighted: sums of w and w^2 over the in-band SFTs.  Rows in which the whole tile is in band
    // advance a warp-uniform float64 pair; only rows that straddle a band edge are counted per lane.
    float w1p[WGT ? R : 1], w2p[WGT ? R : 1];
    double W1u = 0, W2u = 0;
#pragma unroll
    for (int r = 0; r < R; ++r) {
        acc[r] = 0;
        if constexpr (!UNI) df[r] = __dsub_rn(p.f0[min(i0 + r * 32 + lane, i_last)], f_first);
        if (WGT) w1p[r] = w2p[r] = 0.0f;
    }
    // warp w owns the ring slots w, w + NW, w + 2*NW, ... of the chunk; a slot is RB CONSECUTIVE SFT rows, so that one
    // tensor-map copy can fetch it.  Row n of the warp (n = RB*slot + q) is SFT row_of(n); rows at or past j1 do not exist.
    const int jw = j0 + RB * warp;
    auto row_of = [&](int n) { return jw + (NW * RB) * (n / RB) + (n % RB); };

    // Row metadata is computed 32 rows at a time, one row per lane (rows 32*m + lane of this warp),
    // and written to the warp's metadata ring; (g, D) of the next batch are loaded ahead of use.
    double gn = 0, dn = 1;
    float wn = 1.0f;
    if (row_of(lane) < j1) {
        gn = __ldg(g + row_of(lane)); dn = __ldg(d + row_of(lane));
        if (WGT && wr) wn = __ldg(wr + row_of(lane));
    }

    int m_pos = lane;                            // (32*m + lane) mod MR: the row's place in the metadata ring
    int m_slot = (lane / RB) % D;                // ((32*m + lane) / RB) mod D: the ring slot the row is staged in
    const int slot_step = (32 / RB) % D;
    auto compute_batch = [&](int m) {
        const int n = 32 * m + lane;
        const int jn = row_of(n);
        const double gj = gn, dj = dn;
        const double Dp = TPOW2 ? __dmul_rn(dj, p.T) : dj;
        Meta mt;
        mt.c = TPOW2 ? __dmul_rn(gj, Dp) : __dmul_rn(__dmul_rn(gj, dj), p.T);
        mt.Q = 0;
        mt.flags = 0;
        mt.by16 = -1;
        mt.src_lo = mt.src_hi = 0;
        RowWgt mw = {wn, 0u};
        bool full = false;
        if (jn + 32 * NW < j1) {          // row_of(n + 32) = jn + 32*NW
            gn = __ldg(g + jn + 32 * NW); dn = __ldg(d + jn + 32 * NW);
            if (WGT && wr) wn = __ldg(wr + jn + 32 * NW);
        }
        // once the highest template of the tile is below the band for the largest possible Doppler
        // factor, no later SFT can contribute
        int kf = 0, kl = -1, lo_f = 0;
        bool bad = false;                                   // the row's own 1-D window breaks the host's bound
        if (jn < j1 && !(f_last * gj * p.dmaxT < below)) {
            lo_f = bin_lo<TPOW2>(f_first, gj, Dp, p.T);
            kf = lo_f - p.k_min;
            kl = bin_lo<TPOW2>(f_last, gj, Dp, p.T) - p.k_min;
            mt.by16 = 0;
            if (kl >= 0 && kf < p.n_bins) {
                const int a_byte = (BPB * kf) & ~15;                 // rounds towards -inf: may reach into the left padding
                const int e_byte = (BPB * (kl + 1) + 15) & ~15;
                if (kf < -PAD_BINS || kl >= p.n_bins + PAD_BINS) {
                    atomicOr(p.status, 1);  // host-side window bound violated: the search reports TCW_EINTERNAL
                } else {
                    bad = e_byte - a_byte > p.slot_limit;
                    mt.by16 = e_byte - a_byte;
                }
            }
        }
        // A slot whose RB rows are all live and whose windows fit one {128 B x nseg x RB} box travels by ONE
        // tensor-map copy (the rows of a slot are consecutive in memory and the track drifts slowly); otherwise
        // (band edges, gaps in the data, the steep start of a fast spin-down) every row gets its own 1-D copy.
        bool use2d = false;
        int seg0 = 0, nseg = 0;
        if (p.tmaps) {
            int kfm = mt.by16 > 0 ? kf : INT32_MAX, klm = mt.by16 > 0 ? kl : INT32_MIN;
            bool all = mt.by16 > 0;
#pragma unroll
            for (int o = 1; o < RB; o <<= 1) {
                kfm = min(kfm, __shfl_xor_sync(0xffffffffu, kfm, o));
                klm = max(klm, __shfl_xor_sync(0xffffffffu, klm, o));
                all = __shfl_xor_sync(0xffffffffu, (int)all, o) && all;
            }
            if (all) {
                seg0 = ((int)p.pad_bytes + BPB * kfm) >> 7;
                nseg = (((int)p.pad_bytes + BPB * (klm + 1) + 127) >> 7) - seg0;
                use2d = nseg <= p.max_seg && nseg * 128 <= p.slot_limit;
            }
        }
        if (mt.by16 > 0 && bad && !use2d) {
            atomicOr(p.status, 1);
            mt.by16 = 0;
        }
        if (mt.by16 > 0) {
            const int a_byte = use2d ? 128 * seg0 - (int)p.pad_bytes : (BPB * kf) & ~15;   // first staged byte, relative to bin 0
            const uint32_t row_stride = use2d ? (uint32_t)(128 * nseg) : (uint32_t)p.slot_bytes;
            const long src = (long)jn * p.pitch + p.pad_bytes + a_byte;
            mt.src_lo = (uint32_t)src;
            mt.src_hi = (uint32_t)(src >> 32);
            const uint32_t S = slots_s + (uint32_t)m_slot * slot_stride + (uint32_t)(lane % RB) * row_stride;
            // byte address of band-relative bin b: S + BPB*b - a_byte (both multiples of BPB), so the tile's
            // first bin kf sits at element W = (S - a_byte)/BPB + kf of shared memory (W < 2^16)
            const int W = (((int)S - a_byte) >> SH) + kf;
            mt.Q = __dadd_rn(__dadd_rn(__dsub_rn(__dmul_rn(f_first, mt.c), (double)lo_f), p.fix_add + (double)W), TCW_FIX_BASE);
            if constexpr (WGT) {
                full = kf >= 0 && kl < p.n_bins;
                mw.ktest = (uint32_t)(kf - W) - FIX_HC;
            }
        }
        // the first row of every ring slot carries the slot's summary for the consumer
        const unsigned live = __ballot_sync(0xffffffffu, mt.by16 > 0);
        mt.flags = ((live >> (lane & ~(RB - 1))) & ((1u << RB) - 1u)) | (mt.by16 < 0 ? 256u : 0u);
        if (use2d) {
            // the slot's first row carries the box: bytes the copy delivers, first segment, first SFT row
            mt.flags |= 512u | ((uint32_t)nseg << 16);
            if (lane % RB == 0) {
                mt.by16 = 128 * nseg * RB;
                mt.src_lo = (uint32_t)seg0;
                mt.src_hi = (uint32_t)jn;
            }
        }
        if constexpr (WGT) {
            if (full) mt.flags |= 1024u;
            wmeta[m_pos] = mw;
        }
        meta[m_pos] = mt;
        m_pos += 32;
        if (m_pos >= MR) m_pos -= MR;
        m_slot += slot_step;
        if (m_slot >= D) m_slot -= D;
        __syncwarp();
    };

    int ni = 0;                                  // next slot (RB rows) to stage
    uint32_t bar_i = bars_s, slot_i = slots_s, meta_i = meta_s;
    // Stage the rows RB*ni .. RB*ni + RB-1: one elected lane reads the slot's descriptor and issues one
    // tensor-map copy for the slot, or one TMA bulk copy per staged row, counted on the slot's mbarrier.
    auto stage_next = [&]() {
        if ((ni & (32 / RB - 1)) == 0) compute_batch(ni / (32 / RB));
        if (elect_one()) {
            uint32_t u[RB], lo[RB], hi[RB];
            int by[RB], tot = 0;
            {
                uint32_t b;
                lds_v4(meta_i + 16u, u[0], b, lo[0], hi[0]);
                by[0] = (int)b;
            }
            if (u[0] & 512u) {
                mbar_arrive_expect_tx(bar_i, (uint32_t)by[0]);
                tensor3_g2s(slot_i, p.tmaps + ((u[0] >> 16) << 7), (int)lo[0], (int)hi[0], bar_i);
                tot = -1;
            } else {
                tot = max(by[0], 0);
#pragma unroll
                for (int q = 1; q < RB; ++q) {
                    uint32_t b;
                    lds_v4(meta_i + (uint32_t)(q * MB) + 16u, u[q], b, lo[q], hi[q]);
                    by[q] = (int)b;
                    tot += max(by[q], 0);
                }
            }
            if (tot < 0) {
            } else if (tot > 0) {
                mbar_arrive_expect_tx(bar_i, (uint32_t)tot);
#pragma unroll
                for (int q = 0; q < RB; ++q)
                    if (by[q] > 0)
                        bulk_g2s(slot_i + (uint32_t)(q * p.slot_bytes), p.spec_pad + (((size_t)hi[q] << 32) | lo[q]),
                                 (uint32_t)by[q], bar_i);
            } else if (by[0] >= 0) {
                mbar_arrive(bar_i);   // every use of a slot completes one phase of its barrier
            }
        }
        ++ni;
        bar_i += 8u; slot_i += slot_stride; meta_i += RB * MB;
        if (slot_i == slots_e) { slot_i = slots_s; bar_i = bars_s; }
        if (meta_i == meta_e) meta_i = meta_s;
    };

    for (int q = 0; q < D - 1; ++q) stage_next();

    // ---- consumer pieces (all inlined; the arrays live in registers)
    // fast indices of the lane's R templates in the row whose metadata sits at mq: hi[r] = FIX_HC + the element's
    // place in shared memory; returns the smallest fraction word (see the comment at FIX_HC)
    auto fast_row = [&](uint32_t mq, uint32_t (&hi)[R]) -> uint32_t {
        double c, Q;
        lds_v2f64(mq, c, Q);
        uint32_t lo[R];
        if constexpr (UNI) {
            // equally spaced f0: template 32*r + lane sits at y0 + r*step, step = 32*delta*c
            const double y0 = __fma_rn(dlane, c, Q);
            const double step = __dmul_rn(p.d32, c);
            hi[0] = (uint32_t)__double2hiint(y0);
            lo[0] = (uint32_t)__double2loint(y0);
#pragma unroll
            for (int r = 1; r < R; ++r) {
                const double y = __fma_rn(step, (double)r, y0);
                hi[r] = (uint32_t)__double2hiint(y);
                lo[r] = (uint32_t)__double2loint(y);
            }
        } else {
#pragma unroll
            for (int r = 0; r < R; ++r) {
                const double y = __fma_rn(df[r], c, Q);
                hi[r] = (uint32_t)__double2hiint(y);
                lo[r] = (uint32_t)__double2loint(y);
            }
        }
        auto min3 = [](uint32_t x, uint32_t y, uint32_t z) { return min(x, min(y, z)); };
        if constexpr (R == 4) return min(min3(lo[0], lo[1], lo[2]), lo[3]);
        else if constexpr (R == 8) return min3(min3(lo[0], lo[1], lo[2]), min3(lo[3], lo[4], lo[5]), min(lo[6], lo[7]));
        else {
            static_assert(R == 4 || R == 8 || R == 16, "templates per lane");
            const uint32_t a0 = min3(lo[0], lo[1], lo[2]), a1 = min3(lo[3], lo[4], lo[5]), a2 = min3(lo[6], lo[7], lo[8]);
            const uint32_t a3 = min3(lo[9], lo[10], lo[11]), a4 = min3(lo[12], lo[13], lo[14]);
            return min(min3(a0, a1, a2), min3(a3, a4, lo[15]));
        }
    };
    // the same indices by the defining chain (bin_lo): taken where a lookup of this lane lies within thr of a
    // rounding boundary, or always when the fast index is switched off.  S = shared address of the row's slot.
    auto exact_row = [&](int n, uint32_t mc, uint32_t sc_, uint32_t (&hi)[R]) {
        const int j = row_of(n);
        const double gj = __ldg(g + j), dj = __ldg(d + j);
        const double Dp = TPOW2 ? __dmul_rn(dj, p.T) : dj;
        const int lo_f = bin_lo<TPOW2>(f_first, gj, Dp, p.T);
        const int kf = lo_f - p.k_min;
        // where the row was staged: mc = metadata of the slot's first row, sc_ = the slot's first byte
        const uint32_t fl = lds_u32(mc + 16u);
        const bool box = (fl & 512u) != 0;
        const int a_byte = box ? 128 * (int)lds_u32(mc + 24u) - (int)p.pad_bytes : (BPB * kf) & ~15;
        const uint32_t S = sc_ + (uint32_t)(n % RB) * (box ? ((fl >> 16) << 7) : (uint32_t)p.slot_bytes);
        const uint32_t base = FIX_HC + (uint32_t)((((int)S - a_byte) >> SH) + kf) - (uint32_t)lo_f;
#pragma unroll
        for (int r = 0; r < R; ++r)
            hi[r] = base + (uint32_t)bin_lo<TPOW2>(__ldg(p.f0 + min(i0 + r * 32 + lane, i_last)), gj, Dp, p.T);
    };
    // gather the row's elements from its staged window and accumulate: the element with index word hi sits at
    // shared byte address BPB*(hi - FIX_HC)
    const uint32_t addr0 = 0u - ((uint32_t)BPB * FIX_HC);
    auto add_row = [&](uint32_t mq, const uint32_t (&hi)[R]) {
        if constexpr (WGT) {
            const uint32_t wq = wmeta_s + ((mq - meta_s) >> 2);     // the row's RowWgt entry (8 bytes per 32 of RowMeta)
            const float wj = lds_f32(wq);
            if (lds_u32(mq + 16u) & 1024u) {  // warp-uniform: the whole tile is in band
                const double wd = (double)wj;
                W1u = __dadd_rn(W1u, wd);
                W2u = __dadd_rn(W2u, __dmul_rn(wd, wd));
                float v[R];
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    const uint32_t a = addr0 + (hi[r] << SH);
                    v[r] = FMT == FMT_F32 ? lds_f32(a) : (float)lds_u8(a);
                }
#pragma unroll
                for (int r = 0; r < R; r += 2) ffma2(acc[r], acc[r + 1], wj, v[r], v[r + 1], acc[r], acc[r + 1]);
            } else {
                const float wj2 = __fmul_rn(wj, wj);
                const uint32_t ktest = lds_u32(wq + 4u);
                float v[R];
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    const uint32_t a = addr0 + (hi[r] << SH);
                    v[r] = FMT == FMT_F32 ? lds_f32(a) : (float)lds_u8(a);
                    if (hi[r] + ktest < (uint32_t)p.n_bins) fadd2(w1p[r], w2p[r], w1p[r], w2p[r], wj, wj2);   // both counters in one add
                }
#pragma unroll
                for (int r = 0; r < R; r += 2) ffma2(acc[r], acc[r + 1], wj, v[r], v[r + 1], acc[r], acc[r + 1]);
            }
        } else if constexpr (FMT == FMT_F32 && TCW_FADD2) {
            float v[R];
#pragma unroll
            for (int r = 0; r < R; ++r) v[r] = lds_f32(addr0 + (hi[r] << SH));
#pragma unroll
            for (int r = 0; r < R; r += 2) fadd2(acc[r], acc[r + 1], acc[r], acc[r + 1], v[r], v[r + 1]);
        } else {
#pragma unroll
            for (int r = 0; r < R; ++r) {
                const uint32_t a = addr0 + (hi[r] << SH);
                if (FMT == FMT_F32) acc[r] += lds_f32(a);
                else acc[r] += (V)lds_u8(a);
            }
        }
    };

    uint32_t ph = 0;      // parity of the phase the slots complete in this pass over the ring
    uint32_t bar_c = bars_s, meta_c = meta_s, slot_c = slots_s;
    int sc = 0, nc = 0;   // slot of the ring and slot count of the consumer
    for (;;) {
        stage_next();     // refills the slot consumed in the previous iteration
        const uint32_t flags_w = lds_u32(meta_c + 16u);   // bit q: row q of the slot is staged; bit 8: no further rows;
        if (flags_w & 256u) break;                        // bit 9 and bits 16-23: one box copy of that many segments
        const uint32_t flags = flags_w & 255u;
        if (flags) {
            mbar_wait(bar_c, ph);
            if (PAIR && flags == (1u << RB) - 1u) {
                // the usual case, every row of the slot is live: two rows per straight-line block, so the
                // index arithmetic of one row overlaps the shared-memory gathers of the other.  The guard-band
                // branch repeats the gathers instead of merging, which keeps the fast path free of register moves.
#ifdef TCW_PAIR_LOOP
#pragma unroll 1
#else
#pragma unroll
#endif
                for (int q = 0; q < RB; q += 2) {
                    const uint32_t mq0 = meta_c + (uint32_t)(q * MB), mq1 = mq0 + (uint32_t)MB;
                    uint32_t hi0[R], hi1[R];
                    const uint32_t mn0 = fast_row(mq0, hi0);
                    const uint32_t mn1 = fast_row(mq1, hi1);
                    if constexpr (WGT || !UNI) {
                        bool done = false;
                        if constexpr (WGT && FMT == FMT_F32) {
                            if (lds_u32(mq0 + 16u) & lds_u32(mq1 + 16u) & 1024u) {
                                // weighted, the whole tile in band in both rows (warp-uniform): both rows' elements are
                                // gathered with the fast indices before the guard band is consulted, then accumulated
                                // in the order of the one-row path (row q, then row q + 1: bit-identical to it), so the
                                // gathers of one row overlap the arithmetic of the other
                                const uint32_t wq0 = wmeta_s + ((mq0 - meta_s) >> 2);
                                const float wa = lds_f32(wq0), wb = lds_f32(wq0 + (uint32_t)sizeof(RowWgt));
                                float v0[R], v1[R];
#pragma unroll
                                for (int r = 0; r < R; ++r) {
                                    v0[r] = lds_f32(addr0 + (hi0[r] << SH));
                                    v1[r] = lds_f32(addr0 + (hi1[r] << SH));
                                }
                                if (min(mn0, mn1) <= p.thr2) {
                                    uint32_t ex0[R], ex1[R];
                                    exact_row(RB * nc + q, meta_c, slot_c, ex0);
                                    exact_row(RB * nc + q + 1, meta_c, slot_c, ex1);
#pragma unroll
                                    for (int r = 0; r < R; ++r) {
                                        v0[r] = lds_f32(addr0 + (ex0[r] << SH));
                                        v1[r] = lds_f32(addr0 + (ex1[r] << SH));
                                    }
                                }
                                const double wda = (double)wa, wdb = (double)wb;
                                W1u = __dadd_rn(__dadd_rn(W1u, wda), wdb);
                                W2u = __dadd_rn(__dadd_rn(W2u, __dmul_rn(wda, wda)), __dmul_rn(wdb, wdb));
#pragma unroll
                                for (int r = 0; r < R; r += 2) {
                                    ffma2(acc[r], acc[r + 1], wa, v0[r], v0[r + 1], acc[r], acc[r + 1]);
                                    ffma2(acc[r], acc[r + 1], wb, v1[r], v1[r + 1], acc[r], acc[r + 1]);
                                }
                                done = true;
                            }
                        }
                        if (done) {
                        } else if (min(mn0, mn1) <= p.thr2) {
                            uint32_t ex0[R], ex1[R];
                            exact_row(RB * nc + q, meta_c, slot_c, ex0);
                            exact_row(RB * nc + q + 1, meta_c, slot_c, ex1);
                            add_row(mq0, ex0);
                            add_row(mq1, ex1);
                        } else {
                            add_row(mq0, hi0);
                            add_row(mq1, hi1);
                        }
                    } else {
                        // the two rows' elements are gathered with the fast indices and summed BEFORE the guard
                        // band is consulted (a fast index is at most one bin off, still inside the slot), so the
                        // gathers do not wait for the minimum; only the accumulate does.  Fixed order:
                        // acc += (row q + row q+1).
                        V t[R];
                        if constexpr (FMT == FMT_F32 && TCW_FADD2) {
                            float v0[R], v1[R];
#pragma unroll
                            for (int r = 0; r < R; ++r) {
                                v0[r] = lds_f32(addr0 + (hi0[r] << SH));
                                v1[r] = lds_f32(addr0 + (hi1[r] << SH));
                            }
#pragma unroll
                            for (int r = 0; r < R; r += 2) fadd2(t[r], t[r + 1], v0[r], v0[r + 1], v1[r], v1[r + 1]);
                        } else {
#pragma unroll
                            for (int r = 0; r < R; ++r) {
                                const uint32_t a0 = addr0 + (hi0[r] << SH), a1 = addr0 + (hi1[r] << SH);
                                if (FMT == FMT_F32) t[r] = lds_f32(a0) + lds_f32(a1);
                                else t[r] = (V)(lds_u8(a0) + lds_u8(a1));
                            }
                        }
                        if (min(mn0, mn1) <= p.thr2) {
                            uint32_t ex0[R], ex1[R];
                            exact_row(RB * nc + q, meta_c, slot_c, ex0);
                            exact_row(RB * nc + q + 1, meta_c, slot_c, ex1);
#pragma unroll
                            for (int r = 0; r < R; ++r) {
                                const uint32_t a0 = addr0 + (ex0[r] << SH), a1 = addr0 + (ex1[r] << SH);
                                if (FMT == FMT_F32) t[r] = lds_f32(a0) + lds_f32(a1);
                                else t[r] = (V)(lds_u8(a0) + lds_u8(a1));
                            }
                        }
                        if constexpr (FMT == FMT_F32 && TCW_FADD2) {
#pragma unroll
                            for (int r = 0; r < R; r += 2) fadd2(acc[r], acc[r + 1], acc[r], acc[r + 1], t[r], t[r + 1]);
                        } else {
#pragma unroll
                            for (int r = 0; r < R; ++r) acc[r] += t[r];
                        }
                    }
                }
            } else {
#pragma unroll
                for (int q = 0; q < RB; ++q) {
                    if (flags & (1u << q)) {
                        const uint32_t mq = meta_c + (uint32_t)(q * MB);
                        uint32_t hi[R];
                        if (fast_row(mq, hi) <= p.thr2) {
                            uint32_t ex[R];
                            exact_row(RB * nc + q, meta_c, slot_c, ex);
                            add_row(mq, ex);
                        } else {
                            add_row(mq, hi);
                        }
                    }
                }
            }
        }
        __syncwarp();     // every lane has read the slot before the next iteration refills it
        ++nc;
        bar_c += 8u; meta_c += RB * MB; slot_c += slot_stride;
        if (++sc == D) { sc = 0; bar_c = bars_s; slot_c = slots_s; ph ^= 1u; }
        if (meta_c == meta_e) meta_c = meta_s;
    }

    // ---------------- fixed-order combine of the warps' partial sums
    __syncthreads();      // every staged copy has been consumed: the slot region can be reused
    V *red = (V *)slots;
#pragma unroll
    for (int r = 0; r < R; ++r) red[warp * F + r * 32 + lane] = acc[r];
    if constexpr (WGT) {
        float *rw = (float *)slots + NW * F;          // [2][NW][F] per-lane sums, then [NW][2] float64 uniform sums
        double *wu = (double *)((float *)slots + 3 * NW * F);
#pragma unroll
        for (int r = 0; r < R; ++r) {
            rw[warp * F + r * 32 + lane] = w1p[r];
            rw[(NW + warp) * F + r * 32 + lane] = w2p[r];
        }
        if (lane == 0) { wu[2 * warp] = W1u; wu[2 * warp + 1] = W2u; }
    }
    __syncthreads();
    V best_v = lowest<V>();
    int best_i = INT32_MAX;
    const long cbase = ((long)chunk * p.n_groups + grp) * p.n_f0;
    V *dst = p.n_chunks > 1 ? (V *)p.cpart + cbase : (p.out_stat ? (V *)p.out_stat + grp * p.n_f0 : nullptr);
    for (int t = threadIdx.x; t < F; t += STAGED_THREADS) {
        const int i = i0 + t;
        if (i < p.n_f0) {
            V s = red[t];
#pragma unroll
            for (int w = 1; w < NW; ++w) s += red[w * F + t];
            if (dst) dst[i] = s;
            if constexpr (WGT) {
                const float *rw = (const float *)slots + NW * F;
                const double *wu = (const double *)((const float *)slots + 3 * NW * F);
                double W1 = 0, W2 = 0;
#pragma unroll
                for (int w = 0; w < NW; ++w) {
                    W1 += wu[2 * w] + (double)rw[w * F + t];
                    W2 += wu[2 * w + 1] + (double)rw[(NW + w) * F + t];
                }
                if (p.n_chunks > 1) {
                    p.cw1[cbase + i] = W1;
                    p.cw2[cbase + i] = W2;
                } else {
                    s = critical_ratio(s, W1, W2, p.mean1, p.var1);
                    if (p.out_psi) p.out_psi[grp * p.n_f0 + i] = s;
                }
            }
            argmax_step(best_v, best_i, s, i);
        }
    }
    if (p.n_chunks > 1) return;   // chunk_reduce_kernel adds the chunks and finds the tile's best
    __syncthreads();
    block_best<V>(best_v, best_i, (Best<V> *)slots, (Best<V> *)p.partial + grp * p.n_tiles + tile);
    block_done(p, part);
}

// Chunked searches: out_stat[i] = sum over the live SFT chunks, in ascending chunk order, of the
// chunk's partial sum; then the tile's (max, lowest index).  One block per (group, f0 tile).
template <typename V, bool WGT>
__global__ void __launch_bounds__(256)
chunk_reduce_kernel(const SumParams p)
{
    __shared__ Best<V> red[8];
    __shared__ unsigned char live[256];
    const int tile = (int)(blockIdx.x % p.n_tiles);
    const long grp = blockIdx.x / p.n_tiles;
    for (int c = threadIdx.x; c < p.n_chunks; c += blockDim.x)
        live[c] = p.clive[((long)c * p.n_groups + grp) * p.n_tiles + tile];
    __syncthreads();
    V best_v = lowest<V>();
    int best_i = INT32_MAX;
    const long stride = p.n_groups * (long)p.n_f0;
    const V *src = (const V *)p.cpart + grp * p.n_f0;
    for (int t = threadIdx.x; t < p.tile; t += blockDim.x) {
        const int i = tile * p.tile + t;
        if (i < p.n_f0) {
            V s = 0;
            for (int c = 0; c < p.n_chunks; ++c)
                if (live[c]) s += src[c * stride + i];
            if (p.out_stat) ((V *)p.out_stat)[grp * p.n_f0 + i] = s;
            if constexpr (WGT) {
                double W1 = 0, W2 = 0;
                for (int c = 0; c < p.n_chunks; ++c)
                    if (live[c]) {
                        W1 += p.cw1[c * stride + grp * p.n_f0 + i];
                        W2 += p.cw2[c * stride + grp * p.n_f0 + i];
                    }
                s = critical_ratio(s, W1, W2, p.mean1, p.var1);
                if (p.out_psi) p.out_psi[grp * p.n_f0 + i] = s;
            }
            argmax_step(best_v, best_i, s, i);
        }
    }
    block_best<V>(best_v, best_i, red, (Best<V> *)p.partial + grp * p.n_tiles + tile);
}

// --------------------------------------------------------------------------- candidate reduction
// out_best[group] = max over the group's tiles; tiles are in ascending f0, so a strict '>'
// keeps the lowest f0 index on ties (north_star (d)).
template <typename V>
__global__ void __launch_bounds__(128)
best_kernel(const Best<V> *__restrict__ partial, long n_groups, int n_tiles, Best<V> *__restrict__ out_best)
{
    long grp = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (grp >= n_groups) return;
    const Best<V> *q = partial + grp * n_tiles;
    Best<V> b = q[0];
    for (int t = 1; t < n_tiles; ++t) {
        Best<V> c = q[t];
        if (c.stat > b.stat) b = c;
    }
    out_best[grp] = b;
}

// --------------------------------------------------------------------------- index export
// k_j of the listed templates, by the same bin_lo the sum kernels use.
template <bool TPOW2>
__global__ void __launch_bounds__(256)
track_index_kernel(const SumParams p, const long *__restrict__ sel, long n_sel, int n_tau_brk,
                   int *__restrict__ out_k)
{
    long q = (long)blockIdx.x * blockDim.x + threadIdx.x;
    long total = n_sel * p.n_sft;
    if (q >= total) return;
    int j = (int)(q % p.n_sft);
    long lin = sel[q / p.n_sft];
    int i = (int)(lin % p.n_f0);
    long grp = lin / p.n_f0;
    if (j < p.j_begin) {
        out_k[q] = INT32_MIN;
        return;
    }
    double g = p.gtab[(grp % p.n_ab) * (long)p.n_sft + j];
    double d = p.dtab[(grp / p.n_ab) * (long)p.n_sft + j];
    double Dp = TPOW2 ? __dmul_rn(d, p.T) : d;
    out_k[q] = bin_lo<TPOW2>(p.f0[i], g, Dp, p.T) - p.k_min;
}

// --------------------------------------------------------------------------- layout
// Bit-packed number counts (uint32 words, LSB first) -> one byte per bin, rows at `pitch`.
__global__ void __launch_bounds__(256)
expand_bits_kernel(const uint32_t *__restrict__ words, long words_pitch, int n_sft, int n_bins,
                   unsigned char *__restrict__ dst, long pitch)
{
    const long total = (long)n_sft * n_bins;
    for (long q = (long)blockIdx.x * blockDim.x + threadIdx.x; q < total; q += (long)gridDim.x * blockDim.x) {
        const int j = (int)(q / n_bins), k = (int)(q % n_bins);
        const uint32_t w = words[j * words_pitch + (k >> 5)];
        dst[j * pitch + k] = (unsigned char)((w >> (k & 31)) & 1u);
    }
}


// Largest element of a uint8 spectrogram (rows at `pitch`): tells the host whether the packed
// int16 corrections of the two-level sky-block kernel are exact for this data.
__global__ void __launch_bounds__(256)
max_u8_kernel(const unsigned char *__restrict__ src, long pitch, int n_sft, int n_bins, int *__restrict__ out)
{
    const long total = (long)n_sft * n_bins;
    int m = 0;
    for (long q = (long)blockIdx.x * blockDim.x + threadIdx.x; q < total; q += (long)gridDim.x * blockDim.x)
        m = max(m, (int)src[(q / n_bins) * pitch + (q % n_bins)]);
    for (int o = 16; o; o >>= 1) m = max(m, __shfl_xor_sync(0xffffffffu, m, o));
    if ((threadIdx.x & 31) == 0 && m) atomicMax(out, m);
}

}  // namespace tcw
