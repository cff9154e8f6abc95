// tcw_sum.cuh -- bin index, gather-accumulate and candidate reduction kernels (sm_100a).
//
// The statistic is "summed across the data bins selected by the track": for
// template i of group (s, a, b) and SFT j
//     x = ((f0_i * g[a][b][j]) * D[s][j]) * T_sft ,  k = rint(x) - k_min         (eq. (1)-(2))
//     stat_i += spectrogram[j][k]  if 0 <= k < n_bins .
// Two kernels compute it:
//   * sum_staged_kernel -- the product path.  One CTA owns (group, tile of consecutive f0).
//     Consecutive f0 of one group select a narrow contiguous bin window per SFT (g <= 1), so a
//     producer warp stages the [32 SFT x window] slab into shared memory with one TMA bulk copy
//     (cp.async.bulk, mbarrier complete_tx) per SFT row through a multi-stage ring, and eight
//     consumer warps gather from shared memory, each lane carrying R templates.
//   * sum_gather_kernel -- one thread per template gathering from global memory.  It serves f0
//     axes so sparse that the window of a 32-template tile does not fit shared memory, and it is
//     the simple kernel the staged one is checked against.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace tcw {

enum { FMT_F32 = 0, FMT_U8 = 1, FMT_BITS = 2 };

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
    const unsigned char *spec;  // library copy of the spectrogram, rows 16-byte aligned
    long pitch;                 // its row pitch in bytes (multiple of 16)
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
    int stages, pitch_s;        // staged kernel: ring depth, shared-memory row pitch (bytes)
    int *status;                // device status word
};

template <int FMT> struct Acc { typedef int type; };
template <> struct Acc<FMT_F32> { typedef float type; };

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

// --------------------------------------------------------------------------- gather kernel
template <int FMT, bool TPOW2>
__global__ void __launch_bounds__(128)
sum_gather_kernel(const SumParams p)
{
    typedef typename Acc<FMT>::type V;
    __shared__ Best<V> red[4];
    const int tile = blockIdx.x % p.n_tiles;
    const long grp = blockIdx.x / p.n_tiles;
    const int i = tile * p.tile + threadIdx.x;
    const bool valid = i < p.n_f0;
    const double f0 = p.f0[valid ? i : p.n_f0 - 1];
    const double *g = p.gtab + (grp % p.n_ab) * (long)p.n_sft;
    const double *d = p.dtab + (grp / p.n_ab) * (long)p.n_sft;
    V acc = 0;
    for (int j = p.j_begin; j < p.n_sft; ++j) {
        double Dp = TPOW2 ? __dmul_rn(d[j], p.T) : d[j];
        int k = bin_lo<TPOW2>(f0, g[j], Dp, p.T) - p.k_min;
        if ((unsigned)k < (unsigned)p.n_bins) {
            const unsigned char *row = p.spec + (long)j * p.pitch;
            if (FMT == FMT_F32) acc += ((const float *)row)[k];
            else if (FMT == FMT_U8) acc += (V)row[k];
            else acc += (V)((((const uint32_t *)row)[k >> 5] >> (k & 31)) & 1u);
        }
    }
    if (valid && p.out_stat) ((V *)p.out_stat)[grp * p.n_f0 + i] = acc;
    block_best<V>(valid ? acc : lowest<V>(), valid ? i : INT32_MAX, red,
                  (Best<V> *)p.partial + grp * p.n_tiles + tile);
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
__device__ __forceinline__ float lds_f32(uint32_t a)
{
    float v;
    asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(a));
    return v;
}
__device__ __forceinline__ uint32_t lds_u8(uint32_t a)
{
    uint32_t v;
    asm volatile("ld.shared.u8 %0, [%1];" : "=r"(v) : "r"(a));
    return v;
}
__device__ __forceinline__ uint32_t lds_u32(uint32_t a)
{
    uint32_t v;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(a));
    return v;
}

// --------------------------------------------------------------------------- staged kernel
constexpr int ROWS = 32;      // SFT rows per stage (one per producer lane)
constexpr int NCW = 8;        // consumer warps
constexpr int STAGED_THREADS = 32 * (NCW + 1);

// Per staged row: what a consumer lane needs to turn rint(x) into a shared-memory address.
struct __align__(16) RowMeta {
    double g, Dp;   // spin-down factor and Doppler factor (times T_sft when it is a power of two)
    uint32_t rb;    // f32: addr = rb + 4*lo   u8: addr = rb + lo   bits: word addr = rb + 4*((u + d0) >> 5)
    int lo0;        // k_min + first in-band bin of the row window
    int span;       // last - first in-band bin of the window; < 0: nothing to do in this row
    int d0;         // bits: offset of bin lo0 from the first staged bit
};

// dynamic shared memory: [full[S] | empty[S] | ctrl[S] (pad to 16)] [meta S*ROWS] [slab S*ROWS*pitch_s]
__host__ __device__ inline size_t staged_header_bytes(int stages) { return ((size_t)stages * 20 + 15) & ~(size_t)15; }
__host__ __device__ inline size_t staged_smem_bytes(int stages, int pitch_s)
{
    return staged_header_bytes(stages) + (size_t)stages * ROWS * (sizeof(RowMeta) + pitch_s);
}

template <int FMT> __device__ __forceinline__ int byte_of_bin(int k)
{
    return FMT == FMT_F32 ? 4 * k : (FMT == FMT_U8 ? k : (k >> 5) * 4);
}

template <int FMT, int R, bool TPOW2>
__global__ void __launch_bounds__(STAGED_THREADS)
sum_staged_kernel(const SumParams p)
{
    typedef typename Acc<FMT>::type V;
    constexpr int F = 32 * R;  // templates per tile
    extern __shared__ __align__(16) unsigned char smem[];
    const int S = p.stages;
    uint64_t *full = (uint64_t *)smem;
    uint64_t *empty = full + S;
    volatile int *ctrl = (volatile int *)(empty + S);
    RowMeta *meta = (RowMeta *)(smem + staged_header_bytes(S));
    unsigned char *slab = (unsigned char *)(meta + S * ROWS);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    // heavy tiles (high f0 stays in band longest) are launched first
    const int tile = p.n_tiles - 1 - (int)(blockIdx.x % p.n_tiles);
    const long grp = blockIdx.x / p.n_tiles;
    const int i0 = tile * F;
    const int i_last = min(i0 + F, p.n_f0) - 1;

    if (threadIdx.x == 0) {
        for (int s = 0; s < S; ++s) {
            mbar_init(smem_u32(full + s), 32);
            mbar_init(smem_u32(empty + s), NCW);
            ctrl[s] = 0;
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    V acc[R];
#pragma unroll
    for (int r = 0; r < R; ++r) acc[r] = 0;

    if (warp == NCW) {
        // ---------------- producer warp: lane = SFT row of the stage
        const double *g = p.gtab + (grp % p.n_ab) * (long)p.n_sft;
        const double *d = p.dtab + (grp / p.n_ab) * (long)p.n_sft;
        const double f_first = p.f0[i0], f_last = p.f0[i_last];
        const double below = (double)p.k_min - 1.0;
        int st = 0;
        uint32_t ph = 0;
        for (int jt = p.j_begin;; jt += ROWS) {
            const int j = jt + lane;
            const bool in_list = j < p.n_sft;
            const double gj = in_list ? g[j] : 0.0;
            const double dj = in_list ? d[j] : 1.0;
            // g decreases with j, so once the highest template of the tile is below the band
            // for the largest possible Doppler factor, no later SFT can contribute.
            const bool row_dead = !in_list || (f_last * gj * p.dmaxT < below);
            const bool tile_dead = __shfl_sync(0xffffffffu, row_dead, 0);
            mbar_wait(smem_u32(empty + st), ph ^ 1);
            if (tile_dead) {
                if (lane == 0) ctrl[st] = 1;
                __syncwarp();
                mbar_arrive(smem_u32(full + st));
                break;
            }
            RowMeta m;
            m.g = gj;
            m.Dp = TPOW2 ? __dmul_rn(dj, p.T) : dj;
            m.rb = 0; m.lo0 = 0; m.span = -1; m.d0 = 0;
            uint32_t bytes = 0;
            const unsigned char *src = nullptr;
            const uint32_t row_s = smem_u32(slab + (size_t)(st * ROWS + lane) * p.pitch_s);
            if (in_list) {
                int kf = bin_lo<TPOW2>(f_first, gj, m.Dp, p.T) - p.k_min;
                int kl = bin_lo<TPOW2>(f_last, gj, m.Dp, p.T) - p.k_min;
                int kfc = max(kf, 0), klc = min(kl, p.n_bins - 1);
                if (kfc <= klc) {
                    int a_byte = byte_of_bin<FMT>(kfc) & ~15;
                    int e_byte = (byte_of_bin<FMT>(klc) + (FMT == FMT_U8 ? 1 : 4) + 15) & ~15;
                    if (e_byte - a_byte > p.pitch_s) {
                        atomicOr(p.status, 1);  // host-side window bound violated: never expected
                    } else {
                        bytes = (uint32_t)(e_byte - a_byte);
                        src = p.spec + (long)j * p.pitch + a_byte;
                        m.lo0 = p.k_min + kfc;
                        m.span = klc - kfc;
                        if (FMT == FMT_F32) m.rb = row_s - 4u * (uint32_t)(p.k_min + a_byte / 4);
                        else if (FMT == FMT_U8) m.rb = row_s - (uint32_t)(p.k_min + a_byte);
                        else { m.rb = row_s; m.d0 = kfc - a_byte * 8; }
                    }
                }
            }
            meta[st * ROWS + lane] = m;
            if (bytes) {
                mbar_arrive_expect_tx(smem_u32(full + st), bytes);
                bulk_g2s(row_s, src, bytes, smem_u32(full + st));
            } else {
                mbar_arrive(smem_u32(full + st));
            }
            if (++st == S) { st = 0; ph ^= 1; }
        }
    } else {
        // ---------------- consumer warps: lane carries templates i0 + r*32 + lane
        double f0r[R];
#pragma unroll
        for (int r = 0; r < R; ++r) f0r[r] = p.f0[min(i0 + r * 32 + lane, p.n_f0 - 1)];
        int st = 0;
        uint32_t ph = 0;
        for (;;) {
            mbar_wait(smem_u32(full + st), ph);
            if (ctrl[st]) break;
            const RowMeta *ms = meta + st * ROWS;
#pragma unroll 1
            for (int rr = warp; rr < ROWS; rr += NCW) {
                const RowMeta m = ms[rr];
                if (m.span < 0) continue;
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    const int lo = bin_lo<TPOW2>(f0r[r], m.g, m.Dp, p.T);
                    const uint32_t u = (uint32_t)(lo - m.lo0);
                    if (u <= (uint32_t)m.span) {
                        if (FMT == FMT_F32) acc[r] += lds_f32(m.rb + 4u * (uint32_t)lo);
                        else if (FMT == FMT_U8) acc[r] += (V)lds_u8(m.rb + (uint32_t)lo);
                        else {
                            const uint32_t rel = u + (uint32_t)m.d0;
                            acc[r] += (V)((lds_u32(m.rb + 4u * (rel >> 5)) >> (rel & 31u)) & 1u);
                        }
                    }
                }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(smem_u32(empty + st));
            if (++st == S) { st = 0; ph ^= 1; }
        }
    }

    // ---------------- fixed-order combine of the consumer warps' partial sums
    __syncthreads();  // every staged copy has been consumed: the slab can be reused
    V *red = (V *)slab;
    if (warp < NCW) {
#pragma unroll
        for (int r = 0; r < R; ++r) red[warp * F + r * 32 + lane] = acc[r];
    }
    __syncthreads();
    V tot = lowest<V>();
    int idx = INT32_MAX;
    if (threadIdx.x < F) {
        const int i = i0 + threadIdx.x;
        if (i < p.n_f0) {
            V s = red[threadIdx.x];
#pragma unroll
            for (int w = 1; w < NCW; ++w) s += red[w * F + threadIdx.x];
            if (p.out_stat) ((V *)p.out_stat)[grp * p.n_f0 + i] = s;
            tot = s;
            idx = i;
        }
    }
    __syncthreads();
    block_best<V>(tot, idx, (Best<V> *)meta, (Best<V> *)p.partial + grp * p.n_tiles + tile);
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

}  // namespace tcw
