// tcw_select.cuh -- downstream selection over a statistic array (sm_100a).
//
// "a threshold was set on Psi based on the distribution of critical ratios on only noise using
// the same amount of templates (Psi_noise max) ... an injection was considered detected if a
// template close to the injection had Psi > Psi_noise max".  Two exact operations
// over a device array of n statistics (float32 Psi / power sums, or int32 counts):
//   * top-K: the K largest values in descending order, equal values in ascending index order
//     (K = 1 on a noise-only search gives Psi_noise max);
//   * threshold selection: the indices i with value[i] > threshold, ascending.
// Both are HBM-bound streaming passes with integer bookkeeping only, so results are exact and
// run-to-run identical:
//   top-K = radix select of the K-th largest key (three histogram passes over 11 + 11 + 10 bits of
//   an order-preserving uint32 key, shared-memory histograms, integer atomics), then an ordered
//   compaction (per-block counts -> one-block scan -> ordered scatter) of the keys above it plus
//   the lowest-index keys equal to it, then a bitonic sort of the K candidates in one CTA.
//   NaN is never selected; -0.0 equals +0.0.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace tcw {

constexpr int SEL_THREADS = 256;
constexpr int SEL_MAX_BLOCKS = 2048;   // the block-count scan runs in one CTA
constexpr int SEL_MAX_K = 2048;        // candidates sorted in one CTA's shared memory

struct SelState {
    unsigned int prefix;        // high bits of the K-th largest key found so far
    unsigned int k_rem;         // candidates still to take among the keys matching `prefix`
    unsigned int k_eff;         // min(K, number of selectable values)
    unsigned int n_greater;     // keys strictly above the K-th largest (after the last pass)
    unsigned long long count;   // threshold selection: number of values above the threshold
};

// order-preserving key of a float32 (NaN -> 0 = "not selectable"), or of an int32
__device__ __forceinline__ unsigned int sel_key(unsigned int bits, int is_int)
{
    if (is_int) return (bits ^ 0x80000000u) | 0u;
    if ((bits & 0x7fffffffu) > 0x7f800000u) return 0u;           // NaN
    if ((bits << 1) == 0u) bits = 0u;                             // -0.0 == +0.0
    return (bits & 0x80000000u) ? ~bits : (bits | 0x80000000u);
}
// int32 keys can be 0 (INT32_MIN); selectable test is format dependent
__device__ __forceinline__ bool sel_valid(unsigned int bits, int is_int)
{
    return is_int || (bits & 0x7fffffffu) <= 0x7f800000u;
}

struct SelSeg { long begin, end; };
__device__ __forceinline__ SelSeg sel_segment(long n, long seg)
{
    long b = (long)blockIdx.x * seg;
    long e = b + seg < n ? b + seg : n;
    return {b, e};
}

// histogram of one radix digit over the keys whose higher bits equal state->prefix
//   pass 0: bits 31..21 (2048 bins), pass 1: bits 20..10 (2048), pass 2: bits 9..0 (1024)
template <int PASS>
__global__ void __launch_bounds__(SEL_THREADS)
sel_hist_kernel(const unsigned int *__restrict__ vals, long n, long seg, int is_int,
                const SelState *__restrict__ state, unsigned int *__restrict__ hist)
{
    __shared__ unsigned int h[2048];
    for (int t = threadIdx.x; t < 2048; t += SEL_THREADS) h[t] = 0;
    __syncthreads();
    const unsigned int prefix = PASS ? state->prefix : 0u;
    const SelSeg sg = sel_segment(n, seg);
    for (long i = sg.begin + threadIdx.x; i < sg.end; i += SEL_THREADS) {
        const unsigned int bits = vals[i];
        if (!sel_valid(bits, is_int)) continue;
        const unsigned int key = sel_key(bits, is_int);
        if (PASS == 0) atomicAdd(&h[key >> 21], 1u);
        else if (PASS == 1) { if ((key >> 21) == (prefix >> 21)) atomicAdd(&h[(key >> 10) & 2047u], 1u); }
        else { if ((key >> 10) == (prefix >> 10)) atomicAdd(&h[key & 1023u], 1u); }
    }
    __syncthreads();
    for (int t = threadIdx.x; t < 2048; t += SEL_THREADS)
        if (h[t]) atomicAdd(&hist[t], h[t]);
}

// one CTA: walk the digit histogram from the top until the cumulative count reaches k_rem
template <int PASS>
__global__ void __launch_bounds__(1)
sel_pick_kernel(unsigned int *__restrict__ hist, SelState *__restrict__ state, unsigned int K)
{
    const int bins = PASS == 2 ? 1024 : 2048;
    unsigned int k_rem = state->k_rem;
    if (PASS == 0) {
        unsigned long long total = 0;
        for (int b = 0; b < bins; ++b) total += hist[b];
        k_rem = (unsigned int)(total < K ? total : K);
        state->k_eff = k_rem;
        state->prefix = 0;
    }
    unsigned int above = 0;
    int d = bins - 1;
    if (k_rem > 0)
        for (; d > 0; --d) {
            if (above + hist[d] >= k_rem) break;
            above += hist[d];
        }
    const int shift = PASS == 0 ? 21 : (PASS == 1 ? 10 : 0);
    state->prefix |= (unsigned int)d << shift;
    state->k_rem = k_rem - above;          // still to take among the keys with this digit
    if (PASS == 2) state->n_greater = state->k_eff - state->k_rem;
    for (int b = 0; b < bins; ++b) hist[b] = 0;   // ready for the next pass
}

// ---- ordered compaction -------------------------------------------------------------------
// predicate classes of one element: 2 = taken unconditionally, 1 = equal to the K-th key (taken
// while the equal budget lasts, in index order), 0 = not taken
template <bool THR>
__device__ __forceinline__ int sel_class(unsigned int bits, int is_int, unsigned int kth, double thr)
{
    if (THR) {
        const double v = is_int ? (double)(int)bits : (double)__uint_as_float(bits);
        return v > thr ? 2 : 0;                       // NaN compares false
    }
    if (!sel_valid(bits, is_int)) return 0;
    const unsigned int key = sel_key(bits, is_int);
    return key > kth ? 2 : (key == kth ? 1 : 0);
}

template <bool THR>
__global__ void __launch_bounds__(SEL_THREADS)
sel_count_kernel(const unsigned int *__restrict__ vals, long n, long seg, int is_int,
                 const SelState *__restrict__ state, double thr,
                 unsigned int *__restrict__ blk_gt, unsigned int *__restrict__ blk_eq)
{
    __shared__ unsigned int s_gt, s_eq;
    if (threadIdx.x == 0) s_gt = s_eq = 0;
    __syncthreads();
    const unsigned int kth = THR ? 0u : state->prefix;
    const SelSeg sg = sel_segment(n, seg);
    unsigned int gt = 0, eq = 0;
    for (long i = sg.begin + threadIdx.x; i < sg.end; i += SEL_THREADS) {
        const int c = sel_class<THR>(vals[i], is_int, kth, thr);
        gt += c == 2;
        eq += c == 1;
    }
    for (int o = 16; o; o >>= 1) {
        gt += __shfl_xor_sync(0xffffffffu, gt, o);
        eq += __shfl_xor_sync(0xffffffffu, eq, o);
    }
    if ((threadIdx.x & 31) == 0) { atomicAdd(&s_gt, gt); atomicAdd(&s_eq, eq); }
    __syncthreads();
    if (threadIdx.x == 0) { blk_gt[blockIdx.x] = s_gt; blk_eq[blockIdx.x] = s_eq; }
}

// exclusive scan of the per-block counts (one thread: at most SEL_MAX_BLOCKS entries)
__global__ void __launch_bounds__(1)
sel_scan_kernel(unsigned int *__restrict__ blk_gt, unsigned int *__restrict__ blk_eq, int n_blocks,
                unsigned long long *__restrict__ off_gt, unsigned long long *__restrict__ off_eq,
                SelState *__restrict__ state)
{
    unsigned long long a = 0, b = 0;
    for (int q = 0; q < n_blocks; ++q) {
        off_gt[q] = a;
        off_eq[q] = b;
        a += blk_gt[q];
        b += blk_eq[q];
    }
    state->count = a;
}

// block-wide exclusive scan of a 0/1 flag; returns this thread's rank and the block total
__device__ __forceinline__ unsigned int sel_block_rank(bool flag, unsigned int *warp_tot, unsigned int &total)
{
    const unsigned int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const unsigned int m = __ballot_sync(0xffffffffu, flag);
    if (lane == 0) warp_tot[warp] = __popc(m);
    __syncthreads();
    unsigned int base = 0, tot = 0;
    for (unsigned int w = 0; w < SEL_THREADS / 32; ++w) {
        const unsigned int c = warp_tot[w];
        if (w < warp) base += c;
        tot += c;
    }
    __syncthreads();
    total = tot;
    return base + __popc(m & ((1u << lane) - 1u));
}

// THR: out_idx[rank] = i for the values above the threshold, ascending i, up to `capacity`.
// top-K: candidates (raw bits, index) -> cand_bits / cand_idx [k_eff]: the keys above the K-th
// first (any order: they are sorted afterwards), then the lowest-index keys equal to it.
template <bool THR>
__global__ void __launch_bounds__(SEL_THREADS)
sel_scatter_kernel(const unsigned int *__restrict__ vals, long n, long seg, int is_int,
                   const SelState *__restrict__ state, double thr,
                   const unsigned long long *__restrict__ off_gt, const unsigned long long *__restrict__ off_eq,
                   long capacity, unsigned int *__restrict__ cand_bits, long long *__restrict__ out_idx)
{
    __shared__ unsigned int wt[SEL_THREADS / 32];
    const unsigned int kth = THR ? 0u : state->prefix;
    const unsigned long long n_greater = THR ? 0ull : state->n_greater;
    const unsigned long long eq_budget = THR ? 0ull : state->k_rem;
    unsigned long long base_gt = off_gt[blockIdx.x], base_eq = off_eq[blockIdx.x];
    const SelSeg sg = sel_segment(n, seg);
    for (long i0 = sg.begin; i0 < sg.end; i0 += SEL_THREADS) {
        const long i = i0 + threadIdx.x;
        const unsigned int bits = i < sg.end ? vals[i] : 0u;
        const int c = i < sg.end ? sel_class<THR>(bits, is_int, kth, thr) : 0;
        unsigned int tot;
        const unsigned int r2 = sel_block_rank(c == 2, wt, tot);
        if (c == 2) {
            const unsigned long long pos = base_gt + r2;
            if (THR) { if ((long)pos < capacity) out_idx[pos] = i; }
            else { cand_bits[pos] = bits; out_idx[pos] = i; }
        }
        base_gt += tot;
        if (!THR) {
            const unsigned int r1 = sel_block_rank(c == 1, wt, tot);
            if (c == 1 && base_eq + r1 < eq_budget) {
                const unsigned long long pos = n_greater + base_eq + r1;
                cand_bits[pos] = bits;
                out_idx[pos] = i;
            }
            base_eq += tot;
        }
    }
}

// one CTA: bitonic sort of the k_eff candidates by (key descending, index ascending)
__global__ void __launch_bounds__(1024)
sel_sort_kernel(const unsigned int *__restrict__ cand_bits, const long long *__restrict__ cand_idx, int is_int,
                const SelState *__restrict__ state, unsigned int *__restrict__ out_val,
                long long *__restrict__ out_idx, int *__restrict__ out_count)
{
    __shared__ unsigned int key[SEL_MAX_K], raw[SEL_MAX_K];
    __shared__ long long idx[SEL_MAX_K];
    const int k = (int)state->k_eff;
    for (int t = threadIdx.x; t < SEL_MAX_K; t += 1024) {
        if (t < k) { raw[t] = cand_bits[t]; key[t] = sel_key(raw[t], is_int); idx[t] = cand_idx[t]; }
        else { raw[t] = 0; key[t] = 0; idx[t] = 0x7fffffffffffffffLL; }
    }
    __syncthreads();
    for (int size = 2; size <= SEL_MAX_K; size <<= 1)
        for (int stride = size >> 1; stride > 0; stride >>= 1) {
            for (int t = threadIdx.x; t < SEL_MAX_K / 2; t += 1024) {
                const int lo = 2 * t - (t & (stride - 1));
                const int hi = lo + stride;
                // "a before b": larger key first, then smaller index; padding (key 0, index max) sorts last
                const bool a_first = key[lo] > key[hi] || (key[lo] == key[hi] && idx[lo] < idx[hi]);
                const bool desc = (lo & size) == 0;
                if (a_first != desc) {
                    unsigned int tk = key[lo]; key[lo] = key[hi]; key[hi] = tk;
                    unsigned int tr = raw[lo]; raw[lo] = raw[hi]; raw[hi] = tr;
                    long long ti = idx[lo]; idx[lo] = idx[hi]; idx[hi] = ti;
                }
            }
            __syncthreads();
        }
    for (int t = threadIdx.x; t < k; t += 1024) { out_val[t] = raw[t]; out_idx[t] = idx[t]; }
    if (threadIdx.x == 0 && out_count) *out_count = k;
}

}  // namespace tcw
