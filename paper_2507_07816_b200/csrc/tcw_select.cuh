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
// Large arrays take a two-read route first (tcw_topk): a monotone 2048-bin map of the keys, zoomed on
// the upper tail by a small sample, is histogrammed in ONE pass that also stores every CTA's own
// histogram; the bin holding the K-th largest key is picked; a second pass compacts, in index order,
// the keys at or above that bin (a few thousand for typical statistics) together with their indices;
// the exact selection above then runs on the compacted candidates.  If the candidates would exceed
// SEL_MAX_CAND (heavily tied data) the full-array route is taken instead.  Same results either way.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace tcw {

constexpr int SEL_THREADS = 256;
constexpr int SEL_MAX_BLOCKS = 2048;   // the block-count scan runs in one CTA
constexpr int SEL_MAX_K = 2048;        // candidates sorted in one CTA's shared memory
constexpr int SEL_MAX_CAND = 1 << 20;  // two-read route: candidate buffer (key bits + index per entry)
constexpr int SEL_SAMPLE = 2048;       // keys sampled to place the zoom window

struct SelState {
    unsigned int prefix;        // high bits of the K-th largest key found so far
    unsigned int k_rem;         // candidates still to take among the keys matching `prefix`
    unsigned int k_eff;         // min(K, number of selectable values)
    unsigned int n_greater;     // keys strictly above the K-th largest (after the last pass)
    unsigned long long count;   // threshold selection: number of values above the threshold
    // two-read route: monotone bin map  bin(key) = 0 if key < z_lo, else min(((key - z_lo) >> z_shift) + 1, 2047);
    // z_bin = the bin of the K-th largest key; n_cand = keys in bins >= z_bin; cand_ok = 1 when they fit the
    // candidate buffer
    unsigned int z_shift, z_lo, z_bin, n_cand, cand_ok;
    unsigned int z_val_lo;      // raw value (float bits / int) of the lowest key in a bin >= 1: smaller values skip the key arithmetic
    unsigned int z_val_bin;     // raw value of the lowest key in a bin >= z_bin: only values at or above it can be candidates
};

// the monotone bin of a key under the zoom window (non-decreasing in key)
__device__ __forceinline__ unsigned int sel_zoom_bin(unsigned int key, unsigned int z_shift, unsigned int z_lo)
{
    if (key < z_lo) return 0u;
    return min(((key - z_lo) >> z_shift) + 1u, 2047u);
}
// the lowest key of bin d >= 1 (saturating)
__device__ __forceinline__ unsigned int sel_zoom_bin_lo(unsigned int d, unsigned int z_shift, unsigned int z_lo)
{
    const unsigned long long k = (unsigned long long)z_lo + ((unsigned long long)(d - 1u) << z_shift);
    return k > 0xffffffffull ? 0xffffffffu : (unsigned int)k;
}

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

// Kernels of the exact selection are enqueued for both routes; `gate` says which launch is live:
// 0 always; 1 only if the two-read route found too many candidates (full array); 2 only if it did not
// (then the array is the candidate buffer and its length is state->n_cand).
__device__ __forceinline__ bool sel_gate(const SelState *__restrict__ state, int gate, long &n)
{
    if (gate == 0) return true;
    const unsigned int ok = state->cand_ok;
    if (gate == 1) return ok == 0u;
    if (ok == 0u) return false;
    n = (long)state->n_cand < n ? (long)state->n_cand : n;
    return true;
}

// inverse of sel_key (for keys of selectable values)
__device__ __forceinline__ unsigned int sel_unkey(unsigned int key, int is_int)
{
    if (is_int) return key ^ 0x80000000u;
    return (key & 0x80000000u) ? (key & 0x7fffffffu) : ~key;
}
// raw value `b` is certainly below raw value `lim` (false for NaN: those take the exact path)
__device__ __forceinline__ bool sel_raw_below(unsigned int b, unsigned int lim, int is_int)
{
    return is_int ? (int)b < (int)lim : __uint_as_float(b) < __uint_as_float(lim);
}

struct SelSeg { long begin, end; };
__device__ __forceinline__ SelSeg sel_segment(long n, long seg)
{
    long b = (long)blockIdx.x * seg;
    long e = b + seg < n ? b + seg : n;
    return {b, e};
}

// Streaming access: a CTA walks its segment in tiles of 4 * SEL_THREADS elements, thread t owning the
// four consecutive elements tile + 4t .. tile + 4t + 3 (one 16-byte load when the array is 16-byte
// aligned; segments start on multiples of 1024 elements).  nv = how many of the four are in range.
constexpr int SEL_TILE = 4 * SEL_THREADS;
constexpr int SEL_ROW = 128;      // a row: the 128 consecutive values one warp fetches with one 16-byte load per lane
__device__ __forceinline__ void sel_load4(const unsigned int *__restrict__ vals, long i, long end, bool vec,
                                          unsigned int (&b)[4], int &nv)
{
    nv = end - i >= 4 ? 4 : (end > i ? (int)(end - i) : 0);
    if (vec && nv == 4) {
        const uint4 q = __ldg((const uint4 *)(vals + i));
        b[0] = q.x; b[1] = q.y; b[2] = q.z; b[3] = q.w;
    } else {
#pragma unroll
        for (int c = 0; c < 4; ++c) b[c] = c < nv ? __ldg(vals + i + c) : 0u;
    }
}

// histogram of one radix digit over the keys whose higher bits equal state->prefix
//   pass 0: bits 31..21 (2048 bins), pass 1: bits 20..10 (2048), pass 2: bits 9..0 (1024)
// Pass 0 sees every key and statistics cluster in a few dozen digits, so it keeps four copies of
// the histogram, picked by the lane, which cuts same-address atomic conflicts fourfold.
template <int PASS>
__global__ void __launch_bounds__(SEL_THREADS)
sel_hist_kernel(const unsigned int *__restrict__ vals, long n, long seg, int is_int, int vec,
                const SelState *__restrict__ state, unsigned int *__restrict__ hist, int gate = 0)
{
    constexpr int COPIES = PASS == 0 ? 4 : 1;
    __shared__ unsigned int h[COPIES * 2048];
    if (!sel_gate(state, gate, n)) return;
    for (int t = threadIdx.x; t < COPIES * 2048; t += SEL_THREADS) h[t] = 0;
    __syncthreads();
    const unsigned int prefix = PASS ? state->prefix : 0u;
    const SelSeg sg = sel_segment(n, seg);
    unsigned int *hc = h + (threadIdx.x & (COPIES - 1)) * 2048;
    // Passes 1 and 2 only count the keys that share the prefix found so far, a small minority: a
    // cheap value-range test (a superset of the matching keys) skips the key arithmetic for the rest.
    const unsigned int kmask = PASS == 1 ? 0x001fffffu : 0x000003ffu;
    const unsigned int klo = PASS == 1 ? (prefix & ~kmask) : (prefix & ~kmask), khi = klo | kmask;
    float flo = 0.f, fhi = 0.f;
    int ilo = 0, ihi = 0;
    if (PASS) {
        if (is_int) { ilo = (int)(klo ^ 0x80000000u); ihi = (int)(khi ^ 0x80000000u); }
        else {
            // clamp the key range to the keys of -inf .. +inf, then map both ends back to float32
            const unsigned int a = klo < 0x007fffffu ? 0x007fffffu : klo, b = khi > 0xff800000u ? 0xff800000u : khi;
            flo = __uint_as_float((a & 0x80000000u) ? (a & 0x7fffffffu) : ~a);
            fhi = __uint_as_float((b & 0x80000000u) ? (b & 0x7fffffffu) : ~b);
        }
    }
    // two tiles per iteration: 32 bytes in flight per thread keep the HBM pipe full
    for (long t0 = sg.begin; t0 < sg.end; t0 += 2 * SEL_TILE) {
        unsigned int b[8];
        int nv[2];
        {
            unsigned int b0[4], b1[4];
            sel_load4(vals, t0 + 4 * threadIdx.x, sg.end, vec != 0, b0, nv[0]);
            sel_load4(vals, t0 + SEL_TILE + 4 * threadIdx.x, sg.end, vec != 0, b1, nv[1]);
#pragma unroll
            for (int c = 0; c < 4; ++c) { b[c] = b0[c]; b[4 + c] = b1[c]; }
        }
#pragma unroll
        for (int c = 0; c < 8; ++c) {
            if (PASS) {
                const bool maybe = is_int ? ((int)b[c] >= ilo && (int)b[c] <= ihi)
                                          : (__uint_as_float(b[c]) >= flo && __uint_as_float(b[c]) <= fhi);
                if (!maybe) continue;
            }
            const bool ok = (c & 3) < nv[c >> 2] && sel_valid(b[c], is_int);
            const unsigned int key = sel_key(b[c], is_int);
            if (PASS == 0) {
                if (ok) atomicAdd(&hc[key >> 21], 1u);
            } else if (PASS == 1) {
                if (ok && (key >> 21) == (prefix >> 21)) atomicAdd(&h[(key >> 10) & 2047u], 1u);
            } else {
                if (ok && (key >> 10) == (prefix >> 10)) atomicAdd(&h[key & 1023u], 1u);
            }
        }
    }
    __syncthreads();
    for (int t = threadIdx.x; t < 2048; t += SEL_THREADS) {
        unsigned int c = h[t];
        for (int q = 1; q < COPIES; ++q) c += h[q * 2048 + t];
        if (c) atomicAdd(&hist[t], c);
    }
}

// one CTA: walk the digit histogram from the top until the cumulative count reaches k_rem
// (thread t sums the 8 bins [8t, 8t + 8); thread 0 walks the 256 partial sums, then the 8 bins)
template <int PASS>
__global__ void __launch_bounds__(256)
sel_pick_kernel(unsigned int *__restrict__ hist, SelState *__restrict__ state, unsigned int K, int gate = 0)
{
    constexpr int bins = PASS == 2 ? 1024 : 2048;
    __shared__ unsigned int part[256];
    { long dummy = 0; if (!sel_gate(state, gate, dummy)) return; }
    unsigned int mine = 0;
    for (int b = 0; b < 8; ++b) { const int q = 8 * threadIdx.x + b; mine += q < bins ? hist[q] : 0u; }
    part[threadIdx.x] = mine;
    __syncthreads();
    if (threadIdx.x == 0) {
        unsigned int k_rem = state->k_rem;
        if (PASS == 0) {
            unsigned long long total = 0;
            for (int t = 0; t < 256; ++t) total += part[t];
            k_rem = (unsigned int)(total < K ? total : K);
            state->k_eff = k_rem;
            state->prefix = 0;
        }
        unsigned int above = 0;
        int d = 0;
        if (k_rem > 0) {
            int t = bins / 8 - 1;
            for (; t > 0; --t) {
                if (above + part[t] >= k_rem) break;
                above += part[t];
            }
            for (d = 8 * t + 7; d > 8 * t; --d) {
                if (above + hist[d] >= k_rem) break;
                above += hist[d];
            }
        }
        constexpr int shift = PASS == 0 ? 21 : (PASS == 1 ? 10 : 0);
        state->prefix |= (unsigned int)d << shift;
        state->k_rem = k_rem - above;          // still to take among the keys with this digit
        if (PASS == 2) state->n_greater = state->k_eff - state->k_rem;
    }
    __syncthreads();
    for (int b = threadIdx.x; b < bins; b += 256) hist[b] = 0;   // ready for the next pass
}

__device__ __forceinline__ unsigned int sel_block_scan(unsigned int cnt, unsigned int *warp_tot, unsigned int &total);

// ---- two-read route -------------------------------------------------------------------------
// One CTA: SEL_SAMPLE keys at a fixed stride, sorted descending.  The zoom window starts at the sample's r-th
// largest key, r as small as still leaves an expected 8 K values above it (2 <= r <= 16): everything below is
// settled by one compare in pass A, and the fewer values reach the window the fewer warps leave that fast path.
// The bins are 1/128 of the spread between the sample's largest and 16th largest key wide, so that 2047 of them
// resolve the tail far above the sample's maximum.  Any window gives exact results; this one gives few candidates.
__global__ void __launch_bounds__(1024)
sel_sample_kernel(const unsigned int *__restrict__ vals, long n, int is_int, unsigned int K, SelState *__restrict__ state)
{
    __shared__ unsigned int key[SEL_SAMPLE];
    const long stride = n / SEL_SAMPLE > 0 ? n / SEL_SAMPLE : 1;
    for (int t = threadIdx.x; t < SEL_SAMPLE; t += 1024) {
        const long i = (long)t * stride;
        const unsigned int b = i < n ? __ldg(vals + i) : 0u;
        key[t] = (i < n && sel_valid(b, is_int)) ? sel_key(b, is_int) : 0u;
    }
    __syncthreads();
    for (int size = 2; size <= SEL_SAMPLE; size <<= 1)
        for (int st = size >> 1; st > 0; st >>= 1) {
            for (int t = threadIdx.x; t < SEL_SAMPLE / 2; t += 1024) {
                const int lo = 2 * t - (t & (st - 1)), hi = lo + st;
                const bool desc = (lo & size) == 0;
                if ((key[lo] > key[hi]) != desc) { const unsigned int k = key[lo]; key[lo] = key[hi]; key[hi] = k; }
            }
            __syncthreads();
        }
    if (threadIdx.x == 0) {
        const unsigned int spread = key[0] - key[15];
        const int bits = spread ? 32 - __clz(spread) : 0;
        const int shift = bits > 7 ? bits - 7 : 0;                   // spread >> shift < 128
        long r = ((long)8 * K * SEL_SAMPLE + n - 1) / n;
        r = r < 2 ? 2 : (r > 16 ? 16 : r);
        state->z_shift = (unsigned int)shift;
        state->z_lo = key[r - 1];
        state->z_val_lo = sel_unkey(key[r - 1], is_int);
        state->z_val_bin = state->z_val_lo;
        state->z_bin = 0;
        state->n_cand = 0;
        state->cand_ok = 0;
    }
}

// Pass A: histogram of the zoom bins over all keys; every CTA also stores its own histogram (2048 words)
// so that the candidates of pass B can be placed in index order without another read of the array.
// Almost every key lies below the zoom window (bin 0): one compare per value settles those, branch-free,
// and counts them in a register; only iterations that hold a value in or above the window take the key
// arithmetic and the shared-memory atomics.
template <int IS_INT>
__global__ void __launch_bounds__(SEL_THREADS)
sel_zoom_hist_kernel(const unsigned int *__restrict__ vals, long n, long seg, int vec,
                     const SelState *__restrict__ state, unsigned int *__restrict__ hist, unsigned int *__restrict__ blk_hist,
                     unsigned short *__restrict__ row_max)
{
    __shared__ unsigned int h[2048];
    for (int t = threadIdx.x; t < 2048; t += SEL_THREADS) h[t] = 0;
    __syncthreads();
    const unsigned int zs = state->z_shift, zl = state->z_lo, vlo = state->z_val_lo;
    const SelSeg sg = sel_segment(n, seg);
    unsigned int below = 0;
    for (long t0 = sg.begin; t0 < sg.end; t0 += 2 * SEL_TILE) {
        unsigned int b[8];
        int nv[2];
        {
            unsigned int b0[4], b1[4];
            sel_load4(vals, t0 + 4 * threadIdx.x, sg.end, vec != 0, b0, nv[0]);
            sel_load4(vals, t0 + SEL_TILE + 4 * threadIdx.x, sg.end, vec != 0, b1, nv[1]);
#pragma unroll
            for (int c = 0; c < 4; ++c) { b[c] = b0[c]; b[4 + c] = b1[c]; }
        }
        unsigned int rest = 0;                                  // bit c: value c needs the exact path
#pragma unroll
        for (int c = 0; c < 8; ++c) {
            const bool inr = (c & 3) < nv[c >> 2];
            const bool lt = sel_raw_below(b[c], vlo, IS_INT);
            below += (inr && lt) ? 1u : 0u;
            rest |= (inr && !lt) ? (1u << c) : 0u;
        }
        unsigned int m0 = 0, m1 = 0;                            // largest zoom bin among this thread's values of either tile
        if (rest) {
#pragma unroll
            for (int c = 0; c < 8; ++c) {
                if ((rest >> c & 1u) && sel_valid(b[c], IS_INT)) {
                    const unsigned int d = sel_zoom_bin(sel_key(b[c], IS_INT), zs, zl);
                    if (d) atomicAdd(&h[d], 1u); else ++below;
                    if (c < 4) m0 = max(m0, d); else m1 = max(m1, d);
                }
            }
        }
        // the largest bin of each ROW (the 128 consecutive values one warp loads): pass B opens only the rows that can
        // hold a candidate, a few thousand of three million, instead of reading the array again
        // (row_max is zeroed by the host; only warps that met the window write)
        if (__any_sync(0xffffffffu, rest != 0u)) {
            m0 = __reduce_max_sync(0xffffffffu, m0);
            m1 = __reduce_max_sync(0xffffffffu, m1);
            if ((threadIdx.x & 31) == 0) {
                const long r0 = (t0 >> 7) + (threadIdx.x >> 5), r1 = r0 + SEL_TILE / SEL_ROW;
                if (m0) row_max[r0] = (unsigned short)m0;
                if (m1) row_max[r1] = (unsigned short)m1;
            }
        }
    }
    for (int o = 16; o; o >>= 1) below += __shfl_xor_sync(0xffffffffu, below, o);
    if ((threadIdx.x & 31) == 0 && below) atomicAdd(&h[0], below);
    __syncthreads();
    for (int t = threadIdx.x; t < 2048; t += SEL_THREADS) {
        const unsigned int c = h[t];
        blk_hist[(long)blockIdx.x * 2048 + t] = c;
        if (c) atomicAdd(&hist[t], c);
    }
}

// One CTA: the bin of the K-th largest key, the number of candidates (keys in bins >= it), whether they fit
__global__ void __launch_bounds__(256)
sel_zoom_pick_kernel(unsigned int *__restrict__ hist, SelState *__restrict__ state, unsigned int K, int is_int)
{
    __shared__ unsigned int part[256];
    unsigned int mine = 0;
    for (int b = 0; b < 8; ++b) mine += hist[8 * threadIdx.x + b];
    part[threadIdx.x] = mine;
    __syncthreads();
    if (threadIdx.x == 0) {
        unsigned long long total = 0;
        for (int t = 0; t < 256; ++t) total += part[t];
        const unsigned long long k = total < K ? total : K;
        unsigned long long above = 0;
        int d = 0;
        if (k > 0) {
            int t = 255;
            for (; t > 0; --t) {
                if (above + part[t] >= k) break;
                above += part[t];
            }
            for (d = 8 * t + 7; d > 8 * t; --d) {
                if (above + hist[d] >= k) break;
                above += hist[d];
            }
        }
        const unsigned long long n_cand = above + hist[d];
        state->z_bin = (unsigned int)d;
        {
            // the lowest key of bin d (d >= 1) as a raw value: pass B tests values against it before any key arithmetic
            state->z_val_bin = sel_unkey(sel_zoom_bin_lo((unsigned int)(d > 0 ? d : 1), state->z_shift, state->z_lo), is_int);
        }
        state->n_cand = n_cand > 0xffffffffull ? 0xffffffffu : (unsigned int)n_cand;
        state->cand_ok = (k > 0 && n_cand <= (unsigned long long)SEL_MAX_CAND) ? 1u : 0u;
    }
    __syncthreads();
    for (int b = threadIdx.x; b < 2048; b += 256) hist[b] = 0;
}

// per-CTA candidate counts from the stored histograms: one warp per CTA of pass A
__global__ void __launch_bounds__(256)
sel_zoom_count_kernel(const unsigned int *__restrict__ blk_hist, int n_blocks, const SelState *__restrict__ state,
                      unsigned int *__restrict__ blk_cnt)
{
    const unsigned int d0 = state->z_bin;
    const int b = blockIdx.x * 8 + (threadIdx.x >> 5), lane = threadIdx.x & 31;
    if (b >= n_blocks) return;
    unsigned int c = 0;
    for (unsigned int d = d0 + lane; d < 2048u; d += 32) c += blk_hist[(long)b * 2048 + d];
    for (int o = 16; o; o >>= 1) c += __shfl_xor_sync(0xffffffffu, c, o);
    if (lane == 0) blk_cnt[b] = c;
}
// their exclusive scan (one CTA, <= 2048 entries: thread t owns 8)
__global__ void __launch_bounds__(256)
sel_zoom_scan_kernel(const unsigned int *__restrict__ blk_cnt, int n_blocks, unsigned int *__restrict__ blk_off)
{
    __shared__ unsigned int pa[256];
    unsigned int a = 0;
    for (int c = 0; c < 8; ++c) { const int q = 8 * threadIdx.x + c; a += q < n_blocks ? blk_cnt[q] : 0u; }
    pa[threadIdx.x] = a;
    __syncthreads();
    if (threadIdx.x == 0) {
        unsigned int s = 0;
        for (int t = 0; t < 256; ++t) { const unsigned int v = pa[t]; pa[t] = s; s += v; }
    }
    __syncthreads();
    a = pa[threadIdx.x];
    for (int c = 0; c < 8; ++c) {
        const int q = 8 * threadIdx.x + c;
        if (q < n_blocks) { blk_off[q] = a; a += blk_cnt[q]; }
    }
}

// Rows: a row is SEL_ROW = 128 consecutive values, what one warp fetches with one 16-byte load per lane.  The
// streaming passes leave one small summary per row (largest zoom bin, or number of selected values); the passes
// below read only the summaries and open the few rows that matter.  Warp w of a CTA owns a contiguous run of
// the CTA's rows, lanes scan 32 summaries at a time, and an open row is loaded by the whole warp: lane order,
// then the four values of a lane, is index order.
//   open(r)  -> the row may hold a wanted value     take(bits) -> the value is wanted
//   WRITE = false: returns the number of wanted values in the warp's rows (warp-uniform);
//   WRITE = true:  emit(rank, bits, index) for each of them, ranks ascending from `pos`.
template <bool WRITE, class Open, class Take, class Emit>
__device__ __forceinline__ unsigned int sel_walk_rows(const unsigned int *__restrict__ vals, long end, bool vec, long w0, long w1,
                                                      Open open, Take take, unsigned long long pos, Emit emit)
{
    const unsigned int lane = threadIdx.x & 31, lt = (1u << lane) - 1u;
    unsigned int total = 0;
    for (long rb = w0; rb < w1; rb += 32) {
        const long r = rb + lane;
        unsigned int m = __ballot_sync(0xffffffffu, r < w1 && open(r));
        while (m) {
            const long row = rb + (__ffs(m) - 1);
            m &= m - 1;
            const long i = row * SEL_ROW + 4 * lane;
            unsigned int b[4];
            int nv;
            sel_load4(vals, i, end, vec, b, nv);
            unsigned int c = 0, t[4];
#pragma unroll
            for (int q = 0; q < 4; ++q) { t[q] = (q < nv && take(b[q])) ? 1u : 0u; c += t[q]; }
            if (!WRITE) {
                total += __reduce_add_sync(0xffffffffu, c);
            } else {
                // exclusive prefix of c over the lanes: four ballots of the per-value flags, counted below the lane
                unsigned int before = 0, all = 0;
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    const unsigned int bm = __ballot_sync(0xffffffffu, t[q] != 0u);
                    before += __popc(bm & lt);
                    all += __popc(bm);
                }
                unsigned long long at = pos + before;
#pragma unroll
                for (int q = 0; q < 4; ++q)
                    if (t[q]) { emit(at, b[q], i + q); ++at; }
                pos += all;
                total += all;
            }
        }
    }
    return total;
}
// the contiguous run of rows warp `warp` of this CTA owns
__device__ __forceinline__ void sel_warp_rows(const SelSeg &sg, long &w0, long &w1)
{
    const long r_begin = sg.begin / SEL_ROW, r_end = (sg.end + SEL_ROW - 1) / SEL_ROW;
    const long rpw = (r_end - r_begin + SEL_THREADS / 32 - 1) / (SEL_THREADS / 32);
    w0 = min(r_begin + rpw * (threadIdx.x >> 5), r_end);
    w1 = min(w0 + rpw, r_end);
}

// Pass B: the keys in bins >= z_bin with their indices, in index order, into the candidate buffer.  It does not
// read the array again: pass A left the largest bin of every row, and only rows whose maximum reaches z_bin are
// opened (counted first, then written behind the per-CTA offsets from the stored histograms).
template <int IS_INT>
__global__ void __launch_bounds__(SEL_THREADS)
sel_zoom_compact_kernel(const unsigned int *__restrict__ vals, long n, long seg, int vec,
                        const SelState *__restrict__ state, const unsigned int *__restrict__ blk_off,
                        const unsigned short *__restrict__ row_max,
                        unsigned int *__restrict__ cand_bits, long long *__restrict__ cand_idx)
{
    __shared__ unsigned int wt[SEL_THREADS / 32];
    if (!state->cand_ok) return;
    const unsigned int zs = state->z_shift, zl = state->z_lo, d0 = state->z_bin, vbin = state->z_val_bin;
    const SelSeg sg = sel_segment(n, seg);
    long w0, w1;
    sel_warp_rows(sg, w0, w1);
    auto open = [&](long r) { return (unsigned int)row_max[r] >= d0; };
    auto take = [&](unsigned int bits) {
        return (d0 == 0u || !sel_raw_below(bits, vbin, IS_INT)) && sel_valid(bits, IS_INT) &&
               sel_zoom_bin(sel_key(bits, IS_INT), zs, zl) >= d0;
    };
    auto emit = [&](unsigned long long at, unsigned int bits, long i) { cand_bits[at] = bits; cand_idx[at] = i; };
    const unsigned int cnt = sel_walk_rows<false>(vals, sg.end, vec != 0, w0, w1, open, take, 0ull, emit);
    if ((threadIdx.x & 31) == 0) wt[threadIdx.x >> 5] = cnt;
    __syncthreads();
    unsigned long long pos = blk_off[blockIdx.x];
    for (unsigned int w = 0; w < (threadIdx.x >> 5); ++w) pos += wt[w];
    if (cnt) sel_walk_rows<true>(vals, sg.end, vec != 0, w0, w1, open, take, pos, emit);
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
    if (is_int) {
        const int v = (int)bits, kv = (int)(kth ^ 0x80000000u);
        return v > kv ? 2 : (v == kv ? 1 : 0);
    }
    // float32: comparing the values is comparing the keys (NaN compares false; -0.0 == +0.0 as in sel_key)
    const float kf = __uint_as_float((kth & 0x80000000u) ? (kth & 0x7fffffffu) : ~kth);
    const float v = __uint_as_float(bits);
    return v > kf ? 2 : (v == kf ? 1 : 0);
}

template <bool THR>
__global__ void __launch_bounds__(SEL_THREADS)
sel_count_kernel(const unsigned int *__restrict__ vals, long n, long seg, int is_int, int vec,
                 const SelState *__restrict__ state, double thr,
                 unsigned int *__restrict__ blk_gt, unsigned int *__restrict__ blk_eq, int gate = 0,
                 unsigned char *__restrict__ row_cnt = nullptr)
{
    __shared__ unsigned int s_gt, s_eq;
    if (!THR && !sel_gate(state, gate, n)) return;
    if (threadIdx.x == 0) s_gt = s_eq = 0;
    __syncthreads();
    const unsigned int kth = THR ? 0u : state->prefix;
    const SelSeg sg = sel_segment(n, seg);
    unsigned int gt = 0, eq = 0;
    for (long t0 = sg.begin; t0 < sg.end; t0 += 2 * SEL_TILE) {
        unsigned int b0[4], b1[4];
        int n0, n1;
        sel_load4(vals, t0 + 4 * threadIdx.x, sg.end, vec != 0, b0, n0);
        sel_load4(vals, t0 + SEL_TILE + 4 * threadIdx.x, sg.end, vec != 0, b1, n1);
        unsigned int g0 = 0, g1 = 0;
#pragma unroll
        for (int c = 0; c < 4; ++c) {
            const int c0 = c < n0 ? sel_class<THR>(b0[c], is_int, kth, thr) : 0;
            const int c1 = c < n1 ? sel_class<THR>(b1[c], is_int, kth, thr) : 0;
            g0 += c0 == 2;
            g1 += c1 == 2;
            eq += (c0 == 1) + (c1 == 1);
        }
        gt += g0 + g1;
        if (THR && row_cnt) {
            // how many values of each ROW (128 consecutive values, one warp's load) are selected: the scatter pass
            // then opens only the rows that hold one instead of reading the array again
            // (row_cnt is zeroed by the host; only warps that hold a selected value write)
            if (__any_sync(0xffffffffu, (g0 | g1) != 0u)) {
                g0 = __reduce_add_sync(0xffffffffu, g0);
                g1 = __reduce_add_sync(0xffffffffu, g1);
                if ((threadIdx.x & 31) == 0) {
                    const long r0 = (t0 >> 7) + (threadIdx.x >> 5), r1 = r0 + SEL_TILE / SEL_ROW;
                    if (g0) row_cnt[r0] = (unsigned char)g0;
                    if (g1) row_cnt[r1] = (unsigned char)g1;
                }
            }
        }
    }
    for (int o = 16; o; o >>= 1) {
        gt += __shfl_xor_sync(0xffffffffu, gt, o);
        eq += __shfl_xor_sync(0xffffffffu, eq, o);
    }
    if ((threadIdx.x & 31) == 0) { atomicAdd(&s_gt, gt); atomicAdd(&s_eq, eq); }
    __syncthreads();
    if (threadIdx.x == 0) { blk_gt[blockIdx.x] = s_gt; blk_eq[blockIdx.x] = s_eq; }
}

// exclusive scan of the per-block counts (at most SEL_MAX_BLOCKS = 8 * 256 entries: thread t owns 8)
__global__ void __launch_bounds__(256)
sel_scan_kernel(unsigned int *__restrict__ blk_gt, unsigned int *__restrict__ blk_eq, int n_blocks,
                unsigned long long *__restrict__ off_gt, unsigned long long *__restrict__ off_eq,
                SelState *__restrict__ state, int gate = 0)
{
    __shared__ unsigned long long pa[256], pb[256];
    { long dummy = 0; if (!sel_gate(state, gate, dummy)) return; }
    unsigned long long a = 0, b = 0;
    for (int c = 0; c < 8; ++c) {
        const int q = 8 * threadIdx.x + c;
        if (q < n_blocks) { a += blk_gt[q]; b += blk_eq[q]; }
    }
    pa[threadIdx.x] = a;
    pb[threadIdx.x] = b;
    __syncthreads();
    if (threadIdx.x == 0) {
        unsigned long long sa = 0, sb = 0;
        for (int t = 0; t < 256; ++t) {
            const unsigned long long ta = pa[t], tb = pb[t];
            pa[t] = sa; pb[t] = sb;
            sa += ta; sb += tb;
        }
        state->count = sa;
    }
    __syncthreads();
    a = pa[threadIdx.x];
    b = pb[threadIdx.x];
    for (int c = 0; c < 8; ++c) {
        const int q = 8 * threadIdx.x + c;
        if (q < n_blocks) { off_gt[q] = a; off_eq[q] = b; a += blk_gt[q]; b += blk_eq[q]; }
    }
}

// block-wide exclusive scan of a small per-thread count; returns this thread's offset and the block total
__device__ __forceinline__ unsigned int sel_block_scan(unsigned int cnt, unsigned int *warp_tot, unsigned int &total)
{
    const unsigned int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    unsigned int inc = cnt;
    for (int o = 1; o < 32; o <<= 1) {
        const unsigned int up = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= (unsigned int)o) inc += up;
    }
    if (lane == 31) warp_tot[warp] = inc;
    __syncthreads();
    unsigned int base = 0, tot = 0;
    for (unsigned int w = 0; w < SEL_THREADS / 32; ++w) {
        const unsigned int c = warp_tot[w];
        if (w < warp) base += c;
        tot += c;
    }
    __syncthreads();
    total = tot;
    return base + inc - cnt;
}

// THR: out_idx[rank] = i for the values above the threshold, ascending i, up to `capacity`.
// top-K: candidates (raw bits, index) -> cand_bits / cand_idx [k_eff]: the keys above the K-th
// first (in index order; they are sorted afterwards), then the lowest-index keys equal to it.
// A CTA whose segment holds no candidate (known from the count pass) reads nothing; a tile with no
// candidate costs one vector load and one barrier.
template <bool THR>
__global__ void __launch_bounds__(SEL_THREADS)
sel_scatter_kernel(const unsigned int *__restrict__ vals, long n, long seg, int is_int, int vec,
                   const SelState *__restrict__ state, double thr,
                   const unsigned int *__restrict__ blk_gt, const unsigned int *__restrict__ blk_eq,
                   const unsigned long long *__restrict__ off_gt, const unsigned long long *__restrict__ off_eq,
                   long capacity, unsigned int *__restrict__ cand_bits, long long *__restrict__ out_idx,
                   const long long *__restrict__ idx_map = nullptr, int gate = 0)
{
    __shared__ unsigned int wt[SEL_THREADS / 32];
    if (!THR && !sel_gate(state, gate, n)) return;
    const unsigned int kth = THR ? 0u : state->prefix;
    const unsigned long long n_greater = THR ? 0ull : state->n_greater;
    const unsigned long long eq_budget = THR ? 0ull : state->k_rem;
    unsigned long long base_gt = off_gt[blockIdx.x], base_eq = off_eq[blockIdx.x];
    const bool want_eq = !THR && blk_eq[blockIdx.x] != 0 && base_eq < eq_budget;
    if (blk_gt[blockIdx.x] == 0 && !want_eq) return;
    if (THR && (long)base_gt >= capacity) return;
    const SelSeg sg = sel_segment(n, seg);
    for (long t0 = sg.begin; t0 < sg.end; t0 += SEL_TILE) {
        const long i = t0 + 4 * threadIdx.x;
        unsigned int b[4];
        int nv, cls[4];
        sel_load4(vals, i, sg.end, vec != 0, b, nv);
        unsigned int c2 = 0, c1 = 0;
#pragma unroll
        for (int c = 0; c < 4; ++c) {
            cls[c] = c < nv ? sel_class<THR>(b[c], is_int, kth, thr) : 0;
            c2 += cls[c] == 2;
            c1 += cls[c] == 1;
        }
        if (!__syncthreads_or((int)(c2 | c1))) continue;
        unsigned int tot;
        unsigned int r2 = sel_block_scan(c2, wt, tot);
        const unsigned int tot2 = tot;
        unsigned int r1 = 0, tot1 = 0;
        if (!THR) { r1 = sel_block_scan(c1, wt, tot); tot1 = tot; }
#pragma unroll
        for (int c = 0; c < 4; ++c) {
            if (cls[c] == 2) {
                const unsigned long long pos = base_gt + r2++;
                if (THR) { if ((long)pos < capacity) out_idx[pos] = i + c; }
                else { cand_bits[pos] = b[c]; out_idx[pos] = idx_map ? idx_map[i + c] : i + c; }
            } else if constexpr (!THR) {
                if (cls[c] == 1) {
                    const unsigned long long q = base_eq + r1++;
                    if (q < eq_budget) { cand_bits[n_greater + q] = b[c]; out_idx[n_greater + q] = idx_map ? idx_map[i + c] : i + c; }
                }
            }
        }
        base_gt += tot2;
        base_eq += tot1;
    }
}

// Threshold selection, second pass: out_idx[rank] = i for the values above the threshold, ascending i, up to
// `capacity`.  Reads the per-row counts of the count pass (n/128 bytes) and opens only the rows that hold a selected
// value (sel_walk_rows).
__global__ void __launch_bounds__(SEL_THREADS)
sel_scatter_rows_kernel(const unsigned int *__restrict__ vals, long n, long seg, int is_int, int vec, double thr,
                        const unsigned char *__restrict__ row_cnt, const unsigned long long *__restrict__ off_gt,
                        long capacity, long long *__restrict__ out_idx)
{
    __shared__ unsigned int wt[SEL_THREADS / 32];
    const SelSeg sg = sel_segment(n, seg);
    long w0, w1;
    sel_warp_rows(sg, w0, w1);
    unsigned int cnt = 0;
    for (long r = w0 + (threadIdx.x & 31); r < w1; r += 32) cnt += row_cnt[r];
    cnt = __reduce_add_sync(0xffffffffu, cnt);
    if ((threadIdx.x & 31) == 0) wt[threadIdx.x >> 5] = cnt;
    __syncthreads();
    unsigned long long pos = off_gt[blockIdx.x];
    for (unsigned int w = 0; w < (threadIdx.x >> 5); ++w) pos += wt[w];
    if (cnt == 0) return;
    auto open = [&](long r) { return row_cnt[r] != 0; };
    auto take = [&](unsigned int bits) { return sel_class<true>(bits, is_int, 0u, thr) == 2; };
    auto emit = [&](unsigned long long at, unsigned int, long i) { if ((long)at < capacity) out_idx[at] = i; };
    sel_walk_rows<true>(vals, sg.end, vec != 0, w0, w1, open, take, pos, emit);
}

// one CTA: bitonic sort of the k_eff candidates by (key descending, index ascending)
__global__ void __launch_bounds__(1024)
sel_sort_kernel(const unsigned int *__restrict__ cand_bits, const long long *__restrict__ cand_idx, int is_int,
                const SelState *__restrict__ state, unsigned int *__restrict__ out_val,
                long long *__restrict__ out_idx, int *__restrict__ out_count, int gate = 0)
{
    __shared__ unsigned int key[SEL_MAX_K], raw[SEL_MAX_K];
    __shared__ long long idx[SEL_MAX_K];
    { long dummy = 0; if (!sel_gate(state, gate, dummy)) return; }
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
