// tcw_peaks.cuh -- microbenchmarks of the limits that bind the track-sum kernels on this GPU (sm_100a).
//
// The gather-accumulate kernels are bound by warp-instruction issue, the FP64 pipe and shared-memory
// gathers, not by HBM; MEASURED_PEAKS.json has no entry for any of those
// ("the builder must micro-benchmark those").  tcw_measure_peaks times, with
// CUDA events, kernels that do nothing but
//   * independent FP64 instructions (DFMA, DMUL, DADD) -- the FP64 pipe's warp-instruction rate,
//   * independent FP32 FFMA                            -- the schedulers' warp-instruction issue rate,
//   * independent LDS.32 gathers of the access pattern the staged kernel has (lanes on consecutive
//     templates read words at a stride below one) -- the shared-memory gather rate,
//   * the bare lookup chain of the staged kernel as it ships (one DFMA, one address LEA, one LDS.32, half a FADD2,
//     half a VIMNMX3 per lookup, two rows of 16 lookups per straight-line block) -- the speed of light of the
//     design's instruction mix, in lookups per second.
//   * the staged kernel's ring alone (no consumer): four 1-D bulk copies per slot against one tensor-map copy per
//     slot -- the L2 -> shared-memory staging rate, in bytes per second.
// Rates are whole-GPU, per second.  The numbers are only as good as the clocks of the moment; bench.py
// measures them in the same process as the timed search and prints the SM clock beside them.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "tcw_sum.cuh"   // fadd2

namespace tcw {

constexpr int PEAK_THREADS = 256;
constexpr int PEAK_ILP = 8;

// kind 0: DFMA, 1: DMUL, 2: DADD.  PEAK_ILP independent chains per thread, `iters` rounds.
template <int KIND>
__global__ void __launch_bounds__(PEAK_THREADS)
peak_fp64_kernel(int iters, double seed, double *out)
{
    double a[PEAK_ILP];
#pragma unroll
    for (int i = 0; i < PEAK_ILP; ++i) a[i] = seed + (double)(threadIdx.x + i);
    const double m = 1.0 + seed * 1e-9, c = seed * 1e-3;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < 4; ++u) {
#pragma unroll
            for (int i = 0; i < PEAK_ILP; ++i) {
                if (KIND == 0) a[i] = __fma_rn(a[i], m, c);
                else if (KIND == 1) a[i] = __dmul_rn(a[i], m);
                else a[i] = __dadd_rn(a[i], c);
            }
        }
    }
    double s = 0;
#pragma unroll
    for (int i = 0; i < PEAK_ILP; ++i) s += a[i];
    if (s == 12345.678) out[0] = s;          // never true: keeps the chains alive
}

// Independent FP32 FFMA chains: one warp instruction per scheduler per cycle is the issue limit.
__global__ void __launch_bounds__(PEAK_THREADS)
peak_issue_kernel(int iters, float seed, float *out)
{
    float a[PEAK_ILP];
#pragma unroll
    for (int i = 0; i < PEAK_ILP; ++i) a[i] = seed + (float)(threadIdx.x + i);
    const float m = 1.0f + seed * 1e-6f, c = seed * 1e-3f;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < 4; ++u) {
#pragma unroll
            for (int i = 0; i < PEAK_ILP; ++i) a[i] = __fmaf_rn(a[i], m, c);
        }
    }
    float s = 0;
#pragma unroll
    for (int i = 0; i < PEAK_ILP; ++i) s += a[i];
    if (s == 12345.678f) out[0] = s;
}

// LDS.32 gathers with the staged kernel's pattern: lane l, lookup r reads word (l*s + r*32*s) of a
// 2 KB window, s = 0.93 (a spin-down factor times a Doppler factor); 16 independent loads per block,
// four blocks per round at different immediate offsets (so that no two loads of a round coincide and
// none can be merged), each load followed by the FADD that consumes it.
template <int OFF>
__device__ __forceinline__ float peak_lds_off(uint32_t a)
{
    float v;
    asm volatile("ld.shared.f32 %0, [%1+%2];" : "=f"(v) : "r"(a), "n"(OFF));
    return v;
}
__global__ void __launch_bounds__(PEAK_THREADS)
peak_lds_kernel(int iters, float *out)
{
    __shared__ float win[8 * 640 + 64];
    for (int i = threadIdx.x; i < 8 * 640 + 64; i += PEAK_THREADS) win[i] = (float)i * 1e-6f;
    __syncthreads();
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const uint32_t base = (uint32_t)__cvta_generic_to_shared(win);
    uint32_t a[16];
#pragma unroll
    for (int r = 0; r < 16; ++r) a[r] = base + 4u * ((uint32_t)(warp * 640) + (uint32_t)((lane + 32 * r) * 0.93f));
    float acc[16];
#pragma unroll
    for (int r = 0; r < 16; ++r) acc[r] = 0.0f;
    for (int it = 0; it < iters; it += 4) {
#pragma unroll
        for (int r = 0; r < 16; ++r) acc[r] += peak_lds_off<0>(a[r]);
#pragma unroll
        for (int r = 0; r < 16; ++r) acc[r] += peak_lds_off<64>(a[r]);
#pragma unroll
        for (int r = 0; r < 16; ++r) acc[r] += peak_lds_off<128>(a[r]);
#pragma unroll
        for (int r = 0; r < 16; ++r) acc[r] += peak_lds_off<192>(a[r]);
    }
    float s = 0;
#pragma unroll
    for (int r = 0; r < 16; ++r) s += acc[r];
    if (s == 12345.678f) out[0] = s;
}

// The bare lookup chain of sum_staged_kernel as it ships: two rows per straight-line block, per row 16 x { DFMA,
// address, LDS.32 } plus the minimum of the fraction words, the two rows' elements added pairwise and accumulated
// with packed float32 adds (FADD2); nothing else (no staging, no metadata, no band edges).
__global__ void __launch_bounds__(128, 3)
peak_chain_kernel(int rows, double c0, double q0, float *out)
{
    __shared__ float win[4 * 640];
    for (int i = threadIdx.x; i < 4 * 640; i += 128) win[i] = (float)i * 1e-6f;
    __syncthreads();
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const uint32_t base = (uint32_t)__cvta_generic_to_shared(win) + (uint32_t)(warp * 640 * 4) - 4u * 0x41380000u;
    const double dlane = 0.125 * lane;
    float acc[16];
#pragma unroll
    for (int r = 0; r < 16; ++r) acc[r] = 0.0f;
    uint32_t mn_all = 0xffffffffu;
    double c = c0, q = q0;
    for (int j = 0; j < rows; j += 2) {
        uint32_t hi[2][16], lo[2][16];
#pragma unroll
        for (int z = 0; z < 2; ++z) {
            // c drifts a little from row to row like g*D does; q keeps y in [2^20 + 2^19, +600)
            c = __dadd_rn(c, -1e-9);
            const double y0 = __fma_rn(dlane, c, q);
            const double step = __dmul_rn(4.0, c);
            hi[z][0] = (uint32_t)__double2hiint(y0);
            lo[z][0] = (uint32_t)__double2loint(y0);
#pragma unroll
            for (int r = 1; r < 16; ++r) {
                const double y = __fma_rn(step, (double)r, y0);
                hi[z][r] = (uint32_t)__double2hiint(y);
                lo[z][r] = (uint32_t)__double2loint(y);
            }
            uint32_t m = min(lo[z][0], min(lo[z][1], lo[z][2]));
#pragma unroll
            for (int r = 3; r + 1 < 16; r += 2) m = min(m, min(lo[z][r], lo[z][r + 1]));
            mn_all = min(mn_all, min(m, lo[z][15]));
        }
        float v0[16], v1[16], t[16];
#pragma unroll
        for (int r = 0; r < 16; ++r) {
            asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v0[r]) : "r"(base + (hi[0][r] << 2)));
            asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v1[r]) : "r"(base + (hi[1][r] << 2)));
        }
#pragma unroll
        for (int r = 0; r < 16; r += 2) fadd2(t[r], t[r + 1], v0[r], v0[r + 1], v1[r], v1[r + 1]);
#pragma unroll
        for (int r = 0; r < 16; r += 2) fadd2(acc[r], acc[r + 1], acc[r], acc[r + 1], t[r], t[r + 1]);
    }
    float s = 0;
#pragma unroll
    for (int r = 0; r < 16; ++r) s += acc[r];
    if (s == 12345.678f || mn_all == 1u) out[0] = s;
}

// The count formats' lookup chain with one byte per bin (PACKED = false: the layout the kernels use; a
// bit-packed input is expanded by tcw_create) against one BIT per bin (PACKED = true: byte = window[k >> 3],
// value = (byte >> (k & 7)) & 1).  Same index arithmetic, 16 lookups per row; the two rates settle whether
// gathering from packed words could pay on a kernel that is bound by instruction issue.
template <bool PACKED>
__global__ void __launch_bounds__(128, 3)
peak_count_chain_kernel(int rows, double c0, double q0, int *out)
{
    __shared__ unsigned char win[4 * 1024];
    for (int i = threadIdx.x; i < 4 * 1024; i += 128) win[i] = (unsigned char)((i * 2654435761u) >> 24 & (PACKED ? 255u : 1u));
    __syncthreads();
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const uint32_t base = (uint32_t)__cvta_generic_to_shared(win) + (uint32_t)(warp * 1024);
    const double dlane = 0.125 * lane;
    int acc[16];
#pragma unroll
    for (int r = 0; r < 16; ++r) acc[r] = 0;
    uint32_t mn_all = 0xffffffffu;
    double c = c0;
    for (int j = 0; j < rows; ++j) {
        c = __dadd_rn(c, -1e-9);
        const double y0 = __fma_rn(dlane, c, q0);
        const double step = __dmul_rn(4.0, c);
        uint32_t hi[16], lo[16];
        hi[0] = (uint32_t)__double2hiint(y0);
        lo[0] = (uint32_t)__double2loint(y0);
#pragma unroll
        for (int r = 1; r < 16; ++r) {
            const double y = __fma_rn(step, (double)r, y0);
            hi[r] = (uint32_t)__double2hiint(y);
            lo[r] = (uint32_t)__double2loint(y);
        }
        uint32_t m = min(lo[0], min(lo[1], lo[2]));
#pragma unroll
        for (int r = 3; r + 1 < 16; r += 2) m = min(m, min(lo[r], lo[r + 1]));
        mn_all = min(mn_all, min(m, lo[15]));
#pragma unroll
        for (int r = 0; r < 16; ++r) {
            const uint32_t k = hi[r] - 0x41380000u;          // bin inside the window, < 640
            uint32_t v;
            if (PACKED) {
                asm volatile("ld.shared.u8 %0, [%1];" : "=r"(v) : "r"(base + (k >> 3)));
                v = (v >> (k & 7u)) & 1u;
            } else {
                asm volatile("ld.shared.u8 %0, [%1];" : "=r"(v) : "r"(base + k));
            }
            acc[r] += (int)v;
        }
    }
    int s = 0;
#pragma unroll
    for (int r = 0; r < 16; ++r) s += acc[r];
    if (s == 123456789 || mn_all == 1u) out[0] = s;
}

// Staging alone: every warp runs the staged kernel's two-slot ring over a spectrogram-like array (rows of a 20 000-bin
// float32 band, windows drifting like a track) and consumes nothing.  BOX = false: four 1-D bulk copies of `bytes`
// per slot (round 1's staging); BOX = true: one tensor-map copy of {128 B, nseg, RB rows} per slot.  The rate is the
// L2 -> shared-memory throughput the ring can draw with twelve warps per SM.
constexpr int PEAK_STAGE_ROW = 2304;     // shared-memory bytes per staged row
template <bool BOX>
__global__ void __launch_bounds__(128, 3)
peak_stage_kernel(const unsigned char *spec, long pitch, int n_rows, int slots, int bytes, const unsigned char *tmaps, int nseg, unsigned *out)
{
    extern __shared__ __align__(128) unsigned char peak_smem[];
    const int warp = (int)__reduce_or_sync(0xffffffffu, threadIdx.x >> 5), lane = threadIdx.x & 31;
    const uint32_t bar0 = smem_u32(peak_smem) + 16u * warp;
    unsigned char *ring = peak_smem + 128 + (size_t)warp * 2 * RB * PEAK_STAGE_ROW;
    const uint32_t ring0 = smem_u32(ring);
    if (lane == 0) {
        mbar_init(bar0, 1);
        mbar_init(bar0 + 8u, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncwarp();
    const long gw = (long)blockIdx.x * 4 + warp;
    const int row = (int)((gw * 37) % (n_rows - RB * slots - 8));
    const int col = 4096 + (int)((gw * 53) % 4096) * 16;      // byte offset in the row, 16-byte aligned
    unsigned acc = 0;
    uint32_t ph = 0;
    auto issue = [&](int s, int n) {
        if (elect_one()) {
            const int r0 = row + RB * n, c0 = col - 48 * n;
            const uint32_t bar = bar0 + 8u * s, dst = ring0 + (uint32_t)(s * RB * PEAK_STAGE_ROW);
            if (!BOX) {
                mbar_arrive_expect_tx(bar, (uint32_t)(RB * bytes));
#pragma unroll
                for (int q = 0; q < RB; ++q)
                    bulk_g2s(dst + q * PEAK_STAGE_ROW, spec + (long)(r0 + q) * pitch + c0 - 16 * q, (uint32_t)bytes, bar);
            } else {
                mbar_arrive_expect_tx(bar, (uint32_t)(RB * 128 * nseg));
                tensor3_g2s(dst, tmaps + 128 * nseg, c0 >> 7, r0, bar);
            }
        }
    };
    issue(0, 0);
    for (int n = 0; n < slots; ++n) {
        const int s = n & 1;
        if (n + 1 < slots) issue(s ^ 1, n + 1);
        mbar_wait(bar0 + 8u * s, ph);
        acc += *(volatile unsigned *)(ring + (size_t)s * RB * PEAK_STAGE_ROW + 4 * lane);
        __syncwarp();
        if (s == 1) ph ^= 1u;
    }
    if (acc == 0x12345678u) out[0] = acc;
}

}  // namespace tcw
