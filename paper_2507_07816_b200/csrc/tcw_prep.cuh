// tcw_prep.cuh -- strain -> Hann-windowed SFTs -> normalised power / number count (sm_100a).
//
// "The data used in this study are 8-second Han-windowed Short Fourier Transforms (SFTs), which are
// processed into either normalized power rho_j or number count nu_j".  Reading Q24
// (DESIGN.md): non-overlapping segments of N = fs*T_sft samples, w[t] = 0.5 - 0.5 cos(2 pi t/N),
// P_j[k] = |DFT(w x_j)[k]|^2, m_j[k] = running median of P_j over W = 2h + 1 bins centred on k,
// rho_j[k] = P_j[k] ln 2 / m_j[k], nu_j[k] = (rho_j[k] > threshold).
//
// The DFT itself is a plain batched real-to-complex transform and is left to cuFFT (a library
// primitive, like a GEMM left to cuBLAS).  Everything around it is here:
//   * prep_window_kernel: window multiply into the batch buffer cuFFT reads (float32);
//   * prep_normalise_kernel: up to four SFTs per CTA: |X|^2 of the band and its two half-windows into shared
//     memory, then every thread walks a run of consecutive bins keeping the running median by
//     counting (see the kernel), and writes rho (float32), nu (uint8) or nu bit-packed (uint32
//     words, LSB first) straight into the spectrogram layout tcw_create reads.  (A per-thread sliding
//     median with amortised O(1) updates -- counters plus the nearest elements on either side of the
//     median in registers, window re-scan only when a list runs dry -- was built and measured in round 2:
//     exact, but 3.9x SLOWER on B200 (616 against 160 us per 512 SFTs), because under SIMT a warp pays for
//     the union of its lanes' branches and a re-scan that is rare per lane happens in most warps on most
//     slides.  The counting form below, identical work in every lane, stays.)
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace tcw {

constexpr int PREP_THREADS = 256;
constexpr int PREP_MAX_W = 1025;      // median window limit (odd)

// w[t] = 0.5 - 0.5 cos(2 pi t / N), evaluated once per call in binary64 and stored as float32
__global__ void __launch_bounds__(256)
prep_window_table_kernel(int N, float *__restrict__ w)
{
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t < N) w[t] = (float)(0.5 - 0.5 * cospi(2.0 * (double)t / (double)N));
}

// out[b][t] = x[b*N + t] * w[t]   (out may alias x: each element is read and written by one thread)
// Scalar version: any N, any alignment.
__global__ void __launch_bounds__(256)
prep_window_kernel(const float *x, const float *__restrict__ w, int n_batch, int N, float *out)
{
    const long total = (long)n_batch * N;
    for (long q = (long)blockIdx.x * blockDim.x + threadIdx.x; q < total; q += (long)gridDim.x * blockDim.x)
        out[q] = x[q] * __ldg(w + (int)(q % N));
}
// Vector version (N a multiple of 4, 16-byte aligned buffers): a thread keeps four window values in
// registers and walks the segments blockIdx.y, blockIdx.y + gridDim.y, ...: 16-byte loads and stores,
// no index arithmetic per element.  One read and one write of the batch, at HBM rate.
__global__ void __launch_bounds__(256)
prep_window4_kernel(const float *x, const float *__restrict__ w, int n_batch, int N, float *out)
{
    const int t4 = blockIdx.x * blockDim.x + threadIdx.x;
    if (4 * t4 >= N) return;
    const float4 wv = __ldg((const float4 *)w + t4);
    for (int b = blockIdx.y; b < n_batch; b += gridDim.y) {
        float4 v = *((const float4 *)(x + (long)b * N) + t4);
        v.x *= wv.x; v.y *= wv.y; v.z *= wv.z; v.w *= wv.w;
        *((float4 *)(out + (long)b * N) + t4) = v;
    }
}

struct PrepParams {
    const float2 *spec;     // cuFFT output of this batch: [n_batch][N/2 + 1] complex
    int n_half;             // N/2 + 1
    int k_min, n_bins, h;   // band start bin, band bins, median half-window
    float threshold;
    int out_format;         // 0 float32 rho, 1 uint8 nu, 2 bit-packed nu
    unsigned char *out;     // row 0 of this batch in the output spectrogram
    long out_pitch;         // bytes
};

// One CTA normalises spc SFTs (4 when their bands fit two CTAs' worth of shared memory, else 2 or 1), 256/spc
// threads each: the selection of a thread's first window costs as much as thirteen slides, so long runs (few
// threads per SFT) pay, and several SFTs per CTA keep the SM full.  Dynamic shared memory per SFT:
// float P[n_bins + 2h] (16-byte rounded), then (count formats) unsigned char nu[n_bins rounded up to 32].
constexpr int PREP_SPC = 4;
__host__ __device__ inline size_t prep_sft_smem(int n_bins, int h)
{
    return ((((size_t)(n_bins + 2 * h) * 4 + 15) & ~(size_t)15) + (((size_t)n_bins + 31) & ~(size_t)31) + 127) & ~(size_t)127;
}

__global__ void __launch_bounds__(PREP_THREADS)
prep_normalise_kernel(const PrepParams p, int n_batch, int spc)
{
    extern __shared__ __align__(128) unsigned char smem[];
    const int tps = PREP_THREADS / spc;            // threads per SFT
    const int sub = threadIdx.x / tps, t = threadIdx.x % tps;
    const int sft = blockIdx.x * spc + sub;
    unsigned char *mine = smem + (size_t)sub * prep_sft_smem(p.n_bins, p.h);
    float *P = (float *)mine;
    const int n_in = p.n_bins + 2 * p.h;
    unsigned char *nu = mine + (((size_t)n_in * 4 + 15) & ~(size_t)15);
    const bool live = sft < n_batch;
    if (live) {
        const float2 *row = p.spec + (long)sft * p.n_half + (p.k_min - p.h);
        for (int q = t; q < n_in; q += tps) {
            const float2 c = row[q];
            P[q] = c.x * c.x + c.y * c.y;
        }
    }
    __syncthreads();

    // Running median without per-thread sorted arrays (those live in local memory and serialise):
    // the first bin of a thread's run selects the rank-h value of its window by a bitwise binary
    // search on the float bits (P >= 0, so the bits order like the values); every further bin
    // re-counts the slid window against the previous median m.  One element left and one entered,
    // so #(x < m) <= h + 1 and #(x <= m) >= h: the new median is m, or the largest element below it,
    // or the smallest element above it.  All reads are conflict-free shared-memory loads.
    const int W = 2 * p.h + 1, h = p.h;
    // an odd run length: lanes then start 'run' words apart, which visits all 32 banks (no conflicts)
    const int run = ((p.n_bins + tps - 1) / tps) | 1;
    const int k0 = min(t * run, p.n_bins), k1 = min(k0 + run, p.n_bins);
    unsigned char *orow = p.out + (long)sft * p.out_pitch;
    if (live && k0 < k1) {
        const unsigned int *Pu = (const unsigned int *)P;
        unsigned int key = 0;
        for (int bit = 30; bit >= 0; --bit) {
            const unsigned int cand = key | (1u << bit);
            int c = 0;
            for (int q = 0; q < W; ++q) c += Pu[k0 + q] < cand;
            if (c <= h) key = cand;
        }
        // Slides.  With L = #(x < mu) and LE = #(x <= mu) over the slid window, the new median is the largest element
        // below mu if L > h, the smallest above it if LE <= h, else mu.  Every slide scans the window once, branch-free
        // and identical in every lane, for three things: pred - mu (the unsigned maximum of x - mu is attained by the
        // largest x < mu, whose difference wraps to the top of the range), succ - mu - 1 (the unsigned minimum of
        // x - mu - 1: elements <= mu wrap to the top), and ONE of the two counts, C = #(x < mu + s), from the sign of
        // x - mu - s (keys are float bits of non-negative numbers, below 2^31).  The other count K is carried: it moves
        // by (entering element) - (leaving element), and when the median moves it is known exactly -- moving down to
        // pred gives LE(pred) = L, so K := L and the scans count L (s = 0); moving up to succ gives L(succ) = LE, so
        // K := LE and the scans count LE (s = 1).
        unsigned int mu = key;
        unsigned int sflag = 0u;
        int K = 0;
        for (int q = 0; q < W; ++q) K += Pu[k0 + q] <= mu;          // LE of the first window
        for (int k = k0; k < k1; ++k) {
            if (k > k0) {
                const unsigned int *wq = Pu + k;
                const unsigned int x_out = wq[-1], x_in = wq[W - 1];
                const unsigned int mk = mu + 1u - sflag;            // K = #(x < mk)
                K += (int)(x_in < mk) - (int)(x_out < mk);
                const unsigned int nmu = 0u - mu, nmu1 = nmu - 1u, nms = nmu - sflag;
                unsigned int maxd0 = 0u, maxd1 = 0u, mine0 = 0xffffffffu, mine1 = 0xffffffffu;
                unsigned int c0 = 0u, c1 = 0u;
#pragma unroll 4
                for (int q = 0; q + 1 < W; q += 2) {
                    const unsigned int x0 = wq[q], x1 = wq[q + 1];
                    maxd0 = max(maxd0, x0 + nmu);
                    maxd1 = max(maxd1, x1 + nmu);
                    mine0 = min(mine0, x0 + nmu1);
                    mine1 = min(mine1, x1 + nmu1);
                    c0 += (x0 + nms) >> 31;
                    c1 += (x1 + nms) >> 31;
                }
                {
                    const unsigned int x0 = wq[W - 1];              // W is odd
                    maxd0 = max(maxd0, x0 + nmu);
                    mine0 = min(mine0, x0 + nmu1);
                    c0 += (x0 + nms) >> 31;
                }
                const int C = (int)(c0 + c1);
                const int L = sflag ? K : C, LE = sflag ? C : K;
                if (L > h) { mu += max(maxd0, maxd1); K = L; sflag = 0u; }
                else if (LE <= h) { mu += 1u + min(mine0, mine1); K = LE; sflag = 1u; }
            }
            const float m = __uint_as_float(mu);
            const float rho = P[k + h] * 0.69314718055994531f / m;
            if (p.out_format == 0) ((float *)orow)[k] = rho;
            else nu[k] = rho > p.threshold ? 1 : 0;
        }
    }
    if (p.out_format == 0) return;
    __syncthreads();
    if (!live) return;
    if (p.out_format == 1) {
        for (int k = t; k < p.n_bins; k += tps) orow[k] = nu[k];
    } else {
        const int n_words = (p.n_bins + 31) / 32;
        for (int wd = t; wd < n_words; wd += tps) {
            uint32_t bits = 0;
            for (int b = 0; b < 32; ++b) {
                const int k = 32 * wd + b;
                if (k < p.n_bins && nu[k]) bits |= 1u << b;
            }
            ((uint32_t *)orow)[wd] = bits;
        }
    }
}

}  // namespace tcw
