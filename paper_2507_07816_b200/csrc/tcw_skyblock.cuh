// tcw_skyblock.cuh -- exact sky-shared gather-accumulate for number counts (sm_100a).
//
// The statistic of template (f0, tau, n, n-hat_s) is "summed across the data bins selected by the
// track" with the bin k = rint((f0*g)*(D_s*T)) - k_min of eqs. (1)-(2)
// (PAPER.md:25, 32).  Only the Doppler factor D_s depends on the sky point, and it moves the track
// by a fraction of a bin across neighbouring sky points, so most sky points of a patch select the
// SAME bin for a given (f0, tau, n, SFT).  This kernel uses that without approximating anything:
//
//   * IEEE multiplication by a positive number, the magic-add rounding and hence rint(a*d) are
//     monotone non-decreasing in d.  For a block B of sky points and one SFT j, with
//     d_min = min_{s in B} D_s(j)*T and d_max = max_{s in B} D_s(j)*T (taken over the very doubles
//     the per-sky path multiplies by), every s in B has lo(a*d_min) <= lo(a*D_s*T) <= lo(a*d_max).
//   * If the two ends agree, all sky points of the block select that bin: one lookup serves the
//     whole block (it is added to a per-template base sum).  If they are adjacent bins holding the
//     same value, likewise.  Otherwise the lookup is resolved per sky point (lanes = sky points)
//     and the difference to the base value goes to a per-(template, sky) correction in shared
//     memory.  stat[s] = base + corr[s] in exact integer arithmetic, so the result is bit-identical
//     to the per-sky evaluation whatever the order of the additions.
//
// The host sorts the sky points by their Doppler shift at the middle SFT and cuts the sorted list
// into blocks of S = 32*SC points, which keeps d_max - d_min (and so the fraction of lookups that
// must be resolved) small for any sky grid, ordered or not.  Integer accumulation only: the
// float32 power format keeps the per-sky staged kernel (a fixed summation order is part of its
// contract).
//
// One CTA owns (sky block, (tau, n), tile of 32*R consecutive f0).  As in sum_staged_kernel every
// warp owns the SFT rows j = j_begin + warp + NWS*n and runs a private TMA ring; a ring slot holds
// the block's S Doppler factors of the row followed by the spectrogram window of the row.
#pragma once
#include "tcw_sum.cuh"
#include "tcw_tables.cuh"

namespace tcw {

constexpr int NWS = 16;                 // warps per CTA
constexpr int SKY_THREADS = 32 * NWS;

struct SkyParams {
    const double *dts;     // [n_blocks][n_sft][S]  D_s(j) (times T_sft when it is a power of two), block order
    const double *dmm;     // [n_blocks][n_sft][2]  {min, max} of the row above
    const int *slot_sky;   // [n_blocks*S] sky index of each slot; slots >= n_sky repeat the last sky point
    int n_sky, n_blocks;
};

// ---------------------------------------------------------------------------- block tables
// One warp per (block, SFT): lanes run over the block's sky points.
template <int SC, bool TPOW2>
__global__ void __launch_bounds__(256)
skyblock_table_kernel(const double *__restrict__ vel, int n_sft, const double *__restrict__ sky,
                      const int *__restrict__ slot_sky, int n_blocks, double T,
                      double *__restrict__ dts, double *__restrict__ dmm)
{
    constexpr int S = 32 * SC;
    const long wq = ((long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (wq >= (long)n_blocks * n_sft) return;
    const int j = (int)(wq % n_sft);
    const int b = (int)(wq / n_sft);
    const double *v = vel + 3 * (long)j;
    double lo = 0, hi = 0;
#pragma unroll
    for (int c = 0; c < SC; ++c) {
        const int s = slot_sky[b * S + c * 32 + lane];
        double d = doppler_factor(v, sky + 3 * (long)s);
        if (TPOW2) d = __dmul_rn(d, T);
        dts[wq * S + c * 32 + lane] = d;
        lo = c ? fmin(lo, d) : d;
        hi = c ? fmax(hi, d) : d;
    }
#pragma unroll
    for (int o = 16; o; o >>= 1) {
        lo = fmin(lo, __shfl_xor_sync(0xffffffffu, lo, o));
        hi = fmax(hi, __shfl_xor_sync(0xffffffffu, hi, o));
    }
    if (lane == 0) {
        dmm[2 * wq] = lo;
        dmm[2 * wq + 1] = hi;
    }
}

// ---------------------------------------------------------------------------- sum kernel
__device__ __forceinline__ double lds_f64(uint32_t a)
{
    double v;
    asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(a));
    return v;
}
__device__ __forceinline__ void red_shared_add(uint32_t a, int v)
{
    asm volatile("red.shared.add.s32 [%0], %1;" ::"r"(a), "r"(v) : "memory");
}

constexpr int ITEM_GENERIC = 0x10000;   // item.pk >= this: generic resolve, pk - ITEM_GENERIC is the base value
// one unresolved lookup: a = f0*g, pk, shared address of the template's correction row
__device__ __forceinline__ void sts_item(uint32_t addr, double a, int pk, uint32_t c_s)
{
    asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "r"(__double2loint(a)), "r"(__double2hiint(a)),
                 "r"(pk), "r"(c_s) : "memory");
}
__device__ __forceinline__ void lds_item(uint32_t addr, double &a, int &pk, uint32_t &c_s)
{
    int lo, hi;
    asm volatile("ld.shared.v4.b32 {%0, %1, %2, %3}, [%4];" : "=r"(lo), "=r"(hi), "=r"(pk), "=r"(c_s) : "r"(addr));
    a = __hiloint2double(hi, lo);
}

struct __align__(16) SkyRowMeta {
    double g, d0, d1;   // spin-down factor; min and max Doppler factor of the block in this row
    uint32_t rb;        // shared address of bin (0 - k_min) of the staged window: addr = rb + rint(x)
    int live;           // 1 staged row, 0 row with no in-band bin, -1 no further rows
    int pad[2];
};

// dynamic shared memory: [mbarrier NWS*D][SkyRowMeta NWS*D][item lists NWS*32*16 B][f0 tile F double]
//                        [corr F*(S+1) int][slots NWS*D*slot_bytes]
__host__ __device__ inline size_t sky_header_bytes(int stages) { return (size_t)NWS * stages * (8 + sizeof(SkyRowMeta)); }
__host__ __device__ inline size_t sky_corr_bytes(int tile, int S) { return (((size_t)tile * (S + 1) * 4) + 127) & ~(size_t)127; }
__host__ __device__ inline size_t sky_items_off(int stages) { return (sky_header_bytes(stages) + 127) & ~(size_t)127; }
__host__ __device__ inline size_t sky_f0_off(int stages) { return sky_items_off(stages) + (size_t)NWS * 32 * 16; }
__host__ __device__ inline size_t sky_smem_bytes(int stages, int slot_bytes, int tile, int S)
{
    size_t ring = (size_t)NWS * stages * (size_t)slot_bytes;
    size_t red = (size_t)NWS * tile * 4 + 128;
    return sky_f0_off(stages) + (size_t)tile * 8 + sky_corr_bytes(tile, S) + (ring > red ? ring : red);
}

template <bool TPOW2>
__device__ __forceinline__ int lo_of(double a, double d, double T)
{
    double x = __dmul_rn(a, d);
    if (!TPOW2) x = __dmul_rn(x, T);
    return __double2loint(__dadd_rn(x, TCW_MAGIC));
}

template <int R, int SC, bool TPOW2>
__global__ void __launch_bounds__(SKY_THREADS, 1)
sum_skyblock_kernel(const SumParams p, const SkyParams q)
{
    constexpr int F = 32 * R;       // templates per tile
    constexpr int S = 32 * SC;      // sky points per block
    constexpr int CS = S + 1;       // corr row stride in words: odd, so both access patterns are conflict-free
    constexpr uint32_t FULL = 0xffffffffu;
    extern __shared__ __align__(128) unsigned char smem[];
    const int D = p.stages;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    uint64_t *bars = (uint64_t *)smem + warp * D;
    SkyRowMeta *metas = (SkyRowMeta *)(smem + (size_t)NWS * D * 8) + warp * D;
    double *f0t = (double *)(smem + sky_f0_off(D));          // the tile's f0, lane-interleaved: f0t[r*32 + lane]
    int *corr = (int *)(f0t + F);
    unsigned char *slots = (unsigned char *)corr + sky_corr_bytes(F, S);
    const uint32_t slots_s = smem_u32(slots) + (uint32_t)(warp * D * p.slot_bytes);
    const uint32_t bars_s = smem_u32(bars);
    const uint32_t corr_s = smem_u32(corr);
    const uint32_t f0_s = smem_u32(f0t) + 8u * lane;
    const uint32_t items_s = smem_u32(smem + sky_items_off(D)) + (uint32_t)(warp * 32 * 16);

    // heavy tiles (high f0 stays in band longest) are launched first
    int blk, ab, tile_raw, part;
    block_map(p, blockIdx.x, q.n_blocks, blk, ab, tile_raw, part);
    const int tile = p.n_tiles - 1 - tile_raw;
    const int i0 = tile * F;
    const int i_last = min(i0 + F, p.n_f0) - 1;

    if (lane == 0) {
        for (int s = 0; s < D; ++s) mbar_init(bars_s + 8u * s, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    for (int t = threadIdx.x; t < F * CS; t += SKY_THREADS) corr[t] = 0;
    for (int t = threadIdx.x; t < F; t += SKY_THREADS) f0t[t] = p.f0[min(i0 + t, i_last)];
    __syncthreads();

    int acc[R];
#pragma unroll
    for (int r = 0; r < R; ++r) acc[r] = 0;
    const double f_first = p.f0[i0], f_last = p.f0[i_last];
    const double below = (double)p.k_min - 1.0;
    const double *g = p.gtab + (long)ab * p.n_sft;
    const double *mm = q.dmm + 2 * (long)blk * p.n_sft;
    const double *dts = q.dts + (long)blk * p.n_sft * S;
    const int jw = p.j_begin + warp;
    const int n_rows = jw < p.n_sft ? (p.n_sft - jw + NWS - 1) / NWS : 0;
    const unsigned char *spec_w = p.spec + (long)jw * p.pitch;
    const long pitch_w = (long)NWS * p.pitch;

    // Row metadata is computed 32 rows at a time, one row per lane (rows 32*m + lane of this warp).
    double b_g = 0, b_d0 = 0, b_d1 = 0;
    int b_abyte = 0, b_bytes = 0, b_live = -1;   // first staged byte of the row's window, bytes staged
    double gn = 0, d0n = 1, d1n = 1;
    if (lane < n_rows) {
        const int j = jw + NWS * lane;
        gn = __ldg(g + j); d0n = __ldg(mm + 2 * j); d1n = __ldg(mm + 2 * j + 1);
    }

    auto compute_batch = [&](int m) {
        const int n = 32 * m + lane;
        b_g = gn; b_d0 = d0n; b_d1 = d1n;
        if (n + 32 < n_rows) {
            const int j = jw + NWS * (n + 32);
            gn = __ldg(g + j); d0n = __ldg(mm + 2 * j); d1n = __ldg(mm + 2 * j + 1);
        }
        b_live = -1;
        b_bytes = 0;
        // g decreases with j: once the tile's highest template is below the band for the largest
        // possible Doppler factor, no later SFT can contribute.
        if (n < n_rows && !(f_last * b_g * p.dmaxT < below)) {
            const int kf = lo_of<TPOW2>(__dmul_rn(f_first, b_g), b_d0, p.T) - p.k_min;
            const int kl = lo_of<TPOW2>(__dmul_rn(f_last, b_g), b_d1, p.T) - p.k_min;
            b_live = 0;
            if (kl >= 0 && kf < p.n_bins) {
                const int a_byte = kf & ~15;                      // rounds towards -inf: may reach into the left padding
                const int e_byte = (kl + 1 + 15) & ~15;
                if (e_byte - a_byte + 8 * S > p.slot_limit || kf < -PAD_BINS || kl >= p.n_bins + PAD_BINS) {
                    atomicOr(p.status, 1);  // host-side window bound violated: never expected
                } else {
                    b_bytes = e_byte - a_byte;
                    b_abyte = a_byte;
                    b_live = 1;
                }
            }
        }
    };

    int ni = 0, si = 0;   // next row to stage and its ring slot
    auto stage_next = [&]() {
        if ((ni & 31) == 0) compute_batch(ni >> 5);
        if (lane == (ni & 31)) {
            const uint32_t slot_s = slots_s + (uint32_t)(si * p.slot_bytes);
            SkyRowMeta m;
            m.g = b_g; m.d0 = b_d0; m.d1 = b_d1; m.live = b_live; m.pad[0] = m.pad[1] = 0;
            m.rb = slot_s + (uint32_t)(8 * S) - (uint32_t)(p.k_min + b_abyte);
            metas[si] = m;
            if (b_live > 0) {
                mbar_arrive_expect_tx(bars_s + 8u * si, (uint32_t)(b_bytes + 8 * S));
                bulk_g2s(slot_s, dts + (long)(jw + NWS * ni) * S, (uint32_t)(8 * S), bars_s + 8u * si);
                bulk_g2s(slot_s + 8u * S, spec_w + (long)ni * pitch_w + b_abyte, (uint32_t)b_bytes, bars_s + 8u * si);
            } else if (b_live == 0) {
                mbar_arrive(bars_s + 8u * si);
            }
        }
        __syncwarp();
        ++ni;
        if (++si == D) si = 0;
    };

    for (int s = 0; s < D - 1; ++s) stage_next();

    uint32_t ph = 0;
    int sc = 0;
    for (;;) {
        stage_next();
        const SkyRowMeta m = metas[sc];
        if (m.live <= 0) {
            if (m.live < 0) break;
        } else {
            mbar_wait(bars_s + 8u * sc, ph);
            const uint32_t dt_s = slots_s + (uint32_t)(sc * p.slot_bytes) + 8u * lane;
            // Phase A (lanes = templates): every template against the two ends of the block.  The R
            // chains are independent and issue back to back; a lane notes which of its templates
            // the block does not agree on.
            uint32_t bits = 0;
#pragma unroll
            for (int r = 0; r < R; ++r) {
                const double a = __dmul_rn(lds_f64(f0_s + 256u * r), m.g);
                const int lo0 = lo_of<TPOW2>(a, m.d0, p.T);
                const int lo1 = lo_of<TPOW2>(a, m.d1, p.T);
                const int v0 = (int)lds_u8(m.rb + (uint32_t)lo0);
                const int v1 = (int)lds_u8(m.rb + (uint32_t)lo1);
                acc[r] += v0;
                // unanimous if both ends agree (then v1 is v0 read twice) or are adjacent bins of equal value
                if ((v1 != v0) | ((uint32_t)(lo1 - lo0) > 1u)) bits |= 1u << r;
            }
            // Phase B: the few lookups the block does not agree on.  Owners publish one lookup each
            // (a, what to add, where) in the warp's item list; then lanes = sky points resolve the
            // listed lookups one after the other.  Usually one round of a handful of items.
            for (;;) {
                const unsigned own = __ballot_sync(FULL, bits != 0);
                if (own == 0) break;
                if (bits) {
                    const int r = __ffs(bits) - 1;
                    bits &= bits - 1;
                    const double a = __dmul_rn(lds_f64(f0_s + 256u * r), m.g);
                    const int lo0 = lo_of<TPOW2>(a, m.d0, p.T);
                    const int lo1 = lo_of<TPOW2>(a, m.d1, p.T);
                    const int v0 = (int)lds_u8(m.rb + (uint32_t)lo0);
                    // two candidate bins: (value difference, parity of the low bin); else: the base value
                    const int pk = lo1 - lo0 == 1 ? 2 * ((int)lds_u8(m.rb + (uint32_t)lo1) - v0) + (lo0 & 1) : ITEM_GENERIC + v0;
                    sts_item(items_s + 16u * __popc(own & ((1u << lane) - 1u)), a, pk,
                             corr_s + 4u * (uint32_t)((r * 32 + lane) * CS));
                }
                __syncwarp();
                const int n_items = __popc(own);
#pragma unroll 2
                for (int i = 0; i < n_items; ++i) {
                    double a;
                    int pk;
                    uint32_t c_s;
                    lds_item(items_s + 16u * i, a, pk, c_s);
                    c_s += 4u * lane;
                    if (pk < ITEM_GENERIC) {
                        // a sky point reads the high bin iff its bin's parity differs from the low bin's
                        const int dv = pk >> 1;
#pragma unroll
                        for (int c = 0; c < SC; ++c) {
                            const int lo = lo_of<TPOW2>(a, lds_f64(dt_s + 256u * c), p.T);
                            red_shared_add(c_s + 128u * c, ((lo ^ pk) & 1) * dv);
                        }
                    } else {
                        // ends several bins apart (wide sky blocks, high bands): every sky point looks its bin up
                        const int v0 = pk - ITEM_GENERIC;
#pragma unroll
                        for (int c = 0; c < SC; ++c) {
                            const uint32_t lo = (uint32_t)lo_of<TPOW2>(a, lds_f64(dt_s + 256u * c), p.T);
                            red_shared_add(c_s + 128u * c, (int)lds_u8(m.rb + lo) - v0);
                        }
                    }
                }
                __syncwarp();     // the list is rewritten by the next round
            }
        }
        __syncwarp();     // every lane has read slot sc before the next iteration refills it
        if (++sc == D) { sc = 0; ph ^= 1u; }
    }

    // ---------------- combine: base[t] = sum over warps (integers: any order is exact)
    __syncthreads();      // every staged copy has been consumed and every correction has landed
    int *red = (int *)slots;
#pragma unroll
    for (int r = 0; r < R; ++r) red[warp * F + r * 32 + lane] = acc[r];
    __syncthreads();
    for (int t = threadIdx.x; t < F; t += SKY_THREADS) {
        int s = red[t];
        for (int w = 1; w < NWS; ++w) s += red[w * F + t];
        red[t] = s;
    }
    __syncthreads();
    // ---------------- stat[s][t] = base[t] + corr[t][s]; warp w serves the block's slots w, w + NWS, ...
    for (int sl = warp; sl < S; sl += NWS) {
        const int slot = blk * S + sl;
        if (slot >= q.n_sky) break;           // padding slots repeat the last sky point; no output
        const long grp = (long)q.slot_sky[slot] * p.n_ab + ab;
        int best_v = INT32_MIN, best_i = INT32_MAX;
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const int t = r * 32 + lane;
            const int i = i0 + t;
            if (i < p.n_f0) {
                const int s = red[t] + corr[t * CS + sl];
                if (p.out_stat) ((int *)p.out_stat)[grp * p.n_f0 + i] = s;
                argmax_step(best_v, best_i, s, i);
            }
        }
#pragma unroll
        for (int o = 16; o; o >>= 1) {
            const int ov = __shfl_xor_sync(FULL, best_v, o);
            const int oi = __shfl_xor_sync(FULL, best_i, o);
            argmax_step(best_v, best_i, ov, oi);
        }
        if (lane == 0) ((Best<int> *)p.partial)[grp * p.n_tiles + tile] = {best_v, best_i == INT32_MAX ? 0 : best_i};
    }
    block_done(p, part);
}

}  // namespace tcw
