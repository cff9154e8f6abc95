// tcw_skyblock2.cuh -- two-level exact sky sharing for bit-packed number counts (sm_100a).
//
// Same statistic and the same exactness argument as tcw_skyblock.cuh (IEEE multiplication by a
// positive number followed by the magic-add rounding is monotone in the Doppler factor, so the
// bins of a set of sky points lie between the bins of the set's smallest and largest factor).
// Here a CTA owns a block of S = 256 sky points made of Q = 4 sub-blocks of 64:
//   level 0  every (template, SFT) is tested against the two ends of the whole block: if they select
//            the same bin, or adjacent bins of equal value, ONE lookup serves all 256 sky points;
//   level 1  the lookups the block does not agree on (about one in seven at 1 kHz in a 10-degree
//            patch) are compacted into a per-warp list and re-tested, lanes = list entries, against
//            the ends of each sub-block; an agreeing sub-block adds its value minus the block's
//            base value to a per-(template, sub-block) sum;
//   level 2  what a sub-block does not agree on is resolved per sky point exactly as in
//            tcw_skyblock.cuh (lanes = sky points), into per-(template, sky) corrections.
// stat[s] = base + sub[q(s)] + corr[s], all integers, hence bit-identical to the per-sky evaluation.
// The corrections are int16 pairs packed in 32-bit words (there is no 16-bit shared-memory atomic):
// adding dv * 65536^(s & 1) to the word and decoding low = sext16(word), high = (word - low) >> 16 is
// exact while |corr| < 2^15, which holds for 0/1 data with at most 32767 SFTs: the host takes this
// kernel for bit-packed input only.
#pragma once
#include "tcw_skyblock.cuh"

namespace tcw {

constexpr int S2 = 256, Q2 = 4, R2 = 8, F2 = 32 * R2;   // sky points per block, sub-blocks, templates per lane / tile
constexpr int NW2 = 16, SKY2_THREADS = 32 * NW2, D2 = 2; // warps per CTA, ring depth per warp (shared memory: 129 KB of
                                                         // corrections leave room for 16 two-deep rings of 2.4 KB rows)
constexpr int CW2 = S2 / 2 + 1;                          // corr row stride in 32-bit words (odd)
constexpr int DTS2_BYTES = 8 * S2 + 64;                  // staged per row: 256 Doppler factors + 4 {min, max} pairs

// One warp per (block, SFT): the block's 256 Doppler factors in slot order followed by the
// {min, max} of each 64-point sub-block; dmm gets the {min, max} of the whole block.
template <bool TPOW2>
__global__ void __launch_bounds__(256)
skyblock2_table_kernel(const double *__restrict__ vel, int n_sft, const double *__restrict__ sky,
                       const int *__restrict__ slot_sky, int n_blocks, double T,
                       double *__restrict__ dts, double *__restrict__ dmm)
{
    const long wq = ((long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (wq >= (long)n_blocks * n_sft) return;
    const int j = (int)(wq % n_sft);
    const int b = (int)(wq / n_sft);
    const double *v = vel + 3 * (long)j;
    double *row = dts + wq * (DTS2_BYTES / 8);
    double blo = 0, bhi = 0;
#pragma unroll
    for (int q = 0; q < Q2; ++q) {
        double lo = 0, hi = 0;
#pragma unroll
        for (int c = 0; c < 2; ++c) {
            const int sl = q * 64 + c * 32 + lane;
            double d = doppler_factor(v, sky + 3 * (long)slot_sky[b * S2 + sl]);
            if (TPOW2) d = __dmul_rn(d, T);
            row[sl] = d;
            lo = c ? fmin(lo, d) : d;
            hi = c ? fmax(hi, d) : d;
        }
#pragma unroll
        for (int o = 16; o; o >>= 1) {
            lo = fmin(lo, __shfl_xor_sync(0xffffffffu, lo, o));
            hi = fmax(hi, __shfl_xor_sync(0xffffffffu, hi, o));
        }
        if (lane == 0) { row[S2 + 2 * q] = lo; row[S2 + 2 * q + 1] = hi; }
        blo = q ? fmin(blo, lo) : lo;
        bhi = q ? fmax(bhi, hi) : hi;
    }
    if (lane == 0) { dmm[2 * wq] = blo; dmm[2 * wq + 1] = bhi; }
}

// dynamic shared memory layout (bytes)
__host__ __device__ inline size_t sky2_off_items() { return ((size_t)NW2 * D2 * (8 + sizeof(SkyRowMeta)) + 127) & ~(size_t)127; }
__host__ __device__ inline size_t sky2_off_list() { return sky2_off_items() + (size_t)NW2 * 32 * 16; }
__host__ __device__ inline size_t sky2_off_f0() { return sky2_off_list() + (size_t)NW2 * F2; }
__host__ __device__ inline size_t sky2_off_sub() { return sky2_off_f0() + (size_t)F2 * 8; }
__host__ __device__ inline size_t sky2_off_corr() { return sky2_off_sub() + (size_t)F2 * Q2 * 4; }
__host__ __device__ inline size_t sky2_off_slots() { return (sky2_off_corr() + (size_t)F2 * CW2 * 4 + 127) & ~(size_t)127; }
__host__ __device__ inline size_t sky2_smem_bytes(int slot_bytes)
{
    size_t ring = (size_t)NW2 * D2 * (size_t)slot_bytes;
    size_t red = (size_t)NW2 * F2 * 4 + 128;
    return sky2_off_slots() + (ring > red ? ring : red);
}


template <bool TPOW2>
__global__ void __launch_bounds__(SKY2_THREADS, 1)
sum_skyblock2_kernel(const SumParams p, const SkyParams q)
{
    constexpr uint32_t FULL = 0xffffffffu;
    extern __shared__ __align__(128) unsigned char smem[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    uint64_t *bars = (uint64_t *)smem + warp * D2;
    SkyRowMeta *metas = (SkyRowMeta *)(smem + (size_t)NW2 * D2 * 8) + warp * D2;
    const uint32_t items_s = smem_u32(smem + sky2_off_items()) + (uint32_t)(warp * 32 * 16);
    unsigned char *list = smem + sky2_off_list() + warp * F2;     // level-1 entries: template index within the tile
    double *f0t = (double *)(smem + sky2_off_f0());               // f0t[r*32 + lane]
    int *sub = (int *)(smem + sky2_off_sub());                    // [F2][Q2]
    int *corr = (int *)(smem + sky2_off_corr());                  // [F2][CW2], two int16 per word
    unsigned char *slots = smem + sky2_off_slots();
    const uint32_t slots_s = smem_u32(slots) + (uint32_t)(warp * D2 * p.slot_bytes);
    const uint32_t bars_s = smem_u32(bars);
    const uint32_t corr_s = smem_u32(corr), sub_s = smem_u32(sub);
    const uint32_t f0_s = smem_u32(f0t);

    int blk, ab, tile_raw, part;
    block_map(p, blockIdx.x, q.n_blocks, blk, ab, tile_raw, part);
    const int tile = p.n_tiles - 1 - tile_raw;                        // heavy tiles (high f0) first
    const int i0 = tile * F2;
    const int i_last = min(i0 + F2, p.n_f0) - 1;

    if (lane == 0) {
        for (int s = 0; s < D2; ++s) mbar_init(bars_s + 8u * s, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    for (int t = threadIdx.x; t < F2 * CW2; t += SKY2_THREADS) corr[t] = 0;
    for (int t = threadIdx.x; t < F2 * Q2; t += SKY2_THREADS) sub[t] = 0;
    for (int t = threadIdx.x; t < F2; t += SKY2_THREADS) f0t[t] = p.f0[min(i0 + t, i_last)];
    __syncthreads();

    int acc[R2];
#pragma unroll
    for (int r = 0; r < R2; ++r) acc[r] = 0;
    const double f_first = p.f0[i0], f_last = p.f0[i_last];
    const double below = (double)p.k_min - 1.0;
    const double *g = p.gtab + (long)ab * p.n_sft;
    const double *mm = q.dmm + 2 * (long)blk * p.n_sft;
    const double *dts = q.dts + (long)blk * p.n_sft * (DTS2_BYTES / 8);
    const int jw = p.j_begin + warp;
    const int n_rows = jw < p.n_sft ? (p.n_sft - jw + NW2 - 1) / NW2 : 0;
    const unsigned char *spec_w = p.spec + (long)jw * p.pitch;
    const long pitch_w = (long)NW2 * p.pitch;

    // row metadata, 32 rows at a time (lane = row), as in sum_skyblock_kernel
    double b_g = 0, b_d0 = 0, b_d1 = 0;
    int b_abyte = 0, b_bytes = 0, b_live = -1;
    double gn = 0, d0n = 1, d1n = 1;
    if (lane < n_rows) {
        const int j = jw + NW2 * lane;
        gn = __ldg(g + j); d0n = __ldg(mm + 2 * j); d1n = __ldg(mm + 2 * j + 1);
    }
    auto compute_batch = [&](int m) {
        const int n = 32 * m + lane;
        b_g = gn; b_d0 = d0n; b_d1 = d1n;
        if (n + 32 < n_rows) {
            const int j = jw + NW2 * (n + 32);
            gn = __ldg(g + j); d0n = __ldg(mm + 2 * j); d1n = __ldg(mm + 2 * j + 1);
        }
        b_live = -1;
        b_bytes = 0;
        if (n < n_rows && !(f_last * b_g * p.dmaxT < below)) {
            const int kf = lo_of<TPOW2>(__dmul_rn(f_first, b_g), b_d0, p.T) - p.k_min;
            const int kl = lo_of<TPOW2>(__dmul_rn(f_last, b_g), b_d1, p.T) - p.k_min;
            b_live = 0;
            if (kl >= 0 && kf < p.n_bins) {
                const int a_byte = kf & ~15;
                const int e_byte = (kl + 1 + 15) & ~15;
                if (e_byte - a_byte + DTS2_BYTES > p.slot_limit || kf < -PAD_BINS || kl >= p.n_bins + PAD_BINS) {
                    atomicOr(p.status, 1);
                } else {
                    b_bytes = e_byte - a_byte;
                    b_abyte = a_byte;
                    b_live = 1;
                }
            }
        }
    };
    int ni = 0, si = 0;
    auto stage_next = [&]() {
        if ((ni & 31) == 0) compute_batch(ni >> 5);
        if (lane == (ni & 31)) {
            const uint32_t slot_s = slots_s + (uint32_t)(si * p.slot_bytes);
            SkyRowMeta m;
            m.g = b_g; m.d0 = b_d0; m.d1 = b_d1; m.live = b_live; m.pad[0] = m.pad[1] = 0;
            m.rb = slot_s + (uint32_t)DTS2_BYTES - (uint32_t)(p.k_min + b_abyte);
            metas[si] = m;
            if (b_live > 0) {
                mbar_arrive_expect_tx(bars_s + 8u * si, (uint32_t)(b_bytes + DTS2_BYTES));
                bulk_g2s(slot_s, dts + (long)(jw + NW2 * ni) * (DTS2_BYTES / 8), (uint32_t)DTS2_BYTES, bars_s + 8u * si);
                bulk_g2s(slot_s + (uint32_t)DTS2_BYTES, spec_w + (long)ni * pitch_w + b_abyte, (uint32_t)b_bytes, bars_s + 8u * si);
            } else if (b_live == 0) {
                mbar_arrive(bars_s + 8u * si);
            }
        }
        __syncwarp();
        ++ni;
        if (++si == D2) si = 0;
    };
    for (int s = 0; s < D2 - 1; ++s) stage_next();

    uint32_t ph = 0;
    int sc = 0;
    const uint32_t lt_mask = (1u << lane) - 1u;
    for (;;) {
        stage_next();
        const SkyRowMeta m = metas[sc];
        if (m.live <= 0) {
            if (m.live < 0) break;
        } else {
            mbar_wait(bars_s + 8u * sc, ph);
            const uint32_t dt_s = slots_s + (uint32_t)(sc * p.slot_bytes);   // the row's 256 Doppler factors, then 4 {min, max}
            // ---- level 0 (lanes = templates): the two ends of the whole block
            int n1 = 0;
#pragma unroll
            for (int r = 0; r < R2; ++r) {
                const double a = __dmul_rn(lds_f64(f0_s + 8u * (uint32_t)(r * 32 + lane)), m.g);
                const int lo0 = lo_of<TPOW2>(a, m.d0, p.T);
                const int lo1 = lo_of<TPOW2>(a, m.d1, p.T);
                const int v0 = (int)lds_u8(m.rb + (uint32_t)lo0);
                const int v1 = (int)lds_u8(m.rb + (uint32_t)lo1);
                acc[r] += v0;
                const bool fail = (v1 != v0) | ((uint32_t)(lo1 - lo0) > 1u);
                const unsigned mask = __ballot_sync(FULL, fail);
                if (fail) list[n1 + __popc(mask & lt_mask)] = (unsigned char)(r * 32 + lane);
                n1 += __popc(mask);
            }
            __syncwarp();
            // ---- level 1 (lanes = list entries): the two ends of each 64-point sub-block
            for (int e0 = 0; e0 < n1; e0 += 32) {
                const bool has = e0 + lane < n1;
                const int t = has ? (int)list[e0 + lane] : 0;
                const double a = __dmul_rn(lds_f64(f0_s + 8u * (uint32_t)t), m.g);
                const int vb = (int)lds_u8(m.rb + (uint32_t)lo_of<TPOW2>(a, m.d0, p.T));   // the block's base value
#pragma unroll 1
                for (int qq = 0; qq < Q2; ++qq) {
                    const double dq0 = lds_f64(dt_s + (uint32_t)(8 * S2 + 16 * qq));
                    const double dq1 = lds_f64(dt_s + (uint32_t)(8 * S2 + 16 * qq + 8));
                    const int l0 = lo_of<TPOW2>(a, dq0, p.T);
                    const int l1 = lo_of<TPOW2>(a, dq1, p.T);
                    const int w0 = (int)lds_u8(m.rb + (uint32_t)l0);
                    const int w1 = (int)lds_u8(m.rb + (uint32_t)l1);
                    // every sky point of the sub-block gets at least w0 - vb; the rest is per sky point
                    if (has && w0 != vb) red_shared_add(sub_s + 4u * (uint32_t)(t * Q2 + qq), w0 - vb);
                    const bool open = has & ((w1 != w0) | ((uint32_t)(l1 - l0) > 1u));
                    const unsigned own = __ballot_sync(FULL, open);
                    if (own == 0) continue;
                    const bool far = open & (l1 - l0 != 1);        // ends several bins apart: rare
                    const unsigned any_far = __ballot_sync(FULL, far);
                    if (open) {
                        const int pk = far ? ITEM_GENERIC + w0 : 2 * (w1 - w0) + (l0 & 1);
                        sts_item(items_s + 16u * __popc(own & lt_mask), a, pk, corr_s + 4u * (uint32_t)(t * CW2));
                    }
                    __syncwarp();
                    // ---- level 2 (lanes = pairs of sky points of the sub-block: slots 2*lane and 2*lane + 1
                    // of it, whose int16 corrections share one word: one 16-byte load of the two Doppler
                    // factors and one shared-memory add per lane and item)
                    const int n_items = __popc(own);
                    const uint32_t d2_s = dt_s + 16u * (uint32_t)(qq * 32 + lane);
                    const uint32_t w_off = 4u * (uint32_t)(qq * 32 + lane);
                    double da, db;
                    asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(da), "=d"(db) : "r"(d2_s));
                    if (any_far == 0) {
                        // the usual case: every listed lookup has two candidate bins, the high one iff the
                        // parity of the sky point's bin differs from the low bin's
#pragma unroll 2
                        for (int i = 0; i < n_items; ++i) {
                            double ai;
                            int pk;
                            uint32_t c_s;
                            lds_item(items_s + 16u * i, ai, pk, c_s);
                            const int loa = lo_of<TPOW2>(ai, da, p.T);
                            const int lob = lo_of<TPOW2>(ai, db, p.T);
                            const int dv = pk >> 1;
                            red_shared_add(c_s + w_off, ((loa ^ pk) & 1) * dv + ((lob ^ pk) & 1) * (dv * 65536));
                        }
                    } else {
                        for (int i = 0; i < n_items; ++i) {
                            double ai;
                            int pk;
                            uint32_t c_s;
                            lds_item(items_s + 16u * i, ai, pk, c_s);
                            const int loa = lo_of<TPOW2>(ai, da, p.T);
                            const int lob = lo_of<TPOW2>(ai, db, p.T);
                            int dva, dvb;
                            if (pk < ITEM_GENERIC) {
                                const int dv = pk >> 1;
                                dva = ((loa ^ pk) & 1) * dv;
                                dvb = ((lob ^ pk) & 1) * dv;
                            } else {                      // every sky point looks its bin up
                                const int w0i = pk - ITEM_GENERIC;
                                dva = (int)lds_u8(m.rb + (uint32_t)loa) - w0i;
                                dvb = (int)lds_u8(m.rb + (uint32_t)lob) - w0i;
                            }
                            red_shared_add(c_s + w_off, dva + dvb * 65536);
                        }
                    }
                    __syncwarp();     // the item list is rewritten by the next sub-block
                }
            }
        }
        __syncwarp();     // every lane has read slot sc (and the entry list) before they are reused
        if (++sc == D2) { sc = 0; ph ^= 1u; }
    }

    // ---------------- combine: base[t] = sum over warps (integers: any order is exact)
    __syncthreads();      // every staged copy has been consumed and every correction has landed
    int *red = (int *)slots;
#pragma unroll
    for (int r = 0; r < R2; ++r) red[warp * F2 + r * 32 + lane] = acc[r];
    __syncthreads();
    for (int t = threadIdx.x; t < F2; t += SKY2_THREADS) {
        int s = red[t];
        for (int w = 1; w < NW2; ++w) s += red[w * F2 + t];
        red[t] = s;
    }
    __syncthreads();
    // ---------------- stat[s][t] = base[t] + sub[t][q(s)] + corr[t][s]; warp w serves the slots w, w + NW2, ...
    for (int sl = warp; sl < S2; sl += NW2) {
        const int slot = blk * S2 + sl;
        if (slot >= q.n_sky) break;           // padding slots repeat the last sky point; no output
        const long grp = (long)q.slot_sky[slot] * p.n_ab + ab;
        int best_v = INT32_MIN, best_i = INT32_MAX;
#pragma unroll
        for (int r = 0; r < R2; ++r) {
            const int t = r * 32 + lane;
            const int i = i0 + t;
            if (i < p.n_f0) {
                const int word = corr[t * CW2 + (sl >> 1)];
                const int low = (int)(short)(word & 0xffff);
                const int c = (sl & 1) ? (word - low) >> 16 : low;
                const int s = red[t] + sub[t * Q2 + (sl >> 6)] + c;
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
