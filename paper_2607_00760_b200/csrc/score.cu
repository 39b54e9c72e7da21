// score.cu — step 2a of the hot path: block scores on the packed block keys (PAPER.md:182,
// 214-216): s_b = reduce_h sum_{c kept} q_h[c] * kbar_b[c], directly on the packed keys.  sm_100a.
//
// Design: a streaming kernel over the block-key arena.
//   * Work item = 8 block keys of one segment (one item per segment at L = 64).  Items are taken in
//     pairs (16 keys = the M of one mma.sync tile); the pairs of all units form one stream that is
//     cut into equal contiguous ranges, one per warp of a one-CTA-per-SM grid.  Warps are
//     independent (no __syncthreads in the main loop).
//   * Each pair's payload (position bitmaps + kept bf16 values, DESIGN.md format) is copied into a
//     per-warp shared-memory stage with 16-byte cp.async (LDGSTS, L1 bypass), several pairs in flight.
//   * The packed keys are expanded straight into mma.sync A fragments by the same walk as
//     PackedAttention's QK (mkv_walk.cuh): S = Kbar q^T, keys = M, heads = N, channels = K, fp32
//     accumulate; the group reduction (max or sum over the G heads) is two shuffles.
#include <cstdlib>

#include "mkv_internal.cuh"
#include "mkv_walk.cuh"

namespace mkv {

namespace {

using namespace walk;

constexpr int kItemRing = 64;       // item descriptors kept per warp (32 pairs)
constexpr int kScoreStage = 4096;   // two items: 2 x (128 B of bitmaps + 16 r_k B of values), or 2 x 2048 B dense

struct __align__(16) Item {  // 8 block keys of one segment
    uint32_t src16;          // payload offset of the item's bitmaps (values if dense) in the slice, 16-B units
    uint32_t val16;          // offset of the item's values, 16-B units
    uint32_t out;            // index of its first score: unit * score_stride + block index
    uint16_t unit;
    uint8_t r_k, nb;         // nb = 0: nothing there (segment past the unit's end)
};

__host__ __device__ constexpr int score_warp_smem(int nstage) { return nstage * kScoreStage + kItemRing * 16 + nstage * 16; }

struct __align__(16) SMeta {  // one in-flight group (<= 2 items of one unit with equal r_k)
    int32_t unit;
    uint32_t rknb;            // r_k | nb0 << 8 | nb1 << 16 | n << 24 (n = 0: end of the range)
    uint32_t out0, out1;
};

// ------------------------------------------------------------------------------------------
// one CTA per SM, kWarps independent warps; warp gw owns items [gw I / GW, (gw+1) I / GW) of the
// I = n_units * items_per_unit items of the layer (items_per_unit = S_max * subs).
// ------------------------------------------------------------------------------------------
template <int NSTAGE, int kWarps>
__global__ void __launch_bounds__(kWarps * 32, 1)
mkv_score_kernel(CacheGeom g, LayerView lv, const uint16_t* __restrict__ q, int reduce, int subs,
                 unsigned items_per_unit, float* __restrict__ scores) {
    extern __shared__ __align__(128) uint8_t smem[];
    constexpr int kWS = score_warp_smem(NSTAGE);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int gq = lane >> 2, qq = lane & 3;
    const int G = g.group;

    const unsigned long long I = (unsigned long long)g.n_units * items_per_unit;
    const unsigned GW = gridDim.x * kWarps, gw = blockIdx.x * kWarps + warp;
    const unsigned long long lo = I * gw / GW, hi = I * (gw + 1) / GW;
    const int n_total = (int)(hi - lo);
    if (n_total <= 0) return;

    uint8_t* wbase = smem + warp * kWS;
    const uint32_t stage0 = smem_u32(wbase);
    Item* ring = reinterpret_cast<Item*>(wbase + NSTAGE * kScoreStage);
    SMeta* gmeta = reinterpret_cast<SMeta*>(wbase + NSTAGE * kScoreStage + kItemRing * 16);

    int pos = 0, built = 0;

    auto build = [&](int count) {
        if (lane < count) {
            const unsigned long long it = lo + (unsigned)(built + lane);
            const unsigned u = (unsigned)(it / items_per_unit);
            const unsigned rem = (unsigned)(it - (unsigned long long)u * items_per_unit);
            const unsigned seg = subs == 1 ? rem : rem / (unsigned)subs;
            const unsigned sub = rem - seg * (unsigned)subs;
            Item d;
            d.src16 = 0; d.val16 = 0; d.out = 0; d.unit = (uint16_t)u; d.r_k = 0; d.nb = 0;
            if ((int)seg < lv.unit_nseg[u]) {
                const size_t e = (size_t)u * lv.S_max + seg;
                const StratRec rec = lv.strat[e];
                const int nblk = ((int)rec.n_tok + kB - 1) / kB;
                const int nb = min(8, nblk - 8 * (int)sub);
                if (nb > 0) {
                    const uint32_t off = lv.bk_off[e];
                    d.r_k = rec.r_k; d.nb = (uint8_t)nb;
                    if (rec.r_k == kD) { d.src16 = off + 128u * sub; d.val16 = d.src16; }
                    else { d.src16 = off + 8u * sub; d.val16 = off + (uint32_t)nblk + (uint32_t)rec.r_k * sub; }
                    d.out = u * (unsigned)g.score_stride + seg * (unsigned)g.blocks_per_seg + 8u * sub;
                }
            }
            ring[(built + lane) & (kItemRing - 1)] = d;
        }
        built += count;
        __syncwarp();
    };

    // form the next group and start its copies into stage s
    auto issue = [&](int s) {
        for (;;) {
            if (built - pos <= 8 && built < n_total) build(min(32, n_total - built));
            if (pos >= n_total || ring[pos & (kItemRing - 1)].nb != 0) break;
            ++pos;  // nothing there: a segment past the unit's end
        }
        if (pos >= n_total) {
            if (lane == 0) { SMeta m; m.unit = -1; m.rknb = 0; m.out0 = m.out1 = 0; gmeta[s] = m; }
            cp_async_commit();
            return;
        }
        const Item d0 = ring[pos & (kItemRing - 1)];
        Item d1 = d0;
        bool two = false;
        if (pos + 1 < n_total) {
            d1 = ring[(pos + 1) & (kItemRing - 1)];
            two = d1.nb != 0 && d1.unit == d0.unit && d1.r_k == d0.r_k && (d0.r_k == kD || d0.r_k <= 120);
        }
        if (lane == 0) {
            SMeta m;
            m.unit = d0.unit;
            m.rknb = (uint32_t)d0.r_k | ((uint32_t)d0.nb << 8) | ((two ? (uint32_t)d1.nb : 0u) << 16) | ((two ? 2u : 1u) << 24);
            m.out0 = d0.out; m.out1 = d1.out;
            gmeta[s] = m;
        }
        const unsigned long long base = reinterpret_cast<unsigned long long>(lv.slice);
        const uint32_t dst = stage0 + s * kScoreStage;
        const int r = d0.r_k;
#pragma unroll 1
        for (int t = 0; t < (two ? 2 : 1); ++t) {
            const Item& d = t ? d1 : d0;
            const uint32_t dd = dst + t * 2048;
            if (r == kD) {
                const unsigned long long src = base + ((unsigned long long)d.src16 << 4);
                for (int i = lane; i < 16 * d.nb; i += 32) cp_async_16(dd + 16 * i, src + 16 * i);
            } else {
                const unsigned long long sb = base + ((unsigned long long)d.src16 << 4);
                const unsigned long long sv = base + ((unsigned long long)d.val16 << 4);
                const int nv = (2 * r * d.nb + 15) >> 4, nbm = d.nb;
                for (int i = lane; i < nbm + nv; i += 32) {
                    if (i < nbm) cp_async_16(dd + 16 * i, sb + 16 * i);
                    else cp_async_16(dd + 128 + 16 * (i - nbm), sv + 16 * (i - nbm));
                }
            }
        }
        cp_async_commit();
        pos += two ? 2 : 1;
    };

    uint32_t qa[8][2];
    int cur_unit = -1;

#pragma unroll 1
    for (int k = -NSTAGE;; ++k) {
        const int s = (k + NSTAGE) % NSTAGE;
        if (k >= 0) {
            __syncwarp();
            const SMeta meta = gmeta[s];
            const int n = (int)(meta.rknb >> 24);
            if (n == 0) break;
            if (meta.unit != cur_unit) {
                cur_unit = meta.unit;
                const int bi = cur_unit / g.n_kv_heads, hk = cur_unit % g.n_kv_heads;
                const uint4* qrow = reinterpret_cast<const uint4*>(
                    q + ((size_t)bi * g.n_q_heads + (size_t)hk * G + gq) * kD + 32 * qq);
#pragma unroll
                for (int h = 0; h < 4; ++h) {
                    uint4 v = make_uint4(0u, 0u, 0u, 0u);
                    if (gq < G) v = __ldg(qrow + h);
                    qa[2 * h][0] = v.x; qa[2 * h][1] = v.y; qa[2 * h + 1][0] = v.z; qa[2 * h + 1][1] = v.w;
                }
            }
            const int r_k = (int)(meta.rknb & 255u), nb0 = (int)((meta.rknb >> 8) & 255u), nb1 = (int)((meta.rknb >> 16) & 255u);
            const uint32_t sp0 = stage0 + s * kScoreStage, sp1 = sp0 + 2048;
            const bool full = nb0 == 8 && (n == 1 || nb1 == 8);

            cp_async_wait<NSTAGE - 1>();
            __syncwarp();

            float S[4] = {0.f, 0.f, 0.f, 0.f};  // rows gq / gq+8 = key gq of item 0 / 1, columns = heads 2qq, 2qq+1
            if (r_k == kD && full) {
                const uint32_t a0 = sp0 + 256 * gq + 64 * qq, a1 = sp1 + 256 * gq + 64 * qq;
#pragma unroll
                for (int h = 0; h < 4; ++h) {
                    const uint4 x = lds_128(a0 + 16 * h);
                    uint4 y = make_uint4(0u, 0u, 0u, 0u);
                    if (n == 2) y = lds_128(a1 + 16 * h);
                    mma_bf16(S, x.x, y.x, x.y, y.y, qa[2 * h][0], qa[2 * h][1]);
                    mma_bf16(S, x.z, y.z, x.w, y.w, qa[2 * h + 1][0], qa[2 * h + 1][1]);
                }
            } else {
                uint32_t w0 = 0u, w1 = 0u, p0, p1, st0 = 2u, st1 = 2u;
                if (r_k == kD) {  // ragged dense item: all slots kept, no bitmap stored
                    w0 = gq < nb0 ? 0xffffffffu : 0u;
                    w1 = (n == 2 && gq < nb1) ? 0xffffffffu : 0u;
                    p0 = sp0 + 256 * gq + 64 * qq;
                    p1 = sp1 + 256 * gq + 64 * qq;
                } else {
                    if (gq < nb0) w0 = lds_u32(sp0 + 4 * lane);
                    if (n == 2 && gq < nb1) w1 = lds_u32(sp1 + 4 * lane);
                    uint32_t cnt = (uint32_t)__popc(w0) | ((uint32_t)__popc(w1) << 16), inc = cnt, t;
                    t = __shfl_up_sync(kFull, inc, 1); if (qq >= 1) inc += t;
                    t = __shfl_up_sync(kFull, inc, 2); if (qq >= 2) inc += t;
                    const uint32_t ex = inc - cnt;
                    st0 = 2u * nb0; st1 = 2u * nb1;  // values rank-major within the item (compress.cu)
                    p0 = sp0 + 128 + st0 * (ex & 0xffffu) + 2 * gq;
                    p1 = sp1 + 128 + st1 * (ex >> 16) + 2 * gq;
                }
                k_walk_mma<0>(S, w0, w1, p0, p1, st0, st1, qa);
                k_walk_mma<1>(S, w0, w1, p0, p1, st0, st1, qa);
                k_walk_mma<2>(S, w0, w1, p0, p1, st0, st1, qa);
                k_walk_mma<3>(S, w0, w1, p0, p1, st0, st1, qa);
            }
            __syncwarp();  // every lane is done reading stage s

            // reduce over the group's heads (columns 2qq, 2qq+1 of the four lanes of a row)
            const bool hA = 2 * qq < G, hB = 2 * qq + 1 < G;
            float v0, v1;
            if (reduce == 1) {
                v0 = (hA ? S[0] : 0.f) + (hB ? S[1] : 0.f);
                v1 = (hA ? S[2] : 0.f) + (hB ? S[3] : 0.f);
                v0 += __shfl_xor_sync(kFull, v0, 1); v1 += __shfl_xor_sync(kFull, v1, 1);
                v0 += __shfl_xor_sync(kFull, v0, 2); v1 += __shfl_xor_sync(kFull, v1, 2);
            } else {
                v0 = fmaxf(hA ? S[0] : -INFINITY, hB ? S[1] : -INFINITY);
                v1 = fmaxf(hA ? S[2] : -INFINITY, hB ? S[3] : -INFINITY);
                v0 = fmaxf(v0, __shfl_xor_sync(kFull, v0, 1)); v1 = fmaxf(v1, __shfl_xor_sync(kFull, v1, 1));
                v0 = fmaxf(v0, __shfl_xor_sync(kFull, v0, 2)); v1 = fmaxf(v1, __shfl_xor_sync(kFull, v1, 2));
            }
            if (qq == 0) {
                if (gq < nb0) scores[meta.out0 + gq] = v0 + 0.0f;
                if (n == 2 && gq < nb1) scores[meta.out1 + gq] = v1 + 0.0f;
            }
        }
        issue(s);
    }
}

}  // namespace

template <int NSTAGE, int NWARPS>
static cudaError_t launch_score_cfg(const CacheGeom& g, const LayerView& lv, const uint16_t* q, int reduce,
                                    float* scores, int sm_count, cudaStream_t s) {
    const int smem = NWARPS * score_warp_smem(NSTAGE);
    static int configured = 0;
    if (smem > configured) {
        cudaError_t e = cudaFuncSetAttribute(mkv_score_kernel<NSTAGE, NWARPS>,
                                             cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
        if (e != cudaSuccess) return e;
        configured = smem;
    }
    const int subs = (g.blocks_per_seg + 7) / 8;
    mkv_score_kernel<NSTAGE, NWARPS><<<sm_count, NWARPS * 32, smem, s>>>(g, lv, q, reduce, subs,
                                                                         (unsigned)g.S_max * (unsigned)subs, scores);
    return cudaGetLastError();
}

cudaError_t launch_score(const CacheGeom& g, const LayerView& lv, const uint16_t* q, int reduce, float* scores,
                         int sm_count, cudaStream_t s) {
    static int cfg = -1;  // tuning knob (stages * 100 + warps); default chosen from measurements
    if (cfg < 0) {
        const char* e = getenv("MKV_SCORE_CFG");
        cfg = e ? atoi(e) : 316;
    }
#define MKV_CFG(S, W) \
    case S * 100 + W: return launch_score_cfg<S, W>(g, lv, q, reduce, scores, sm_count, s);
    switch (cfg) {
        MKV_CFG(3, 16) MKV_CFG(2, 16) MKV_CFG(4, 12) MKV_CFG(4, 8) MKV_CFG(6, 8)
        default: return launch_score_cfg<3, 16>(g, lv, q, reduce, scores, sm_count, s);
    }
#undef MKV_CFG
}

}  // namespace mkv
