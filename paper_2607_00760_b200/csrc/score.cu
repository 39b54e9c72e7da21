// score.cu — step 2a of the hot path: block scores on the packed block keys (PAPER.md:182,
// 214-216): s_b = reduce_h sum_{c kept} q_h[c] * kbar_b[c], directly on the packed keys.  sm_100a.
//
// Design: a streaming kernel over the block-key arena.
//   * Work item = 8 block keys of one segment (one item per segment at L = 64).  Items are taken in
//     pairs (16 keys = the M of one mma.sync tile); the items of all units form one stream that is
//     cut into equal contiguous ranges, one per warp of a one-CTA-per-SM grid.  Warps are
//     independent (no __syncthreads at all).
//   * Staging: an item's position bitmaps and its kept values (DESIGN.md format) are contiguous
//     16-B-aligned chunks (usually the whole pair is one); every lane moves 16 bytes at a time with
//     cp.async, one commit group per stage, NSTAGE groups in flight per warp.  Full dense items are
//     placed with their 16-byte chunks swizzled so that the LDS.128 path has no bank conflicts.
//   * The packed keys are expanded straight into mma.sync A fragments by the same walk as
//     PackedAttention's QK (mkv_walk.cuh): S = Kbar q^T, keys = M, heads = N, channels = K, fp32
//     accumulate; the group reduction (max or sum over the G heads) is two shuffles.
#include "mkv_internal.cuh"
#include "mkv_walk.cuh"

namespace mkv {

namespace {

using namespace walk;

constexpr int kRing = 64;           // group descriptors kept per warp
constexpr int kScoreStage = 2176;   // one item of any r_k (<= 128 + 16 * 127 B), or two items with r_k <= kPairMaxR
constexpr int kItem1 = 1024;        // stage offset of the second item of a pair
constexpr uint32_t kPairMaxR = 56;  // 128 + 16 r_k <= kItem1

// One group: <= 2 consecutive items (8 block keys each) of one unit with the same r_k.
struct __align__(16) SDesc {
    uint32_t bm0, val0, bm1, val1;  // chunk offsets in the layer slice, 16-B units (dense: bm = the keys, val unused)
    uint32_t out0, out1;            // index of each item's first score: unit * score_stride + block index
    uint32_t meta;                  // r_k | nb0 << 8 | nb1 << 12 | merged << 16 (the group is ONE contiguous chunk of the slice)
                                    // | its size / 16 << 17 | pairs << 30 (element groups g >= 2: values pair-major, mkv_walk.cuh)
    uint32_t unit;                  // unit | (stage offset of item 1 / 16) << 24
};

__device__ __forceinline__ unsigned lanemask_le() {
    unsigned m;
    asm("mov.u32 %0, %%lanemask_le;" : "=r"(m));
    return m;
}
__device__ __forceinline__ unsigned lanemask_lt() {
    unsigned m;
    asm("mov.u32 %0, %%lanemask_lt;" : "=r"(m));
    return m;
}

__host__ __device__ constexpr int score_warp_smem(int nstage) { return nstage * kScoreStage + kRing * 32 + 64; }

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

    pdl_wait();               // the cache and q are complete; the previous reader of `scores` is done
    pdl_launch_dependents();
    const unsigned I = (unsigned)g.n_units * items_per_unit;  // < 2^32: checked by the launcher
    const unsigned GW = gridDim.x * kWarps, gw = blockIdx.x * kWarps + warp;
    const unsigned ib = I / GW, ir = I - ib * GW;             // the first ir warps hold one more item
    const unsigned lo = gw * ib + min(gw, ir);
    const int n_total = (int)(ib + (gw < ir ? 1u : 0u));
    if (n_total <= 0) return;

    uint8_t* wbase = smem + warp * kWS;
    const uint32_t stage0 = smem_u32(wbase);
    SDesc* ring = reinterpret_cast<SDesc*>(wbase + NSTAGE * kScoreStage);

    int ibuilt = 0;                        // items described
    int gposc = 0, gposi = 0, gbuilt = 0;  // groups consumed / issued / described

    // Describe the next <= 32 items of the range (one per lane) and pair them into groups: item i
    // follows item i - 1 in a group if both hold keys, belong to one unit and have the same r_k;
    // runs of such items are paired greedily from their start.  Items past a unit's end hold no keys.
    auto build = [&](int count) {
        uint32_t bm = 0u, val = 0u, out = 0u, r_k = 0u, nb = 0u, u = 0u, pairs = 0u;
        uint32_t sz = 0u;  // 16-B units of the item when its bitmaps and values are one chunk (one item per segment), else 0
        if (lane < count) {
            const unsigned it = lo + (unsigned)(ibuilt + lane);
            u = it / items_per_unit;
            const unsigned rem = it - u * items_per_unit;
            const unsigned seg = subs == 1 ? rem : rem / (unsigned)subs;
            const unsigned sub = rem - seg * (unsigned)subs;
            if ((int)seg < lv.unit_nseg[u]) {
                const size_t e = (size_t)u * lv.S_max + seg;
                const StratRec rec = lv.strat[e];
                const int nblk = ((int)rec.n_tok + g.B - 1) / g.B;
                const int n = min(8, nblk - 8 * (int)sub);
                if (n > 0) {
                    const uint32_t off = lv.bk_off[e];
                    r_k = rec.r_k; nb = (uint32_t)n;
                    pairs = rec.g >= 2 && rec.r_k != kD ? 1u : 0u;
                    if (rec.r_k == kD) { bm = off + 128u * sub; val = bm; }
                    else { bm = off + 8u * sub; val = off + (uint32_t)nblk + (uint32_t)rec.r_k * sub; }
                    out = u * (unsigned)g.score_stride + seg * (unsigned)g.blocks_per_seg + 8u * sub;
                    if (rec.r_k != kD && nblk <= 8) sz = nb + ((nb * 2u * r_k + 15u) >> 4);
                }
            }
        }
        const uint32_t pu = __shfl_up_sync(kFull, u, 1), prk = __shfl_up_sync(kFull, r_k | (pairs << 8), 1), pnb = __shfl_up_sync(kFull, nb, 1);
        const bool follows = lane > 0 && nb != 0u && pnb != 0u && u == pu && (r_k | (pairs << 8)) == prk && r_k <= kPairMaxR;  // two items must fit one stage
        const unsigned fm = __ballot_sync(kFull, follows);
        const int start = 31 - __clz((int)(~fm & lanemask_le()));  // first item of this lane's run (bit 0 of ~fm is set)
        const bool first = nb != 0u && ((lane - start) & 1) == 0;
        const bool two = first && ((fm >> 1) >> lane & 1u);
        const unsigned gm = __ballot_sync(kFull, first);
        const uint32_t bm1 = __shfl_down_sync(kFull, bm, 1), val1 = __shfl_down_sync(kFull, val, 1);
        const uint32_t out1 = __shfl_down_sync(kFull, out, 1), nb1 = __shfl_down_sync(kFull, nb, 1);
        const uint32_t sz1 = __shfl_down_sync(kFull, sz, 1);
        // segments compressed by one call lie back to back in the slice (plan kernel): the usual group is one chunk
        const bool merged = two && sz != 0u && sz1 != 0u && bm1 == bm + sz;
        if (first) {
            SDesc d;
            d.bm0 = bm; d.val0 = val; d.bm1 = two ? bm1 : 0u; d.val1 = two ? val1 : 0u;
            d.out0 = out; d.out1 = two ? out1 : 0u;
            d.meta = r_k | (nb << 8) | ((two ? nb1 : 0u) << 12) | (merged ? (1u << 16) | ((sz + sz1) << 17) : 0u) | (pairs << 30);
            d.unit = u | ((merged ? sz : (uint32_t)(kItem1 / 16)) << 24);  // (units < 2^24: checked by the launcher)
            ring[(gbuilt + __popc(gm & lanemask_lt())) & (kRing - 1)] = d;
        }
        gbuilt += __popc(gm);
        ibuilt += count;
        __syncwarp();
    };

    // start the copies of the next group into stage s: every lane moves 16 bytes at a time (cp.async), one commit group
    // per call (empty when nothing is left, so that "all but the newest NSTAGE - 1 groups" always means "group k")
    const unsigned long long slice = reinterpret_cast<unsigned long long>(lv.slice);
    auto copy_chunk = [&](uint32_t dst, uint32_t src16, uint32_t bytes) {
        const unsigned long long src = slice + ((unsigned long long)src16 << 4);
#pragma unroll 1
        for (uint32_t x = 16u * (uint32_t)lane; x < bytes; x += 512u) cp_async_16(dst + x, src + x);
    };
    auto issue = [&](int s) {
#pragma unroll 1
        while (gposi == gbuilt && ibuilt < n_total) build(min(32, n_total - ibuilt));
        if (gposi != gbuilt) {
            const SDesc d = ring[gposi & (kRing - 1)];
            const uint32_t dst = stage0 + s * kScoreStage;
            if (d.meta & (1u << 16)) {  // item 1 lands right behind item 0: one chunk of <= kScoreStage bytes
                const uint32_t bytes = ((d.meta >> 17) & 0xffu) << 4, x = 16u * (uint32_t)lane;
                const unsigned long long src = slice + ((unsigned long long)d.bm0 << 4) + x;
#pragma unroll
                for (uint32_t i = 0; i < (kScoreStage + 511) / 512; ++i)  // (straight line: constant offsets, no loop counter)
                    if (x + 512u * i < bytes) cp_async_16(dst + x + 512u * i, src + 512u * i);
            } else {
                const uint32_t r = d.meta & 255u, nb0 = (d.meta >> 8) & 15u, nb1 = (d.meta >> 12) & 15u;
                // bitmaps nb x 16 B, then the values padded to 16 B; dense: nb x 256 B in one chunk
                const uint32_t bb0 = r == (uint32_t)kD ? nb0 * 256u : nb0 * 16u, vb0 = r == (uint32_t)kD ? 0u : pad16u(nb0 * 2u * r);
                const uint32_t bb1 = r == (uint32_t)kD ? nb1 * 256u : nb1 * 16u, vb1 = r == (uint32_t)kD ? 0u : pad16u(nb1 * 2u * r);
                if (r == (uint32_t)kD && nb0 == 8u && nb1 == 0u) {
                    // a full dense item takes the LDS.128 path below: its 16-byte chunks are placed so that the eight lanes
                    // of a load phase (two keys x four 64-byte quarters) hit eight different bank groups (rows are 256 B
                    // apart, i.e. in the same banks): chunk c of key t goes to chunk c ^ 2 (c >> 3) ^ (t & 1)
                    const unsigned long long src = slice + ((unsigned long long)d.bm0 << 4);
#pragma unroll
                    for (uint32_t i = 0; i < 4u; ++i) {
                        const uint32_t ci = (uint32_t)lane + 32u * i, t = ci >> 4, c = ci & 15u;
                        cp_async_16(dst + 256u * t + 16u * (c ^ ((c >> 3) << 1) ^ (t & 1u)), src + 16u * ci);
                    }
                } else
                    copy_chunk(dst, d.bm0, bb0);
                copy_chunk(dst + bb0, d.val0, vb0);
                copy_chunk(dst + kItem1, d.bm1, bb1);
                copy_chunk(dst + kItem1 + bb1, d.val1, vb1);
            }
            ++gposi;
        }
        cp_async_commit();
    };

    uint32_t qa[8][2];
    int cur_unit = -1;

    // ---- main loop.  Iteration k >= 0 consumes group k from stage k % NSTAGE and refills that stage
    // with group k + NSTAGE; iterations k < 0 only fill the pipeline (one call site for issue()).
    int s = 0;
#pragma unroll 1
    for (int k = -NSTAGE;; ++k) {
        if (k >= 0) {
            if (gposc == gbuilt) break;  // issue() runs ahead: nothing described means nothing left
            const SDesc d = ring[gposc & (kRing - 1)];
            if ((int)(d.unit & 0xffffffu) != cur_unit) {
                cur_unit = (int)(d.unit & 0xffffffu);
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
            const int r_k = (int)(d.meta & 255u), nb0 = (int)((d.meta >> 8) & 15u), nb1 = (int)((d.meta >> 12) & 15u);
            const uint32_t sp0 = stage0 + s * kScoreStage;
            const uint32_t sp1 = sp0 + ((d.unit >> 24) << 4);

            cp_async_wait<NSTAGE - 1>();  // this lane's copies of the group have landed ...
            __syncwarp();                 // ... and every other lane's

            float S[4] = {0.f, 0.f, 0.f, 0.f};  // rows gq / gq+8 = key gq of item 0 / 1, columns = heads 2qq, 2qq+1
            if (r_k == kD && nb0 == 8 && nb1 == 0) {  // (dense items are never paired: two do not fit a stage)
                const uint32_t a0 = sp0 + 256 * gq + 64 * qq, sw = (uint32_t)(2 * (qq >> 1)) ^ (uint32_t)(gq & 1);  // (swizzle of issue())
#pragma unroll
                for (int h = 0; h < 4; ++h) {
                    const uint4 x = lds_128(a0 + 16 * ((uint32_t)h ^ sw));
                    mma_bf16(S, x.x, 0u, x.y, 0u, qa[2 * h][0], qa[2 * h][1]);
                    mma_bf16(S, x.z, 0u, x.w, 0u, qa[2 * h + 1][0], qa[2 * h + 1][1]);
                }
            } else {
                uint32_t w0 = 0u, w1 = 0u, p0, p1, st0 = 2u, st1 = 2u;
                if (r_k == kD) {  // ragged dense item: all slots kept, no bitmap stored
                    w0 = gq < nb0 ? 0xffffffffu : 0u;
                    w1 = gq < nb1 ? 0xffffffffu : 0u;
                    p0 = sp0 + 256 * gq + 64 * qq;
                    p1 = sp1 + 256 * gq + 64 * qq;
                } else {  // bitmaps nb x 16 B, then the values rank-major within the item (compress.cu)
                    if (gq < nb0) w0 = lds_u32(sp0 + 4 * lane);
                    if (gq < nb1) w1 = lds_u32(sp1 + 4 * lane);
                    uint32_t cnt = (uint32_t)__popc(w0) | ((uint32_t)__popc(w1) << 16), inc = cnt, t;
                    t = __shfl_up_sync(kFull, inc, 1); if (qq >= 1) inc += t;
                    t = __shfl_up_sync(kFull, inc, 2); if (qq >= 2) inc += t;
                    const uint32_t ex = inc - cnt;
                    st0 = 2u * nb0; st1 = 2u * nb1;
                    p0 = sp0 + 16 * nb0 + st0 * (ex & 0xffffu) + 2 * gq;
                    p1 = sp1 + 16 * nb1 + st1 * (ex >> 16) + 2 * gq;
                }
                if ((d.meta >> 30) & 1u) {  // element groups g >= 2: pair pi = rank / 2 of key t at byte 4 (pi n + t)
                    p0 += 2 * gq; p1 += 2 * gq;
                    st0 *= 2u; st1 *= 2u;
                    k_walk_mma_pairs<0>(S, w0, w1, p0, p1, st0, st1, qa);
                    k_walk_mma_pairs<1>(S, w0, w1, p0, p1, st0, st1, qa);
                    k_walk_mma_pairs<2>(S, w0, w1, p0, p1, st0, st1, qa);
                    k_walk_mma_pairs<3>(S, w0, w1, p0, p1, st0, st1, qa);
                } else {
                    k_walk_mma<0>(S, w0, w1, p0, p1, st0, st1, qa);
                    k_walk_mma<1>(S, w0, w1, p0, p1, st0, st1, qa);
                    k_walk_mma<2>(S, w0, w1, p0, p1, st0, st1, qa);
                    k_walk_mma<3>(S, w0, w1, p0, p1, st0, st1, qa);
                }
            }
            __syncwarp();  // every lane is done reading stage s

            // reduce over the group's heads (columns 2qq, 2qq+1 of the four lanes of a row)
            const bool hA = 2 * qq < G, hB = 2 * qq + 1 < G;
            float v0, v1;
            if (reduce == 1) {
                v0 = (hA ? S[0] : 0.f) + (hB ? S[1] : 0.f);
                v1 = (hA ? S[2] : 0.f) + (hB ? S[3] : 0.f);
                v0 += __shfl_xor_sync(kFull, v0, 1); v1 += __shfl_xor_sync(kFull, v1, 1);
                if (G > 4) { v0 += __shfl_xor_sync(kFull, v0, 2); v1 += __shfl_xor_sync(kFull, v1, 2); }  // (G <= 4: lanes qq = 2, 3 hold nothing)
            } else {
                v0 = fmaxf(hA ? S[0] : -INFINITY, hB ? S[1] : -INFINITY);
                v1 = fmaxf(hA ? S[2] : -INFINITY, hB ? S[3] : -INFINITY);
                v0 = fmaxf(v0, __shfl_xor_sync(kFull, v0, 1)); v1 = fmaxf(v1, __shfl_xor_sync(kFull, v1, 1));
                if (G > 4) { v0 = fmaxf(v0, __shfl_xor_sync(kFull, v0, 2)); v1 = fmaxf(v1, __shfl_xor_sync(kFull, v1, 2)); }
            }
            // (after the reduction every lane of a row holds both results: lane qq = 0 stores item 0's, qq = 1 item 1's)
            if (qq < 2 && gq < (qq == 0 ? nb0 : nb1)) scores[(qq == 0 ? d.out0 : d.out1) + gq] = (qq == 0 ? v0 : v1) + 0.0f;
            ++gposc;
        }
        issue(s);  // stage s is free (or, for k < 0, still empty): start the copies of group k + NSTAGE
        if (++s == NSTAGE) s = 0;
    }
}

}  // namespace

template <int NSTAGE, int NWARPS>
static cudaError_t launch_score_cfg(const CacheGeom& g, const LayerView& lv, const uint16_t* q, int reduce,
                                    float* scores, int sm_count, cudaStream_t s) {
    const int smem = NWARPS * score_warp_smem(NSTAGE);
    // (a per-device attribute of the function: set on every launch, see attention.cu)
    cudaError_t e = cudaFuncSetAttribute(mkv_score_kernel<NSTAGE, NWARPS>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    if (e != cudaSuccess) return e;
    const int subs = (g.blocks_per_seg + 7) / 8;
    if ((unsigned long long)g.n_units * g.S_max * subs >= (1ull << 32) || g.n_units >= (1 << 24)) return cudaErrorInvalidValue;
    return launch_pdl(mkv_score_kernel<NSTAGE, NWARPS>, dim3(sm_count), dim3(NWARPS * 32), (size_t)smem, s, g, lv, q, reduce,
                      subs, (unsigned)g.S_max * (unsigned)subs, scores);
}

// two stages x 32 warps: the kernel needs 64 registers, and warps are what hides the walk's dependent loads
cudaError_t launch_score(const CacheGeom& g, const LayerView& lv, const uint16_t* q, int reduce, float* scores,
                         int sm_count, cudaStream_t s) {
    return launch_score_cfg<2, 32>(g, lv, q, reduce, scores, sm_count, s);
}

}  // namespace mkv
