// attention.cu — step 3 of the hot path: PackedAttention: QK over the
// selected packed keys, online softmax, PV over the packed values, split-K combine.  sm_100a.
//
// Design:
//   * The selected blocks of all units form one stream of T blocks; it is cut into equal ranges,
//     one per warp of a one-CTA-per-SM grid (warps are fully independent: no __syncthreads in
//     the main loop).  A warp walks its range in groups of <= 2 token blocks (16 tokens).
//   * Staging: every token block is one contiguous 16-B-aligned chunk (DESIGN.md format); one lane
//     moves it into the warp's shared-memory stage with ONE 1-D bulk copy (cp.async.bulk, the TMA
//     engine) that completes on the stage's mbarrier; kStages groups are in flight per warp.
//   * Packed vectors are expanded STRAIGHT INTO mma.sync fragments — no dense tile in shared
//     memory.  QK: S = K q^T with the group's 16 tokens = M (rows 0-7 block 0, rows 8-15 block
//     1), heads = N, channels = K; lane (gq, qq) owns token gq of each block and bitmap word qq
//     (32 channels) and walks its 32 slots in order: a set bit loads the next kept bf16 of its
//     run and bumps the run pointer (mkv_walk.cuh).  The channel order inside a k-step is a fixed
//     permutation applied to q's B fragments as well.
//     PV: O^T = V^T P^T with channels = M, heads = N, the 16 tokens of the group = K; lane
//     (gq, qq) owns tokens 2qq, 2qq+1 of each block and the 16-channel half-word gq, so a
//     fragment register pairs two TOKENS of one channel, as the contraction over tokens needs.
//     P is split into bf16 hi + lo (fp32-class accuracy) and transposed into the B fragment
//     layout with movmatrix.  Dense vectors (r = D) skip the walk: their fragments are 16-byte
//     shared loads.
//   * Step 3d (split-K combine) is fused: a unit wholly inside one warp's range is normalised and
//     written directly; otherwise the warp leaves an (m, l, O) partial (<= 2 per warp), every
//     thread of the CTA folds the partials of a unit for its own output element with the LSE rule,
//     and a unit that spans several CTAs is finished by the last CTA to arrive at a per-unit
//     ticket (no second kernel).
#include <cstdlib>

#include "mkv_internal.cuh"
#include "mkv_walk.cuh"

namespace mkv {

#ifdef MKV_DBG_TIMING
__device__ unsigned long long g_dbg_t[160 * 8];
__device__ __forceinline__ unsigned long long dbg_now() { unsigned long long t; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t)); return t; }
#define MKV_T(k) do { if (threadIdx.x == 0) g_dbg_t[blockIdx.x * 8 + (k)] = dbg_now(); } while (0)
#else
#define MKV_T(k) do {} while (0)
#endif

namespace {

using namespace walk;
constexpr float kLog2e = 1.4426950408889634f;
constexpr float kLn2 = 0.6931471805599453f;

constexpr int kMaxWarps = 16;      // upper bound on warps per CTA (sizes the partial-slot scratch)
constexpr int kStageBytes = 4096;  // one dense block (4096 B) or two packed blocks with r <= 56
constexpr int kDescRing = 64;      // block descriptors kept per warp
constexpr int kMaxUnitsSmem = 2048;

struct __align__(16) Desc {  // one selected token block
    uint32_t off16;          // payload offset in the layer slice, 16-B units
    uint32_t bytes;          // payload bytes (multiple of 16); 0 = skip (invalid entry)
    int32_t unit;
    uint32_t rr;             // r_k | r_v << 8 | nb << 16
};

// prefix sums of the clamped selection counts -> s_cum[0..n_units]; returns the total T
__device__ __forceinline__ int scan_counts(const int32_t* __restrict__ sel_count, int n_units, int k_max,
                                            int* s_cum) {
    __shared__ int s_carry;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (warp == 0) {
        int carry = 0;
        for (int i0 = 0; i0 < n_units; i0 += 32) {
            const int i = i0 + lane;
            int c = (i < n_units) ? min(max(sel_count[i], 0), k_max) : 0;
            int inc = c;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int v = __shfl_up_sync(kFull, inc, o);
                if (lane >= o) inc += v;
            }
            if (i < n_units) s_cum[i] = carry + inc - c;
            carry += __shfl_sync(kFull, inc, 31);
        }
        if (lane == 0) { s_cum[n_units] = carry; s_carry = carry; }
    }
    __syncthreads();
    return s_carry;
}

// largest u with s_cum[u] <= i (i < T guaranteed; zero-count units are skipped by construction)
__device__ __forceinline__ int find_unit(const int* s_cum, int n_units, int i) {
    int lo = 0, hi = n_units;  // invariant: s_cum[lo] <= i < s_cum[hi]
    while (hi - lo > 1) {
        const int mid = (lo + hi) >> 1;
        if (s_cum[mid] <= i) lo = mid; else hi = mid;
    }
    return lo;
}

// per warp: the stages, the descriptor ring, one mbarrier per stage (64 B reserved)
__host__ __device__ constexpr int warp_smem_bytes(int nstage) { return nstage * kStageBytes + kDescRing * 16 + 64; }

// ------------------------------------------------------------------------------------------
// main kernel: one CTA per SM, kWarps independent warps, each owning the block range
// [gw*T/GW, (gw+1)*T/GW) of the concatenated selection lists.
// ------------------------------------------------------------------------------------------
template <int NSTAGE, int kWarps>
__global__ void __launch_bounds__(kWarps * 32, 1)
mkv_packed_attention_kernel(CacheGeom g, LayerView lv, const uint16_t* __restrict__ q,
                            const int32_t* __restrict__ sel, const int32_t* __restrict__ sel_count, int k_max,
                            float scale_log2, float* __restrict__ out, float* __restrict__ lse,
                            float* __restrict__ part_o, float* __restrict__ part_ml, int32_t* __restrict__ ticket) {
    extern __shared__ __align__(128) uint8_t smem[];
    constexpr int kWS = warp_smem_bytes(NSTAGE);
    constexpr int kNT = kWarps * 32;
    constexpr int kRec = 2 * kWarps;  // partial records of the CTA: warp w -> 2w (head), 2w + 1 (tail)
    int* s_cum = reinterpret_cast<int*>(smem + kWarps * kWS);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int gq = lane >> 2, qq = lane & 3;  // mma fragment coordinates (groupID, threadID_in_group)

    MKV_T(0);
    __shared__ int s_unit[kRec];                 // unit of each partial record, -1 = none
    __shared__ const float* s_po[kRec];          // its unnormalised O [G][D] (shared memory, or global scratch)
    __shared__ float s_ml[kRec][kMaxGroup][2];   // its (max in log2 units, sum) per head
    __shared__ int s_last[2], s_cf[2], s_cl[2];
    __shared__ int s_clo, s_chi;
    __shared__ size_t s_row[2];

    uint8_t* wbase = smem + warp * kWS;
    const uint32_t stage0 = smem_u32(wbase);
    Desc* ring = reinterpret_cast<Desc*>(wbase + NSTAGE * kStageBytes);
    const uint32_t bar0 = stage0 + NSTAGE * kStageBytes + kDescRing * 16;
    if (lane == 0) {
#pragma unroll
        for (int s = 0; s < NSTAGE; ++s) mbar_init(bar0 + 8 * s, 1);
        mbar_init_fence();
    }
    if (lane < 2) s_unit[warp * 2 + lane] = -1;

    const int T = scan_counts(sel_count, g.n_units, k_max, s_cum);  // (block barrier inside)
    // Gd CTAs share the T blocks (every one of them owns >= 1 block); CTA c owns [c T / Gd, (c+1) T / Gd),
    // cut evenly again over its warps: warp gw of GW owns [gw T / GW, (gw+1) T / GW)
    const unsigned Gd = min(gridDim.x, (unsigned)max(T, 1));
    const unsigned GW = Gd * kWarps, gw = blockIdx.x * kWarps + warp;
    const float inv_GW = 1.f / (float)GW;
    int lo = 0, hi = 0;
    if (blockIdx.x < Gd) {
        lo = (int)div_floor((unsigned long long)gw * (unsigned)T, GW, inv_GW);
        hi = (int)div_floor((unsigned long long)(gw + 1) * (unsigned)T, GW, inv_GW);
    }
    if (lane == 0 && warp == 0) s_clo = lo;
    if (lane == 0 && warp == kWarps - 1) s_chi = hi;
    const int n_total = hi - lo;
    const int G = g.group;
    if (blockIdx.x == 0) {  // units with an empty selection: out = 0, lse = -inf
        for (int u = warp; u < g.n_units; u += kWarps) {
            if (s_cum[u + 1] != s_cum[u]) continue;
            const size_t row = (size_t)(u / g.n_kv_heads) * g.n_q_heads + (size_t)(u % g.n_kv_heads) * G;
            for (int e = lane; e < G * kD; e += 32) out[row * kD + e] = 0.f;
            if (lse != nullptr && lane < G) lse[row + lane] = -INFINITY;
        }
    }

    int posc = 0, posi = 0, built = 0;  // next block to consume / to issue / to describe

    // descriptors of the next <= 32 blocks of the range, one per lane
    auto build = [&](int count) {
        if (lane < count) {
            const int idx = built + lane;
            const int gi = lo + idx;
            const int u = find_unit(s_cum, g.n_units, gi);
            const int j = gi - s_cum[u];
            const int t0 = sel[(size_t)u * k_max + j];
            Desc d;
            d.unit = u; d.off16 = 0; d.bytes = 0; d.rr = 0;
            const int ntok = lv.unit_ntok[u];
            if (t0 >= 0 && t0 < ntok && (t0 & (kB - 1)) == 0) {
                const int seg = t0 / g.L, in_seg = t0 - seg * g.L;
                const size_t e = (size_t)u * lv.S_max + seg;
                const StratRec rec = lv.strat[e];
                const int nb = min(kB, (int)rec.n_tok - in_seg);
                d.off16 = lv.tok_off[e] + (uint32_t)(in_seg >> 3) * (tokblock_bytes(rec.r_k, rec.r_v, kB) >> 4);
                d.bytes = tokblock_bytes(rec.r_k, rec.r_v, nb);
                d.rr = (uint32_t)rec.r_k | ((uint32_t)rec.r_v << 8) | ((uint32_t)nb << 16);
            }
            ring[idx & (kDescRing - 1)] = d;
        }
        built += count;
        __syncwarp();
    };

    // the group starting at block p: <= 2 blocks of one unit with the same strategy that fit one
    // stage.  A pure function of the ring, evaluated identically when issuing and when consuming.
    auto group_at = [&](int p, Desc& d0, Desc& d1) -> bool {
        d0 = ring[p & (kDescRing - 1)];
        d1 = d0;
        if (p + 1 >= n_total) return false;
        d1 = ring[(p + 1) & (kDescRing - 1)];
        return d1.unit == d0.unit && ((d1.rr ^ d0.rr) & 0xffffu) == 0u && d0.bytes != 0u && d1.bytes != 0u &&
               d0.bytes + d1.bytes <= (uint32_t)kStageBytes;
    };

    // start the copies of the next group into stage s: one bulk copy per block, issued by lane 0,
    // completing on the stage's mbarrier
    const unsigned long long slice = reinterpret_cast<unsigned long long>(lv.slice);
    auto issue = [&](int s) {
        if (posi >= n_total) return;
        if (built - posi < 2 && built < n_total) build(min(32, n_total - built));
        Desc d0, d1;
        const bool two = group_at(posi, d0, d1);
        if (lane == 0) {
            const uint32_t bar = bar0 + 8 * s, dst = stage0 + s * kStageBytes;
            mbar_expect_tx(bar, d0.bytes + (two ? d1.bytes : 0u));
            if (d0.bytes) bulk_g2s(dst, slice + ((unsigned long long)d0.off16 << 4), d0.bytes, bar);
            if (two) bulk_g2s(dst + d0.bytes, slice + ((unsigned long long)d1.off16 << 4), d1.bytes, bar);
        }
        posi += two ? 2 : 1;
    };

    // per-unit state.  qa: B fragments of q (column gq = head gq of the unit's group).
    // acc[i] = O^T tile i: rows gq / gq+8 = channels 16gq + 2i / + 1, columns 2qq, 2qq+1 = heads.
    uint32_t qa[8][2];
    float acc[8][4];
    // heads hA = 2qq, hB = 2qq+1: running max (log2 units) and this lane's share of the sum
    float mA = -INFINITY, mB = -INFINITY, lA = 0.f, lB = 0.f;
    int cur_unit = -1;

    // end of a unit inside this warp's range.  `last` = the call after the main loop: the stages are
    // idle, so the partial may live in this warp's own shared memory (record 2w + 1); a unit that
    // ends inside the range while copies are in flight leaves its partial in global scratch (2w).
    auto flush = [&](bool last) {
        const int u = cur_unit;
        const int a = s_cum[u], b = s_cum[u + 1];
#pragma unroll
        for (int o = 4; o < 32; o <<= 1) {
            lA += __shfl_xor_sync(kFull, lA, o);
            lB += __shfl_xor_sync(kFull, lB, o);
        }
        const int hA = 2 * qq, hB = 2 * qq + 1;
        if (lo <= a && b <= hi) {  // the whole unit was processed by this warp: final result
            const int bi = u / g.n_kv_heads, hk = u % g.n_kv_heads;
            const size_t row = (size_t)bi * g.n_q_heads + (size_t)hk * G;
            const float iA = lA > 0.f ? 1.f / lA : 0.f, iB = lB > 0.f ? 1.f / lB : 0.f;
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                const int ch = 16 * gq + 2 * i;
                if (hA < G) *reinterpret_cast<float2*>(out + (row + hA) * kD + ch) = make_float2(acc[i][0] * iA, acc[i][2] * iA);
                if (hB < G) *reinterpret_cast<float2*>(out + (row + hB) * kD + ch) = make_float2(acc[i][1] * iB, acc[i][3] * iB);
            }
            if (lse != nullptr && gq == 0) {
                if (hA < G) lse[row + hA] = lA > 0.f ? (mA + log2f(lA)) * kLn2 : -INFINITY;
                if (hB < G) lse[row + hB] = lB > 0.f ? (mB + log2f(lB)) * kLn2 : -INFINITY;
            }
        } else {
            const int rec = warp * 2 + (last ? 1 : 0);
            float* po = last ? reinterpret_cast<float*>(wbase) : part_o + (size_t)gw * 2 * (size_t)(G * kD);
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                const int ch = 16 * gq + 2 * i;
                if (hA < G) *reinterpret_cast<float2*>(po + hA * kD + ch) = make_float2(acc[i][0], acc[i][2]);
                if (hB < G) *reinterpret_cast<float2*>(po + hB * kD + ch) = make_float2(acc[i][1], acc[i][3]);
            }
            if (gq == 0) {
                if (hA < G) { s_ml[rec][hA][0] = mA; s_ml[rec][hA][1] = lA; }
                if (hB < G) { s_ml[rec][hB][0] = mB; s_ml[rec][hB][1] = lB; }
            }
            if (lane == 0) { s_unit[rec] = u; s_po[rec] = po; }
        }
    };

    // ---- main loop: consume group k from stage k % NSTAGE, then refill that stage with group k + NSTAGE
#pragma unroll 1
    for (int s = 0; s < NSTAGE; ++s) issue(s);
    int s = 0;
    uint32_t parity = 0u;
#pragma unroll 1
    while (posc < n_total) {
        Desc d0, d1;
        const bool two = group_at(posc, d0, d1);
        const int n = two ? 2 : 1;
        if (d0.unit != cur_unit) {
            if (cur_unit >= 0) flush(false);
            cur_unit = d0.unit;
            const int bi = cur_unit / g.n_kv_heads, hk = cur_unit % g.n_kv_heads;
            // q[head gq][32qq .. 32qq+31]: k-step ks uses channels 32qq + 4ks .. + 3
            const uint4* qrow = reinterpret_cast<const uint4*>(
                q + ((size_t)bi * g.n_q_heads + (size_t)hk * g.group + gq) * kD + 32 * qq);
#pragma unroll
            for (int h = 0; h < 4; ++h) {
                uint4 v = make_uint4(0u, 0u, 0u, 0u);
                if (gq < g.group) v = __ldg(qrow + h);
                qa[2 * h][0] = v.x; qa[2 * h][1] = v.y; qa[2 * h + 1][0] = v.z; qa[2 * h + 1][1] = v.w;
            }
#pragma unroll
            for (int i = 0; i < 8; ++i) acc[i][0] = acc[i][1] = acc[i][2] = acc[i][3] = 0.f;
            mA = mB = -INFINITY;
            lA = lB = 0.f;
        }
        const int r_k = (int)(d0.rr & 255u), r_v = (int)((d0.rr >> 8) & 255u);
        const int nb0 = (int)(d0.rr >> 16), nb1 = two ? (int)(d1.rr >> 16) : 0;
        const uint32_t sp0 = stage0 + s * kStageBytes, sp1 = sp0 + d0.bytes;
        const bool full = nb0 == kB && (n == 1 || nb1 == kB);

        mbar_wait(bar0 + 8 * s, parity);  // the group's bulk copies have landed
#ifdef MKV_DBG_NOMATH
        if (r_k != 1) { __syncwarp(); posc += n; issue(s); if (++s == NSTAGE) { s = 0; parity ^= 1u; } continue; }
#endif

        // ---- QK: S (tokens x heads); rows 0-7 = block 0, rows 8-15 = block 1
        float S[4] = {0.f, 0.f, 0.f, 0.f};
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
            // run of (token gq, word qq): starts after the kept elements of the lower words
            uint32_t w0 = 0u, w1 = 0u, p0, p1, st0 = 2u, st1 = 2u;
            if (r_k == kD) {  // ragged dense block: all slots kept, no bitmap stored
                w0 = gq < nb0 ? 0xffffffffu : 0u;
                w1 = (n == 2 && gq < nb1) ? 0xffffffffu : 0u;
                p0 = sp0 + 256 * gq + 64 * qq;
                p1 = sp1 + 256 * gq + 64 * qq;
            } else {  // values rank-major: rank rho of token t at element rho * nb + t
                if (gq < nb0) w0 = lds_u32(sp0 + 4 * lane);
                if (n == 2 && gq < nb1) w1 = lds_u32(sp1 + 4 * lane);
                uint32_t cnt = (uint32_t)__popc(w0) | ((uint32_t)__popc(w1) << 16), inc = cnt, t;
                t = __shfl_up_sync(kFull, inc, 1); if (qq >= 1) inc += t;
                t = __shfl_up_sync(kFull, inc, 2); if (qq >= 2) inc += t;
                const uint32_t ex = inc - cnt;
                st0 = 2u * nb0; st1 = 2u * nb1;
                p0 = sp0 + 16 * nb0 + st0 * (ex & 0xffffu) + 2 * gq;
                p1 = sp1 + 16 * nb1 + st1 * (ex >> 16) + 2 * gq;
            }
            k_walk_mma<0>(S, w0, w1, p0, p1, st0, st1, qa);
            k_walk_mma<1>(S, w0, w1, p0, p1, st0, st1, qa);
            k_walk_mma<2>(S, w0, w1, p0, p1, st0, st1, qa);
            k_walk_mma<3>(S, w0, w1, p0, p1, st0, st1, qa);
        }

        // ---- online softmax in the exp2 domain; this lane: token gq of each block, heads 2qq, 2qq+1
        const bool v0 = gq < nb0, v1 = n == 2 && gq < nb1;
        const float sA0 = v0 ? S[0] * scale_log2 : -INFINITY, sB0 = v0 ? S[1] * scale_log2 : -INFINITY;
        const float sA1 = v1 ? S[2] * scale_log2 : -INFINITY, sB1 = v1 ? S[3] * scale_log2 : -INFINITY;
        float mxA = fmaxf(sA0, sA1), mxB = fmaxf(sB0, sB1);
#pragma unroll
        for (int o = 4; o < 32; o <<= 1) {
            mxA = fmaxf(mxA, __shfl_xor_sync(kFull, mxA, o));
            mxB = fmaxf(mxB, __shfl_xor_sync(kFull, mxB, o));
        }
        const float mnA = fmaxf(mA, mxA), mnB = fmaxf(mB, mxB);
        const float bA = mnA == -INFINITY ? 0.f : mnA, bB = mnB == -INFINITY ? 0.f : mnB;
        const float cA = ex2(mA - bA), cB = ex2(mB - bB);
        if (__any_sync(kFull, mnA != mA || mnB != mB)) {
#pragma unroll
            for (int i = 0; i < 8; ++i) { acc[i][0] *= cA; acc[i][1] *= cB; acc[i][2] *= cA; acc[i][3] *= cB; }
        }
        mA = mnA; mB = mnB;
        const float eA0 = ex2(sA0 - bA), eB0 = ex2(sB0 - bB), eA1 = ex2(sA1 - bA), eB1 = ex2(sB1 - bB);
        lA = lA * cA + (eA0 + eA1);
        lB = lB * cB + (eB0 + eB1);
        // P split into bf16 hi + lo, transposed into the B fragment layout of PV (k = token, n = head)
        const uint32_t h0 = pack_bf16(eA0, eB0), h1 = pack_bf16(eA1, eB1);
        const uint32_t l0 = pack_bf16(eA0 - __uint_as_float(h0 << 16), eB0 - __uint_as_float(h0 & 0xffff0000u));
        const uint32_t l1 = pack_bf16(eA1 - __uint_as_float(h1 << 16), eB1 - __uint_as_float(h1 & 0xffff0000u));
        const uint32_t ph0 = movmatrix_trans(h0), ph1 = movmatrix_trans(h1);
        const uint32_t pl0 = movmatrix_trans(l0), pl1 = movmatrix_trans(l1);

        // ---- PV: O^T += V^T P^T (channels x heads), K = the group's 16 tokens
        const uint32_t bmk = r_k == kD ? 0u : (uint32_t)kBitmapBytes;
        const uint32_t vb0 = sp0 + nb0 * (bmk + 2 * r_k), vb1 = sp1 + nb1 * (bmk + 2 * r_k);  // V part of each block
        if (r_v == kD && full) {
            const uint32_t rA0 = vb0 + 256 * (2 * qq) + 32 * gq, rA1 = vb1 + 256 * (2 * qq) + 32 * gq;
#pragma unroll
            for (int h = 0; h < 2; ++h) {  // 16-byte chunk h = channel slots 8h .. 8h+7 = tiles 4h .. 4h+3
                const uint4 xa = lds_128(rA0 + 16 * h), xb = lds_128(rA0 + 256 + 16 * h);
                uint4 ya = make_uint4(0u, 0u, 0u, 0u), yb = ya;
                if (n == 2) { ya = lds_128(rA1 + 16 * h); yb = lds_128(rA1 + 256 + 16 * h); }
                const uint32_t xav[4] = {xa.x, xa.y, xa.z, xa.w}, xbv[4] = {xb.x, xb.y, xb.z, xb.w};
                const uint32_t yav[4] = {ya.x, ya.y, ya.z, ya.w}, ybv[4] = {yb.x, yb.y, yb.z, yb.w};
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    const uint32_t a0 = prmt(xav[j], xbv[j], 0x5410u), a1 = prmt(xav[j], xbv[j], 0x7632u);
                    const uint32_t a2 = prmt(yav[j], ybv[j], 0x5410u), a3 = prmt(yav[j], ybv[j], 0x7632u);
                    mma_bf16(acc[4 * h + j], a0, a1, a2, a3, ph0, ph1);
                    mma_bf16(acc[4 * h + j], a0, a1, a2, a3, pl0, pl1);
                }
            }
        } else {
            const int tA = 2 * qq, tB = 2 * qq + 1;
            uint32_t hA0 = 0u, hB0 = 0u, hA1 = 0u, hB1 = 0u, pA0, pB0, pA1, pB1, st0 = 2u, st1 = 2u;
            if (r_v == kD) {  // ragged dense block
                hA0 = tA < nb0 ? 0xffffu : 0u; hB0 = tB < nb0 ? 0xffffu : 0u;
                hA1 = (n == 2 && tA < nb1) ? 0xffffu : 0u; hB1 = (n == 2 && tB < nb1) ? 0xffffu : 0u;
                pA0 = vb0 + 256 * tA + 32 * gq; pB0 = pA0 + 256;
                pA1 = vb1 + 256 * tA + 32 * gq; pB1 = pA1 + 256;
            } else {
                if (tA < nb0) hA0 = lds_u16(vb0 + 16 * tA + 2 * gq);
                if (tB < nb0) hB0 = lds_u16(vb0 + 16 * tB + 2 * gq);
                if (n == 2 && tA < nb1) hA1 = lds_u16(vb1 + 16 * tA + 2 * gq);
                if (n == 2 && tB < nb1) hB1 = lds_u16(vb1 + 16 * tB + 2 * gq);
                // exclusive prefix over the lower half-words (lanes gq' < gq, stride 4); four byte counters
                const uint32_t cnt = (uint32_t)__popc(hA0) | ((uint32_t)__popc(hB0) << 8) |
                                     ((uint32_t)__popc(hA1) << 16) | ((uint32_t)__popc(hB1) << 24);
                uint32_t inc = cnt, t;
                t = __shfl_up_sync(kFull, inc, 4); if (gq >= 1) inc += t;
                t = __shfl_up_sync(kFull, inc, 8); if (gq >= 2) inc += t;
                t = __shfl_up_sync(kFull, inc, 16); if (gq >= 4) inc += t;
                const uint32_t ex = inc - cnt;
                st0 = 2u * nb0; st1 = 2u * nb1;
                pA0 = vb0 + 16 * nb0 + st0 * (ex & 255u) + 2 * tA;
                pB0 = vb0 + 16 * nb0 + st0 * ((ex >> 8) & 255u) + 2 * tB;
                pA1 = vb1 + 16 * nb1 + st1 * ((ex >> 16) & 255u) + 2 * tA;
                pB1 = vb1 + 16 * nb1 + st1 * (ex >> 24) + 2 * tB;
            }
            v_walk_mma<0>(acc, hA0, hB0, hA1, hB1, pA0, pB0, pA1, pB1, st0, st1, ph0, ph1, pl0, pl1);
            v_walk_mma<1>(acc, hA0, hB0, hA1, hB1, pA0, pB0, pA1, pB1, st0, st1, ph0, ph1, pl0, pl1);
        }
        __syncwarp();  // every lane is done reading stage s
        posc += n;
        issue(s);      // stage s is free: start the copies of group k + NSTAGE
        if (++s == NSTAGE) { s = 0; parity ^= 1u; }
    }
#ifdef MKV_DBG_TIMING
    if (lane == 0) { atomicMin(&g_dbg_t[blockIdx.x * 8 + 5], dbg_now()); atomicMax(&g_dbg_t[blockIdx.x * 8 + 6], dbg_now()); }
#endif
    if (cur_unit >= 0) flush(true);  // every issued group was consumed: the stages are idle

    // ---- step 3d, fused: fold the warps' partials; finish units that span several CTAs.
    // Records are in warp order (2w = head, 2w + 1 = tail), hence in non-decreasing unit order: the
    // partials of one unit form a run.  Thread tid owns output elements e = tid + j kNT of [G][D]
    // and folds a run with the LSE rule (pinned by oracle pin P10).
    __syncthreads();  // orders the warps' partials (shared memory, or global scratch from flush(false))
    MKV_T(1);
    constexpr int kEPT = (kMaxGroup * kD + kNT - 1) / kNT;
    const int clo = s_clo, chi = s_chi, GD = G * kD;
    const size_t cta_slot_base = (size_t)gridDim.x * kMaxWarps * 2;
    const int tid = threadIdx.x;
    int sh_u[2] = {-1, -1};  // units this CTA shares with others (<= 2: one entering, one leaving its range)
    int n_shared = 0;
    float M[kEPT], L[kEPT], O[kEPT];
    int run = -1;
#pragma unroll 1
    for (int r = 0; r <= kRec; ++r) {
        const int u = r < kRec ? s_unit[r] : -2;  // -2: sentinel that closes the last run
        if (u == -1) continue;
        if (u != run) {
            if (run >= 0) {  // close the run: final result, or this CTA's partial of a shared unit
                const int a = s_cum[run], b = s_cum[run + 1];
                const bool whole = clo <= a && b <= chi;
                const size_t row = (size_t)(run / g.n_kv_heads) * g.n_q_heads + (size_t)(run % g.n_kv_heads) * G;
                const size_t slot = cta_slot_base + blockIdx.x * 2 + (a < clo ? 0 : 1);
#pragma unroll
                for (int j = 0; j < kEPT; ++j) {
                    const int e = tid + j * kNT;
                    if (e >= GD) continue;
                    const int h = e >> 7;
                    if (whole) {
                        out[row * kD + e] = L[j] > 0.f ? O[j] / L[j] : 0.f;
                        if (lse != nullptr && (e & (kD - 1)) == 0)
                            lse[row + h] = L[j] > 0.f ? (M[j] + log2f(L[j])) * kLn2 : -INFINITY;
                    } else {
                        part_o[slot * GD + e] = O[j];
                        if ((e & (kD - 1)) == 0) {
                            part_ml[slot * (2 * kMaxGroup) + 2 * h] = M[j];
                            part_ml[slot * (2 * kMaxGroup) + 2 * h + 1] = L[j];
                        }
                    }
                }
                if (!whole && n_shared < 2) {
                    if (tid == 0) s_row[n_shared] = row;
                    sh_u[n_shared++] = run;
                }
            }
            if (u == -2) break;
            run = u;
#pragma unroll
            for (int j = 0; j < kEPT; ++j) { M[j] = -INFINITY; L[j] = 0.f; O[j] = 0.f; }
        }
        const float* po = s_po[r];
#pragma unroll
        for (int j = 0; j < kEPT; ++j) {
            const int e = tid + j * kNT;
            if (e >= GD) continue;
            const int h = e >> 7;
            const float m = s_ml[r][h][0], l = s_ml[r][h][1], o = po[e];
            const float Mn = fmaxf(M[j], m), Mb = Mn == -INFINITY ? 0.f : Mn;
            const float c = ex2(M[j] - Mb), w = ex2(m - Mb);
            L[j] = fmaf(l, w, L[j] * c);
            O[j] = fmaf(o, w, O[j] * c);
            M[j] = Mn;
        }
    }
    MKV_T(2);
    if (n_shared == 0) return;  // uniform over the CTA

    // CTA c owns block x  <=>  c T < (x+1) Gd <= (c+1) T.  Every thread releases its part of the CTA's
    // partial (fence, then the barrier); one thread per shared unit finds the sharers c_first .. c_last
    // (all non-empty: T >= Gd) and takes a ticket.  A sharer's slot is 1 for c_first (the unit starts
    // inside it), else 0.
    __threadfence();
    __syncthreads();
    if ((tid == 0 || tid == 32) && (tid >> 5) < n_shared) {
        const int k = tid >> 5, u = sh_u[k];
        const float inv_T = 1.f / (float)T;
        int cf = (int)blockIdx.x, cl = (int)blockIdx.x;
        if (s_cum[u] < clo) cf = (int)div_floor((unsigned long long)(s_cum[u] + 1) * Gd - 1, (unsigned)T, inv_T);
        if (s_cum[u + 1] > chi) cl = (int)div_floor((unsigned long long)s_cum[u + 1] * Gd - 1, (unsigned)T, inv_T);
        s_cf[k] = cf; s_cl[k] = cl;
        const int old = atomicAdd(&ticket[u], 1);
        s_last[k] = old == cl - cf;
        if (old == cl - cf) ticket[u] = 0;  // self-cleaning: every sharer has arrived
    }
    __syncthreads();
    MKV_T(3);
#pragma unroll 1
    for (int k = 0; k < n_shared; ++k) {
        if (!s_last[k]) continue;  // uniform over the CTA
        // last arriver: merge the CTA partials (acquire fence; read with ld.global.cg: L2, never a stale L1 line)
        __threadfence();
        const int c_first = s_cf[k], c_last = s_cl[k];
        const size_t row = s_row[k];
#pragma unroll 1
        for (int e = tid; e < GD; e += kNT) {
            const int h = e >> 7;
            float Mx = -INFINITY, Lx = 0.f, Ox = 0.f;
#pragma unroll 1
            for (int c0 = c_first; c0 <= c_last; c0 += 4) {  // four partials' loads in flight at once
                float pm[4], pl[4], po[4];
#pragma unroll
                for (int t = 0; t < 4; ++t) {
                    const int c = c0 + t;
                    pm[t] = -INFINITY; pl[t] = 0.f; po[t] = 0.f;
                    if (c <= c_last) {
                        const size_t sl = cta_slot_base + (size_t)c * 2 + (c == c_first ? 1 : 0);
                        pm[t] = __ldcg(part_ml + sl * (2 * kMaxGroup) + 2 * h);
                        pl[t] = __ldcg(part_ml + sl * (2 * kMaxGroup) + 2 * h + 1);
                        po[t] = __ldcg(part_o + sl * (size_t)GD + e);
                    }
                }
                const float Mn = fmaxf(fmaxf(Mx, fmaxf(pm[0], pm[1])), fmaxf(pm[2], pm[3]));
                const float Mb = Mn == -INFINITY ? 0.f : Mn;
                const float c_old = ex2(Mx - Mb);
                Lx *= c_old; Ox *= c_old; Mx = Mn;
#pragma unroll
                for (int t = 0; t < 4; ++t) {
                    const float w = ex2(pm[t] - Mb);
                    Lx = fmaf(pl[t], w, Lx);
                    Ox = fmaf(po[t], w, Ox);
                }
            }
            out[row * kD + e] = Lx > 0.f ? Ox / Lx : 0.f;
            if (lse != nullptr && (e & (kD - 1)) == 0) lse[row + h] = Lx > 0.f ? (Mx + log2f(Lx)) * kLn2 : -INFINITY;
        }
    }
    MKV_T(4);
}

}  // namespace

#ifdef MKV_DBG_TIMING
extern "C" __attribute__((visibility("default"))) int mkv_dbg_timing(unsigned long long* host, int reset) {
    if (reset) { static unsigned long long init[160 * 8]; for (int i = 0; i < 160 * 8; ++i) init[i] = (i % 8 == 5) ? ~0ull : 0ull; return (int)cudaMemcpyToSymbol(g_dbg_t, init, sizeof(init)); }
    return (int)cudaMemcpyFromSymbol(host, g_dbg_t, sizeof(unsigned long long) * 160 * 8);
}
#endif

int attention_partial_slots(int sm_count) { return sm_count * kMaxWarps * 2 + sm_count * 2; }

template <int NSTAGE, int NWARPS>
static cudaError_t launch_attention_cfg(const CacheGeom& g, const LayerView& lv, const uint16_t* q, const int32_t* sel,
                                        const int32_t* sel_count, int k_max, float scale, float* out, float* lse,
                                        const AttnScratch& scr, int sm_count, cudaStream_t s) {
    const int smem = NWARPS * warp_smem_bytes(NSTAGE) + (g.n_units + 1) * 4;
    static int configured = 0;  // largest dynamic shared-memory size opted into so far
    if (smem > configured) {
        cudaError_t e = cudaFuncSetAttribute(mkv_packed_attention_kernel<NSTAGE, NWARPS>,
                                             cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
        if (e != cudaSuccess) return e;
        configured = smem;
    }
    mkv_packed_attention_kernel<NSTAGE, NWARPS><<<sm_count, NWARPS * 32, smem, s>>>(
        g, lv, q, sel, sel_count, k_max, scale * kLog2e, out, lse, scr.part_o, scr.part_ml, scr.ticket);
    return cudaGetLastError();
}

cudaError_t launch_attention(const CacheGeom& g, const LayerView& lv, const uint16_t* q, const int32_t* sel,
                             const int32_t* sel_count, int k_max, float scale, float* out, float* lse,
                             const AttnScratch& scr, int sm_count, cudaStream_t s, int* n_kernels) {
    if (g.n_units > kMaxUnitsSmem) return cudaErrorInvalidValue;
    if (n_kernels) *n_kernels = 1;
    static int cfg = -1;  // tuning knob (stages * 100 + warps); default chosen from measurements
    if (cfg < 0) {
        const char* e = getenv("MKV_ATTN_CFG");
        cfg = e ? atoi(e) : 316;
    }
#define MKV_CFG(S, W) \
    case S * 100 + W: return launch_attention_cfg<S, W>(g, lv, q, sel, sel_count, k_max, scale, out, lse, scr, sm_count, s);
    switch (cfg) {
        MKV_CFG(3, 16) MKV_CFG(2, 16) MKV_CFG(4, 12) MKV_CFG(3, 12) MKV_CFG(4, 8) MKV_CFG(6, 8)
        default: return launch_attention_cfg<3, 16>(g, lv, q, sel, sel_count, k_max, scale, out, lse, scr, sm_count, s);
    }
#undef MKV_CFG
}

}  // namespace mkv
