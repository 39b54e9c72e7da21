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
//     written directly; otherwise the warp leaves a (ref, l, O) partial (<= 2 per warp), the
//     threads of the CTA fold the partials of a unit (four output channels each, straight-line
//     code) with the LSE rule, and a unit that spans several CTAs is finished by the last CTA to
//     arrive at a per-unit ticket (no second kernel).
//   * Softmax is lazy: 2^(s - ref) with a reference that moves only when a score exceeds it by
//     more than 60 (log2 units); the common group needs no max reduction and no rescale.
#include <cstdlib>

#include "mkv_internal.cuh"
#include "mkv_walk.cuh"

namespace mkv {

#ifdef MKV_DBG_TIMING
__device__ unsigned long long g_dbg_t[160 * 16];
__device__ __forceinline__ unsigned long long dbg_now() { unsigned long long t; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t)); return t; }
#define MKV_T(k) do { if (threadIdx.x == 0) g_dbg_t[blockIdx.x * 16 + (k)] = dbg_now(); } while (0)
#define MKV_TV(k, v) do { if (threadIdx.x == 0 && (v) != -12345) g_dbg_t[blockIdx.x * 16 + (k)] = dbg_now(); } while (0)
#else
#define MKV_T(k) do {} while (0)
#define MKV_TV(k, v) do {} while (0)
#endif

namespace {

using namespace walk;
constexpr float kLog2e = 1.4426950408889634f;
constexpr float kLn2 = 0.6931471805599453f;

constexpr int kMaxWarps = 24;      // upper bound on warps per CTA (sizes the partial-slot scratch)
constexpr int kStageBytes = 4096;  // one dense block (4096 B) or two packed blocks with r <= 56
constexpr int kDescRing = 64;      // block descriptors kept per warp
constexpr int kMaxUnitsSmem = 2048;
// A group of the KV update buffer: nb0 <= 8 uncompressed recent tokens, attended as one dense
// block; off0 / off1 are its K rows / V rows in the buffer arrays (two chunks, staged back to back).
constexpr uint32_t kUpdFlag = 1u << 26;

// One group of the stream: <= 2 consecutive selected token blocks of one unit with the same
// strategy that fit one stage (16 tokens = the M of one mma tile).
struct __align__(16) GDesc {
    uint32_t off0, off1;  // payload offsets in the layer slice, 16-B units
    uint32_t z;           // bytes0 / 16 | bytes1 / 16 << 9 | nb0 << 18 | nb1 << 22 | kUpdFlag   (bytes 0: invalid entry)
    uint32_t w;           // unit | r_k << 16 | r_v << 24
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

// prefix sums of the clamped selection counts -> s_cum[0..n_units]; returns the total T
__device__ __forceinline__ int scan_counts(const int32_t* __restrict__ sel_count, int n_units, int k_max, int extra,
                                            int* s_cum) {
    __shared__ int s_carry;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (warp == 0) {
        int carry = 0;
#pragma unroll 1
        for (int i0 = 0; i0 < n_units; i0 += 32) {
            const int i = i0 + lane;
            int c = (i < n_units) ? min(max(sel_count[i], 0), k_max) + extra : 0;  // + blocks of the update buffer
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
#pragma unroll 1
    while (hi - lo > 1) {
        const int mid = (lo + hi) >> 1;
        if (s_cum[mid] <= i) lo = mid; else hi = mid;
    }
    return lo;
}

// per warp: the stages, the group-descriptor ring, one mbarrier per stage (64 B reserved)
__host__ __device__ constexpr int warp_smem_bytes(int nstage) { return nstage * kStageBytes + kDescRing * 16 + 64; }

// Even split of n items over p parts: part i owns [i b + min(i, r), ...) with b = n / p, r = n % p
// (the first r parts hold one more).  One runtime division per level.
struct Split {
    unsigned b, r;
    __device__ __forceinline__ unsigned begin(unsigned i) const { return i * b + min(i, r); }
    // the part that owns item x (x < n)
    __device__ __forceinline__ unsigned owner(unsigned x) const {
        const unsigned big = r * (b + 1);
        return x < big ? x / (b + 1) : r + (x - big) / b;
    }
};

// ------------------------------------------------------------------------------------------
// main kernel: one CTA per SM, kWarps independent warps.  The T selected blocks are split evenly
// over the CTAs, a CTA's range evenly over its warps; every warp owns one contiguous range.
// ------------------------------------------------------------------------------------------
// kGatherOnly: calibration build of the same kernel (mkv_calibrate_gather): every selected payload is staged
// exactly as in the real run, one word per lane and group is read back, and all arithmetic is skipped.
template <int NSTAGE, int kWarps, bool kGatherOnly>
__global__ void __launch_bounds__(kWarps * 32, 1)
mkv_packed_attention_kernel(CacheGeom g, LayerView lv, const uint16_t* __restrict__ q,
                            const int32_t* __restrict__ sel, const int32_t* __restrict__ sel_count, int k_max,
                            float scale_log2, float* __restrict__ out, float* __restrict__ lse,
                            float* __restrict__ part_o, float* __restrict__ part_ml, int32_t* __restrict__ ticket,
                            const uint16_t* __restrict__ upd_k, const uint16_t* __restrict__ upd_v,
                            const int32_t* __restrict__ upd_count) {
    extern __shared__ __align__(128) uint8_t smem[];
    constexpr int kWS = warp_smem_bytes(NSTAGE);
    constexpr int kNT = kWarps * 32;
    constexpr int kRec = 2 * kWarps;  // partial records of the CTA: warp w -> 2w (head), 2w + 1 (tail)
    int* s_cum = reinterpret_cast<int*>(smem + kWarps * kWS);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int gq = lane >> 2, qq = lane & 3;  // mma fragment coordinates (groupID, threadID_in_group)

    MKV_T(0);
    __shared__ int s_unit[kRec];                 // unit of each partial record, -1 = none
    __shared__ __align__(8) float s_ml[kRec][kMaxGroup][2];   // its (max in log2 units, sum) per head
    __shared__ int s_last[2], s_cf[2], s_cl[2];
    __shared__ size_t s_row[2];

    uint8_t* wbase = smem + warp * kWS;
    const uint32_t stage0 = smem_u32(wbase);
    GDesc* ring = reinterpret_cast<GDesc*>(wbase + NSTAGE * kStageBytes);
    const uint32_t bar0 = stage0 + NSTAGE * kStageBytes + kDescRing * 16;
    if (lane == 0) {
#pragma unroll
        for (int s = 0; s < NSTAGE; ++s) mbar_init(bar0 + 8 * s, 1);
        mbar_init_fence();
    }
    if (lane < 2) s_unit[warp * 2 + lane] = -1;
    pdl_wait();               // the producer of sel / sel_count / the cache (and the previous user of the scratch) is done
    pdl_launch_dependents();  // the next kernel may be scheduled as SMs free up

    // tokens in the layer's update buffer: device-resident, so a captured graph stays valid across appends
    const int n_buf = min(max(*upd_count, 0), g.L);
    const int upd_blocks = (n_buf + kB - 1) / kB;  // every unit ends with the blocks of its update buffer
    const int T = scan_counts(sel_count, g.n_units, k_max, upd_blocks, s_cum);  // (block barrier inside)
    // The stream is split in units of two positions, so every range starts at an even position: with even
    // selection counts (units then start at even positions too) a range never holds two odd runs, which
    // would cost an extra half-empty group -- the slowest warp sets the kernel's time.
    const unsigned P = ((unsigned)T + 1u) >> 1;                     // position pairs
    const unsigned Gd = min(gridDim.x, max(P, 1u));                 // CTAs that own >= 1 pair
    Split cs;                                                       // pairs over CTAs
    cs.b = P / Gd; cs.r = P - cs.b * Gd;
    int clo = 0, chi = 0;
    unsigned cplo = 0, cphi = 0;
    if (blockIdx.x < Gd) { cplo = cs.begin(blockIdx.x); cphi = cs.begin(blockIdx.x + 1); }
    clo = (int)(2u * cplo); chi = min((int)(2u * cphi), T);
    Split ws;                                                       // the CTA's pairs over its warps
    ws.b = (cphi - cplo) / kWarps; ws.r = (cphi - cplo) % kWarps;
    const int lo = min(clo + 2 * (int)ws.begin(warp), chi), hi = min(clo + 2 * (int)ws.begin(warp + 1), chi);
    const unsigned gw = blockIdx.x * kWarps + warp;
    const int n_total = hi - lo;
    const int G = g.group;
    if (blockIdx.x == 0) {  // units with an empty selection: out = 0, lse = -inf
#pragma unroll 1
        for (int u = warp; u < g.n_units; u += kWarps) {
            if (s_cum[u + 1] != s_cum[u]) continue;
            const size_t row = (size_t)(u / g.n_kv_heads) * g.n_q_heads + (size_t)(u % g.n_kv_heads) * G;
#pragma unroll 1
            for (int e = lane; e < G * kD; e += 32) out[row * kD + e] = 0.f;
            if (lse != nullptr && lane < G) lse[row + lane] = -INFINITY;
        }
    }

    int bposc = 0, bposi = 0, bbuilt = 0;  // blocks consumed / issued / described
    int gposc = 0, gposi = 0, gbuilt = 0;  // groups consumed / issued / described

    // Describe the next <= 32 blocks of the range (one per lane) and pair them into groups: block i
    // follows block i - 1 in a group if both belong to one unit, have the same strategy and fit one
    // stage together; runs of such blocks are paired greedily from their start.
    auto build = [&](int count) {
        uint32_t off16 = 0u, bytes = 0u, rr = 0u, nb = 0u;
        int u = -1;
        if (lane < count) {
            const int gi = lo + bbuilt + lane;
            u = find_unit(s_cum, g.n_units, gi);
            const int j = gi - s_cum[u], jb = j - (s_cum[u + 1] - s_cum[u] - upd_blocks);
            if (jb >= 0) {  // block jb of the unit's update buffer: raw rows [u][8 jb ..][128] of upd_k / upd_v
                nb = (uint32_t)min(kB, n_buf - kB * jb);
                off16 = (uint32_t)(((size_t)u * g.L + (size_t)kB * jb) * (kD * 2 / 16));
                bytes = nb * (uint32_t)(kD * 2);
                rr = (uint32_t)kD | ((uint32_t)kD << 8) | 0x10000u;  // bit 16: update-buffer block
            }
            const int t0 = jb >= 0 ? -1 : sel[(size_t)u * k_max + j];
            const int ntok = lv.unit_ntok[u];
            if (t0 >= 0 && t0 < ntok && (t0 & (kB - 1)) == 0) {
                const int seg = t0 / g.L, in_seg = t0 - seg * g.L;
                const size_t e = (size_t)u * lv.S_max + seg;
                const StratRec rec = lv.strat[e];
                nb = (uint32_t)min(kB, (int)rec.n_tok - in_seg);
                off16 = lv.tok_off[e] + (uint32_t)(in_seg >> 3) * (tokblock_bytes(rec.r_k, rec.r_v, kB) >> 4);
                bytes = tokblock_bytes(rec.r_k, rec.r_v, (int)nb);
                rr = (uint32_t)rec.r_k | ((uint32_t)rec.r_v << 8);
            }
        }
        const int pu = __shfl_up_sync(kFull, u, 1);
        const uint32_t prr = __shfl_up_sync(kFull, rr, 1), pbytes = __shfl_up_sync(kFull, bytes, 1);
        const bool follows = lane > 0 && lane < count && u == pu && rr == prr && bytes != 0u && pbytes != 0u &&
                             bytes + pbytes <= (uint32_t)kStageBytes && !(rr & 0x10000u);
        const unsigned fm = __ballot_sync(kFull, follows);
        const int start = 31 - __clz((int)(~fm & lanemask_le()));  // first block of this lane's run (bit 0 of ~fm is set)
        const bool first = lane < count && ((lane - start) & 1) == 0;
        const bool two = first && ((fm >> 1) >> lane & 1u);        // lane + 1 follows (and is therefore < count)
        const unsigned gm = __ballot_sync(kFull, first);
        const uint32_t off1 = __shfl_down_sync(kFull, off16, 1), bytes1 = __shfl_down_sync(kFull, bytes, 1);
        const uint32_t nb1 = __shfl_down_sync(kFull, nb, 1);
        if (first) {
            GDesc d;
            d.off0 = off16; d.off1 = two ? off1 : 0u;
            d.z = (bytes >> 4) | ((two ? bytes1 >> 4 : 0u) << 9) | (nb << 18) | ((two ? nb1 : 0u) << 22);
            if (rr & 0x10000u) {  // K rows and V rows: two chunks of the same size at the same offset
                d.off1 = off16;
                d.z |= ((bytes >> 4) << 9) | kUpdFlag;
            }
            d.w = (uint32_t)u | ((rr & 0xffffu) << 16);
            ring[(gbuilt + __popc(gm & lanemask_lt())) & (kDescRing - 1)] = d;
        }
        gbuilt += __popc(gm);
        bbuilt += count;
        __syncwarp();
    };

    // start the copies of the next group into stage s: one bulk copy per block, issued by lane 0,
    // completing on the stage's mbarrier
    const unsigned long long slice = reinterpret_cast<unsigned long long>(lv.slice);
    auto issue = [&](int s) {
        if (bposi >= n_total) return;
        if (gposi == gbuilt) build(min(32, n_total - bbuilt));
        const GDesc d = ring[gposi & (kDescRing - 1)];
        const uint32_t b0 = (d.z & 511u) << 4, b1 = ((d.z >> 9) & 511u) << 4;
        if (lane == 0) {
            const uint32_t bar = bar0 + 8 * s, dst = stage0 + s * kStageBytes;
            const bool upd = d.z & kUpdFlag;
            const unsigned long long src0 = upd ? reinterpret_cast<unsigned long long>(upd_k) : slice;
            const unsigned long long src1 = upd ? reinterpret_cast<unsigned long long>(upd_v) : slice;
            mbar_expect_tx(bar, b0 + b1);
            if (b0) bulk_g2s(dst, src0 + ((unsigned long long)d.off0 << 4), b0, bar);
            if (b1) bulk_g2s(dst + b0, src1 + ((unsigned long long)d.off1 << 4), b1, bar);
        }
        ++gposi;
        bposi += (b1 && !(d.z & kUpdFlag)) ? 2 : 1;
    };

    // per-unit state.  qa: B fragments of q (column gq = head gq of the unit's group).
    // acc[i] = O^T tile i: rows gq / gq+8 = channels 16gq + 2i / + 1, columns 2qq, 2qq+1 = heads.
    uint32_t qa[8][2];
    float acc[8][4];
    // heads hA = 2qq, hB = 2qq+1: reference exponent (log2 units; -inf = not set yet) and this lane's
    // share of the sum.  Softmax is LAZY: probabilities are 2^(s - ref) with a reference that only
    // moves when a score exceeds it by more than kRefSlack, so the common group needs no max
    // reduction and no rescale of the accumulators (fp32 has the exponent range to spare).
    constexpr float kRefSlack = 60.f;
    float mA = -INFINITY, mB = -INFINITY, lA = 0.f, lB = 0.f;
    int cur_unit = -1;

    // end of a unit inside this warp's range.  `last`: the range is finished and the stages are
    // idle, so the partial lives in this warp's own shared memory (record 2w + 1); a unit that
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
        const bool whole = lo <= a && b <= hi;  // the whole unit was processed by this warp: final result
        float fA = 1.f, fB = 1.f;
        float* po;
        if (whole) {
            po = out + ((size_t)(u / g.n_kv_heads) * g.n_q_heads + (size_t)(u % g.n_kv_heads) * G) * kD;
            fA = lA > 0.f ? 1.f / lA : 0.f;
            fB = lB > 0.f ? 1.f / lB : 0.f;
        } else {
            po = last ? reinterpret_cast<float*>(wbase) : part_o + (size_t)gw * 2 * (size_t)(G * kD);
        }
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            const int ch = 16 * gq + 2 * i;
            if (hA < G) *reinterpret_cast<float2*>(po + hA * kD + ch) = make_float2(acc[i][0] * fA, acc[i][2] * fA);
            if (hB < G) *reinterpret_cast<float2*>(po + hB * kD + ch) = make_float2(acc[i][1] * fB, acc[i][3] * fB);
        }
        if (whole) {
            if (lse != nullptr && gq == 0) {
                float* pl = lse + (size_t)(u / g.n_kv_heads) * g.n_q_heads + (size_t)(u % g.n_kv_heads) * G;
                if (hA < G) pl[hA] = lA > 0.f ? (mA + log2f(lA)) * kLn2 : -INFINITY;
                if (hB < G) pl[hB] = lB > 0.f ? (mB + log2f(lB)) * kLn2 : -INFINITY;
            }
        } else {
            const int rec = warp * 2 + (last ? 1 : 0);
            if (gq == 0) {
                if (hA < G) { s_ml[rec][hA][0] = mA; s_ml[rec][hA][1] = lA; }
                if (hB < G) { s_ml[rec][hB][0] = mB; s_ml[rec][hB][1] = lB; }
            }
            if (lane == 0) s_unit[rec] = u;
        }
    };

    // ---- main loop.  Iteration k >= 0 consumes group k from stage k % NSTAGE and refills that stage
    // with group k + NSTAGE; iterations k < 0 only fill the pipeline.  One call site each for
    // issue() and flush(): code executed once costs ~4 cycles per instruction (instruction fetch).
    int s = 0;
    uint32_t parity = 0u, calib = 0u;
#pragma unroll 1
    for (int k = -NSTAGE;; ++k) {
        if (k >= 0) {
            const bool end = bposc >= n_total;
            GDesc d;
            d.off0 = d.off1 = d.z = 0u; d.w = 0xffffu;
            if (!end) d = ring[gposc & (kDescRing - 1)];
            if (kGatherOnly) {
                if (end) break;
                mbar_wait(bar0 + 8 * s, parity);
                calib ^= lds_u32(stage0 + s * kStageBytes + 4 * lane);
                __syncwarp();
                bposc += ((d.z >> 22) & 15u) ? 2 : 1;
                ++gposc;
                issue(s);
                if (++s == NSTAGE) { s = 0; parity ^= 1u; }
                continue;
            }
            const int u = end ? -1 : (int)(d.w & 0xffffu);
            if (u != cur_unit) {
                if (cur_unit >= 0) flush(end);
                if (end) break;
                cur_unit = u;
                const int bi = u / g.n_kv_heads, hk = u % g.n_kv_heads;
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
            } else if (end) {
                break;  // empty range
            }
            const int r_k = (int)((d.w >> 16) & 255u), r_v = (int)(d.w >> 24);
            const int nb0 = (int)((d.z >> 18) & 15u), nb1 = (int)((d.z >> 22) & 15u);
            const uint32_t sp0 = stage0 + s * kStageBytes, sp1 = sp0 + ((d.z & 511u) << 4);
            const bool two = nb1 != 0;
            const bool full = nb0 == kB && (!two || nb1 == kB);

            mbar_wait(bar0 + 8 * s, parity);  // the group's bulk copies have landed

            // ---- QK: S (tokens x heads); rows 0-7 = block 0, rows 8-15 = block 1
            float S[4] = {0.f, 0.f, 0.f, 0.f};
            if (r_k == kD && full) {
                const uint32_t a0 = sp0 + 256 * gq + 64 * qq, a1 = sp1 + 256 * gq + 64 * qq;
#pragma unroll
                for (int h = 0; h < 4; ++h) {
                    const uint4 x = lds_128(a0 + 16 * h);
                    uint4 y = make_uint4(0u, 0u, 0u, 0u);
                    if (two) y = lds_128(a1 + 16 * h);
                    mma_bf16(S, x.x, y.x, x.y, y.y, qa[2 * h][0], qa[2 * h][1]);
                    mma_bf16(S, x.z, y.z, x.w, y.w, qa[2 * h + 1][0], qa[2 * h + 1][1]);
                }
            } else {
                // run of (token gq, word qq): starts after the kept elements of the lower words
                uint32_t w0 = 0u, w1 = 0u, p0, p1, st0 = 2u, st1 = 2u;
                if (r_k == kD) {  // ragged dense block: all slots kept, no bitmap stored
                    w0 = gq < nb0 ? 0xffffffffu : 0u;
                    w1 = gq < nb1 ? 0xffffffffu : 0u;
                    p0 = sp0 + 256 * gq + 64 * qq;
                    p1 = sp1 + 256 * gq + 64 * qq;
                } else {  // values rank-major: rank rho of token t at element rho * nb + t
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
                k_walk_mma<0>(S, w0, w1, p0, p1, st0, st1, qa);
                k_walk_mma<1>(S, w0, w1, p0, p1, st0, st1, qa);
                k_walk_mma<2>(S, w0, w1, p0, p1, st0, st1, qa);
                k_walk_mma<3>(S, w0, w1, p0, p1, st0, st1, qa);
            }

            // ---- lazy softmax in the exp2 domain; this lane: token gq of each block, heads 2qq, 2qq+1
            const bool v0 = gq < nb0, v1 = gq < nb1;
            const float sA0 = v0 ? S[0] * scale_log2 : -INFINITY, sB0 = v0 ? S[1] * scale_log2 : -INFINITY;
            const float sA1 = v1 ? S[2] * scale_log2 : -INFINITY, sB1 = v1 ? S[3] * scale_log2 : -INFINITY;
            float mxA = fmaxf(sA0, sA1), mxB = fmaxf(sB0, sB1);
            if (__any_sync(kFull, mxA > mA + kRefSlack || mxB > mB + kRefSlack)) {
                // move the reference (always taken by the first group of a unit: ref = -inf)
#pragma unroll
                for (int o = 4; o < 32; o <<= 1) {
                    mxA = fmaxf(mxA, __shfl_xor_sync(kFull, mxA, o));
                    mxB = fmaxf(mxB, __shfl_xor_sync(kFull, mxB, o));
                }
                const float mnA = fmaxf(mA, mxA), mnB = fmaxf(mB, mxB);
                const float cA = ex2(mA - (mnA == -INFINITY ? 0.f : mnA)), cB = ex2(mB - (mnB == -INFINITY ? 0.f : mnB));
#pragma unroll
                for (int i = 0; i < 8; ++i) { acc[i][0] *= cA; acc[i][1] *= cB; acc[i][2] *= cA; acc[i][3] *= cB; }
                lA *= cA; lB *= cB;
                mA = mnA; mB = mnB;
            }
            const float bA = mA == -INFINITY ? 0.f : mA, bB = mB == -INFINITY ? 0.f : mB;
            const float eA0 = ex2(sA0 - bA), eB0 = ex2(sB0 - bB), eA1 = ex2(sA1 - bA), eB1 = ex2(sB1 - bB);
            lA += eA0 + eA1;
            lB += eB0 + eB1;
            // P split into bf16 hi + lo, transposed into the B fragment layout of PV (k = token, n = head)
            const uint32_t h0 = pack_bf16(eA0, eB0), h1 = pack_bf16(eA1, eB1);
            const uint32_t l0 = pack_bf16(eA0 - __uint_as_float(h0 << 16), eB0 - __uint_as_float(h0 & 0xffff0000u));
            const uint32_t l1 = pack_bf16(eA1 - __uint_as_float(h1 << 16), eB1 - __uint_as_float(h1 & 0xffff0000u));
            const uint32_t ph0 = movmatrix_trans(h0), ph1 = movmatrix_trans(h1);
            const uint32_t pl0 = movmatrix_trans(l0), pl1 = movmatrix_trans(l1);

            // ---- PV: O^T += V^T P^T (channels x heads), K = the group's 16 tokens
            {
                const uint32_t bmk = r_k == kD ? 0u : (uint32_t)kBitmapBytes;
                const uint32_t vb0 = sp0 + nb0 * (bmk + 2 * r_k), vb1 = sp1 + nb1 * (bmk + 2 * r_k);  // V part of each block
                if (r_v == kD && full) {
                    const uint32_t rA0 = vb0 + 256 * (2 * qq) + 32 * gq, rA1 = vb1 + 256 * (2 * qq) + 32 * gq;
#pragma unroll
                    for (int h = 0; h < 2; ++h) {  // 16-byte chunk h = channel slots 8h .. 8h+7 = tiles 4h .. 4h+3
                        const uint4 xa = lds_128(rA0 + 16 * h), xb = lds_128(rA0 + 256 + 16 * h);
                        uint4 ya = make_uint4(0u, 0u, 0u, 0u), yb = ya;
                        if (two) { ya = lds_128(rA1 + 16 * h); yb = lds_128(rA1 + 256 + 16 * h); }
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
                        hA1 = tA < nb1 ? 0xffffu : 0u; hB1 = tB < nb1 ? 0xffffu : 0u;
                        pA0 = vb0 + 256 * tA + 32 * gq; pB0 = pA0 + 256;
                        pA1 = vb1 + 256 * tA + 32 * gq; pB1 = pA1 + 256;
                    } else {
                        if (tA < nb0) hA0 = lds_u16(vb0 + 16 * tA + 2 * gq);
                        if (tB < nb0) hB0 = lds_u16(vb0 + 16 * tB + 2 * gq);
                        if (tA < nb1) hA1 = lds_u16(vb1 + 16 * tA + 2 * gq);
                        if (tB < nb1) hB1 = lds_u16(vb1 + 16 * tB + 2 * gq);
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
            }
            __syncwarp();  // every lane is done reading stage s
            bposc += two ? 2 : 1;
            ++gposc;
        }
        issue(s);  // stage s is free (or, for k < 0, still empty): start the copies of group k + NSTAGE
        if (++s == NSTAGE) { s = 0; if (k >= 0) parity ^= 1u; }
    }
#ifdef MKV_DBG_TIMING
    if (lane == 0) { atomicMin(&g_dbg_t[blockIdx.x * 16 + 5], dbg_now()); atomicMax(&g_dbg_t[blockIdx.x * 16 + 6], dbg_now()); }
#endif
    if (kGatherOnly) {  // keep the read-back alive; nothing else is written
        if (calib == 0x9e3779b9u && lane == 0) part_ml[(size_t)gw * 2 * (2 * kMaxGroup)] = 0.f;
        return;
    }

    // ---- step 3d, fused: fold the warps' partials; finish units that span several CTAs.
    // Records are in warp order (2w = head, 2w + 1 = tail), hence in non-decreasing unit order: the
    // partials of one unit form a run.  Thread tid owns output elements e = tid + j kNT of [G][D]
    // and folds a run with the LSE rule (pinned by oracle pin P10).
    __syncthreads();  // orders the warps' partials (shared memory, or global scratch from flush(false))
    MKV_TV(1, *(volatile int*)&s_unit[1]);
    const int GD = G * kD;
    const size_t cta_slot_base = (size_t)gridDim.x * kMaxWarps * 2;
    const int tid = threadIdx.x;
    int sh_u0 = -1, sh_u1 = -1;  // units this CTA shares with others (<= 2: one entering, one leaving its range)
    int n_shared = 0;
    // GD / 4 threads fold one unit (four consecutive channels of one head each), so a CTA folds
    // kNT / (GD / 4) units side by side: usually all of them (1 or 2 per CTA) in one pass.
    const int tpr = GD / 4, nslots = max(1, kNT / tpr);
    const int rs = tid / tpr, e = 4 * (tid - rs * tpr), h = e >> 7;
    // each lane keeps the units of records lane and lane + 32: searches and membership are votes
    const int myu0 = lane < kRec ? s_unit[lane] : -1, myu1 = lane + 32 < kRec ? s_unit[lane + 32] : -1;
    int run = -1;
#pragma unroll 1
    for (;;) {
        // the next <= nslots units with partial records, ascending; `mine` = the one this thread folds
        int mine = -1, last = run;
#pragma unroll 1
        for (int k = 0; k < nslots; ++k) {
            const int c0 = myu0 > last ? myu0 : 0x7fffffff, c1 = myu1 > last ? myu1 : 0x7fffffff;
            const int nxt = __reduce_min_sync(kFull, min(c0, c1));
            if (nxt == 0x7fffffff) break;
            last = nxt;
            if (k == rs) mine = nxt;
            if (!(clo <= s_cum[nxt] && s_cum[nxt + 1] <= chi) && n_shared < 2) {  // shared with other CTAs
                if (tid == 0) s_row[n_shared] = (size_t)(nxt / g.n_kv_heads) * g.n_q_heads + (size_t)(nxt % g.n_kv_heads) * G;
                if (n_shared == 0) sh_u0 = nxt; else sh_u1 = nxt;
                ++n_shared;
            }
        }
        if (last == run) break;
        run = last;
        if (mine < 0) continue;  // uniform over a warp: GD / 4 is a multiple of 32
        // records of this unit: bit r of `recs` (tail partials are the odd records, head partials the even ones)
        const unsigned long long recs = (unsigned long long)__ballot_sync(kFull, myu0 == mine) |
                                        ((unsigned long long)__ballot_sync(kFull, myu1 == mine) << 32);
        unsigned heads = 0u;  // warps that hold a head partial (record 2w, in global scratch) of this unit: rare
#pragma unroll
        for (int w = 0; w < kWarps; ++w) heads |= (unsigned)((recs >> (2 * w)) & 1ull) << w;
        const int a = s_cum[mine], b = s_cum[mine + 1];
        const bool whole = clo <= a && b <= chi;
        const size_t row = (size_t)(mine / g.n_kv_heads) * g.n_q_heads + (size_t)(mine % g.n_kv_heads) * G;
        const size_t slot = cta_slot_base + blockIdx.x * 2 + (a < clo ? 0 : 1);
        {
            // tail partials (record 2w + 1, in warp w's shared memory): straight-line, every load independent
            float mw[kWarps], lw[kWarps];
            float4 ow[kWarps];
            float Mr = -INFINITY;
#pragma unroll
            for (int w = 0; w < kWarps; ++w) {
                const bool mem = (recs >> (2 * w + 1)) & 1ull;
                const float2 ml = *reinterpret_cast<const float2*>(&s_ml[2 * w + 1][h][0]);
                ow[w] = *reinterpret_cast<const float4*>(smem + w * kWS + 4 * e);
                mw[w] = mem ? ml.x : -INFINITY;
                lw[w] = mem ? ml.y : 0.f;
                Mr = fmaxf(Mr, mw[w]);
            }
#pragma unroll 1
            for (unsigned m = heads; m; m &= m - 1u) Mr = fmaxf(Mr, s_ml[2 * (__ffs(m) - 1)][h][0]);
            const float Mb = Mr == -INFINITY ? 0.f : Mr;
            float4 O = make_float4(0.f, 0.f, 0.f, 0.f);
            float Lr = 0.f;
#pragma unroll
            for (int w = 0; w < kWarps; ++w) {
                const float wt = ex2(mw[w] - Mb);  // 0 for a record of another unit (its O may be stale bits)
                Lr = fmaf(lw[w], wt, Lr);
                if (wt != 0.f) { O.x = fmaf(ow[w].x, wt, O.x); O.y = fmaf(ow[w].y, wt, O.y); O.z = fmaf(ow[w].z, wt, O.z); O.w = fmaf(ow[w].w, wt, O.w); }
            }
#pragma unroll 1
            for (unsigned m = heads; m; m &= m - 1u) {
                const int w = __ffs(m) - 1;
                const float wt = ex2(s_ml[2 * w][h][0] - Mb);
                Lr = fmaf(s_ml[2 * w][h][1], wt, Lr);
                const float4 o = __ldcg(reinterpret_cast<const float4*>(
                    part_o + ((size_t)blockIdx.x * kWarps + w) * 2 * (size_t)GD + e));
                O.x = fmaf(o.x, wt, O.x); O.y = fmaf(o.y, wt, O.y); O.z = fmaf(o.z, wt, O.z); O.w = fmaf(o.w, wt, O.w);
            }
            if (whole) {
                const float inv = Lr > 0.f ? 1.f / Lr : 0.f;
                *reinterpret_cast<float4*>(out + row * kD + e) = make_float4(O.x * inv, O.y * inv, O.z * inv, O.w * inv);
                if (lse != nullptr && (e & (kD - 1)) == 0) lse[row + h] = Lr > 0.f ? (Mr + log2f(Lr)) * kLn2 : -INFINITY;
            } else {
                *reinterpret_cast<float4*>(part_o + slot * GD + e) = O;
                if ((e & (kD - 1)) == 0) {
                    part_ml[slot * (2 * kMaxGroup) + 2 * h] = Mr;
                    part_ml[slot * (2 * kMaxGroup) + 2 * h + 1] = Lr;
                }
            }
        }
    }
    MKV_T(2);
    if (n_shared == 0) return;  // uniform over the CTA

    // One thread per shared unit releases the CTA's partial (the barrier orders the other threads'
    // stores before its fence), finds the sharers c_first .. c_last (CTAs whose ranges meet the unit)
    // and takes a ticket.  A sharer's slot is 1 for c_first (the unit starts inside it), else 0.
    __syncthreads();
    if ((tid == 0 || tid == 32) && (tid >> 5) < n_shared) {
        const int k = tid >> 5, u = k == 0 ? sh_u0 : sh_u1;
        int cf = (int)blockIdx.x, cl = (int)blockIdx.x;
        if (s_cum[u] < clo) cf = (int)cs.owner((unsigned)s_cum[u] >> 1);
        if (s_cum[u + 1] > chi) cl = (int)cs.owner(((unsigned)s_cum[u + 1] - 1u) >> 1);
        s_cf[k] = cf; s_cl[k] = cl;
        int old;  // release this CTA's partial (ordered by the barrier), acquire the other sharers'
        asm volatile("atom.acq_rel.gpu.global.add.s32 %0, [%1], 1;" : "=r"(old) : "l"(ticket + u) : "memory");
        s_last[k] = old == cl - cf;
        if (old == cl - cf) ticket[u] = 0;  // self-cleaning: every sharer has arrived
    }
    __syncthreads();
    MKV_T(3);
    // last arrivers: thread group rs merges the CTA partials of shared unit rs (read with ld.global.cg: L2,
    // never a stale L1 line); with nslots = 1 (G = 8 on a small CTA) the groups take the units in turn
#pragma unroll 1
    for (int k = rs < nslots ? rs : n_shared; k < n_shared; k += nslots) {
        if (!s_last[k]) continue;
        const int c_first = s_cf[k], c_last = s_cl[k];
        const size_t row = s_row[k];
        float Mx = -INFINITY, Lx = 0.f;
        float4 Ox = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll 1
        for (int c0 = c_first; c0 <= c_last; c0 += 4) {  // four partials' loads in flight at once
            float pm[4], pl[4];
            float4 po[4];
#pragma unroll
            for (int t = 0; t < 4; ++t) {
                const int c = min(c0 + t, c_last);  // a repeated partial gets weight 0 below
                const size_t sl = cta_slot_base + (size_t)c * 2 + (c == c_first ? 1 : 0);
                pm[t] = __ldcg(part_ml + sl * (2 * kMaxGroup) + 2 * h);
                pl[t] = __ldcg(part_ml + sl * (2 * kMaxGroup) + 2 * h + 1);
                po[t] = __ldcg(reinterpret_cast<const float4*>(part_o + sl * (size_t)GD + e));
                if (c0 + t > c_last) { pm[t] = -INFINITY; pl[t] = 0.f; }
            }
            const float Mn = fmaxf(fmaxf(Mx, fmaxf(pm[0], pm[1])), fmaxf(pm[2], pm[3]));
            const float Mb = Mn == -INFINITY ? 0.f : Mn;
            const float c_old = ex2(Mx - Mb);
            Lx *= c_old; Ox.x *= c_old; Ox.y *= c_old; Ox.z *= c_old; Ox.w *= c_old; Mx = Mn;
#pragma unroll
            for (int t = 0; t < 4; ++t) {
                const float w = ex2(pm[t] - Mb);
                Lx = fmaf(pl[t], w, Lx);
                Ox.x = fmaf(po[t].x, w, Ox.x); Ox.y = fmaf(po[t].y, w, Ox.y);
                Ox.z = fmaf(po[t].z, w, Ox.z); Ox.w = fmaf(po[t].w, w, Ox.w);
            }
        }
        const float inv = Lx > 0.f ? 1.f / Lx : 0.f;
        *reinterpret_cast<float4*>(out + row * kD + e) = make_float4(Ox.x * inv, Ox.y * inv, Ox.z * inv, Ox.w * inv);
        if (lse != nullptr && (e & (kD - 1)) == 0) lse[row + h] = Lx > 0.f ? (Mx + log2f(Lx)) * kLn2 : -INFINITY;
    }
    MKV_T(4);
}

}  // namespace

#ifdef MKV_DBG_TIMING
extern "C" __attribute__((visibility("default"))) int mkv_dbg_timing(unsigned long long* host, int reset) {
    if (reset) { static unsigned long long init[160 * 16]; for (int i = 0; i < 160 * 16; ++i) init[i] = (i % 16 == 5) ? ~0ull : 0ull; return (int)cudaMemcpyToSymbol(g_dbg_t, init, sizeof(init)); }
    return (int)cudaMemcpyFromSymbol(host, g_dbg_t, sizeof(unsigned long long) * 160 * 16);
}
#endif

int attention_partial_slots(int sm_count) { return sm_count * kMaxWarps * 2 + sm_count * 2; }

template <int NSTAGE, int NWARPS, bool GATHER>
static cudaError_t launch_attention_cfg(const CacheGeom& g, const LayerView& lv, const uint16_t* q, const int32_t* sel,
                                        const int32_t* sel_count, int k_max, float scale, float* out, float* lse,
                                        const AttnScratch& scr, const uint16_t* upd_k, const uint16_t* upd_v,
                                        const int32_t* upd_count, int sm_count, cudaStream_t s) {
    const int smem = NWARPS * warp_smem_bytes(NSTAGE) + (g.n_units + 1) * 4;
    static int configured = 0;  // largest dynamic shared-memory size opted into so far
    if (smem > configured) {
        cudaError_t e = cudaFuncSetAttribute(mkv_packed_attention_kernel<NSTAGE, NWARPS, GATHER>,
                                             cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
        if (e != cudaSuccess) return e;
        configured = smem;
    }
    return launch_pdl(mkv_packed_attention_kernel<NSTAGE, NWARPS, GATHER>, dim3(sm_count), dim3(NWARPS * 32), (size_t)smem, s,
                      g, lv, q, sel, sel_count, k_max, scale * kLog2e, out, lse, scr.part_o, scr.part_ml, scr.ticket, upd_k,
                      upd_v, upd_count);
}

cudaError_t launch_attention(const CacheGeom& g, const LayerView& lv, const uint16_t* q, const int32_t* sel,
                             const int32_t* sel_count, int k_max, float scale, float* out, float* lse,
                             const AttnScratch& scr, const uint16_t* upd_k, const uint16_t* upd_v,
                             const int32_t* upd_count, int sm_count, cudaStream_t s, int* n_kernels, bool gather_only) {
    if (g.n_units > kMaxUnitsSmem) return cudaErrorInvalidValue;
    if (n_kernels) *n_kernels = 1;
    if (gather_only)
        return launch_attention_cfg<3, 16, true>(g, lv, q, sel, sel_count, k_max, scale, out, lse, scr, upd_k, upd_v, upd_count,
                                                 sm_count, s);
    static int cfg = -1;  // tuning knob (stages * 100 + warps); default chosen from measurements
    if (cfg < 0) {
        const char* e = getenv("MKV_ATTN_CFG");
        cfg = e ? atoi(e) : 316;
    }
#define MKV_CFG(S, W) \
    case S * 100 + W: return launch_attention_cfg<S, W, false>(g, lv, q, sel, sel_count, k_max, scale, out, lse, scr, upd_k, upd_v, upd_count, sm_count, s);
    switch (cfg) {
        MKV_CFG(3, 16) MKV_CFG(2, 16) MKV_CFG(2, 20) MKV_CFG(2, 24) MKV_CFG(4, 12) MKV_CFG(4, 8)
        default: return launch_attention_cfg<3, 16, false>(g, lv, q, sel, sel_count, k_max, scale, out, lse, scr, upd_k, upd_v, upd_count, sm_count, s);
    }
#undef MKV_CFG
}

}  // namespace mkv
