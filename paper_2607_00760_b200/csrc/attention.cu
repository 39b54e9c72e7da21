// attention.cu — step 3 of the hot path: PackedAttention: QK over the
// selected packed keys, softmax, PV over the packed values, split-K combine.  sm_100a.
//
// Design: one launch; every unit is attended by ONE thread-block
// cluster of C CTAs (C = 2 for 64 units on 148 SMs, 8 for 8 units), one CTA per SM.
//   * The unit's selected blocks are cut into equal ranges, one per warp of the cluster.  A warp
//     walks its range in groups of <= 2 token blocks (16 tokens = the M of one mma tile).  What a
//     block is (payload offset, tokens, r_k, r_v) comes from the plan record mkv_select wrote next
//     to `sel`, verified against the `sel` entry; a record that does not match is replaced by the
//     table lookup.
//   * Staging: a block's K part and its V part are contiguous chunks (DESIGN.md format); one lane
//     moves a chunk into the warp's shared-memory ring with ONE 1-D bulk copy (cp.async.bulk, the
//     TMA engine) that completes on the slot's mbarrier.  The ring is byte-granular (a group takes
//     what it needs); up to kSlots groups are in flight per warp.
//   * Phase 1 (QK): S = K q^T with the group's 16 tokens = M, heads = N, channels = K; packed
//     vectors are expanded straight into mma.sync fragments (mkv_walk.cuh).  The scaled logits go
//     to the warp's logit cache (shared memory; global scratch beyond its capacity), the warp's
//     per-head maxima into the CTA's table (shared-memory atomic max).
//   * The CTAs of the cluster exchange their maxima through distributed shared memory: every CTA
//     sends its table to each peer with asynchronous remote stores counted on the receiver's mbarrier
//     (st.async, no fence, no cluster barrier).  Every warp then knows the unit's exact maximum M:
//     probabilities are 2^(z - M), nothing is ever rescaled, and partial results simply add.
//   * Phase 2 (PV, deferred): the softmax sum runs over every selected token; the V part of a block
//     is fetched and walked only if one of its probabilities is >= 2^-40 (error bound).
//     O^T = V^T P^T with channels = M, heads = N, the group's 16 tokens = K; P is split into bf16
//     hi + lo (fp32-class accuracy).  Dense vectors (r = D) skip the walk.  When every range of the
//     cluster is short, each warp lists the groups of its range that matter and the lists are dealt
//     out over all warps of the CTA (which warps hold those groups is an accident of the data).
//   * Step 3d (split-K combine): the warps' partials are added inside the CTA (shared memory), the
//     CTAs' partials by the cluster's first CTA (sent into its shared memory by the second CTA of a
//     cluster of two, again with counted asynchronous stores, after which the sender leaves; pulled
//     through distributed shared memory behind a cluster barrier otherwise), in a fixed order: no
//     global scratch, no atomics, no second kernel, bit-reproducible.
#include "mkv_internal.cuh"
#include "mkv_walk.cuh"

namespace mkv {

namespace {

using namespace walk;
constexpr float kLog2e = 1.4426950408889634f;
constexpr float kLn2 = 0.6931471805599453f;

constexpr int kWarps = 16;         // warps per CTA (one CTA per SM)
constexpr int kRingBytes = 8192;   // per-warp staging ring: two dense groups or five groups at r = 38
constexpr int kSlots = 8;          // groups in flight per warp (one mbarrier each)
constexpr int kGroupMax16 = 256;   // largest group in 16-B units: two dense K (or V) parts
constexpr int kDesc = 32;          // group descriptors kept per warp and phase
constexpr int kDescribe = 24;      // blocks described per call: kDescribe + kSlots <= kDesc
constexpr int kZBytes = 4096;      // per-warp logit cache: 32 blocks at G = 4
constexpr int kMaxCluster = 16;
constexpr float kSkip = 40.f;      // a block whose probabilities are all < 2^-40 is not walked in phase 2

// -DMKV_TRACE (python -m paper_2607_00760_b200.trace; never defined in libmkv.so): lane 0 of every warp stamps %globaltimer
// at the phase boundaries of the LAST launch into a file-scope array that mkv_trace_read copies out.  The stamps are the
// committed evidence for "where the time of a launch goes" (profiles/r3/trace_attention_config2.md).
#ifdef MKV_TRACE
constexpr int kTraceCtas = 160, kTraceStamps = 16;
__device__ unsigned long long g_trace[kTraceCtas][kWarps][kTraceStamps];
__device__ __forceinline__ unsigned long long trace_now() {
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t)::"memory");
    return t;
}
#define MKV_STAMP(i)                                                                                         \
    do {                                                                                                     \
        if ((threadIdx.x & 31) == 0 && blockIdx.x < kTraceCtas) g_trace[blockIdx.x][threadIdx.x >> 5][i] = trace_now(); \
    } while (0)
#else
#define MKV_STAMP(i) do { } while (0)
#endif

// One group of the stream: <= 2 consecutive selected token blocks with the same strategy whose K parts and V
// parts each fit kGroupMax16.  Every size the hot loops need is worked out once, by the describing lane.
struct __align__(16) GDesc {
    // phase 1 (K parts)                                     phase 2 (V parts)
    uint32_t off0, off1;  // chunk offsets, 16-B units       first 16-B unit of each V part
    uint32_t x;           // kc0 | kc1 << 8 | nb0 << 16      vc0 | vc1 << 8 | skew0 << 16 | skew1 << 20 | r_v << 24
                          //   | nb1 << 20 | r_k << 24         (chunk sizes in 16-B units; skew: bytes before the V part)
    uint32_t y;           // upd                              upd | nb0 << 4 | nb1 << 8
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
__device__ __forceinline__ uint32_t vecb(uint32_t r) { return r == (uint32_t)kD ? 256u : 16u + 2u * r; }
// order-preserving map fp32 -> u32 and back (larger float <=> larger key; every key of a float is > 0)
__device__ __forceinline__ uint32_t fkey(float f) {
    const uint32_t u = __float_as_uint(f);
    return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}
__device__ __forceinline__ float funkey(uint32_t k) {
    return __uint_as_float((k & 0x80000000u) ? (k & 0x7fffffffu) : ~k);
}
__device__ __forceinline__ void sts_f32(uint32_t a, float v) { asm volatile("st.shared.f32 [%0], %1;" ::"r"(a), "f"(v) : "memory"); }
__device__ __forceinline__ float2 lds_f32x2(uint32_t a) {
    float2 v;
    asm volatile("ld.shared.v2.f32 {%0,%1}, [%2];" : "=f"(v.x), "=f"(v.y) : "r"(a));
    return v;
}
// ---- thread-block cluster: rank, barrier, distributed shared memory
__device__ __forceinline__ uint32_t cluster_ctarank() {
    uint32_t r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
__device__ __forceinline__ void cluster_sync() {  // also orders shared-memory accesses cluster-wide (release / acquire)
    asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
__device__ __forceinline__ void cluster_arrive_relaxed() { asm volatile("barrier.cluster.arrive.relaxed.aligned;" ::: "memory"); }
__device__ __forceinline__ void cluster_wait() { asm volatile("barrier.cluster.wait.aligned;" ::: "memory"); }
// 4 bytes into another CTA's shared memory, counted on an mbarrier of THAT CTA when they have landed: the receiver waits on
// its own mbarrier and then sees the data.  No fence on either side (a cluster-scope release, which is what a plain remote
// store followed by barrier.cluster needs, is a MEMBAR.ALL.GPU on this machine: it waits for every outstanding access).
__device__ __forceinline__ void st_async_b32(uint32_t dst, uint32_t v, uint32_t mbar) {
    asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.b32 [%0], %1, [%2];" ::"r"(dst), "r"(v), "r"(mbar) : "memory");
}
__device__ __forceinline__ uint32_t dsmem_addr(uint32_t local, uint32_t rank) {  // the same offset in CTA `rank` of the cluster
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(local), "r"(rank));
    return r;
}
__device__ __forceinline__ uint32_t ld_dsmem_u32(uint32_t a) {
    uint32_t v;
    asm volatile("ld.shared::cluster.u32 %0, [%1];" : "=r"(v) : "r"(a) : "memory");
    return v;
}
__device__ __forceinline__ void st_dsmem_f32(uint32_t a, float v) {
    asm volatile("st.shared::cluster.f32 [%0], %1;" ::"r"(a), "f"(v) : "memory");
}
__device__ __forceinline__ float ld_dsmem_f32(uint32_t a) {
    float v;
    asm volatile("ld.shared::cluster.f32 %0, [%1];" : "=f"(v) : "r"(a) : "memory");
    return v;
}

// per warp: staging ring | phase-1 descriptors | phase-2 descriptors | logit cache | slot table (offset, bytes) |
// mbarriers | groups in flight in phase 2
constexpr int kOffD1 = kRingBytes, kOffD2 = kOffD1 + kDesc * 16, kOffZ = kOffD2 + kDesc * 16, kOffSlot = kOffZ + kZBytes;
constexpr int kOffBar = kOffSlot + kSlots * 8, kOffGrp = kOffBar + kSlots * 8, kWS = kOffGrp + kSlots * 16;

// Even split of n items over p parts: part i owns [i b + min(i, r), ...) with b = n / p, r = n % p
// (the first r parts hold one more).
struct Split {
    unsigned b, r;
    __device__ __forceinline__ unsigned begin(unsigned i) const { return i * b + min(i, r); }
};

// Where element e = head * 128 + channel of a partial O sits in shared memory: channel 16 a + 2 i + p of head h at
// h * 128 + ((16 i + 2 a + p + 8 (h / 2)) mod 128) -- a bijection per head that makes the warps' fragment stores (lane
// (a, qq) holds channels 16 a + 2 i, + 1 of heads 2 qq, 2 qq + 1) free of bank conflicts.
__device__ __forceinline__ int o_slot(int e) {
    const int h = e >> 7, ch = e & 127;
    return (e & ~127) | ((((ch & 15) >> 1) * 16 + (ch >> 4) * 2 + (ch & 1) + 8 * (h >> 1)) & 127);
}

// QK of one group in flight: S (16 tokens x 8 heads) += K q^T with the group's tokens = M (rows 0-7 = block 0, rows 8-15 =
// block 1), heads = N, channels = K.  sp0 / sp1: the K parts of its blocks in shared memory; qa: q[head gq][32qq .. 32qq+31]
// as B fragments.  Packed vectors are expanded straight into A fragments (mkv_walk.cuh); dense vectors skip the walk.
// pairs: the vectors were kept in element groups g >= 2 and their values are stored pair-major (k_walk_mma_pairs).
__device__ __forceinline__ void qk_group(float (&S)[4], int r_k, int nb0, int nb1, uint32_t sp0, uint32_t sp1,
                                         const uint32_t (&qa)[8][2], int lane, bool pairs) {
    const int gq = lane >> 2, qq = lane & 3;
    const bool two = nb1 != 0;
    const bool full = nb0 == kPhys && (!two || nb1 == kPhys);
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
            if (pairs) {  // pair pi = rank / 2 of token t at byte 4 (pi n + t): the same 2 n bytes per kept element before it
                p0 = sp0 + 16 * nb0 + st0 * (ex & 0xffffu) + 4 * gq;
                p1 = sp1 + 16 * nb1 + st1 * (ex >> 16) + 4 * gq;
                st0 *= 2u; st1 *= 2u;
                k_walk_mma_pairs<0>(S, w0, w1, p0, p1, st0, st1, qa);
                k_walk_mma_pairs<1>(S, w0, w1, p0, p1, st0, st1, qa);
                k_walk_mma_pairs<2>(S, w0, w1, p0, p1, st0, st1, qa);
                k_walk_mma_pairs<3>(S, w0, w1, p0, p1, st0, st1, qa);
                return;
            }
            p0 = sp0 + 16 * nb0 + st0 * (ex & 0xffffu) + 2 * gq;
            p1 = sp1 + 16 * nb1 + st1 * (ex >> 16) + 2 * gq;
        }
        k_walk_mma<0>(S, w0, w1, p0, p1, st0, st1, qa);
        k_walk_mma<1>(S, w0, w1, p0, p1, st0, st1, qa);
        k_walk_mma<2>(S, w0, w1, p0, p1, st0, st1, qa);
        k_walk_mma<3>(S, w0, w1, p0, p1, st0, st1, qa);
    }
}

// PV of one group in flight: O^T += V^T P^T with channels = M, heads = N, the group's <= 16 tokens = K.  vb0 / vb1: the
// V parts of its blocks in shared memory; ph / pl: probabilities of head gq, tokens 2qq, 2qq+1 of each block, split into
// bf16 hi + lo (exactly the B fragments: k = token, n = head).  Dense vectors (r = D) skip the walk.
__device__ __forceinline__ void pv_group(float (&acc)[8][4], int r_v, int nb0, int nb1, uint32_t vb0, uint32_t vb1,
                                         uint32_t ph0, uint32_t ph1, uint32_t pl0, uint32_t pl1, int gq, int qq) {
    const bool two = nb1 != 0;
    const bool full = nb0 == kPhys && (!two || nb1 == kPhys);
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

// ------------------------------------------------------------------------------------------
// grid = n_units clusters of C CTAs; cluster u attends unit u.
// kGatherOnly: calibration build of the same kernel (mkv_calibrate_gather): every K part and every
// V part of the selection is staged exactly as in the real run (nothing is skipped), one word per
// lane and group is read back, and all arithmetic, synchronisation and output are left out.
// ------------------------------------------------------------------------------------------
template <bool kGatherOnly>
__global__ void __launch_bounds__(kWarps * 32, 1)
mkv_packed_attention_kernel(CacheGeom g, LayerView lv, const uint16_t* __restrict__ q,
                            const int32_t* __restrict__ sel, const int32_t* __restrict__ sel_count, int k_max,
                            float scale_log2, float* __restrict__ out, float* __restrict__ lse, AttnScratch scr,
                            const uint16_t* __restrict__ upd_k, const uint16_t* __restrict__ upd_v,
                            const int32_t* __restrict__ upd_count, int C) {
    extern __shared__ __align__(128) uint8_t smem[];
    constexpr int kNT = kWarps * 32;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int gq = lane >> 2, qq = lane & 3;  // mma fragment coordinates (groupID, threadID_in_group)
    const int G = g.group;

    __shared__ uint32_t s_max[kMaxGroup];                 // the CTA's per-head maxima (keys); read by the whole cluster
    __shared__ float s_l[kWarps][kMaxGroup];              // the warps' softmax sums
    __shared__ float s_cta_l[kMaxGroup];                  // the CTA's partial sums (its partial O: s_cta_o)
    __shared__ float s_peer_l[kMaxGroup];                 // clusters of two: the second CTA's sums, pushed into the first
    __shared__ float s_M[kMaxGroup];                      // the unit's per-head maxima after the exchange
    __shared__ unsigned s_active;                         // warps of the CTA that hold a partial result
    __shared__ unsigned s_stat[2];                        // V blocks / V bytes this CTA fetched (mkv_attention_stats)
    __shared__ __align__(8) unsigned long long s_xbar[2]; // mbarriers: [0] the peers' maxima have landed; [1] (first CTA of a
                                                          // cluster of two) the second CTA's partial has landed
    __shared__ uint32_t s_peer_max[kMaxCluster][kMaxGroup];  // maxima (keys) sent by the other CTAs of the cluster
    __shared__ uint32_t s_q[kWarps][kDesc];               // phase 2: the groups of each warp's range that matter ...
    __shared__ int s_qn[kWarps];                          // ... and how many
    float* s_cta_o = reinterpret_cast<float*>(smem + kWarps * kWS);  // [G][128] floats behind the warps' regions
    float* s_peer_o = s_cta_o + kMaxGroup * kD;                      // clusters of two: the second CTA's partial O

    uint8_t* wbase = smem + warp * kWS;
    const uint32_t ring0 = smem_u32(wbase);
    GDesc* d1 = reinterpret_cast<GDesc*>(wbase + kOffD1);
    GDesc* d2 = reinterpret_cast<GDesc*>(wbase + kOffD2);
    const uint32_t zs0 = ring0 + kOffZ;
    uint2* slot_tab = reinterpret_cast<uint2*>(wbase + kOffSlot);
    const uint32_t bar0 = ring0 + kOffBar;
    GDesc* slot_grp = reinterpret_cast<GDesc*>(wbase + kOffGrp);
    if (lane == 0) {
#pragma unroll
        for (int s = 0; s < kSlots; ++s) mbar_init(bar0 + 8 * s, 1);
        mbar_init_fence();
    }
    if (threadIdx.x < kMaxGroup) s_max[threadIdx.x] = 0u;  // below the key of every float
    if (threadIdx.x == 0) {
        s_active = 0u; s_stat[0] = s_stat[1] = 0u;
        // what the peers will send: (C - 1) x 8 maxima; to the first CTA of a cluster of two also G x 128 floats + G sums
        mbar_init(smem_u32(&s_xbar[0]), 1);
        mbar_init(smem_u32(&s_xbar[1]), 1);
        mbar_init_fence();
        if (C > 1) mbar_expect_tx(smem_u32(&s_xbar[0]), (uint32_t)(C - 1) * kMaxGroup * 4u);
        if (C == 2) mbar_expect_tx(smem_u32(&s_xbar[1]), (uint32_t)G * (kD + 1) * 4u);
    }
    const int u = (int)blockIdx.x / C;                      // the cluster's unit
    const unsigned rank = cluster_ctarank();
    __syncthreads();
    MKV_STAMP(0);             // scheduled, barriers initialised
    pdl_wait();               // the producer of sel / sel_count / the plan / the cache is done
    pdl_launch_dependents();  // the next kernel may be scheduled as SMs free up
    MKV_STAMP(1);             // griddepcontrol.wait returned

    // tokens in the layer's update buffer: device-resident, so a captured graph stays valid across appends
    const int n_buf = min(max(__ldg(upd_count), 0), g.L);
    const int upd_blocks = (n_buf + kPhys - 1) / kPhys;  // the unit's stream ends with the blocks of its update buffer
    const int ppb = g.ppb;                                // device blocks per selected token block (2 at B = 16)
    // device blocks selected: at most sel_cap = blocks per unit + 1 entries of `sel` are attended (plan_stride = sel_cap
    // * ppb), which is also what the unit's share of the logit scratch is sized for; a caller-built selection longer
    // than that (k_max beyond sel_cap, duplicates) is cut there instead of running into the next unit's scratch
    const int cnt = min(min(max(__ldg(sel_count + u), 0), k_max) * ppb, scr.plan_stride);
    const int T = cnt + upd_blocks;                       // device blocks of the unit's stream
    MKV_STAMP(2);                                         // counts known
    const size_t row = (size_t)(u / g.n_kv_heads) * g.n_q_heads + (size_t)(u % g.n_kv_heads) * G;
    if (T == 0) {  // (uniform over the cluster) empty selection: out = 0, lse = -inf
        if (rank == 0 && !kGatherOnly) {
            for (int e = threadIdx.x; e < G * kD; e += kNT) out[row * kD + e] = 0.f;
            if (lse != nullptr && threadIdx.x < G) lse[row + threadIdx.x] = -INFINITY;
        }
        return;
    }
    // this CTA's mbarriers are ready for its peers: arrive here, wait (for every peer's arrival) right before the first send
    if (!kGatherOnly && C > 1) cluster_arrive_relaxed();
    // The stream is split in units of two positions, so every range starts at an even position: a range never
    // holds two odd runs, which would cost an extra half-empty group.
    const unsigned P = ((unsigned)T + 1u) >> 1;  // position pairs, over the C * kWarps warps of the cluster
    Split ws;
    ws.b = P / (unsigned)(C * kWarps); ws.r = P % (unsigned)(C * kWarps);
    const unsigned wi = rank * kWarps + (unsigned)warp;
    const int lo = min(2 * (int)ws.begin(wi), T), hi = min(2 * (int)ws.begin(wi + 1), T);
    const int n_total = hi - lo;
    const uint32_t zstride = 32u * (uint32_t)G;         // bytes of one block's logits: [head][token] floats
    const int zcap = kZBytes / (int)zstride;            // blocks of the range whose logits stay in shared memory
    float* zglob = scr.zbuf + ((size_t)u * scr.z_unit_stride + (size_t)lo) * (size_t)(8 * G);

    int bbuilt = 0, gbuilt = 0;  // blocks / groups described so far

    // Describe the next <= kDescribe blocks of the range (one per lane) and pair them into groups: block i
    // follows block i - 1 in a group if both have the same strategy and their K parts and V parts fit one group;
    // runs of such blocks are paired greedily from their start.  A pure function of the inputs: when phase 2
    // has to describe a long range again it gets the same groups.
    auto describe = [&](int count) {
        uint32_t off16 = 0u, meta = 0u, updf = 0u;
        if (lane < count) {
            const int j = lo + bbuilt + lane, jb = j - cnt;
            if (jb >= 0) {  // block jb of the unit's update buffer: raw rows [u][8 jb ..][128] of upd_k / upd_v
                const uint32_t nb = (uint32_t)min(kPhys, n_buf - kPhys * jb);
                off16 = (uint32_t)(((size_t)u * g.L + (size_t)kPhys * jb) * (kD * 2 / 16));
                meta = (uint32_t)kD | ((uint32_t)kD << 8) | (nb << 16);
                updf = 1u;
            } else {
                const int ts = __ldg(sel + (size_t)u * k_max + (j >> (ppb - 1)));  // ppb is 1 or 2
                const int t0 = (ts < 0 || (ts & (g.B - 1))) ? -1 : ts + kPhys * (j & (ppb - 1));  // (j odd: second half of 16 tokens)
                PlanRec pr;
                pr.t0 = -1; pr.off16 = 0u; pr.meta = 0u; pr.tag = 0u;
                if (scr.plan != nullptr && j < scr.plan_stride) {
                    const uint4 v = __ldg(reinterpret_cast<const uint4*>(scr.plan + (size_t)u * scr.plan_stride + j));
                    pr.t0 = (int32_t)v.x; pr.off16 = v.y; pr.meta = v.z; pr.tag = v.w;
                }
                if (pr.tag == scr.plan_tag && pr.t0 == t0 && t0 >= 0) { off16 = pr.off16; meta = pr.meta; }
                else plan_lookup(g, lv, u, t0, off16, meta);
            }
        }
        const uint32_t nb = (meta >> 16) & 15u, rk = meta & 255u, rv = (meta >> 8) & 255u, kpairs = (meta >> 24) & 1u;
        const uint32_t kb = nb * vecb(rk);                      // bytes of the K part
        const uint32_t sk = updf ? 0u : (kb & 15u);             // bytes between the last 16-B boundary and the V part
        const uint32_t kc = (kb + 15u) >> 4, vc = (sk + nb * vecb(rv) + 15u) >> 4;  // 16-B units staged in phase 1 / 2
        const uint32_t voff = updf ? off16 : off16 + (kb >> 4);
        const uint32_t pmeta = __shfl_up_sync(kFull, meta, 1), pkc = __shfl_up_sync(kFull, kc, 1);
        const uint32_t pvc = __shfl_up_sync(kFull, vc, 1), pupd = __shfl_up_sync(kFull, updf, 1);
        const bool follows = lane > 0 && lane < count && ((meta ^ pmeta) & 0x0100ffffu) == 0u && nb != 0u &&
                             ((pmeta >> 16) & 15u) != 0u && kc + pkc <= (uint32_t)kGroupMax16 && vc + pvc <= (uint32_t)kGroupMax16 &&
                             !updf && !pupd;
        const unsigned fm = __ballot_sync(kFull, follows);
        const int start = 31 - __clz((int)(~fm & lanemask_le()));  // first block of this lane's run (bit 0 of ~fm is set)
        const bool first = lane < count && ((lane - start) & 1) == 0;
        const bool two = first && ((fm >> 1) >> lane & 1u);        // lane + 1 follows (and is therefore < count)
        const unsigned gm = __ballot_sync(kFull, first);
        const uint32_t off1 = __shfl_down_sync(kFull, off16, 1), nb1 = __shfl_down_sync(kFull, nb, 1);
        const uint32_t kc1 = __shfl_down_sync(kFull, kc, 1), vc1 = __shfl_down_sync(kFull, vc, 1);
        const uint32_t voff1 = __shfl_down_sync(kFull, voff, 1), sk1 = __shfl_down_sync(kFull, sk, 1);
        if (first) {
            const int slot = (gbuilt + __popc(gm & lanemask_lt())) & (kDesc - 1);
            GDesc a, b;
            a.off0 = off16; a.off1 = two ? off1 : 0u;
            a.x = kc | ((two ? kc1 : 0u) << 8) | (nb << 16) | ((two ? nb1 : 0u) << 20) | (rk << 24);
            a.y = updf | (kpairs << 1);
            b.off0 = voff; b.off1 = two ? voff1 : 0u;
            b.x = vc | ((two ? vc1 : 0u) << 8) | (sk << 16) | ((two ? sk1 : 0u) << 20) | (rv << 24);
            b.y = updf | (nb << 4) | ((two ? nb1 : 0u) << 8);
            d1[slot] = a;
            d2[slot] = b;
        }
        gbuilt += __popc(gm);
        bbuilt += count;
        __syncwarp();
    };

    // ---- staging ring (all scalars below are warp-uniform)
    uint32_t rhead = 0u, rused = 0u, parbits = 0u;
    int pend = 0, si = 0, sc = 0;
    const unsigned long long slice = reinterpret_cast<unsigned long long>(lv.slice);
    // claim `sz` bytes (a multiple of 16, <= 4096) for the next group; false: no room yet
    auto ring_alloc = [&](uint32_t sz, uint32_t& off) -> bool {
        uint32_t need = sz, h = pend == 0 ? 0u : rhead;  // an idle ring restarts at its beginning
        if (h + sz > (uint32_t)kRingBytes) { need += (uint32_t)kRingBytes - h; h = 0u; }  // wrap: the tail stays unused
        if (pend == kSlots || rused + need > (uint32_t)kRingBytes) return false;
        off = h;
        rhead = h + sz;
        rused += need;
        if (lane == 0) slot_tab[si] = make_uint2(h, need);
        return true;
    };
    auto ring_commit = [&]() {
        si = (si + 1) & (kSlots - 1);
        ++pend;
        __syncwarp();  // the slot table entry is visible to the whole warp
    };
    // start the copies of one group (<= 2 chunks, 16-byte units) into ring offset `off`; `landed()` returns when the OLDEST
    // group in flight is complete (groups complete in issue order)
    auto stage = [&](const unsigned long long src, uint32_t off, uint32_t off0, uint32_t c0, uint32_t off1, uint32_t c1) {
        // (one lane, one bulk copy per chunk on the slot's mbarrier; staging by all lanes with cp.async, which pays in the
        // score kernel, was measured here too: 24.4 against 23.6 us/layer)
        if (lane == 0) {
            const uint32_t bar = bar0 + 8 * si, dst = ring0 + off;
            mbar_expect_tx(bar, c0 + c1);
            if (c0) bulk_g2s(dst, src + ((unsigned long long)off0 << 4), c0, bar);
            if (c1) bulk_g2s(dst + c0, src + ((unsigned long long)off1 << 4), c1, bar);
        }
    };
    auto landed = [&]() { mbar_wait(bar0 + 8 * sc, (parbits >> sc) & 1u); };
    auto ring_release = [&]() {  // the oldest group has been consumed
        rused -= slot_tab[sc].y;
        parbits ^= 1u << sc;
        sc = (sc + 1) & (kSlots - 1);
        --pend;
    };

    // =====================================================================================
    // Phase 1: QK.  Logits (log2 domain, scaled) -> logit cache; per-head maxima -> the CTA's table.
    // =====================================================================================
    float mxA = -INFINITY, mxB = -INFINITY;  // this lane's maxima for heads 2qq, 2qq+1
    uint32_t twomask = 0u;                   // bit i: group i of the range holds two blocks (short ranges: phase 2 deals them out)
    uint32_t calib = 0u;
    // this lane's slots inside a block's logits ([head][token] floats): phase 1 writes token gq of heads 2qq, 2qq+1;
    // phase 2 reads tokens 2qq, 2qq+1 of head gq
    const uint32_t zw = (uint32_t)(16 * qq + gq) * 4u, zr = (uint32_t)(8 * gq + 2 * qq) * 4u;

    if (n_total > 0) {
        // q[head gq][32qq .. 32qq+31]: k-step ks uses channels 32qq + 4ks .. + 3
        uint32_t qa[8][2];
        {
            const uint4* qrow = reinterpret_cast<const uint4*>(q + (row + gq) * kD + 32 * qq);
#pragma unroll
            for (int h = 0; h < 4; ++h) {
                uint4 v = make_uint4(0u, 0u, 0u, 0u);
                if (gq < G) v = __ldg(qrow + h);
                qa[2 * h][0] = v.x; qa[2 * h][1] = v.y; qa[2 * h + 1][0] = v.z; qa[2 * h + 1][1] = v.w;
            }
        }
        int bposi = 0, gposi = 0, gposc = 0, bposc = 0;
#pragma unroll 1
        for (;;) {
            // ---- issue: K parts of the next groups while the ring has room
#pragma unroll 1
            while (bposi < n_total) {
                if (gposi == gbuilt) {
                    describe(min(kDescribe, n_total - bbuilt));
#ifdef MKV_TRACE
                    if (gposi == 0) MKV_STAMP(3);  // first blocks described
#endif
                }
                const GDesc d = d1[gposi & (kDesc - 1)];
                const uint32_t c0 = (d.x & 255u) << 4, c1 = ((d.x >> 8) & 255u) << 4;
                uint32_t off;
                if (!ring_alloc(c0 + c1, off)) break;
                stage((d.y & 1u) ? reinterpret_cast<unsigned long long>(upd_k) : slice, off, d.off0, c0, d.off1, c1);
                ring_commit();
                ++gposi;
                bposi += c1 ? 2 : 1;
                // two groups are in flight and the oldest has landed: walk it now, issue the rest between the walks (at
                // the start of the kernel every warp of the SM is issuing and nothing else hides the cost of it)
                if (pend >= 2 && mbar_test(bar0 + 8 * sc, (parbits >> sc) & 1u)) break;
            }
            if (pend == 0) break;  // nothing in flight and nothing left to issue

            // ---- consume the oldest group
            const GDesc d = d1[gposc & (kDesc - 1)];
            const int r_k = (int)(d.x >> 24);
            const int nb0 = (int)((d.x >> 16) & 15u), nb1 = (int)((d.x >> 20) & 15u);
            const bool two = nb1 != 0;
            const uint32_t sp0 = ring0 + slot_tab[sc].x, sp1 = sp0 + ((d.x & 255u) << 4);
            if (kGatherOnly) {
                landed();
                calib ^= lds_u32(sp0 + 4 * lane);
                __syncwarp();
                ring_release();
                ++gposc;
                bposc += two ? 2 : 1;
                continue;
            }
            const bool full = nb0 == kPhys && (!two || nb1 == kPhys);

            landed();  // the group's K parts have landed
#ifdef MKV_TRACE
            if (gposc == 0) MKV_STAMP(4);  // first K part landed
#endif

            // ---- QK: S (tokens x heads); rows 0-7 = block 0, rows 8-15 = block 1.  (A position that holds no block -- an
            // invalid `sel` entry, the missing second half of a ragged 16-token block -- still gets its logits: -inf, so
            // that whoever reads the cache in phase 2 sees "no token" instead of stale shared memory.)
            {
                float S[4] = {0.f, 0.f, 0.f, 0.f};
                if (nb0 != 0) qk_group(S, r_k, nb0, nb1, sp0, sp1, qa, lane, (d.y & 2u) != 0u);
                // ---- scaled logits of token gq of each block, heads 2qq, 2qq+1 -> cache [head][token]
                const bool v0 = gq < nb0, v1 = gq < nb1;
                const float zA0 = v0 ? S[0] * scale_log2 : -INFINITY, zB0 = v0 ? S[1] * scale_log2 : -INFINITY;
                const float zA1 = v1 ? S[2] * scale_log2 : -INFINITY, zB1 = v1 ? S[3] * scale_log2 : -INFINITY;
                mxA = fmaxf(mxA, fmaxf(zA0, zA1));
                mxB = fmaxf(mxB, fmaxf(zB0, zB1));
                // block i of the range keeps its logits in shared memory iff i < zcap, else in global scratch
                if (bposc < zcap) {
                    const uint32_t za = zs0 + (uint32_t)bposc * zstride + zw;
                    if (2 * qq < G) sts_f32(za, zA0);
                    if (2 * qq + 1 < G) sts_f32(za + 32, zB0);
                } else {
                    float* z0 = zglob + (size_t)bposc * (size_t)(8 * G) + (zw >> 2);
                    if (2 * qq < G) z0[0] = zA0;
                    if (2 * qq + 1 < G) z0[8] = zB0;
                }
                if (two) {
                    if (bposc + 1 < zcap) {
                        const uint32_t za = zs0 + (uint32_t)(bposc + 1) * zstride + zw;
                        if (2 * qq < G) sts_f32(za, zA1);
                        if (2 * qq + 1 < G) sts_f32(za + 32, zB1);
                    } else {
                        float* z1 = zglob + (size_t)(bposc + 1) * (size_t)(8 * G) + (zw >> 2);
                        if (2 * qq < G) z1[0] = zA1;
                        if (2 * qq + 1 < G) z1[8] = zB1;
                    }
                }
            }
            __syncwarp();  // every lane is done reading the slot
            ring_release();
            if (two && gposc < 32) twomask |= 1u << gposc;
            ++gposc;
            bposc += two ? 2 : 1;
        }
        if (!kGatherOnly) {  // the warp's maxima -> the CTA's table
#pragma unroll
            for (int o = 4; o < 32; o <<= 1) {
                mxA = fmaxf(mxA, __shfl_xor_sync(kFull, mxA, o));
                mxB = fmaxf(mxB, __shfl_xor_sync(kFull, mxB, o));
            }
            if (gq == 0) {  // lanes 0..3 hold heads 2qq, 2qq+1
                if (2 * qq < G) atomicMax(&s_max[2 * qq], fkey(mxA));
                if (2 * qq + 1 < G) atomicMax(&s_max[2 * qq + 1], fkey(mxB));
            }
        }
    }

    // =====================================================================================
    // The cluster's CTAs exchange their maxima through distributed shared memory.
    // =====================================================================================
    float Mraw = -INFINITY;  // the unit's maximum logit of head gq (log2 domain)
    MKV_STAMP(5);            // phase 1 of this warp done
    if (!kGatherOnly) {
        __syncthreads();  // the CTA's table is complete
        if (C > 1) {
            // every CTA SENDS its eight maxima to each peer (asynchronous remote stores counted on the receiver's mbarrier)
            // and waits for the C - 1 sets sent to it: no cluster barrier, no fence, no remote load
            cluster_wait();  // every peer has initialised its mbarriers (it arrived at the start of its kernel)
            if (warp == 0) {
                for (int i = lane; i < (C - 1) * kMaxGroup; i += 32) {
                    const int p = i / kMaxGroup, j = i % kMaxGroup;
                    const uint32_t r = (uint32_t)(p >= (int)rank ? p + 1 : p);
                    st_async_b32(dsmem_addr(smem_u32(&s_peer_max[rank][j]), r), s_max[j], dsmem_addr(smem_u32(&s_xbar[0]), r));
                }
            }
            mbar_wait(smem_u32(&s_xbar[0]), 0u);
        }
        MKV_STAMP(6);    // maxima exchanged
        if (gq < G) {
            uint32_t k = s_max[gq];
            for (int r = 0; r < C; ++r)
                if (r != (int)rank) k = max(k, s_peer_max[r][gq]);
            Mraw = k == 0u ? -INFINITY : funkey(k);
            if (warp == 0 && qq == 0) s_M[gq] = Mraw;
        }
    }
    const float Mh = Mraw == -INFINITY ? 0.f : Mraw;  // 0 if the unit holds no valid token
    // A warp whose own maxima all lie more than kSkip below the unit's takes no further part: each of its tokens has a
    // probability < 2^-40, which neither the sums nor the output can see (error bound).
    bool active = kGatherOnly;
    if (!kGatherOnly) {
        const float MA = __shfl_sync(kFull, Mraw, 8 * qq), MB = __shfl_sync(kFull, Mraw, 8 * qq + 4);  // heads 2qq, 2qq+1
        active = __any_sync(kFull, (2 * qq < G && mxA - MA >= -kSkip) || (2 * qq + 1 < G && mxB - MB >= -kSkip));
    }

    // =====================================================================================
    // Phase 2: softmax sums over every selected token, PV over the blocks that matter.
    // =====================================================================================
    float acc[8][4];    // O^T tile i: rows gq / gq+8 = channels 16gq + 2i / + 1, columns 2qq, 2qq+1 = heads
#pragma unroll
    for (int i = 0; i < 8; ++i) acc[i][0] = acc[i][1] = acc[i][2] = acc[i][3] = 0.f;
    float lsum = 0.f;   // this lane's share of the softmax sum of head gq
    unsigned st_vblocks = 0u, st_vbytes = 0u;

    // logits of head gq, tokens 2qq, 2qq+1 of block i of the range (shared-memory cache, or global scratch beyond it)
    auto z_pair = [&](int i) -> float2 {
        if (i < zcap) return lds_f32x2(zs0 + (uint32_t)i * zstride + zr);
        return __ldcg(reinterpret_cast<const float2*>(zglob + (size_t)i * (size_t)(8 * G) + (zr >> 2)));
    };

    // Short ranges (every range of the cluster fits its descriptor ring and its logit cache): phase 2 is a handful of
    // blocks, and which warps hold them is an accident of the data.  Every warp lists the groups of its range that matter
    // (and adds up its softmax sums); the lists are then dealt out over all warps of the CTA, so no warp walks more than
    // ceil(groups that matter / warps) of them.  The order is a function of the data only: results are reproducible.
    const bool redist = !kGatherOnly && 2 * ((int)ws.b + 1) <= min(kDesc, zcap);
    bool walked = false;  // this warp holds a partial O
    if (redist) {
        int qn = 0;
        if (n_total > 0 && active) {
            // softmax sums and "this block matters" flags of the range's blocks, four blocks at a time (independent loads,
            // exponentials and votes); then one entry per group with a block that matters
            uint32_t needmask = 0u;
#pragma unroll 1
            for (int b0 = 0; b0 < n_total; b0 += 4) {
                float2 z[4];
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    z[j] = make_float2(-INFINITY, -INFINITY);
                    if (gq < G && b0 + j < n_total) z[j] = lds_f32x2(zs0 + (uint32_t)(b0 + j) * zstride + zr);
                }
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    lsum += ex2(z[j].x - Mh) + ex2(z[j].y - Mh);
                    if (__any_sync(kFull, fmaxf(z[j].x, z[j].y) - Mh >= -kSkip)) needmask |= 1u << (b0 + j);
                }
            }
            int bpos = 0;
#pragma unroll 1
            for (int gi = 0; gi < gbuilt; ++gi) {
                const bool two = (twomask >> gi) & 1u;
                const uint32_t nd = (needmask >> bpos) & (two ? 3u : 1u);
                if (nd != 0u) {
                    if (lane == 0) s_q[warp][qn] = (uint32_t)gi | (nd << 8) | ((uint32_t)bpos << 10);
                    ++qn;
                }
                bpos += two ? 2 : 1;
            }
        }
        if (lane == 0) s_qn[warp] = qn;
        __syncthreads();
        // inclusive prefix of the warps' counts (lane w: warps 0..w)
        int incl = lane < kWarps ? s_qn[lane] : 0;
#pragma unroll
        for (int o = 1; o < kWarps; o <<= 1) {
            const int t = __shfl_up_sync(kFull, incl, o);
            if (lane >= o) incl += t;
        }
        const int Q = __shfl_sync(kFull, incl, kWarps - 1);
        int e = warp;  // this warp walks entries warp, warp + kWarps, ...
#pragma unroll 1
        for (;;) {
            // ---- start the V copies of this warp's next entries while the ring has room
#pragma unroll 1
            while (e < Q) {
                const int owner = __popc(__ballot_sync(kFull, lane < kWarps && incl <= e));
                const int excl = owner == 0 ? 0 : __shfl_sync(kFull, incl, owner - 1);
                const uint32_t ent = s_q[owner][e - excl];
                const GDesc d = *reinterpret_cast<const GDesc*>(smem + owner * kWS + kOffD2 + 16 * (int)(ent & 255u));
                uint32_t nb0 = (d.y >> 4) & 15u, nb1 = (d.y >> 8) & 15u;
                const bool need0 = (ent >> 8) & 1u, need1 = (ent >> 9) & 1u;
                // a group with one block that matters becomes a one-block group
                uint32_t off0 = d.off0, off1 = d.off1, c0 = (d.x & 255u) << 4, c1 = ((d.x >> 8) & 255u) << 4;
                uint32_t sk0 = (d.x >> 16) & 15u, sk1 = (d.x >> 20) & 15u, shift = 0u;
                if (!need0) { off0 = off1; c0 = c1; sk0 = sk1; nb0 = nb1; nb1 = 0u; c1 = 0u; shift = 1u; }
                else if (!need1) { nb1 = 0u; c1 = 0u; }
                uint32_t off;
                if (!ring_alloc(c0 + c1, off)) break;
                stage((d.y & 1u) ? reinterpret_cast<unsigned long long>(upd_v) : slice, off, off0, c0, off1, c1);
                if (lane == 0) {
                    GDesc g2;
                    g2.off0 = sk0 | (sk1 << 4) | (c0 << 8);                  // skews of the V parts, bytes of the first chunk
                    g2.off1 = (ent >> 10) + shift;                           // index of the first WALKED block in the owner's range
                    g2.x = d.x;
                    g2.y = nb0 | (nb1 << 4) | ((uint32_t)owner << 8);
                    slot_grp[si] = g2;
                }
                st_vblocks += nb1 ? 2u : 1u;
                st_vbytes += c0 + c1;
                ring_commit();
                e += kWarps;
            }
            if (pend == 0) break;
            // ---- consume the oldest group in flight: PV with the owner's logits
            const GDesc d = slot_grp[sc];
            const int r_v = (int)(d.x >> 24);
            const int nb0 = (int)(d.y & 15u), nb1 = (int)((d.y >> 4) & 15u), pos = (int)d.off1;
            const bool two = nb1 != 0;
            const uint32_t vb0 = ring0 + slot_tab[sc].x + (d.off0 & 15u);
            const uint32_t vb1 = ring0 + slot_tab[sc].x + (d.off0 >> 8) + ((d.off0 >> 4) & 15u);
            const uint32_t zo = smem_u32(smem + (d.y >> 8) * kWS) + kOffZ + zr;
            float2 za = make_float2(-INFINITY, -INFINITY), zb = za;
            if (gq < G) {
                za = lds_f32x2(zo + (uint32_t)pos * zstride);
                if (two) zb = lds_f32x2(zo + (uint32_t)(pos + 1) * zstride);
            }
            const float e00 = ex2(za.x - Mh), e01 = ex2(za.y - Mh), e10 = ex2(zb.x - Mh), e11 = ex2(zb.y - Mh);
            const uint32_t ph0 = pack_bf16(e00, e01), ph1 = pack_bf16(e10, e11);
            const uint32_t pl0 = pack_bf16(e00 - __uint_as_float(ph0 << 16), e01 - __uint_as_float(ph0 & 0xffff0000u));
            const uint32_t pl1 = pack_bf16(e10 - __uint_as_float(ph1 << 16), e11 - __uint_as_float(ph1 & 0xffff0000u));
            landed();  // the group's V parts have landed
            pv_group(acc, r_v, nb0, nb1, vb0, vb1, ph0, ph1, pl0, pl1, gq, qq);
            walked = true;
            __syncwarp();  // every lane is done reading the slot
            ring_release();
        }
    } else if (n_total > 0 && active) {
        walked = true;
        // the range's descriptors are still in shared memory unless it was longer than one ring: then describe again
        const bool redo = gbuilt > kDesc;
        if (redo) { bbuilt = 0; gbuilt = 0; }
        const int gtotal = gbuilt;
        int bposd = 0, gposd = 0;  // blocks / groups decided
#pragma unroll 1
        for (;;) {
            // ---- decide: softmax sums of the next groups; start the V copies of the groups that matter
#pragma unroll 1
            while (bposd < n_total) {
                if (redo) { if (gposd == gbuilt) describe(min(kDescribe, n_total - bbuilt)); }
                else if (gposd == gtotal) break;
                const GDesc d = d2[gposd & (kDesc - 1)];
                uint32_t nb0 = (d.y >> 4) & 15u, nb1 = (d.y >> 8) & 15u;
                const bool two = nb1 != 0u;
                bool need0 = nb0 != 0u, need1 = two;
                float add = 0.f;
                if (!kGatherOnly && nb0 != 0u) {
                    // lane (gq, qq): head gq, tokens 2qq, 2qq+1 of each block
                    float2 za = make_float2(-INFINITY, -INFINITY), zb = za;
                    if (gq < G) {
                        za = z_pair(bposd);
                        if (two) zb = z_pair(bposd + 1);
                    }
                    add = (ex2(za.x - Mh) + ex2(za.y - Mh)) + (ex2(zb.x - Mh) + ex2(zb.y - Mh));
                    need0 = __any_sync(kFull, fmaxf(za.x, za.y) - Mh >= -kSkip);
                    need1 = __any_sync(kFull, fmaxf(zb.x, zb.y) - Mh >= -kSkip);
                }
                if (need0 || need1) {
                    // a group with one block that matters becomes a one-block group
                    uint32_t off0 = d.off0, off1 = d.off1, c0 = (d.x & 255u) << 4, c1 = ((d.x >> 8) & 255u) << 4;
                    uint32_t sk0 = (d.x >> 16) & 15u, sk1 = (d.x >> 20) & 15u, shift = 0u;
                    if (!need0) { off0 = off1; c0 = c1; sk0 = sk1; nb0 = nb1; nb1 = 0u; c1 = 0u; shift = 1u; }
                    else if (!need1) { nb1 = 0u; c1 = 0u; }
                    uint32_t off;
                    if (!ring_alloc(c0 + c1, off)) break;  // no room yet: decide this group again after a consume
                    stage((d.y & 1u) ? reinterpret_cast<unsigned long long>(upd_v) : slice, off, off0, c0, off1, c1);
                    if (lane == 0) {
                        GDesc e;
                        e.off0 = sk0 | (sk1 << 4) | (c0 << 8);                   // skews of the V parts, bytes of the first chunk
                        e.off1 = (uint32_t)bposd + shift;                        // index of the first WALKED block in the range
                        e.x = d.x;
                        e.y = nb0 | (nb1 << 4);
                        slot_grp[si] = e;
                    }
                    st_vblocks += nb1 ? 2u : 1u;
                    st_vbytes += c0 + c1;
                    ring_commit();
                }
                lsum += add;
                ++gposd;
                bposd += two ? 2 : 1;
            }
            if (pend == 0) break;  // (nothing in flight means the decide loop ran to the end of the range)

            // ---- consume the oldest group in flight: PV
            const GDesc d = slot_grp[sc];
            const int r_v = (int)(d.x >> 24);
            const int nb0 = (int)(d.y & 15u), nb1 = (int)((d.y >> 4) & 15u), pos = (int)d.off1;
            const bool two = nb1 != 0;
            const uint32_t vb0 = ring0 + slot_tab[sc].x + (d.off0 & 15u);
            const uint32_t vb1 = ring0 + slot_tab[sc].x + (d.off0 >> 8) + ((d.off0 >> 4) & 15u);
            if (kGatherOnly) {
                landed();
                calib ^= lds_u32((vb0 & ~3u) + 4 * lane);
                __syncwarp();
                ring_release();
                continue;
            }
            // probabilities of head gq, tokens 2qq, 2qq+1 of each block, split into bf16 hi + lo:
            // exactly the B fragments of O^T += V^T P^T (k = token, n = head)
            float2 za = make_float2(-INFINITY, -INFINITY), zb = za;
            if (gq < G) {
                za = z_pair(pos);
                if (two) zb = z_pair(pos + 1);
            }
            const float e00 = ex2(za.x - Mh), e01 = ex2(za.y - Mh), e10 = ex2(zb.x - Mh), e11 = ex2(zb.y - Mh);
            const uint32_t ph0 = pack_bf16(e00, e01), ph1 = pack_bf16(e10, e11);
            const uint32_t pl0 = pack_bf16(e00 - __uint_as_float(ph0 << 16), e01 - __uint_as_float(ph0 & 0xffff0000u));
            const uint32_t pl1 = pack_bf16(e10 - __uint_as_float(ph1 << 16), e11 - __uint_as_float(ph1 & 0xffff0000u));
            landed();  // the group's V parts have landed
            pv_group(acc, r_v, nb0, nb1, vb0, vb1, ph0, ph1, pl0, pl1, gq, qq);
            __syncwarp();  // every lane is done reading the slot
            ring_release();
        }
    }
    if (kGatherOnly) {  // keep the read-back alive; nothing else is written
        if (calib == 0x9e3779b9u && lane == 0) scr.stats[7] = 1ull;
        return;
    }
    MKV_STAMP(7);  // phase 2 of this warp done (sums, lists, V parts fetched and walked)
    // counters of mkv_attention_stats: added up per CTA in shared memory; the CTA's three global reductions are issued
    // at the very end (4224 same-address reductions per launch, two per warp, used to sit in front of the cluster
    // barrier's release fence, which waits for them)
    if (lane == 0 && st_vblocks != 0u) {
        atomicAdd(&s_stat[0], st_vblocks);
        atomicAdd(&s_stat[1], st_vbytes);
    }

    // =====================================================================================
    // Step 3d.  Every partial of the unit is relative to the same maximum, so combining is plain addition (the
    // split-K rule of oracle pin P10 with equal references), always in the same order: warps inside the CTA, then
    // the cluster's CTAs.
    // =====================================================================================
    lsum += __shfl_xor_sync(kFull, lsum, 1);
    lsum += __shfl_xor_sync(kFull, lsum, 2);  // lanes (gq, *): the warp's sum of head gq (0 if it added nothing)
    if (qq == 0 && gq < G) s_l[warp][gq] = lsum;
    if (walked) {
        // the warp's partial: O^T fragments -> [head][channel] floats in the warp's (now idle) ring
        if (lane == 0) atomicOr(&s_active, 1u << warp);
        // Partials live in a swizzled order (o_slot): stored plainly, the 32 lanes of one of these stores would hit two
        // bank pairs (channel stride 16 floats over gq, head stride 128 floats over qq), 16 wavefronts each -- measured:
        // 2 us of shared-memory pipe per launch.  In o_slot order a half-warp's float2 stores cover 32 banks.  The sums
        // below run element-wise in that order; only the final store to `out` maps back.
        float* po = reinterpret_cast<float*>(wbase);
        const int hA = 2 * qq, hB = 2 * qq + 1;
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            const int in = (16 * i + 2 * gq + 8 * qq) & (kD - 1);  // o_slot of channel 16 gq + 2 i for heads 2 qq, 2 qq + 1
            if (hA < G) *reinterpret_cast<float2*>(po + hA * kD + in) = make_float2(acc[i][0], acc[i][2]);
            if (hB < G) *reinterpret_cast<float2*>(po + hB * kD + in) = make_float2(acc[i][1], acc[i][3]);
        }
    }
    __syncthreads();
    MKV_STAMP(8);  // warps' partials stored, CTA barrier passed
    const int GD = G * kD;
    // A cluster of two (64 units on 148 SMs): the second CTA PUSHES its partial into the first one's shared memory, so
    // after the barrier the first CTA adds two local arrays and the second one is free to leave: no remote loads on the
    // critical path and no third barrier.  Larger clusters are pulled by the first CTA (no room for 16 partials).
    const bool push = C == 2;
    const unsigned wmask = s_active;  // (in warp order: the sums are reproducible)
    const uint32_t peer_o = dsmem_addr(smem_u32(s_peer_o), 0u), peer_l = dsmem_addr(smem_u32(s_peer_l), 0u);
    const uint32_t peer_bar = dsmem_addr(smem_u32(&s_xbar[1]), 0u);
    auto flush_stats = [&]() {  // (s_stat is complete since the CTA barrier above)
        if (threadIdx.x == 0) {
            if (s_stat[0] != 0u) {
                atomicAdd(scr.stats + 1, (unsigned long long)s_stat[0]);
                atomicAdd(scr.stats + 2, (unsigned long long)s_stat[1]);
            }
            if (rank == 0) atomicAdd(scr.stats + 0, (unsigned long long)T);
        }
    };
    for (int e = threadIdx.x; e < GD; e += kNT) {  // the CTA's partial
        float o = 0.f, v[kWarps];
#pragma unroll
        for (int w = 0; w < kWarps; ++w) v[w] = (wmask >> w) & 1u ? *reinterpret_cast<const float*>(smem + w * kWS + 4 * e) : 0.f;
#pragma unroll
        for (int w = 0; w < kWarps; ++w) o += v[w];  // (warp order, as ever: an idle warp adds +0)
        if (push && rank != 0) st_async_b32(peer_o + 4u * (uint32_t)e, __float_as_uint(o), peer_bar);
        else s_cta_o[e] = o;
    }
    MKV_STAMP(12);  // (between 8 and 9) the CTA's partial O summed
    if (threadIdx.x < G) {
        float l = 0.f;
#pragma unroll
        for (int w = 0; w < kWarps; ++w) l += s_l[w][threadIdx.x];
        if (push && rank != 0) st_async_b32(peer_l + 4u * threadIdx.x, __float_as_uint(l), peer_bar);
        else s_cta_l[threadIdx.x] = l;
    }
    MKV_STAMP(9);    // CTA partial summed (and pushed)
    if (push) {
        // A cluster of two: the second CTA has sent its partial (asynchronous remote stores counted on the first CTA's
        // mbarrier) and leaves; the first waits for the G x 129 floats to land.  No cluster barrier, no fence.
        if (rank == 0) {
            __syncthreads();  // s_cta_o / s_cta_l of this CTA are complete
            mbar_wait(smem_u32(&s_xbar[1]), 0u);
        }
        MKV_STAMP(10);   // (first CTA) the peer's partial has landed
        flush_stats();
        if (rank == 0) {
            for (int e = threadIdx.x; e < GD; e += kNT) {
                const int h = e >> 7, es = o_slot(e);
                const float o = s_cta_o[es] + s_peer_o[es], l = s_cta_l[h] + s_peer_l[h];
                out[row * kD + e] = l > 0.f ? o / l : 0.f;
                if (lse != nullptr && (e & (kD - 1)) == 0) lse[row + h] = l > 0.f ? (s_M[h] + log2f(l)) * kLn2 : -INFINITY;
            }
        }
        MKV_STAMP(11);  // output stored (rank 0) / leaving (rank 1)
        return;
    }
    cluster_sync();  // every CTA's partial is complete and visible to the cluster
    MKV_STAMP(10);   // second cluster barrier passed
    flush_stats();
    if (rank == 0) {
        const uint32_t ao = smem_u32(s_cta_o), al = smem_u32(s_cta_l);
        for (int e = threadIdx.x; e < GD; e += kNT) {
            const int h = e >> 7, es = o_slot(e);
            float o = 0.f, l = 0.f;
#pragma unroll 1
            for (int r0 = 0; r0 < C; r0 += 4) {  // (eight remote loads in flight; ranks past the cluster add nothing)
                float vo[4], vl[4];
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    const uint32_t r = (uint32_t)min(r0 + j, C - 1);
                    vo[j] = ld_dsmem_f32(dsmem_addr(ao + 4u * (uint32_t)es, r));
                    vl[j] = ld_dsmem_f32(dsmem_addr(al + 4u * (uint32_t)h, r));
                }
#pragma unroll
                for (int j = 0; j < 4; ++j)
                    if (r0 + j < C) { o += vo[j]; l += vl[j]; }
            }
            out[row * kD + e] = l > 0.f ? o / l : 0.f;
            if (lse != nullptr && (e & (kD - 1)) == 0) lse[row + h] = l > 0.f ? (s_M[h] + log2f(l)) * kLn2 : -INFINITY;
        }
    }
    cluster_sync();  // no CTA leaves (and releases its shared memory) before the first one has read it
    MKV_STAMP(11);   // output stored, third cluster barrier passed
}


// calibration row (i) of SURVEY 8(d): a plain streaming read of `bytes` bytes in the attention kernel's launch shape
__global__ void __launch_bounds__(kWarps * 32, 1)
mkv_stream_read_kernel(const uint4* __restrict__ base, unsigned long long n16, unsigned long long* __restrict__ sink) {
    pdl_wait();
    pdl_launch_dependents();
    const unsigned long long stride = (unsigned long long)gridDim.x * blockDim.x;
    uint32_t acc = 0u;
    unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;
#pragma unroll 1
    for (; i + 3ull * stride < n16; i += 4ull * stride) {  // four independent 16-byte loads in flight per thread
        uint4 v[4];
#pragma unroll
        for (int j = 0; j < 4; ++j)
            asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];"
                         : "=r"(v[j].x), "=r"(v[j].y), "=r"(v[j].z), "=r"(v[j].w) : "l"(base + i + j * stride));
#pragma unroll
        for (int j = 0; j < 4; ++j) acc ^= v[j].x ^ v[j].y ^ v[j].z ^ v[j].w;
    }
#pragma unroll 1
    for (; i < n16; i += stride) {
        uint4 v;
        asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];"
                     : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(base + i));
        acc ^= v.x ^ v.y ^ v.z ^ v.w;
    }
    if (acc == 0x9e3779b9u) *sink = acc;  // keeps the loads alive
}


// calibration row (iii): the QK expansion alone.  Every warp copies the K parts of ONE group of the real selection (two
// consecutive selected blocks of a unit) into shared memory and then runs qk_group() on it `reps` times: no staging, no
// logits, no softmax, no output.  (t(reps2) - t(reps1)) / (reps2 - reps1) / kWarps is the time one SM needs per group
// when nothing but the expansion runs: the floor the shared-memory pipe sets for phase 1 (and for the score kernel).
__global__ void __launch_bounds__(kWarps * 32, 1)
mkv_walk_probe_kernel(CacheGeom g, LayerView lv, const uint16_t* __restrict__ q, const int32_t* __restrict__ sel,
                      const int32_t* __restrict__ sel_count, int k_max, int reps, unsigned long long* __restrict__ sink) {
    extern __shared__ __align__(128) uint8_t smem[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, gq = lane >> 2, qq = lane & 3;
    const int wi = blockIdx.x * kWarps + warp;
    const int u = wi % g.n_units;
    const int cnt = min(min(max(__ldg(sel_count + u), 0), k_max), g.score_stride + 1) * g.ppb;  // as mkv_packed_attention cuts it
    const int pairs = cnt >> 1;
    if (pairs == 0) return;
    const int j = 2 * ((wi / g.n_units) % pairs);
    uint32_t off[2], meta[2];
#pragma unroll
    for (int i = 0; i < 2; ++i) {
        const int ts = __ldg(sel + (size_t)u * k_max + ((j + i) >> (g.ppb - 1)));
        plan_lookup(g, lv, u, ts < 0 ? -1 : ts + kPhys * ((j + i) & (g.ppb - 1)), off[i], meta[i]);
    }
    uint8_t* mine = smem + warp * 4096;
    const uint32_t sp0 = smem_u32(mine), sp1 = sp0 + 2048;
#pragma unroll
    for (int i = 0; i < 2; ++i) {
        const uint32_t nb = (meta[i] >> 16) & 15u, kb = (nb * vecb(meta[i] & 255u) + 15u) >> 4;  // 16-B units of the K part (<= 128)
        const uint4* src = reinterpret_cast<const uint4*>(lv.slice) + off[i];
        for (uint32_t x = lane; x < kb; x += 32) reinterpret_cast<uint4*>(mine + 2048 * i)[x] = __ldg(src + x);
    }
    __syncwarp();
    const int r_k = (int)(meta[0] & 255u);
    const int nb0 = (int)((meta[0] >> 16) & 15u);
    const int nb1 = ((meta[1] ^ meta[0]) & 0x010000ffu) == 0u ? (int)((meta[1] >> 16) & 15u) : 0;
    const size_t row = (size_t)(u / g.n_kv_heads) * g.n_q_heads + (size_t)(u % g.n_kv_heads) * g.group;
    uint32_t qa[8][2];
    {
        const uint4* qrow = reinterpret_cast<const uint4*>(q + (row + gq) * kD + 32 * qq);
#pragma unroll
        for (int h = 0; h < 4; ++h) {
            uint4 v = make_uint4(0u, 0u, 0u, 0u);
            if (gq < g.group) v = __ldg(qrow + h);
            qa[2 * h][0] = v.x; qa[2 * h][1] = v.y; qa[2 * h + 1][0] = v.z; qa[2 * h + 1][1] = v.w;
        }
    }
    float acc = 0.f;
#pragma unroll 1
    for (int it = 0; it < reps; ++it) {
        float S[4] = {0.f, 0.f, 0.f, 0.f};
        qk_group(S, r_k, nb0, nb1, sp0, sp1, qa, lane, (meta[0] >> 24) & 1u);
        acc += (S[0] + S[1]) + (S[2] + S[3]);
        qa[0][0] ^= __float_as_uint(acc) & 0x10000u;  // loop-carried: the walk cannot be hoisted out of the loop
    }
    if (acc == 1234.56789f) *sink = 1ull;  // keeps the arithmetic alive
}

}  // namespace

// logit scratch: per unit one entry of 8 G floats per position of its block stream (selected + update-buffer blocks)
size_t attention_z_unit_stride(const CacheGeom& g) { return ((size_t)g.score_stride + 1) * g.ppb + (size_t)(g.L + kPhys - 1) / kPhys; }
size_t attention_zbuf_floats(const CacheGeom& g) { return (size_t)g.n_units * attention_z_unit_stride(g) * 8 * (size_t)g.group; }

// Cluster size for a layer of n_units units: the largest power of two C <= 16 with n_units * C <= SMs whose clusters
// can all be resident at once (one CTA per SM; a cluster lives inside one GPC), else 1.  (Sizes that are not powers of
// two were tried for 8 units: 10 CTAs per unit are schedulable, 16 are not, and 10 was no faster than 8.)
template <bool GATHER>
static int pick_cluster(const CacheGeom& g, int smem, int sm_count) {
    cudaFuncSetAttribute(mkv_packed_attention_kernel<GATHER>, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
    for (int C = kMaxCluster; C > 1; C >>= 1) {
        if ((long long)g.n_units * C > sm_count) continue;
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3(g.n_units * C); cfg.blockDim = dim3(kWarps * 32); cfg.dynamicSmemBytes = smem;
        cudaLaunchAttribute attr[1];
        attr[0].id = cudaLaunchAttributeClusterDimension;
        attr[0].val.clusterDim.x = C; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
        cfg.attrs = attr; cfg.numAttrs = 1;
        int n = 0;
        if (cudaOccupancyMaxActiveClusters(&n, mkv_packed_attention_kernel<GATHER>, &cfg) == cudaSuccess && n >= g.n_units)
            return C;
        cudaGetLastError();
    }
    return 1;
}

template <bool GATHER>
static cudaError_t launch_attention_cfg(const CacheGeom& g, const LayerView& lv, const uint16_t* q, const int32_t* sel,
                                        const int32_t* sel_count, int k_max, float scale, float* out, float* lse,
                                        const AttnScratch& scr, const uint16_t* upd_k, const uint16_t* upd_v,
                                        const int32_t* upd_count, int sm_count, int* cluster_cache, cudaStream_t s) {
    const int smem = kWarps * kWS + 2 * kMaxGroup * kD * 4;
    // the dynamic shared-memory opt-in is a per-device attribute of the function: set it on every launch (a cheap
    // host-side call) so that caches on different devices of one process are independent
    cudaError_t e = cudaFuncSetAttribute(mkv_packed_attention_kernel<GATHER>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    if (e != cudaSuccess) return e;
    if (*cluster_cache == 0) *cluster_cache = pick_cluster<GATHER>(g, smem, sm_count);  // (normally chosen at cache creation)
    const int C = *cluster_cache;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(g.n_units * C); cfg.blockDim = dim3(kWarps * 32); cfg.dynamicSmemBytes = smem; cfg.stream = s;
    cudaLaunchAttribute attr[2];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    attr[1].id = cudaLaunchAttributeClusterDimension;
    attr[1].val.clusterDim.x = C; attr[1].val.clusterDim.y = 1; attr[1].val.clusterDim.z = 1;
    cfg.attrs = attr; cfg.numAttrs = 2;
    return cudaLaunchKernelEx(&cfg, mkv_packed_attention_kernel<GATHER>, g, lv, q, sel, sel_count, k_max, scale * kLog2e, out,
                              lse, scr, upd_k, upd_v, upd_count, C);
}

cudaError_t launch_attention(const CacheGeom& g, const LayerView& lv, const uint16_t* q, const int32_t* sel,
                             const int32_t* sel_count, int k_max, float scale, float* out, float* lse,
                             const AttnScratch& scr, const uint16_t* upd_k, const uint16_t* upd_v,
                             const int32_t* upd_count, int sm_count, int* cluster_cache, cudaStream_t s, int* n_kernels,
                             bool gather_only) {
    if (n_kernels) *n_kernels = 1;
    if (gather_only)
        return launch_attention_cfg<true>(g, lv, q, sel, sel_count, k_max, scale, out, lse, scr, upd_k, upd_v, upd_count,
                                          sm_count, cluster_cache + 1, s);
    return launch_attention_cfg<false>(g, lv, q, sel, sel_count, k_max, scale, out, lse, scr, upd_k, upd_v, upd_count,
                                       sm_count, cluster_cache, s);
}

// choose the cluster sizes of both kernels for this cache (occupancy queries: host-side, not capturable)
cudaError_t attention_prepare(const CacheGeom& g, int sm_count, int* cluster_cache) {
    const int smem = kWarps * kWS + 2 * kMaxGroup * kD * 4;
    cudaError_t e = cudaFuncSetAttribute(mkv_packed_attention_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(mkv_packed_attention_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    if (e != cudaSuccess) return e;
    cluster_cache[0] = pick_cluster<false>(g, smem, sm_count);
    cluster_cache[1] = pick_cluster<true>(g, smem, sm_count);
    return cudaSuccess;
}

cudaError_t launch_stream_read(const uint8_t* base, unsigned long long bytes, int sm_count, unsigned long long* sink,
                               cudaStream_t s) {
    return launch_pdl(mkv_stream_read_kernel, dim3(sm_count), dim3(kWarps * 32), (size_t)0, s,
                      reinterpret_cast<const uint4*>(base), bytes / 16ull, sink);
}

cudaError_t launch_walk_probe(const CacheGeom& g, const LayerView& lv, const uint16_t* q, const int32_t* sel,
                              const int32_t* sel_count, int k_max, int reps, int sm_count, unsigned long long* sink,
                              cudaStream_t s) {
    const int smem = kWarps * 4096;
    cudaError_t e = cudaFuncSetAttribute(mkv_walk_probe_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    if (e != cudaSuccess) return e;
    mkv_walk_probe_kernel<<<sm_count, kWarps * 32, smem, s>>>(g, lv, q, sel, sel_count, k_max, reps, sink);
    return cudaGetLastError();
}

}  // namespace mkv

#ifdef MKV_TRACE
// trace build only (not in include/mkv.h, not in libmkv.so): the stamps of the last mkv_packed_attention launch on the
// current device, [kTraceCtas = 160][16 warps][16] x u64 nanoseconds of %globaltimer (0 = never written).  Synchronises.
extern "C" __attribute__((visibility("default"))) int mkv_trace_read(unsigned long long* host, unsigned long long cap_bytes,
                                                                     int clear) {
    using namespace mkv;
    if (!host || cap_bytes < sizeof(g_trace)) return MKV_E_ARG;
    if (cudaDeviceSynchronize() != cudaSuccess) return MKV_E_CUDA;
    if (cudaMemcpyFromSymbol(host, g_trace, sizeof(g_trace)) != cudaSuccess) return MKV_E_CUDA;
    if (clear) {
        void* p = nullptr;
        if (cudaGetSymbolAddress(&p, g_trace) != cudaSuccess || cudaMemset(p, 0, sizeof(g_trace)) != cudaSuccess) return MKV_E_CUDA;
    }
    return MKV_OK;
}
#endif
