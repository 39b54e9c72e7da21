// attention.cu — step 3 of the hot path: PackedAttention: QK over the
// selected packed keys, online softmax, PV over the packed values, split-K combine.  sm_100a.
//
// Design:
//   * The selected blocks of all units form one stream of T blocks; it is cut into equal ranges,
//     one per warp of a one-CTA-per-SM grid (warps are fully independent: no __syncthreads in
//     the main loop).  A warp walks its range in groups of <= 4 token blocks (32 tokens).
//   * Each group's packed payloads (one contiguous chunk per block, DESIGN.md format) are brought
//     into a per-warp shared-memory stage by cp.async.bulk (TMA bulk engine) completing on an
//     mbarrier; kStages groups are in flight per warp.
//   * lane = token: every lane expands its token's packed K vector (bitmap + kept bf16) into a
//     dense bf16 row of a [32 tokens][128 ch] tile, the warp runs QK^T on the tensor cores
//     (mma.sync m16n8k16, tokens = M, heads = N), an online softmax in the exp2 domain, expands V
//     into the same tile and runs PV with P split into bf16 hi + lo (fp32-class accuracy).
//   * A unit wholly inside one warp's range is normalised and written directly; otherwise the
//     warp writes an (m, l, O) partial (<= 2 per warp) that the combine kernel merges (step 3d).
#include "mkv_internal.cuh"

namespace mkv {

namespace {

constexpr unsigned kFull = 0xffffffffu;
constexpr float kLog2e = 1.4426950408889634f;
constexpr float kLn2 = 0.6931471805599453f;

constexpr int kWarps = 10;                    // warps per CTA (one CTA per SM)
constexpr int kStages = 2;                    // groups in flight per warp
constexpr int kStageBytes = 6144;             // >= 4 blocks at r = 38 (5888 B), >= 1 dense block (4096 B)
constexpr int kTileStride = 272;              // bytes per token row: 256 + 16 pad (ldmatrix conflict-free)
constexpr int kTileBytes = 32 * kTileStride;  // 8704
constexpr int kDescRing = 64;                 // block descriptors kept per warp
constexpr int kMaxUnitsSmem = 2048;

struct __align__(16) Desc {   // one selected token block
    uint32_t off16;           // payload offset in the layer slice, 16-B units
    uint32_t bytes;           // payload bytes (multiple of 16); 0 = skip (invalid entry)
    int32_t unit;
    uint8_t r_k, r_v, nb, pad;
};
struct __align__(16) GInfo {  // one block of an in-flight group
    uint32_t off;             // byte offset inside the stage
    uint32_t r_k, r_v, nb;
};

// ---- PTX wrappers ---------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(bar),
        "r"(parity)
        : "memory");
}
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
                 "l"(src), "r"(bytes), "r"(bar)
                 : "memory");
}
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void ldmatrix_x4(uint32_t addr, uint32_t (&r)[4]) {
    asm volatile("ldmatrix.sync.aligned.m8n8.x4.shared.b16 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3])
                 : "r"(addr));
}
__device__ __forceinline__ void ldmatrix_x4_trans(uint32_t addr, uint32_t (&r)[4]) {
    asm volatile("ldmatrix.sync.aligned.m8n8.x4.trans.shared.b16 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3])
                 : "r"(addr));
}
__device__ __forceinline__ uint32_t movmatrix_trans(uint32_t a) {
    uint32_t d;
    asm volatile("movmatrix.sync.aligned.m8n8.trans.b16 %0, %1;" : "=r"(d) : "r"(a));
    return d;
}
__device__ __forceinline__ void mma_bf16(float (&c)[4], const uint32_t (&a)[4], uint32_t b0, uint32_t b1) {
    asm volatile(
        "mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
        : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
        : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}
__device__ __forceinline__ float ex2(float x) {
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
// bf16x2 of (lo, hi) rounded to nearest even; lo in the low half
__device__ __forceinline__ uint32_t pack_bf16(float lo, float hi) {
    uint32_t d;
    asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(d) : "f"(hi), "f"(lo));
    return d;
}
__device__ __forceinline__ void sts_u16(uint32_t addr, uint32_t v) {
    asm volatile("st.shared.u16 [%0], %1;" ::"r"(addr), "h"((unsigned short)v));
}
__device__ __forceinline__ uint32_t lds_u16(uint32_t addr) {
    unsigned short v;
    asm volatile("ld.shared.u16 %0, [%1];" : "=h"(v) : "r"(addr));
    return v;
}
__device__ __forceinline__ uint4 lds_128(uint32_t addr) {
    uint4 v;
    asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(addr));
    return v;
}
__device__ __forceinline__ void sts_128(uint32_t addr, uint4 v) {
    asm volatile("st.shared.v4.u32 [%0], {%1,%2,%3,%4};" ::"r"(addr), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w));
}

// ---- lane = token: expand one packed (or dense) vector into this lane's dense tile row ------
// row: shared address of the lane's 256-byte tile row; bm / val: shared addresses in the stage.
// Kept values are consumed from the highest channel down (FLO gives the top set bit directly).
__device__ __forceinline__ void expand_row(uint32_t row, uint32_t bm, uint32_t val, int r, bool valid) {
    const uint4 z4 = make_uint4(0u, 0u, 0u, 0u);
    if (!valid) {
#pragma unroll
        for (int i = 0; i < 16; ++i) sts_128(row + 16 * i, z4);
        return;
    }
    if (r == kD) {
        if ((val & 15u) == 0) {
#pragma unroll
            for (int i = 0; i < 16; ++i) sts_128(row + 16 * i, lds_128(val + 16 * i));
        } else {  // ragged token block: values only 2-byte aligned
            for (int c = 0; c < kD; ++c) sts_u16(row + 2 * c, lds_u16(val + 2 * c));
        }
        return;
    }
#pragma unroll
    for (int i = 0; i < 16; ++i) sts_128(row + 16 * i, z4);
    uint32_t w[4];
    if ((bm & 15u) == 0) {
        const uint4 b = lds_128(bm);
        w[0] = b.x; w[1] = b.y; w[2] = b.z; w[3] = b.w;
    } else {
#pragma unroll
        for (int j = 0; j < 4; ++j) w[j] = lds_u16(bm + 4 * j) | (lds_u16(bm + 4 * j + 2) << 16);
    }
    uint32_t vp = val + 2 * (uint32_t)(r - 1);  // address of the last kept value
#pragma unroll
    for (int j = 3; j >= 0; --j) {
        uint32_t wj = w[j];
        const uint32_t base = row + 64 * j;
        while (wj) {
            const int pos = 31 - __clz(wj);
            wj ^= 1u << pos;
            sts_u16(base + 2 * pos, lds_u16(vp));
            vp -= 2;
        }
    }
}

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

__host__ __device__ constexpr int warp_smem_bytes(int nstage) {
    return nstage * kStageBytes + kTileBytes + kDescRing * 16 + nstage * 64 + 64;
}

// ------------------------------------------------------------------------------------------
// main kernel: one CTA per SM, kWarps independent warps, each owning the block range
// [gw*T/GW, (gw+1)*T/GW) of the concatenated selection lists.
// ------------------------------------------------------------------------------------------
template <int NSTAGE>
__global__ void __launch_bounds__(kWarps * 32, 1)
mkv_packed_attention_kernel(CacheGeom g, LayerView lv, const uint16_t* __restrict__ q,
                            const int32_t* __restrict__ sel, const int32_t* __restrict__ sel_count, int k_max,
                            float scale_log2, float* __restrict__ out, float* __restrict__ lse,
                            float* __restrict__ part_o, float* __restrict__ part_ml) {
    extern __shared__ __align__(128) uint8_t smem[];
    constexpr int kWS = warp_smem_bytes(NSTAGE);
    int* s_cum = reinterpret_cast<int*>(smem + kWarps * kWS);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int gq = lane >> 2, qq = lane & 3;  // mma fragment coordinates

    const int T = scan_counts(sel_count, g.n_units, k_max, s_cum);
    const int GW = gridDim.x * kWarps, gw = blockIdx.x * kWarps + warp;
    const int lo = (int)((unsigned long long)gw * (unsigned)T / (unsigned)GW);
    const int hi = (int)((unsigned long long)(gw + 1) * (unsigned)T / (unsigned)GW);
    if (lo >= hi) return;
    const int n_total = hi - lo;

    uint8_t* wbase = smem + warp * kWS;
    const uint32_t stage0 = smem_u32(wbase);
    const uint32_t tile = stage0 + NSTAGE * kStageBytes;
    Desc* desc = reinterpret_cast<Desc*>(wbase + NSTAGE * kStageBytes + kTileBytes);
    GInfo* ginfo = reinterpret_cast<GInfo*>(wbase + NSTAGE * kStageBytes + kTileBytes + kDescRing * 16);
    int2* gmeta = reinterpret_cast<int2*>(reinterpret_cast<uint8_t*>(ginfo) + NSTAGE * 64);  // (unit, n)
    const uint32_t bar0 = smem_u32(gmeta) + NSTAGE * 8;

    if (lane == 0) {
#pragma unroll
        for (int s = 0; s < NSTAGE; ++s) mbar_init(bar0 + 8 * s, 1);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    fence_proxy_async();
    __syncwarp();

    int pos = 0, built = 0;

    auto build = [&](int count) {
        if (lane < count) {
            const int idx = built + lane;
            const int gi = lo + idx;
            const int u = find_unit(s_cum, g.n_units, gi);
            const int j = gi - s_cum[u];
            const int t0 = sel[(size_t)u * k_max + j];
            Desc d;
            d.unit = u; d.off16 = 0; d.bytes = 0; d.r_k = 0; d.r_v = 0; d.nb = 0; d.pad = 0;
            const int ntok = lv.unit_ntok[u];
            if (t0 >= 0 && t0 < ntok && (t0 & (kB - 1)) == 0) {
                const int seg = t0 / g.L, in_seg = t0 - seg * g.L;
                const size_t e = (size_t)u * lv.S_max + seg;
                const StratRec rec = lv.strat[e];
                const int nb = min(kB, (int)rec.n_tok - in_seg);
                d.off16 = lv.tok_off[e] + (uint32_t)(in_seg >> 3) * (tokblock_bytes(rec.r_k, rec.r_v, kB) >> 4);
                d.bytes = tokblock_bytes(rec.r_k, rec.r_v, nb);
                d.r_k = rec.r_k; d.r_v = rec.r_v; d.nb = (uint8_t)nb;
            }
            desc[idx & (kDescRing - 1)] = d;
        }
        built += count;
        __syncwarp();
    };

    // form the next group (<= 4 blocks of one unit, <= kStageBytes) and start its bulk copies
    auto issue = [&](int s) {
        if (built - pos <= 8 && built < n_total) build(min(32, n_total - built));
        if (pos >= n_total) {
            if (lane == 0) gmeta[s] = make_int2(-1, 0);
            return;
        }
        const bool have = lane < 4 && pos + lane < built;
        Desc d;
        d.unit = -2; d.bytes = 0; d.off16 = 0; d.r_k = 0; d.r_v = 0; d.nb = 0; d.pad = 0;
        if (have) d = desc[(pos + lane) & (kDescRing - 1)];
        const int unit0 = __shfl_sync(kFull, d.unit, 0);
        uint32_t cum = d.bytes;
#pragma unroll
        for (int o = 1; o < 4; o <<= 1) {
            const uint32_t v = __shfl_up_sync(kFull, cum, o);
            if (lane >= o) cum += v;
        }
        const bool ok = have && d.unit == unit0 && cum <= (uint32_t)kStageBytes;
        const unsigned mask = __ballot_sync(kFull, ok) & 0xFu;
        const int n = __ffs(~mask) - 1;  // leading run of ok lanes (lane 0 is always ok)
        const uint32_t total = __shfl_sync(kFull, cum, n - 1);
        if (lane < n) {
            GInfo gi;
            gi.off = cum - d.bytes; gi.r_k = d.r_k; gi.r_v = d.r_v; gi.nb = d.nb;
            ginfo[s * 4 + lane] = gi;
        }
        const uint32_t bar = bar0 + 8 * s;
        if (lane == 0) {
            gmeta[s] = make_int2(unit0, n);
            mbar_expect_tx(bar, total);
        }
        if (lane < n && d.bytes > 0)
            bulk_g2s(stage0 + s * kStageBytes + (cum - d.bytes), lv.slice + ((size_t)d.off16 << 4), d.bytes, bar);
        pos += n;
    };

    build(min(32, n_total));
#pragma unroll
    for (int s = 0; s < NSTAGE; ++s) issue(s);

    // per-unit state
    uint32_t bq[8][2];
    float acc[8][4];
    float m0 = -INFINITY, m1 = -INFINITY, l0 = 0.f, l1 = 0.f;
    int cur_unit = -1;

    auto flush = [&]() {
        const int u = cur_unit;
        const int a = s_cum[u], b = s_cum[u + 1];
#pragma unroll
        for (int o = 4; o < 32; o <<= 1) {
            l0 += __shfl_xor_sync(kFull, l0, o);
            l1 += __shfl_xor_sync(kFull, l1, o);
        }
        const int G = g.group;
        const int h0 = 2 * qq, h1 = 2 * qq + 1;
        if (lo <= a && b <= hi) {  // the whole unit was processed by this warp: final result
            const int bi = u / g.n_kv_heads, hk = u % g.n_kv_heads;
            const size_t row = (size_t)bi * g.n_q_heads + (size_t)hk * G;
            const float i0 = l0 > 0.f ? 1.f / l0 : 0.f, i1 = l1 > 0.f ? 1.f / l1 : 0.f;
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                const int ch = 16 * i + gq;
                if (h0 < G) { out[(row + h0) * kD + ch] = acc[i][0] * i0; out[(row + h0) * kD + ch + 8] = acc[i][2] * i0; }
                if (h1 < G) { out[(row + h1) * kD + ch] = acc[i][1] * i1; out[(row + h1) * kD + ch + 8] = acc[i][3] * i1; }
            }
            if (lse != nullptr && gq == 0) {
                if (h0 < G) lse[row + h0] = l0 > 0.f ? (m0 + log2f(l0)) * kLn2 : -INFINITY;
                if (h1 < G) lse[row + h1] = l1 > 0.f ? (m1 + log2f(l1)) * kLn2 : -INFINITY;
            }
        } else {
            const size_t slot = (size_t)gw * 2 + (a < lo ? 0 : 1);
            float* po = part_o + slot * (size_t)(G * kD);
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                const int ch = 16 * i + gq;
                if (h0 < G) { po[h0 * kD + ch] = acc[i][0]; po[h0 * kD + ch + 8] = acc[i][2]; }
                if (h1 < G) { po[h1 * kD + ch] = acc[i][1]; po[h1 * kD + ch + 8] = acc[i][3]; }
            }
            if (gq == 0) {
                float* pm = part_ml + slot * (size_t)(2 * kMaxGroup);
                if (h0 < G) { pm[2 * h0] = m0; pm[2 * h0 + 1] = l0; }
                if (h1 < G) { pm[2 * h1] = m1; pm[2 * h1 + 1] = l1; }
            }
        }
    };

    const uint32_t my_row = tile + (uint32_t)lane * kTileStride;
    const int mi = lane >> 3, mr = lane & 7;
    // ldmatrix lane addresses: QK (A = K tile rows) and PV (A = V tile transposed)
    const uint32_t a_qk = tile + (uint32_t)(((mi & 1) * 8 + mr) * kTileStride + (mi >> 1) * 16);
    const uint32_t a_pv = tile + (uint32_t)(((mi >> 1) * 8 + mr) * kTileStride + (mi & 1) * 16);

    for (int k = 0;; ++k) {
        const int s = k % NSTAGE;
        __syncwarp();
        const int2 meta = gmeta[s];
        const int n = meta.y;
        if (n == 0) break;
        if (meta.x != cur_unit) {
            if (cur_unit >= 0) flush();
            cur_unit = meta.x;
            const int bi = cur_unit / g.n_kv_heads, hk = cur_unit % g.n_kv_heads;
            const uint32_t* qrow = reinterpret_cast<const uint32_t*>(
                q + ((size_t)bi * g.n_q_heads + (size_t)hk * g.group + gq) * kD);
#pragma unroll
            for (int ks = 0; ks < 8; ++ks) {
                bq[ks][0] = gq < g.group ? __ldg(qrow + ks * 8 + qq) : 0u;
                bq[ks][1] = gq < g.group ? __ldg(qrow + ks * 8 + 4 + qq) : 0u;
            }
#pragma unroll
            for (int i = 0; i < 8; ++i) acc[i][0] = acc[i][1] = acc[i][2] = acc[i][3] = 0.f;
            m0 = m1 = -INFINITY;
            l0 = l1 = 0.f;
        }
        const GInfo gi = ginfo[s * 4 + mi];
        int nbj[4];
#pragma unroll
        for (int j = 0; j < 4; ++j) nbj[j] = j < n ? (int)ginfo[s * 4 + j].nb : 0;
        const bool valid = mi < n && mr < (int)gi.nb;
        const uint32_t bmk = gi.r_k == kD ? 0u : (uint32_t)kBitmapBytes, bmv = gi.r_v == kD ? 0u : (uint32_t)kBitmapBytes;
        const uint32_t sp = stage0 + s * kStageBytes + gi.off;
        const uint32_t k_bm = sp + mr * bmk;
        const uint32_t k_val = sp + gi.nb * bmk + mr * gi.r_k * 2;
        const uint32_t v_bm0 = sp + gi.nb * (bmk + 2 * gi.r_k);
        const uint32_t v_bm = v_bm0 + mr * bmv;
        const uint32_t v_val = v_bm0 + gi.nb * bmv + mr * gi.r_v * 2;

        mbar_wait(bar0 + 8 * s, (uint32_t)(k / NSTAGE) & 1u);

        // ---- K: expand, S = K q^T on the tensor cores (tokens = M, heads = N)
        expand_row(my_row, k_bm, k_val, (int)gi.r_k, valid);
        __syncwarp();
        float S[2][4];
#pragma unroll
        for (int mt = 0; mt < 2; ++mt) {
            S[mt][0] = S[mt][1] = S[mt][2] = S[mt][3] = 0.f;
#pragma unroll
            for (int ks = 0; ks < 8; ++ks) {
                uint32_t a[4];
                ldmatrix_x4(a_qk + mt * 16 * kTileStride + ks * 32, a);
                mma_bf16(S[mt], a, bq[ks][0], bq[ks][1]);
            }
        }
        __syncwarp();  // every lane's ldmatrix reads are done: the tile may be overwritten
        // ---- V: expand into the same tile (overlaps the softmax arithmetic below)
        expand_row(my_row, v_bm, v_val, (int)gi.r_v, valid);
        __syncwarp();
        fence_proxy_async();
        issue(s);  // stage s is free: start the copies of group k + NSTAGE

        // ---- online softmax in the exp2 domain; this lane: tokens 8j + gq (j = 0..3), heads 2qq, 2qq+1
        float mx0 = -INFINITY, mx1 = -INFINITY;
#pragma unroll
        for (int mt = 0; mt < 2; ++mt) {
#pragma unroll
            for (int hf = 0; hf < 2; ++hf) {
                const bool tv = gq < nbj[mt * 2 + hf];
                S[mt][2 * hf] = tv ? S[mt][2 * hf] * scale_log2 : -INFINITY;
                S[mt][2 * hf + 1] = tv ? S[mt][2 * hf + 1] * scale_log2 : -INFINITY;
                mx0 = fmaxf(mx0, S[mt][2 * hf]);
                mx1 = fmaxf(mx1, S[mt][2 * hf + 1]);
            }
        }
#pragma unroll
        for (int o = 4; o < 32; o <<= 1) {
            mx0 = fmaxf(mx0, __shfl_xor_sync(kFull, mx0, o));
            mx1 = fmaxf(mx1, __shfl_xor_sync(kFull, mx1, o));
        }
        const float mn0 = fmaxf(m0, mx0), mn1 = fmaxf(m1, mx1);
        const float b0 = mn0 == -INFINITY ? 0.f : mn0, b1 = mn1 == -INFINITY ? 0.f : mn1;
        const float c0 = ex2(m0 - b0), c1 = ex2(m1 - b1);
        if (__any_sync(kFull, mn0 != m0 || mn1 != m1)) {
#pragma unroll
            for (int i = 0; i < 8; ++i) { acc[i][0] *= c0; acc[i][1] *= c1; acc[i][2] *= c0; acc[i][3] *= c1; }
        }
        m0 = mn0; m1 = mn1;
        l0 *= c0; l1 *= c1;
        uint32_t ph[2][2], pl[2][2];  // [k-step of 16 tokens][b0 / b1], P = hi + lo in bf16
#pragma unroll
        for (int mt = 0; mt < 2; ++mt) {
#pragma unroll
            for (int hf = 0; hf < 2; ++hf) {
                const float p0 = ex2(S[mt][2 * hf] - b0), p1 = ex2(S[mt][2 * hf + 1] - b1);
                l0 += p0; l1 += p1;
                const uint32_t h = pack_bf16(p0, p1);
                const uint32_t lw = pack_bf16(p0 - __uint_as_float(h << 16), p1 - __uint_as_float(h & 0xffff0000u));
                ph[mt][hf] = movmatrix_trans(h);
                pl[mt][hf] = movmatrix_trans(lw);
            }
        }
        // ---- O^T += V^T P  (channels = M, heads = N, tokens = K)
#pragma unroll
        for (int kt = 0; kt < 2; ++kt) {
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                uint32_t a[4];
                ldmatrix_x4_trans(a_pv + kt * 16 * kTileStride + i * 32, a);
                mma_bf16(acc[i], a, ph[kt][0], ph[kt][1]);
                mma_bf16(acc[i], a, pl[kt][0], pl[kt][1]);
            }
        }
    }
    if (cur_unit >= 0) flush();
}

// ------------------------------------------------------------------------------------------
// step 3d: merge the partials of every unit that was shared between warps; units with an empty
// selection get out = 0, lse = -inf; units finished by a single warp are already written.
// grid = n_units, block = 128 (thread = channel).  GW = warps of the main kernel's grid.
// ------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(128) mkv_combine_kernel(CacheGeom g, const int32_t* __restrict__ sel_count, int k_max,
                                                          int GW, const float* __restrict__ part_o,
                                                          const float* __restrict__ part_ml, float* __restrict__ out,
                                                          float* __restrict__ lse) {
    const int u = blockIdx.x, c = threadIdx.x;
    __shared__ int s_a[4], s_t[4];
    int before = 0, total = 0;
    for (int i = c; i < g.n_units; i += 128) {
        const int v = min(max(sel_count[i], 0), k_max);
        total += v;
        if (i < u) before += v;
    }
#pragma unroll
    for (int o = 16; o; o >>= 1) {
        before += __shfl_xor_sync(kFull, before, o);
        total += __shfl_xor_sync(kFull, total, o);
    }
    if ((c & 31) == 0) { s_a[c >> 5] = before; s_t[c >> 5] = total; }
    __syncthreads();
    const int a = s_a[0] + s_a[1] + s_a[2] + s_a[3];
    const long long T = (long long)s_t[0] + s_t[1] + s_t[2] + s_t[3];
    const int b = a + min(max(sel_count[u], 0), k_max);
    const int G = g.group;
    const int bi = u / g.n_kv_heads, hk = u % g.n_kv_heads;
    const size_t row = (size_t)bi * g.n_q_heads + (size_t)hk * G;
    if (b == a) {
        for (int gi = 0; gi < G; ++gi) {
            out[(row + gi) * kD + c] = 0.f;
            if (lse != nullptr && c == 0) lse[row + gi] = -INFINITY;
        }
        return;
    }
    auto lo_of = [&](long long w) { return (int)(w * T / GW); };
    long long first = (long long)a * GW / T;
    while (lo_of(first + 1) <= a) ++first;      // first warp whose range reaches past a
    long long last = (long long)(b - 1) * GW / T;
    while (last + 1 < GW && lo_of(last + 1) < b) ++last;
    while (lo_of(last) >= b) --last;
    if (first == last) return;  // one warp saw the whole unit and wrote the result itself
    for (int gi = 0; gi < G; ++gi) {
        float M = -INFINITY;
        for (long long w = first; w <= last; ++w) {
            const int wl = lo_of(w), wh = lo_of(w + 1);
            if (wl >= wh) continue;
            const size_t slot = (size_t)w * 2 + (a < wl ? 0 : 1);
            M = fmaxf(M, part_ml[slot * (2 * kMaxGroup) + 2 * gi]);
        }
        float L = 0.f, O = 0.f;
        for (long long w = first; w <= last; ++w) {
            const int wl = lo_of(w), wh = lo_of(w + 1);
            if (wl >= wh) continue;
            const size_t slot = (size_t)w * 2 + (a < wl ? 0 : 1);
            const float ms = part_ml[slot * (2 * kMaxGroup) + 2 * gi];
            const float wgt = ms == -INFINITY ? 0.f : ex2(ms - M);
            L = fmaf(part_ml[slot * (2 * kMaxGroup) + 2 * gi + 1], wgt, L);
            O = fmaf(part_o[(slot * G + gi) * kD + c], wgt, O);
        }
        out[(row + gi) * kD + c] = L > 0.f ? O / L : 0.f;
        if (lse != nullptr && c == 0) lse[row + gi] = L > 0.f ? (M + log2f(L)) * kLn2 : -INFINITY;
    }
}

}  // namespace

int attention_partial_slots(int sm_count) { return sm_count * kWarps * 2; }

cudaError_t launch_attention(const CacheGeom& g, const LayerView& lv, const uint16_t* q, const int32_t* sel,
                             const int32_t* sel_count, int k_max, float scale, float* out, float* lse,
                             const AttnScratch& scr, int sm_count, cudaStream_t s, int* n_kernels) {
    if (g.n_units > kMaxUnitsSmem) return cudaErrorInvalidValue;
    const int smem = kWarps * warp_smem_bytes(kStages) + (g.n_units + 1) * 4;
    static int configured = 0;  // largest dynamic shared-memory size opted into so far
    if (smem > configured) {
        cudaError_t e = cudaFuncSetAttribute(mkv_packed_attention_kernel<kStages>,
                                             cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
        if (e != cudaSuccess) return e;
        configured = smem;
    }
    const float scale_log2 = scale * kLog2e;
    mkv_packed_attention_kernel<kStages><<<sm_count, kWarps * 32, smem, s>>>(g, lv, q, sel, sel_count, k_max, scale_log2,
                                                                              out, lse, scr.part_o, scr.part_ml);
    cudaError_t err = cudaGetLastError();
    if (err != cudaSuccess) return err;
    mkv_combine_kernel<<<g.n_units, 128, 0, s>>>(g, sel_count, k_max, sm_count * kWarps, scr.part_o, scr.part_ml, out, lse);
    if (n_kernels) *n_kernels = 2;
    return cudaGetLastError();
}

}  // namespace mkv
