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
#include <cstdlib>

#include "mkv_internal.cuh"

namespace mkv {

namespace {

constexpr unsigned kFull = 0xffffffffu;
constexpr float kLog2e = 1.4426950408889634f;
constexpr float kLn2 = 0.6931471805599453f;

constexpr int kMaxWarps = 16;                 // upper bound on warps per CTA (sizes the partial-slot scratch)
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
__device__ __forceinline__ void cp_async_16(uint32_t dst, unsigned long long src) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() {
    asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory");
}
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
//
// "Row assembly": the lane walks its 128 channel slots in order.  For slot c the bitmap bit (an
// immediate mask, so the test is one LOP3 into a predicate) guards a 2-byte load of the next kept
// value and the advance of the value pointer; a dropped slot keeps the zero its register was
// initialised with.  Eight slots are packed into four registers and stored with one 16-byte store.
// Why this shape: it is uniform across lanes (no divergence, no padding
// to the longest lane), needs no zero-fill pass and no scattered 2-byte stores (bank conflicts),
// no FLO/POPC (XU pipe), and only ~1.5 ALU-pipe instructions per slot; a dense vector (r = D) is
// the same code with an all-ones bitmap.  The 32-slot body exists once (word loop rolled): the
// hot code must stay small, instruction fetch is a shared per-GPC resource.
template <int BIT>
__device__ __forceinline__ void take_slot(uint32_t w, uint32_t& v, uint32_t& vptr) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        ".reg .b32 t;\n"
        "and.b32 t, %2, %3;\n"
        "setp.ne.u32 p, t, 0;\n"
        "@p ld.shared.u16 %0, [%1];\n"
        "@p add.u32 %1, %1, 2;\n"
        "}\n"
        : "+r"(v), "+r"(vptr)
        : "r"(w), "n"(1u << BIT)
        : "memory");
}

template <int OCT>
__device__ __forceinline__ void assemble_octet(uint32_t w, uint32_t& vptr, uint32_t dst) {
    uint32_t v[8];
#pragma unroll
    for (int c = 0; c < 8; ++c) v[c] = 0u;
    take_slot<8 * OCT + 0>(w, v[0], vptr);
    take_slot<8 * OCT + 1>(w, v[1], vptr);
    take_slot<8 * OCT + 2>(w, v[2], vptr);
    take_slot<8 * OCT + 3>(w, v[3], vptr);
    take_slot<8 * OCT + 4>(w, v[4], vptr);
    take_slot<8 * OCT + 5>(w, v[5], vptr);
    take_slot<8 * OCT + 6>(w, v[6], vptr);
    take_slot<8 * OCT + 7>(w, v[7], vptr);
    uint4 o;  // hi * 65536 + lo: an IMAD (FMA pipe), not a PRMT/LOP3 (ALU pipe)
    o.x = v[1] * 65536u + v[0];
    o.y = v[3] * 65536u + v[2];
    o.z = v[5] * 65536u + v[4];
    o.w = v[7] * 65536u + v[6];
    sts_128(dst + 16 * OCT, o);
}

__device__ __noinline__ void expand_row(uint32_t row, uint32_t bm, uint32_t val, int r, bool valid) {
    uint32_t w0 = 0u, w1 = 0u, w2 = 0u, w3 = 0u;
    if (valid) {
        if (r == kD) {
            w0 = w1 = w2 = w3 = 0xffffffffu;
        } else if ((bm & 15u) == 0) {
            const uint4 b = lds_128(bm);
            w0 = b.x; w1 = b.y; w2 = b.z; w3 = b.w;
        } else {  // ragged token block: bitmaps are only 2-byte aligned
            w0 = lds_u16(bm) | (lds_u16(bm + 2) << 16);
            w1 = lds_u16(bm + 4) | (lds_u16(bm + 6) << 16);
            w2 = lds_u16(bm + 8) | (lds_u16(bm + 10) << 16);
            w3 = lds_u16(bm + 12) | (lds_u16(bm + 14) << 16);
        }
    }
    uint32_t vptr = val;  // never dereferenced by a lane whose bitmap is empty
#pragma unroll 1
    for (int j = 0; j < 4; ++j) {
        const uint32_t w = w0;
        w0 = w1; w1 = w2; w2 = w3;
#ifndef MKV_DBG_NO_DECODE
        assemble_octet<0>(w, vptr, row);
        assemble_octet<1>(w, vptr, row);
        assemble_octet<2>(w, vptr, row);
        assemble_octet<3>(w, vptr, row);
#endif
        row += 64;
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
template <int NSTAGE, int kWarps>
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
            cp_async_commit();  // keeps the group count in step with the wait in the main loop
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
        if (lane == 0) gmeta[s] = make_int2(unit0, n);
        // every lane copies 16-byte chunks of each block of the group (LDGSTS, L1 bypass)
        const uint32_t my_dst = stage0 + s * kStageBytes + (cum - d.bytes);
        const unsigned long long my_src = reinterpret_cast<unsigned long long>(lv.slice) + ((unsigned long long)d.off16 << 4);
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            if (i < n) {
                const uint32_t dst = __shfl_sync(kFull, my_dst, i);
                const unsigned long long src = __shfl_sync(kFull, my_src, i);
                const uint32_t nbytes = __shfl_sync(kFull, d.bytes, i);
                for (uint32_t o = 16u * lane; o < nbytes; o += 512u) cp_async_16(dst + o, src + o);
            }
        }
        cp_async_commit();
        pos += n;
    };


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

    // One call site each for issue() and flush() (code size): iterations k < 0 only fill the pipeline.
    uint32_t ph[2][2], pl[2][2];  // P = hi + lo in bf16, [k-step of 16 tokens][b0 / b1]
#pragma unroll 1
    for (int k = -NSTAGE;; ++k) {
        const int s = (k + NSTAGE) % NSTAGE;
        const bool active = k >= 0;
        float S[2][4];
        int nbj[4];
        if (active) {
        __syncwarp();
        const int2 meta = gmeta[s];
        const int n = meta.y;
        if (meta.x != cur_unit) {
            if (cur_unit >= 0) flush();
            if (n == 0) break;
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

        cp_async_wait<NSTAGE - 1>();  // this lane's copies of group k have landed ...
        __syncwarp();                 // ... and so have every other lane's

        // ---- K: expand, S = K q^T on the tensor cores (tokens = M, heads = N)
        expand_row(my_row, k_bm, k_val, (int)gi.r_k, valid);
        __syncwarp();
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
        }  // active
        issue(s);  // stage s is free: start the copies of group k + NSTAGE
        if (!active) continue;

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
}

// ------------------------------------------------------------------------------------------
// step 3d: merge the partials of every unit that was shared between warps; units with an empty
// selection get out = 0, lse = -inf; units finished by a single warp are already written.
// grid = (n_units, G), block = 128 (thread = channel).  GW = warps of the main kernel's grid.
// ------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(128) mkv_combine_kernel(CacheGeom g, const int32_t* __restrict__ sel_count, int k_max,
                                                          int GW, const float* __restrict__ part_o,
                                                          const float* __restrict__ part_ml, float* __restrict__ out,
                                                          float* __restrict__ lse) {
    const int u = blockIdx.x, gi = blockIdx.y, c = threadIdx.x;
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
    const size_t row = (size_t)bi * g.n_q_heads + (size_t)hk * G + gi;
    if (b == a) {
        out[row * kD + c] = 0.f;
        if (lse != nullptr && c == 0) lse[row] = -INFINITY;
        return;
    }
    auto lo_of = [&](long long w) { return (int)(w * T / GW); };
    long long first = (long long)a * GW / T;
    while (lo_of(first + 1) <= a) ++first;      // first warp whose range reaches past a
    long long last = (long long)(b - 1) * GW / T;
    while (last + 1 < GW && lo_of(last + 1) < b) ++last;
    while (lo_of(last) >= b) --last;
    if (first == last) return;  // one warp saw the whole unit and wrote the result itself
    __shared__ int s_slot[128];
    __shared__ float s_m[128], s_l[128];
    float M = -INFINITY, L = 0.f, O = 0.f;
    for (long long w0 = first; w0 <= last; w0 += 128) {
        __syncthreads();
        const long long w = w0 + c;
        int slot = -1;
        if (w <= last) {
            const int wl = lo_of(w), wh = lo_of(w + 1);
            if (wl < wh) slot = (int)(w * 2 + (a < wl ? 0 : 1));
        }
        s_slot[c] = slot;
        s_m[c] = slot >= 0 ? part_ml[(size_t)slot * (2 * kMaxGroup) + 2 * gi] : -INFINITY;
        s_l[c] = slot >= 0 ? part_ml[(size_t)slot * (2 * kMaxGroup) + 2 * gi + 1] : 0.f;
        __syncthreads();
        const int cnt = (int)min((long long)128, last - w0 + 1);
        float mx = M;
        for (int i = 0; i < cnt; ++i) mx = fmaxf(mx, s_m[i]);
        const float bs = mx == -INFINITY ? 0.f : mx;
        const float co = ex2(M - bs);
        L *= co; O *= co; M = mx;
        for (int i0 = 0; i0 < cnt; i0 += 8) {  // eight independent loads in flight
            float os[8];
#pragma unroll
            for (int e = 0; e < 8; ++e) {
                const int sl = i0 + e < cnt ? s_slot[i0 + e] : -1;
                os[e] = sl >= 0 ? part_o[((size_t)sl * G + gi) * kD + c] : 0.f;
            }
#pragma unroll
            for (int e = 0; e < 8; ++e) {
                if (i0 + e < cnt) {
                    const float wgt = ex2(s_m[i0 + e] - bs);
                    L = fmaf(s_l[i0 + e], wgt, L);
                    O = fmaf(os[e], wgt, O);
                }
            }
        }
    }
    out[row * kD + c] = L > 0.f ? O / L : 0.f;
    if (lse != nullptr && c == 0) lse[row] = L > 0.f ? (M + log2f(L)) * kLn2 : -INFINITY;
}

}  // namespace

int attention_partial_slots(int sm_count) { return sm_count * kMaxWarps * 2; }

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
        g, lv, q, sel, sel_count, k_max, scale * kLog2e, out, lse, scr.part_o, scr.part_ml);
    cudaError_t err = cudaGetLastError();
    if (err != cudaSuccess) return err;
    mkv_combine_kernel<<<dim3(g.n_units, g.group), 128, 0, s>>>(g, sel_count, k_max, sm_count * NWARPS, scr.part_o, scr.part_ml,
                                                                 out, lse);
    return cudaGetLastError();
}

cudaError_t launch_attention(const CacheGeom& g, const LayerView& lv, const uint16_t* q, const int32_t* sel,
                             const int32_t* sel_count, int k_max, float scale, float* out, float* lse,
                             const AttnScratch& scr, int sm_count, cudaStream_t s, int* n_kernels) {
    if (g.n_units > kMaxUnitsSmem) return cudaErrorInvalidValue;
    if (n_kernels) *n_kernels = 2;
    static int cfg = -1;  // tuning knob (stages * 100 + warps); default chosen from measurements
    if (cfg < 0) {
        const char* e = getenv("MKV_ATTN_CFG");
        cfg = e ? atoi(e) : 210;
    }
#define MKV_CFG(S, W) \
    case S * 100 + W: return launch_attention_cfg<S, W>(g, lv, q, sel, sel_count, k_max, scale, out, lse, scr, sm_count, s);
    switch (cfg) {
        MKV_CFG(1, 12) MKV_CFG(1, 14) MKV_CFG(2, 8) MKV_CFG(2, 10) MKV_CFG(3, 8) MKV_CFG(2, 4) MKV_CFG(2, 6)
        default: return launch_attention_cfg<2, 10>(g, lv, q, sel, sel_count, k_max, scale, out, lse, scr, sm_count, s);
    }
#undef MKV_CFG
}

}  // namespace mkv
