// compress.cu — step 1 of the hot path: per-vector top-r element selection,
// per-block mean keys, compression loss + strategy choice
// and packing behind a position bitmap.  sm_100a.
//
// Thread mapping: one warp owns one vector at a time; lane l holds channels l, l+32, l+64, l+96,
// so `__ballot_sync` of a per-channel predicate IS bitmap word j of the canonical format and
// the ascending-channel rank of a kept element is popc(words below) + popc(word & lanemask_lt).
#include "mkv_internal.cuh"

namespace mkv {

namespace {

constexpr unsigned kFull = 0xffffffffu;
constexpr unsigned long long kNoBase = ~0ull;
constexpr int kStageBytes = 8 * 2 * (kBitmapBytes + 2 * 127);  // the largest packed token block; a dense one is 4096 B

__device__ __forceinline__ unsigned lanemask_lt() {
    unsigned m;
    asm("mov.u32 %0, %%lanemask_lt;" : "=r"(m));
    return m;
}

// Top-r mask of one 128-channel vector held as 15-bit magnitudes mag[j] (channel lane + 32 j).
// Finds the r-th largest magnitude T by a bitwise binary search (count(mag >= cand) via REDUX),
// keeps everything above T and the lowest-channel elements equal to T until r are kept
// (ties -> lower index).  Returns the four bitmap words in w (identical in all lanes).
__device__ __forceinline__ void topr_mask(const uint32_t (&mag)[4], int r, uint32_t (&w)[4]) {
    uint32_t T = 0;
    // two 15-bit magnitudes per register with bit 15 / 31 set: (pair - cand x 0x10001) keeps that bit exactly
    // where mag >= cand, and no borrow crosses the halves -- four compares in two subtractions
    const uint32_t p01 = mag[0] | (mag[1] << 16) | 0x80008000u, p23 = mag[2] | (mag[3] << 16) | 0x80008000u;
    // (as soon as exactly r magnitudes lie at or above a candidate they ARE the top r: no lower bit can change the set,
    // and no tie straddles its edge -- the warp-uniform early exit saves the last steps of most searches)
#pragma unroll
    for (int bit = 14; bit >= 0; --bit) {
        const uint32_t cand = T | (1u << bit);
        const uint32_t c2 = cand * 0x10001u;
        const uint32_t z = ((p01 - c2) & 0x80008000u) | (((p23 - c2) >> 1) & 0x40004000u);
        const int c = __reduce_add_sync(kFull, __popc(z));
        if (c >= r) T = cand;
        if (c == r) {
#pragma unroll
            for (int j = 0; j < 4; ++j) w[j] = __ballot_sync(kFull, mag[j] >= cand);
            return;
        }
    }
    int ngt = (mag[0] > T) + (mag[1] > T) + (mag[2] > T) + (mag[3] > T);
    ngt = __reduce_add_sync(kFull, ngt);
    const int need = r - ngt;  // >= 1 elements equal to T are kept, lowest channels first
    const unsigned lt = lanemask_lt();
    int seen = 0;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        const bool eq = (mag[j] == T);
        const unsigned e = __ballot_sync(kFull, eq);
        const bool keep = (mag[j] > T) || (eq && (seen + __popc(e & lt) < need));
        seen += __popc(e);
        w[j] = __ballot_sync(kFull, keep);
    }
}

// Element groups ("selects groups of adjacent elements together ... one bit per element group"): the
// r / g groups of g adjacent channels with the largest energy sum_i x_i^2, evaluated in fp32 from left to right
// (R4; the squares of bf16 values are exact in fp32), ties -> lower group.  x[j]: bf16 bits of channel
// lane + 32 j, so a group lives in g adjacent lanes of one j.  Returns the mask EXPANDED to one bit per channel
// (w[j] = channels 32 j .. 32 j + 31): the device keeps 128-bit bitmaps for every g, export packs them (mkv_api.cu).
// energy of this lane's group (g adjacent lanes of one j), fp32 left to right, as an order-preserving integer
__device__ __forceinline__ void group_keys(const uint32_t (&x)[4], int g, int lane, uint32_t (&key)[4]) {
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        const float f = bf16_bits_to_f32(x[j]);
        const float sq = __fmul_rn(f, f);
        const int l0 = lane & ~(g - 1);
        float e = __shfl_sync(kFull, sq, l0);
        e = __fadd_rn(e, __shfl_sync(kFull, sq, l0 + 1));
        if (g == 4) {
            e = __fadd_rn(e, __shfl_sync(kFull, sq, l0 + 2));
            e = __fadd_rn(e, __shfl_sync(kFull, sq, l0 + 3));
        }
        key[j] = __float_as_uint(e);
    }
}

__device__ __forceinline__ void topr_mask_groups(const uint32_t (&x)[4], int r, int g, uint32_t (&w)[4], int lane) {
    uint32_t key[4];  // energy of this lane's group, as an order-preserving integer (non-negative floats)
    group_keys(x, g, lane, key);
    const bool leader = (lane & (g - 1)) == 0;
    const int nk = r / g;
    uint32_t T = 0;
#pragma unroll 1
    for (int bit = 30; bit >= 0; --bit) {
        const uint32_t cand = T | (1u << bit);
        int c = 0;
        if (leader) c = (key[0] >= cand) + (key[1] >= cand) + (key[2] >= cand) + (key[3] >= cand);
        c = __reduce_add_sync(kFull, c);
        if (c >= nk) T = cand;
        if (c == nk) {  // exactly r / g groups at or above the candidate: they are the kept set (see topr_mask)
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const unsigned kl = __ballot_sync(kFull, leader && key[j] >= cand);
                w[j] = kl | (kl << 1) | (g == 4 ? (kl << 2) | (kl << 3) : 0u);
            }
            return;
        }
    }
    int ngt = 0;
    if (leader) ngt = (key[0] > T) + (key[1] > T) + (key[2] > T) + (key[3] > T);
    ngt = __reduce_add_sync(kFull, ngt);
    const int need = nk - ngt;  // >= 1 groups equal to T are kept, lowest groups first
    const unsigned lt = lanemask_lt();
    int seen = 0;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        const bool eq = leader && key[j] == T;
        const unsigned e = __ballot_sync(kFull, eq);
        const bool keep = leader && ((key[j] > T) || (eq && (seen + __popc(e & lt) < need)));
        seen += __popc(e);
        const unsigned kl = __ballot_sync(kFull, keep);            // one bit per leader
        w[j] = kl | (kl << 1) | (g == 4 ? (kl << 2) | (kl << 3) : 0u);  // every channel of a kept group
    }
}

// Write one packed vector: vector t of a group of n <= 8 vectors (the K or the V vectors of a token
// block, or 8 block keys of a segment).  Physical layout of a group:
// the n position bitmaps, then the kept values RANK-MAJOR: the value of rank rho (ascending
// channel) of vector t sits at element rho * n + t, so that the vectors' run pointers advance
// through disjoint shared-memory banks in the decode kernels' walk.  Dense vectors (r = D) carry
// no bitmap and stay vector-major.  x[j]: bf16 bits of channel lane + 32 j.
// bm: this vector's bitmap; val: the GROUP's value area (2-byte aligned).
// cached: a mask found earlier for this vector by mkv_segment_loss (or nullptr).  It is used only if it keeps r elements
// and every kept magnitude is strictly above every dropped one -- then it IS the top-r mask, whatever wrote it.
// pairs: K vectors and block keys kept in element groups g >= 2 store their values PAIR-major instead (the kept channels
// come in aligned pairs; pair pi = rho / 2 of vector t sits at 32-bit element pi * n + t), so that the QK walk loads a whole
// A-fragment register with one aligned LDS.32 (mkv_walk.cuh: k_walk_mma_pairs).  Same bytes, same bitmaps.
__device__ __forceinline__ void pack_vector(const uint32_t (&x)[4], int r, int g, uint8_t* bm, uint8_t* val, int t, int n,
                                            int lane, bool pairs, bool cached = false,
                                            uint4 cw = make_uint4(0u, 0u, 0u, 0u)) {
    uint16_t* v16 = reinterpret_cast<uint16_t*>(val);
    if (r == kD) {
#pragma unroll
        for (int j = 0; j < 4; ++j) v16[t * kD + lane + 32 * j] = (uint16_t)x[j];
        return;
    }
    uint32_t mag[4], w[4];
#pragma unroll
    for (int j = 0; j < 4; ++j) mag[j] = x[j] & 0x7FFFu;
    bool have = false;
    if (g == 1 && cached) {  // (a kept magnitude equal to a dropped one means a tie: searched again, never guessed)
        w[0] = cw.x; w[1] = cw.y; w[2] = cw.z; w[3] = cw.w;
        uint32_t kmin = 0x8000u, dmax = 0u;
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const bool kept = (w[j] >> lane) & 1u;
            kmin = kept ? min(kmin, mag[j]) : kmin;
            dmax = kept ? dmax : max(dmax, mag[j]);
        }
        kmin = __reduce_min_sync(kFull, kmin);
        dmax = __reduce_max_sync(kFull, dmax);
        have = __popc(w[0]) + __popc(w[1]) + __popc(w[2]) + __popc(w[3]) == r && kmin > dmax;
    } else if (cached) {
        // element groups: the cached mask must be made of whole groups, keep r / g of them, and every kept group's energy
        // must lie strictly above every dropped one's
        w[0] = cw.x; w[1] = cw.y; w[2] = cw.z; w[3] = cw.w;
        uint32_t key[4];
        group_keys(x, g, lane, key);
        const bool leader = (lane & (g - 1)) == 0;
        const uint32_t lead = g == 2 ? 0x55555555u : 0x11111111u;
        uint32_t kmin = 0xffffffffu, dmax = 0u;
        bool whole = true;
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const uint32_t m = w[j] & lead;
            whole = whole && w[j] == (m | (m << 1) | (g == 4 ? (m << 2) | (m << 3) : 0u));
            const bool kept = (w[j] >> lane) & 1u;
            if (leader) {
                kmin = kept ? min(kmin, key[j]) : kmin;
                dmax = kept ? dmax : max(dmax, key[j] + 1u);  // (+ 1: a dropped group of energy 0 still counts)
            }
        }
        kmin = __reduce_min_sync(kFull, kmin);
        dmax = __reduce_max_sync(kFull, dmax);
        have = whole && __popc(w[0]) + __popc(w[1]) + __popc(w[2]) + __popc(w[3]) == r && kmin >= dmax;
    }
    if (!have) {
        if (g == 1) topr_mask(mag, r, w);
        else topr_mask_groups(x, r, g, w, lane);
    }
    const unsigned lt = lanemask_lt();
    int base = 0;
    if (!pairs) {  // (warp-uniform: two tight loops instead of one with a select per element)
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            if ((w[j] >> lane) & 1u) v16[(base + __popc(w[j] & lt)) * n + t] = (uint16_t)x[j];
            base += __popc(w[j]);
        }
    } else {
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            if ((w[j] >> lane) & 1u) {
                const int rho = base + __popc(w[j] & lt);
                v16[((rho >> 1) * n + t) * 2 + (rho & 1)] = (uint16_t)x[j];
            }
            base += __popc(w[j]);
        }
    }
    if (lane < 8) {  // 2-byte stores: a ragged token block leaves the V bitmaps only 2-byte aligned
        const int j = lane >> 1;
        const uint32_t wl = j == 0 ? w[0] : j == 1 ? w[1] : j == 2 ? w[2] : w[3];
        reinterpret_cast<uint16_t*>(bm)[lane] = (uint16_t)(wl >> (16 * (lane & 1)));
    }
}

__device__ __forceinline__ bool strat_supported(const mkv_strategy& s, int B) {
    return (s.g == 1 || s.g == 2 || s.g == 4) && s.B == B && s.r_k >= s.g && s.r_k <= kD && s.r_v >= s.g && s.r_v <= kD &&
           s.r_k % s.g == 0 && s.r_v % s.g == 0;
}

// ------------------------------------------------------------------------------------------
// plan: one CTA per unit of the call.  Sizes every segment from its strategy, claims a
// contiguous region [block keys | token blocks] of the layer slice with one atomicAdd, and
// writes the unit's table entries (strategy record, offsets).
// ------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) mkv_plan_kernel(CacheGeom g, LayerView lv, CompressArgs a,
                                                       const mkv_strategy* __restrict__ strat,
                                                       unsigned long long* __restrict__ call_base,
                                                       uint32_t* __restrict__ dev_flags) {
    const int uc = blockIdx.x;
    const int b = a.b0 + uc / g.n_kv_heads, h = uc % g.n_kv_heads;
    const int unit = b * g.n_kv_heads + h;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const mkv_strategy* st = strat + (size_t)uc * a.nseg;

    __shared__ unsigned long long s_tok[8], s_bk[8];
    __shared__ int s_bad[8];
    __shared__ unsigned long long s_base, s_bk_total;

    unsigned long long tokb = 0, bkb = 0;
    int bad = 0;
    for (int i = tid; i < a.nseg; i += 256) {
        const mkv_strategy s = st[i];
        const int n_tok = (i == a.nseg - 1) ? a.n_tok - i * g.L : g.L;
        if (!strat_supported(s, g.B)) { bad = 1; continue; }
        tokb += seg_tok_bytes(s.r_k, s.r_v, n_tok, g.pb);
        bkb += seg_bk_bytes(s.r_k, n_tok, g.B);
    }
#pragma unroll
    for (int o = 16; o; o >>= 1) {
        tokb += __shfl_xor_sync(kFull, tokb, o);
        bkb += __shfl_xor_sync(kFull, bkb, o);
        bad |= __shfl_xor_sync(kFull, bad, o);
    }
    if (lane == 0) { s_tok[warp] = tokb; s_bk[warp] = bkb; s_bad[warp] = bad; }
    __syncthreads();
    if (tid == 0) {
        unsigned long long T = 0, K = 0;
        int B = 0;
        for (int i = 0; i < 8; ++i) { T += s_tok[i]; K += s_bk[i]; B |= s_bad[i]; }
        unsigned long long base = kNoBase;
        if (B || lv.unit_nseg[unit] != a.seg0) {
            // a bad strategy, or an earlier call for this unit was rejected on the device (the host's append
            // state ran ahead): never leave a hole of unwritten table entries behind
            atomicOr(dev_flags, MKV_DEV_BAD_STRATEGY);
        } else {
            base = atomicAdd(lv.bump, T + K);
            if (base + T + K > lv.slice_bytes) {
                atomicOr(dev_flags, MKV_DEV_ARENA_OVERFLOW);
                base = kNoBase;
            } else {
                atomicAdd(lv.used_tok, T);
                atomicAdd(lv.used_bk, K);
                lv.unit_nseg[unit] = a.seg0 + a.nseg;
                lv.unit_ntok[unit] = a.seg0 * g.L + a.n_tok;
            }
        }
        s_base = base;
        s_bk_total = K;
        call_base[uc] = base;
    }
    __syncthreads();
    const unsigned long long base = s_base;
    if (base == kNoBase) return;
    const unsigned long long tok_base = base + s_bk_total;

    // exclusive scan over the segments, 256 at a time, with a running carry
    __shared__ unsigned long long s_wtok[8], s_wbk[8];
    unsigned long long carry_tok = 0, carry_bk = 0;
    for (int i0 = 0; i0 < a.nseg; i0 += 256) {
        const int i = i0 + tid;
        unsigned long long t = 0, k = 0;
        mkv_strategy s = {0, 0, 0, 0};
        int n_tok = 0;
        if (i < a.nseg) {
            s = st[i];
            n_tok = (i == a.nseg - 1) ? a.n_tok - i * g.L : g.L;
            t = seg_tok_bytes(s.r_k, s.r_v, n_tok, g.pb);
            k = seg_bk_bytes(s.r_k, n_tok, g.B);
        }
        unsigned long long it = t, ik = k;  // inclusive warp scan
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const unsigned long long ut = __shfl_up_sync(kFull, it, o);
            const unsigned long long uk = __shfl_up_sync(kFull, ik, o);
            if (lane >= o) { it += ut; ik += uk; }
        }
        if (lane == 31) { s_wtok[warp] = it; s_wbk[warp] = ik; }
        __syncthreads();
        unsigned long long wt = 0, wk = 0, tot_t = 0, tot_k = 0;
        for (int wv = 0; wv < 8; ++wv) {
            if (wv < warp) { wt += s_wtok[wv]; wk += s_wbk[wv]; }
            tot_t += s_wtok[wv];
            tot_k += s_wbk[wv];
        }
        if (i < a.nseg) {
            const size_t e = (size_t)unit * lv.S_max + a.seg0 + i;
            StratRec rec;
            rec.r_k = s.r_k; rec.r_v = s.r_v; rec.g = s.g; rec.B = s.B;
            rec.n_tok = (uint16_t)n_tok;
            rec.flags = (uint16_t)((s.r_k == kD ? 1 : 0) | (s.r_v == kD ? 2 : 0));
            lv.strat[e] = rec;
            lv.tok_off[e] = (uint32_t)((tok_base + carry_tok + wt + it - t) >> 4);
            lv.bk_off[e] = (uint32_t)((base + carry_bk + wk + ik - k) >> 4);
        }
        carry_tok += tot_t;
        carry_bk += tot_k;
        __syncthreads();
    }
}

// ------------------------------------------------------------------------------------------
// compress: CTA = 8 warps = 8 consecutive token blocks of one segment; warp = one token block:
// nb K vectors, nb V vectors, and the block key (fp32 sum in token order, IEEE /nb, RNE bf16).
// ------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256, 4) mkv_compress_kernel(CacheGeom g, LayerView lv, CompressArgs a,
                                                           const unsigned long long* __restrict__ call_base,
                                                           int chunks_per_seg) {
    const int uc = blockIdx.y;
    if (call_base[uc] == kNoBase) return;
    const int b = a.b0 + uc / g.n_kv_heads, h = uc % g.n_kv_heads;
    const int unit = b * g.n_kv_heads + h;
    const int seg_local = blockIdx.x / chunks_per_seg, chunk = blockIdx.x % chunks_per_seg;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const size_t e = (size_t)unit * lv.S_max + a.seg0 + seg_local;
    const StratRec rec = lv.strat[e];
    const int pb = g.pb, B = g.B;
    const int n_tok = rec.n_tok, nblk = (n_tok + pb - 1) / pb;  // device token blocks of the segment
    const int blk = chunk * 8 + warp;
    if (blk >= nblk) return;
    const int nb = min(pb, n_tok - blk * pb);
    const int r_k = rec.r_k, r_v = rec.r_v;
    const uint32_t bmk = (r_k == kD) ? 0u : kBitmapBytes, bmv = (r_v == kD) ? 0u : kBitmapBytes;

    uint8_t* base = lv.slice + ((size_t)lv.tok_off[e] << 4) + (size_t)blk * tokblock_bytes(r_k, r_v, pb);
    // the block is packed in shared memory (2-byte stores at rank-major positions) and leaves in 16-byte stores
    __shared__ __align__(16) uint8_t s_stage[8][kStageBytes];
    uint8_t* k_bm = s_stage[warp];
    uint8_t* k_val = k_bm + nb * bmk;
    uint8_t* v_bm = k_val + nb * r_k * 2;
    uint8_t* v_val = v_bm + nb * bmv;
    uint8_t* bk_base = lv.slice + ((size_t)lv.bk_off[e] << 4);

    const size_t row0 = (size_t)(b - a.b0) * a.stride_b + (size_t)h * a.stride_h +
                        (size_t)(seg_local * g.L + blk * pb) * a.stride_t;
    const uint16_t* ksrc = a.k + row0;
    const uint16_t* vsrc = a.v + row0;
    // masks of this block's vectors as mkv_segment_loss left them, [token][K, V][4 words]: 64 words, two per lane
    const bool mk = a.masks != nullptr;
    uint32_t m0 = 0u, m1 = 0u;
    if (mk) {
        const uint32_t* m32 = reinterpret_cast<const uint32_t*>(
            a.masks + 2 * ((size_t)unit * a.mask_stride + (size_t)(a.seg0 + seg_local) * g.L + blk * pb));
        if (lane < 8 * nb) m0 = __ldg(m32 + lane);
        if (32 + lane < 8 * nb) m1 = __ldg(m32 + 32 + lane);
    }
    auto cached_mask = [&](int t, int which) {  // words 8 t + 4 which .. + 3
        const uint32_t src = t < 4 ? m0 : m1;
        const int l0 = (8 * t + 4 * which) & 31;
        return make_uint4(__shfl_sync(kFull, src, l0), __shfl_sync(kFull, src, l0 + 1), __shfl_sync(kFull, src, l0 + 2),
                          __shfl_sync(kFull, src, l0 + 3));
    };

    float sum[4] = {0.f, 0.f, 0.f, 0.f};
    // token t + 1 is loaded while token t is searched and packed (the loads are what the warp would wait for)
    uint32_t nk[4], nv[4];
#pragma unroll
    for (int j = 0; j < 4; ++j) { nk[j] = __ldg(ksrc + lane + 32 * j); nv[j] = __ldg(vsrc + lane + 32 * j); }
#pragma unroll 1
    for (int t = 0; t < nb; ++t) {
        uint32_t xk[4], xv[4];
#pragma unroll
        for (int j = 0; j < 4; ++j) { xk[j] = nk[j]; xv[j] = nv[j]; }
        if (t + 1 < nb) {
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                nk[j] = __ldg(ksrc + (size_t)(t + 1) * a.stride_t + lane + 32 * j);
                nv[j] = __ldg(vsrc + (size_t)(t + 1) * a.stride_t + lane + 32 * j);
            }
        }
#pragma unroll
        for (int j = 0; j < 4; ++j) sum[j] = __fadd_rn(sum[j], bf16_bits_to_f32(xk[j]));
        pack_vector(xk, r_k, rec.g, k_bm + t * bmk, k_val, t, nb, lane, rec.g >= 2, mk && r_k != kD, cached_mask(t, 0));
        pack_vector(xv, r_v, rec.g, v_bm + t * bmv, v_val, t, nb, lane, false, mk && r_v != kD, cached_mask(t, 1));
    }
    {
        const uint32_t used = (uint32_t)nb * (vec_bytes(r_k) + vec_bytes(r_v));
        const uint32_t padded = pad16u(used);
        for (uint32_t o = used + lane; o < padded; o += 32) s_stage[warp][o] = 0;  // the pad of a ragged token block
        __syncwarp();
        for (uint32_t o = 16u * lane; o < padded; o += 512u)
            *reinterpret_cast<uint4*>(base + o) = *reinterpret_cast<const uint4*>(s_stage[warp] + o);
    }
    // block key of the token block (B tokens): a block of 16 tokens spans two device blocks; the warp of the first one
    // goes on through the keys of the second (fp32 sum in token order over the whole block, R5)
    int nbk = nb;  // tokens averaged
    if (B > pb) {
        if (blk & 1) return;
        const int more = min(pb, n_tok - (blk + 1) * pb);
        for (int t = 0; t < more; ++t) {
#pragma unroll
            for (int j = 0; j < 4; ++j)
                sum[j] = __fadd_rn(sum[j], bf16_bits_to_f32(__ldg(ksrc + (size_t)(pb + t) * a.stride_t + lane + 32 * j)));
        }
        nbk += max(more, 0);
    }
    {
        const int lb = B > pb ? blk >> 1 : blk, nlb = (n_tok + B - 1) / B;  // this token block, token blocks of the segment
        uint32_t x[4];
        const float fnb = (float)nbk;
#pragma unroll
        for (int j = 0; j < 4; ++j) x[j] = f32_to_bf16_bits_rne(__fdiv_rn(sum[j], fnb));
        // the block keys of a segment form groups of 8 (one work item of the score kernel each)
        const int grp = lb >> 3, gn = min(8, nlb - 8 * grp);
        pack_vector(x, r_k, rec.g, bk_base + lb * bmk, bk_base + nlb * bmk + (size_t)grp * 8 * r_k * 2, lb & 7, gn, lane, rec.g >= 2);
        if (lb == nlb - 1) {
            const uint32_t used = (uint32_t)nlb * vec_bytes(r_k);
            const uint32_t padded = pad16u(used);
            for (uint32_t o = used + lane; o < padded; o += 32) bk_base[o] = 0;
        }
    }
}

// ------------------------------------------------------------------------------------------
// loss: CTA = one segment of one unit; warps stride over its tokens.  fp64 sums of the exact
// fp32 squares of the dropped / all elements (R9).
// ------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) mkv_segment_loss_kernel(CacheGeom g, CompressArgs a, int r_k, int r_v, int grp,
                                                               double* __restrict__ loss_k,
                                                               double* __restrict__ loss_v) {
    const int uc = blockIdx.y, seg_local = blockIdx.x;
    const int b = a.b0 + uc / g.n_kv_heads, h = uc % g.n_kv_heads;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int n_tok = (seg_local == a.nseg - 1) ? a.n_tok - seg_local * g.L : g.L;
    const size_t row0 = (size_t)(b - a.b0) * a.stride_b + (size_t)h * a.stride_h +
                        (size_t)(seg_local * g.L) * a.stride_t;
    double acc[4] = {0., 0., 0., 0.};  // dropped_k, total_k, dropped_v, total_v
    const int unit = b * g.n_kv_heads + h;
    uint4* masks = a.masks ? a.masks + 2 * ((size_t)unit * a.mask_stride + (size_t)(a.seg0 + seg_local) * g.L) : nullptr;
    for (int which = 0; which < 2; ++which) {
        const uint16_t* src = (which ? a.v : a.k) + row0;
        const int r = which ? r_v : r_k;
        for (int t = warp; t < n_tok; t += 8) {
            uint32_t x[4], mag[4], w[4];
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                x[j] = __ldg(src + (size_t)t * a.stride_t + lane + 32 * j);
                mag[j] = x[j] & 0x7FFFu;
            }
            if (r == kD) w[0] = w[1] = w[2] = w[3] = kFull;
            else if (grp == 1) {
                topr_mask(mag, r, w);
                if (masks != nullptr && lane == 0) masks[2 * t + which] = make_uint4(w[0], w[1], w[2], w[3]);
            } else {
                topr_mask_groups(x, r, grp, w, lane);
                if (masks != nullptr && lane == 0) masks[2 * t + which] = make_uint4(w[0], w[1], w[2], w[3]);
            }
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const float f = bf16_bits_to_f32(x[j]);
                const double sq = (double)__fmul_rn(f, f);  // exact: 8-bit x 8-bit significands
                acc[2 * which + 1] += sq;
                if (!((w[j] >> lane) & 1u)) acc[2 * which] += sq;
            }
        }
    }
    __shared__ double s_acc[8][4];
#pragma unroll
    for (int i = 0; i < 4; ++i) {
#pragma unroll
        for (int o = 16; o; o >>= 1) acc[i] += __shfl_xor_sync(kFull, acc[i], o);
    }
    if (lane == 0)
        for (int i = 0; i < 4; ++i) s_acc[warp][i] = acc[i];
    __syncthreads();
    if (threadIdx.x == 0) {
        double t[4] = {0., 0., 0., 0.};
        for (int wv = 0; wv < 8; ++wv)
            for (int i = 0; i < 4; ++i) t[i] += s_acc[wv][i];
        const size_t o = (size_t)uc * a.nseg + seg_local;
        loss_k[o] = t[1] > 0. ? t[0] / t[1] : 0.;
        loss_v[o] = t[3] > 0. ? t[2] / t[3] : 0.;
    }
}

// ------------------------------------------------------------------------------------------
// strategy, quantile rule: CTA (chunk, unit) ranks 256 segments of one unit; a segment stays dense iff its
// rank by (importance descending, index ascending) is below n_dense.  Rank by counting against every
// segment of the unit, 1024 at a time through shared memory (a long unit spreads over many CTAs).
// ------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) mkv_strategy_quantile_kernel(const double* __restrict__ loss_k,
                                                                    const double* __restrict__ loss_v,
                                                                    int nseg, int n_dense, mkv_strategy sparse,
                                                                    mkv_strategy* __restrict__ out) {
    const int u = blockIdx.y;
    const double* lk = loss_k + (size_t)u * nseg;
    const double* lvv = loss_v + (size_t)u * nseg;
    constexpr int kTile = 1024;
    __shared__ double s_I[kTile];
    {
        const int i = blockIdx.x * 256 + threadIdx.x;
        const double mine = (i < nseg) ? 0.5 * (lk[i] + lvv[i]) : 0.;
        int rank = 0;
        for (int j0 = 0; j0 < nseg; j0 += kTile) {
            __syncthreads();
            for (int j = threadIdx.x; j < kTile && j0 + j < nseg; j += 256)
                s_I[j] = 0.5 * (lk[j0 + j] + lvv[j0 + j]);
            __syncthreads();
            const int n = min(kTile, nseg - j0);
            for (int j = 0; j < n; ++j) {
                const double o = s_I[j];
                rank += (o > mine) || (o == mine && (j0 + j) < i);
            }
        }
        if (i < nseg) {
            mkv_strategy s = sparse;
            if (rank < n_dense) { s.r_k = kD; s.r_v = kD; }
            out[(size_t)u * nseg + i] = s;
        }
    }
}

struct CandList {
    mkv_strategy c[64];
};
__global__ void mkv_strategy_threshold_kernel(const double* __restrict__ loss_k, const double* __restrict__ loss_v,
                                              int ncand, long long n, const CandList cands, double tau,
                                              mkv_strategy* __restrict__ out) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    mkv_strategy s;
    s.r_k = kD; s.r_v = kD; s.g = 1; s.B = cands.c[ncand - 1].B;
    for (int c = 0; c < ncand; ++c) {
        const double I = 0.5 * (loss_k[(size_t)c * n + i] + loss_v[(size_t)c * n + i]);
        if (I <= tau) { s = cands.c[c]; break; }
    }
    out[i] = s;
}

// ------------------------------------------------------------------------------------------
// KV update buffer: the newest tokens of every unit are held uncompressed, raw
// rows [unit][t][128] bf16, until a whole segment can be compressed.  One warp copies one K row
// and one V row (256 B each, 8 B per lane).
// ------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) mkv_update_copy_kernel(CacheGeom g, CompressArgs a, uint16_t* __restrict__ upd_k,
                                                              uint16_t* __restrict__ upd_v,
                                                              int32_t* __restrict__ upd_count, int n_have) {
    if (blockIdx.x == 0 && threadIdx.x == 0) *upd_count = n_have + a.n_tok;
    const int row = blockIdx.x * 8 + (threadIdx.x >> 5), lane = threadIdx.x & 31;
    if (row >= g.n_units * a.n_tok) return;
    const int unit = row / a.n_tok, t = row - unit * a.n_tok;
    const int b = unit / g.n_kv_heads, h = unit % g.n_kv_heads;
    const size_t src = (size_t)b * a.stride_b + (size_t)h * a.stride_h + (size_t)t * a.stride_t + 4 * lane;
    const size_t dst = ((size_t)unit * g.L + n_have + t) * kD + 4 * lane;
    // rows may be only 2-byte aligned in the caller's tensors: element loads, one 8-byte store
    uint16_t kx[4], vx[4];
#pragma unroll
    for (int j = 0; j < 4; ++j) { kx[j] = a.k[src + j]; vx[j] = a.v[src + j]; }
    *reinterpret_cast<uint2*>(upd_k + dst) = make_uint2(kx[0] | ((uint32_t)kx[1] << 16), kx[2] | ((uint32_t)kx[3] << 16));
    *reinterpret_cast<uint2*>(upd_v + dst) = make_uint2(vx[0] | ((uint32_t)vx[1] << 16), vx[2] | ((uint32_t)vx[3] << 16));
}

}  // namespace

cudaError_t launch_update_copy(const CacheGeom& g, const CompressArgs& a, uint16_t* upd_k, uint16_t* upd_v,
                               int32_t* upd_count, int n_have, cudaStream_t s) {
    const int rows = g.n_units * a.n_tok;
    mkv_update_copy_kernel<<<(rows + 7) / 8, 256, 0, s>>>(g, a, upd_k, upd_v, upd_count, n_have);
    return cudaGetLastError();
}

cudaError_t launch_segment_loss(const CacheGeom& g, const CompressArgs& a, mkv_strategy cand, double* loss_k,
                                double* loss_v, cudaStream_t s) {
    dim3 grid(a.nseg, a.nb * g.n_kv_heads);
    mkv_segment_loss_kernel<<<grid, 256, 0, s>>>(g, a, cand.r_k, cand.r_v, cand.g, loss_k, loss_v);
    return cudaGetLastError();
}

cudaError_t launch_strategy_quantile(const double* loss_k, const double* loss_v, int n_units, int nseg,
                                     int n_dense, mkv_strategy sparse, mkv_strategy* out, cudaStream_t s) {
    if (n_units > 65535) return cudaErrorInvalidValue;
    mkv_strategy_quantile_kernel<<<dim3((nseg + 255) / 256, n_units), 256, 0, s>>>(loss_k, loss_v, nseg, n_dense, sparse, out);
    return cudaGetLastError();
}

cudaError_t launch_strategy_threshold(const double* loss_k, const double* loss_v, int ncand, long long n,
                                      const mkv_strategy* cands_host, double tau, mkv_strategy* out,
                                      cudaStream_t s) {
    const int threads = 256;
    const long long blocks = (n + threads - 1) / threads;
    CandList cl;  // by value: read during this call only, so the call is capturable and needs no staging buffer
    for (int i = 0; i < 64; ++i) cl.c[i] = cands_host[i < ncand ? i : ncand - 1];
    mkv_strategy_threshold_kernel<<<(unsigned)blocks, threads, 0, s>>>(loss_k, loss_v, ncand, n, cl, tau, out);
    return cudaGetLastError();
}

cudaError_t launch_compress(const CacheGeom& g, const LayerView& lv, const CompressArgs& a,
                            const mkv_strategy* strat, unsigned long long* call_base, uint32_t* dev_flags,
                            cudaStream_t s, int* n_kernels) {
    const int units = a.nb * g.n_kv_heads;
    mkv_plan_kernel<<<units, 256, 0, s>>>(g, lv, a, strat, call_base, dev_flags);
    cudaError_t err = cudaGetLastError();
    if (err != cudaSuccess) return err;
    const int chunks = (g.L / g.pb + 7) / 8;  // CTAs of 8 warps per segment: one warp per device token block
    dim3 grid(a.nseg * chunks, units);
    mkv_compress_kernel<<<grid, 256, 0, s>>>(g, lv, a, call_base, chunks);
    if (n_kernels) *n_kernels = 2;
    return cudaGetLastError();
}

}  // namespace mkv
