// mkv_walk.cuh — device helpers shared by the decode kernels (select.cu, attention.cu): PTX
// wrappers and the "walk" that expands packed vectors (kept bf16 values behind a
// position bitmap) straight into mma.sync fragments.  sm_100a.  Not used by the CPU oracle.
#pragma once

#include "mkv_internal.cuh"

namespace mkv {
namespace walk {

constexpr unsigned kFull = 0xffffffffu;

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
__device__ __forceinline__ uint32_t movmatrix_trans(uint32_t a) {
    uint32_t d;
    asm volatile("movmatrix.sync.aligned.m8n8.trans.b16 %0, %1;" : "=r"(d) : "r"(a));
    return d;
}
// D(16x8) += A(16x16) B(16x8), bf16 inputs, fp32 accumulate
__device__ __forceinline__ void mma_bf16(float (&c)[4], uint32_t a0, uint32_t a1, uint32_t a2, uint32_t a3,
                                         uint32_t b0, uint32_t b1) {
    asm volatile(
        "mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
        : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
        : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1));
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
__device__ __forceinline__ uint32_t lds_u16(uint32_t addr) {
    unsigned short v;
    asm volatile("ld.shared.u16 %0, [%1];" : "=h"(v) : "r"(addr));
    return v;
}
__device__ __forceinline__ uint32_t lds_u32(uint32_t addr) {
    uint32_t v;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(addr));
    return v;
}
__device__ __forceinline__ uint4 lds_128(uint32_t addr) {
    uint4 v;
    asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(addr));
    return v;
}
__device__ __forceinline__ uint32_t prmt(uint32_t a, uint32_t b, uint32_t sel) {
    uint32_t d;
    asm("prmt.b32 %0, %1, %2, %3;" : "=r"(d) : "r"(a), "r"(b), "r"(sel));
    return d;
}

// ---- mbarrier + 1-D bulk copy (TMA engine: one instruction moves a whole payload chunk) ------
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_init_fence() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
// global -> this CTA's shared memory; src, dst and bytes are multiples of 16
__device__ __forceinline__ void bulk_g2s(uint32_t dst, unsigned long long src, uint32_t bytes, uint32_t bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
                 "l"(src), "r"(bytes), "r"(bar)
                 : "memory");
}
// has the phase with this parity completed?  (does not block)
__device__ __forceinline__ bool mbar_test(uint32_t bar, uint32_t parity) {
    uint32_t ok;
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "mbarrier.test_wait.parity.shared::cta.b64 p, [%1], %2;\n"
        "selp.u32 %0, 1, 0, p;\n"
        "}\n"
        : "=r"(ok)
        : "r"(bar), "r"(parity)
        : "memory");
    return ok != 0u;
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "MKV_WAIT:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra MKV_DONE;\n"
        "bra MKV_WAIT;\n"
        "MKV_DONE:\n"
        "}\n" ::"r"(bar),
        "r"(parity)
        : "memory");
}

// Eight slots (byte BYTE of the position-bitmap word `w`) of one packed run: a set bit loads the
// next kept bf16 of the run and advances the run pointer by `step` bytes (2 n for a group of n
// vectors stored rank-major, 2 for a dense vector); a clear bit leaves 0.  Written as plain
// bit tests of ONE word in slot order so that ptxas if-converts them (predicated LDS.U16 + add, no
// branch) and derives seven predicates at a time with R2P instead of one LOP3 per slot.  The empty
// asm keeps the values opaque, so the pairing below stays one IMAD on zero-initialised registers.
template <int BYTE>
__device__ __forceinline__ void walk8(uint32_t w, uint32_t& ptr, uint32_t step, uint32_t (&v)[8]) {
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        v[i] = 0u;
        if (w & (1u << (8 * BYTE + i))) {
            v[i] = lds_u16(ptr);
            ptr += step;
        }
    }
#pragma unroll
    for (int i = 0; i < 8; ++i) asm volatile("" : "+r"(v[i]));
}
// hi * 65536 + lo: an IMAD (FMA pipe), not a PRMT/LOP3 (ALU pipe)
__device__ __forceinline__ uint32_t pair16(uint32_t lo, uint32_t hi) { return hi * 65536u + lo; }

// K walk: byte BYTE (8 channels of this lane's 32-channel word) of two runs -- token gq of block 0
// (rows 0-7 of the 16-token M tile) and of block 1 (rows 8-15) -- feeds two k-steps of S = K q^T.
// qa: B fragments of q for the k-steps 2 BYTE and 2 BYTE + 1 (same channel permutation).
template <int BYTE>
__device__ __forceinline__ void k_walk_mma(float (&S)[4], uint32_t w0, uint32_t w1, uint32_t& p0, uint32_t& p1,
                                           uint32_t st0, uint32_t st1, const uint32_t (&qa)[8][2]) {
    uint32_t e[8], f[8];
    walk8<BYTE>(w0, p0, st0, e);
    walk8<BYTE>(w1, p1, st1, f);
    mma_bf16(S, pair16(e[0], e[1]), pair16(f[0], f[1]), pair16(e[2], e[3]), pair16(f[2], f[3]), qa[2 * BYTE][0],
             qa[2 * BYTE][1]);
    mma_bf16(S, pair16(e[4], e[5]), pair16(f[4], f[5]), pair16(e[6], e[7]), pair16(f[6], f[7]), qa[2 * BYTE + 1][0],
             qa[2 * BYTE + 1][1]);
}

// K walk of vectors kept in element groups g = 2 or 4: the kept channels come in aligned pairs, the
// values of a group of vectors are stored PAIR-major (pair pi of vector t at 32-bit element pi * n + t, compress.cu), and
// a pair (c, c + 1) of one token IS one A-fragment register.  Byte BYTE of the (one bit per channel) bitmap word holds
// four pairs: a set even bit loads the pair with one aligned LDS.32 and advances the run pointer by `step` = 4 n bytes.
// Half the slots of the g = 1 walk, no packing of two halves.
template <int BYTE>
__device__ __forceinline__ void walk4_pairs(uint32_t w, uint32_t& ptr, uint32_t step, uint32_t (&v)[4]) {
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        v[i] = 0u;
        if (w & (1u << (8 * BYTE + 2 * i))) {
            v[i] = lds_u32(ptr);
            ptr += step;
        }
    }
#pragma unroll
    for (int i = 0; i < 4; ++i) asm volatile("" : "+r"(v[i]));
}
template <int BYTE>
__device__ __forceinline__ void k_walk_mma_pairs(float (&S)[4], uint32_t w0, uint32_t w1, uint32_t& p0, uint32_t& p1,
                                                 uint32_t st0, uint32_t st1, const uint32_t (&qa)[8][2]) {
    uint32_t e[4], f[4];
    walk4_pairs<BYTE>(w0, p0, st0, e);
    walk4_pairs<BYTE>(w1, p1, st1, f);
    mma_bf16(S, e[0], f[0], e[1], f[1], qa[2 * BYTE][0], qa[2 * BYTE][1]);
    mma_bf16(S, e[2], f[2], e[3], f[3], qa[2 * BYTE + 1][0], qa[2 * BYTE + 1][1]);
}

// V walk: byte BYTE (8 channels of this lane's 16-channel half-word) of four runs -- tokens
// A = 2qq and B = 2qq+1 of block 0 and of block 1 -- feeds four M tiles of O^T += V^T P^T with P
// split into bf16 hi (ph) and lo (pl).  A register pairs two TOKENS of one channel.
template <int BYTE>
__device__ __forceinline__ void v_walk_mma(float (&acc)[8][4], uint32_t hA0, uint32_t hB0, uint32_t hA1, uint32_t hB1,
                                           uint32_t& pA0, uint32_t& pB0, uint32_t& pA1, uint32_t& pB1, uint32_t st0,
                                           uint32_t st1, uint32_t ph0, uint32_t ph1, uint32_t pl0, uint32_t pl1) {
    uint32_t a0[8], b0[8], a1[8], b1[8];
    walk8<BYTE>(hA0, pA0, st0, a0);
    walk8<BYTE>(hB0, pB0, st0, b0);
    walk8<BYTE>(hA1, pA1, st1, a1);
    walk8<BYTE>(hB1, pB1, st1, b1);
#pragma unroll
    for (int j = 0; j < 4; ++j) {  // tile 4 BYTE + j: rows gq / gq+8 = channels 16gq + 8 BYTE + 2j / + 1
        const uint32_t x0 = pair16(a0[2 * j], b0[2 * j]), x1 = pair16(a0[2 * j + 1], b0[2 * j + 1]);
        const uint32_t x2 = pair16(a1[2 * j], b1[2 * j]), x3 = pair16(a1[2 * j + 1], b1[2 * j + 1]);
        mma_bf16(acc[4 * BYTE + j], x0, x1, x2, x3, ph0, ph1);
        mma_bf16(acc[4 * BYTE + j], x0, x1, x2, x3, pl0, pl1);
    }
}

// floor(p / d) for p < 2^56 without the 64-bit division subroutine: fp32 estimate, exact fix-up
__device__ __forceinline__ unsigned div_floor(unsigned long long p, unsigned d, float inv_d) {
    unsigned q = (unsigned)fminf((float)p * inv_d, 4.0e9f);
#pragma unroll 1
    while ((unsigned long long)q * d > p) --q;
#pragma unroll 1
    while ((unsigned long long)(q + 1) * d <= p) ++q;
    return q;
}


}  // namespace walk
}  // namespace mkv
