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

// One slot of a packed run: if bit MASK of the position bitmap `w` is set, load the next kept
// bf16 of the run into `v` (which the caller zero-initialised) and advance the run pointer.
// Predicated, no branch: every lane executes the same instruction stream whatever its bitmap.
template <uint32_t MASK>
__device__ __forceinline__ void take_slot(uint32_t w, uint32_t& v, uint32_t& ptr) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        ".reg .b32 t;\n"
        "and.b32 t, %2, %3;\n"
        "setp.ne.u32 p, t, 0;\n"
        "@p ld.shared.u16 %0, [%1];\n"
        "@p add.u32 %1, %1, 2;\n"
        "}\n"
        : "+r"(v), "+r"(ptr)
        : "r"(w), "n"(MASK)
        : "memory");
}
// hi * 65536 + lo: an IMAD (FMA pipe), not a PRMT/LOP3 (ALU pipe, which the bit tests load)
__device__ __forceinline__ uint32_t pair16(uint32_t lo, uint32_t hi) { return hi * 65536u + lo; }

// K walk, k-step KS (4 slots of this lane's bitmap word) of two runs at once (token gq of block
// 0 and of block 1) -> A fragment a0..a3
template <int KS>
__device__ __forceinline__ void k_step(uint32_t w0, uint32_t w1, uint32_t& p0, uint32_t& p1, uint32_t (&b)[4]) {
    uint32_t e[4] = {0u, 0u, 0u, 0u}, f[4] = {0u, 0u, 0u, 0u};
    take_slot<1u << (4 * KS + 0)>(w0, e[0], p0);
    take_slot<1u << (4 * KS + 0)>(w1, f[0], p1);
    take_slot<1u << (4 * KS + 1)>(w0, e[1], p0);
    take_slot<1u << (4 * KS + 1)>(w1, f[1], p1);
    take_slot<1u << (4 * KS + 2)>(w0, e[2], p0);
    take_slot<1u << (4 * KS + 2)>(w1, f[2], p1);
    take_slot<1u << (4 * KS + 3)>(w0, e[3], p0);
    take_slot<1u << (4 * KS + 3)>(w1, f[3], p1);
    b[0] = pair16(e[0], e[1]);  // row gq   (block 0), k = 2qq, 2qq+1
    b[1] = pair16(f[0], f[1]);  // row gq+8 (block 1)
    b[2] = pair16(e[2], e[3]);  // row gq,   k = 2qq+8, 2qq+9
    b[3] = pair16(f[2], f[3]);  // row gq+8
}

// V walk, M tile I (channel slots 2I, 2I+1 of this lane's half-word) of four runs at once
// (tokens A = 2qq and B = 2qq+1 of block 0 and of block 1) -> A fragment a0..a3
template <int I>
__device__ __forceinline__ void v_step(uint32_t hA0, uint32_t hB0, uint32_t hA1, uint32_t hB1, uint32_t& pA0,
                                       uint32_t& pB0, uint32_t& pA1, uint32_t& pB1, uint32_t (&a)[4]) {
    uint32_t x[8] = {0u, 0u, 0u, 0u, 0u, 0u, 0u, 0u};
    take_slot<1u << (2 * I)>(hA0, x[0], pA0);
    take_slot<1u << (2 * I)>(hB0, x[1], pB0);
    take_slot<1u << (2 * I)>(hA1, x[4], pA1);
    take_slot<1u << (2 * I)>(hB1, x[5], pB1);
    take_slot<1u << (2 * I + 1)>(hA0, x[2], pA0);
    take_slot<1u << (2 * I + 1)>(hB0, x[3], pB0);
    take_slot<1u << (2 * I + 1)>(hA1, x[6], pA1);
    take_slot<1u << (2 * I + 1)>(hB1, x[7], pB1);
    a[0] = pair16(x[0], x[1]);  // row gq   (channel 16gq + 2I),     tokens 2qq, 2qq+1 of block 0
    a[1] = pair16(x[2], x[3]);  // row gq+8 (channel 16gq + 2I + 1), block 0
    a[2] = pair16(x[4], x[5]);  // row gq,   block 1
    a[3] = pair16(x[6], x[7]);  // row gq+8, block 1
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
