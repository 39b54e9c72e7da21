// rotate.cu — per-head rotation fold.  The cache holds K' = K R_k^T and
// V' = V R_v^T (the caller rotates before mkv_compress_segment: the SVD is CPU-side management).  At
// decode the rotation is merged into the single query vector instead of the matrices: q' = q R_k^T feeds mkv_select
// and mkv_packed_attention unchanged, and the attention output is taken back with out = o' R_v.  sm_100a.
#include "mkv_internal.cuh"

namespace mkv {

namespace {

// q'[v][i] = bf16( sum_j q[v][j] * R[h][i][j] ), one fused multiply-add per j in ascending j (R22: q' is an
// input of the bf16 kernels, so its rounding is part of the definition).  CTA = one query vector, thread i = output i;
// the vector sits in shared memory, row i of R streams through 128-bit loads.
__global__ void __launch_bounds__(kD) mkv_rotate_query_kernel(const uint16_t* __restrict__ q, const float* __restrict__ R,
                                                              uint16_t* __restrict__ out, int n_q_heads, int group) {
    __shared__ float s_q[kD];
    const int v = blockIdx.x, i = threadIdx.x;
    const int hk = (v % n_q_heads) / group;
    s_q[i] = bf16_bits_to_f32(q[(size_t)v * kD + i]);
    __syncthreads();
    const float4* row = reinterpret_cast<const float4*>(R + ((size_t)hk * kD + i) * kD);
    float acc = 0.f;
#pragma unroll 8
    for (int j = 0; j < kD / 4; ++j) {
        const float4 r = __ldg(row + j);
        acc = __fmaf_rn(s_q[4 * j], r.x, acc);
        acc = __fmaf_rn(s_q[4 * j + 1], r.y, acc);
        acc = __fmaf_rn(s_q[4 * j + 2], r.z, acc);
        acc = __fmaf_rn(s_q[4 * j + 3], r.w, acc);
    }
    out[(size_t)v * kD + i] = (uint16_t)f32_to_bf16_bits_rne(acc);
}

// out[v][j] = sum_i o[v][i] * R[h][i][j] in fp32 (in place).  CTA = one output vector, thread j = output channel j:
// the loads of row i are coalesced across the CTA.
__global__ void __launch_bounds__(kD) mkv_rotate_output_kernel(float* __restrict__ o, const float* __restrict__ R,
                                                               int n_q_heads, int group) {
    __shared__ float s_o[kD];
    const int v = blockIdx.x, j = threadIdx.x;
    const int hk = (v % n_q_heads) / group;
    s_o[j] = o[(size_t)v * kD + j];
    __syncthreads();
    const float* Rh = R + (size_t)hk * kD * kD + j;
    float acc0 = 0.f, acc1 = 0.f;
#pragma unroll 8
    for (int i = 0; i < kD; i += 2) {
        acc0 = fmaf(s_o[i], __ldg(Rh + (size_t)i * kD), acc0);
        acc1 = fmaf(s_o[i + 1], __ldg(Rh + (size_t)(i + 1) * kD), acc1);
    }
    o[(size_t)v * kD + j] = acc0 + acc1;
}

}  // namespace

cudaError_t launch_rotate_query(const CacheGeom& g, const uint16_t* q, const float* Rk, uint16_t* q_out, cudaStream_t s) {
    mkv_rotate_query_kernel<<<g.batch * g.n_q_heads, kD, 0, s>>>(q, Rk, q_out, g.n_q_heads, g.group);
    return cudaGetLastError();
}

cudaError_t launch_rotate_output(const CacheGeom& g, float* out, const float* Rv, cudaStream_t s) {
    mkv_rotate_output_kernel<<<g.batch * g.n_q_heads, kD, 0, s>>>(out, Rv, g.n_q_heads, g.group);
    return cudaGetLastError();
}

}  // namespace mkv
