// attention.cu — step 3 of the hot path: PackedAttention: QK over the
// selected packed keys, online softmax, PV over the packed values, split-K combine.  sm_100a.
#include "mkv_internal.cuh"

namespace mkv {

namespace {

constexpr unsigned kFull = 0xffffffffu;
constexpr float kLog2e = 1.4426950408889634f;
constexpr float kLn2 = 0.6931471805599453f;

__device__ __forceinline__ unsigned lanemask_lt() {
    unsigned m;
    asm("mov.u32 %0, %%lanemask_lt;" : "=r"(m));
    return m;
}

// Expand one packed (or dense) vector into the lane's four channels lane + 32 j as fp32.
__device__ __forceinline__ void load_vector(const uint8_t* bm, const uint8_t* val, int r, int lane, float (&x)[4]) {
    const uint16_t* v16 = reinterpret_cast<const uint16_t*>(val);
    if (r == kD) {
#pragma unroll
        for (int j = 0; j < 4; ++j) x[j] = bf16_bits_to_f32(v16[lane + 32 * j]);
        return;
    }
    uint32_t w[4];
    if ((reinterpret_cast<uintptr_t>(bm) & 15u) == 0) {
        const uint4 w4 = *reinterpret_cast<const uint4*>(bm);
        w[0] = w4.x; w[1] = w4.y; w[2] = w4.z; w[3] = w4.w;
    } else {  // ragged token block: bitmaps are only 2-byte aligned
        const uint16_t* b16 = reinterpret_cast<const uint16_t*>(bm);
#pragma unroll
        for (int j = 0; j < 4; ++j) w[j] = (uint32_t)b16[2 * j] | ((uint32_t)b16[2 * j + 1] << 16);
    }
    const unsigned lt = lanemask_lt();
    int base = 0;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        x[j] = ((w[j] >> lane) & 1u) ? bf16_bits_to_f32(v16[base + __popc(w[j] & lt)]) : 0.f;
        base += __popc(w[j]);
    }
}

// ------------------------------------------------------------------------------------------
// v0 kernel: CTA = (split, unit), 4 warps; each warp walks whole token blocks of its split,
// one token at a time, lane l owning channels l + 32 j.  Partial (max, sum, o) per CTA.
// ------------------------------------------------------------------------------------------
template <int GP>
__global__ void __launch_bounds__(128) mkv_packed_attention_kernel(CacheGeom g, LayerView lv,
                                                                   const uint16_t* __restrict__ q,
                                                                   const int32_t* __restrict__ sel,
                                                                   const int32_t* __restrict__ sel_count, int k_max,
                                                                   float scale_log2, float* __restrict__ part_o,
                                                                   float* __restrict__ part_ml, int nsplit) {
    const int unit = blockIdx.y, split = blockIdx.x;
    const int b = unit / g.n_kv_heads, h = unit % g.n_kv_heads;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int count = sel_count[unit];
    const int per = (count + nsplit - 1) / nsplit;
    const int lo = split * per, hi = min(count, lo + per);

    float qr[GP][4];
#pragma unroll
    for (int gi = 0; gi < GP; ++gi)
#pragma unroll
        for (int j = 0; j < 4; ++j)
            qr[gi][j] = (gi < g.group)
                            ? bf16_bits_to_f32(q[((size_t)b * g.n_q_heads + (size_t)h * g.group + gi) * kD + lane + 32 * j])
                            : 0.f;
    float m[GP], l[GP], o[GP][4];
#pragma unroll
    for (int gi = 0; gi < GP; ++gi) {
        m[gi] = -INFINITY;
        l[gi] = 0.f;
#pragma unroll
        for (int j = 0; j < 4; ++j) o[gi][j] = 0.f;
    }
    for (int bi = lo + warp; bi < hi; bi += 4) {
        const int t0 = sel[(size_t)unit * k_max + bi];
        const int seg = t0 / g.L, in_seg = t0 % g.L;
        const size_t e = (size_t)unit * lv.S_max + seg;
        const StratRec rec = lv.strat[e];
        const int nb = min(kB, (int)rec.n_tok - in_seg);
        const int r_k = rec.r_k, r_v = rec.r_v;
        const uint32_t bmk = (r_k == kD) ? 0u : kBitmapBytes, bmv = (r_v == kD) ? 0u : kBitmapBytes;
        const uint8_t* base = lv.slice + ((size_t)lv.tok_off[e] << 4) + (size_t)(in_seg / kB) * tokblock_bytes(r_k, r_v, kB);
        const uint8_t* k_bm = base;
        const uint8_t* k_val = k_bm + nb * bmk;
        const uint8_t* v_bm = k_val + nb * r_k * 2;
        const uint8_t* v_val = v_bm + nb * bmv;
        for (int t = 0; t < nb; ++t) {
            float kx[4], vx[4];
            load_vector(k_bm + t * bmk, k_val + t * r_k * 2, r_k, lane, kx);
            load_vector(v_bm + t * bmv, v_val + t * r_v * 2, r_v, lane, vx);
#pragma unroll
            for (int gi = 0; gi < GP; ++gi) {
                float z = qr[gi][0] * kx[0];
                z = fmaf(qr[gi][1], kx[1], z);
                z = fmaf(qr[gi][2], kx[2], z);
                z = fmaf(qr[gi][3], kx[3], z);
#pragma unroll
                for (int off = 16; off; off >>= 1) z += __shfl_xor_sync(kFull, z, off);
                z *= scale_log2;
                const float mn = fmaxf(m[gi], z);
                const float corr = exp2f(m[gi] - mn);
                const float p = exp2f(z - mn);
                l[gi] = l[gi] * corr + p;
#pragma unroll
                for (int j = 0; j < 4; ++j) o[gi][j] = fmaf(p, vx[j], o[gi][j] * corr);
                m[gi] = mn;
            }
        }
    }
    // merge the 4 warps
    __shared__ float s_m[4][GP], s_l[4][GP], s_o[4][GP][kD];
#pragma unroll
    for (int gi = 0; gi < GP; ++gi) {
        if (lane == 0) { s_m[warp][gi] = m[gi]; s_l[warp][gi] = l[gi]; }
#pragma unroll
        for (int j = 0; j < 4; ++j) s_o[warp][gi][lane + 32 * j] = o[gi][j];
    }
    __syncthreads();
    const int c = threadIdx.x;
    for (int gi = 0; gi < g.group; ++gi) {
        float M = -INFINITY;
        for (int w = 0; w < 4; ++w) M = fmaxf(M, s_m[w][gi]);
        float L = 0.f, O = 0.f;
        for (int w = 0; w < 4; ++w) {
            const float wgt = (s_m[w][gi] == -INFINITY) ? 0.f : exp2f(s_m[w][gi] - M);
            L = fmaf(s_l[w][gi], wgt, L);
            O = fmaf(s_o[w][gi][c], wgt, O);
        }
        const size_t p = ((size_t)unit * nsplit + split) * g.group + gi;
        part_o[p * kD + c] = O;
        if (c == 0) { part_ml[2 * p] = M; part_ml[2 * p + 1] = L; }
    }
}

// step 3d: merge the split partials of a unit, normalise, write out / lse
__global__ void __launch_bounds__(128) mkv_combine_kernel(CacheGeom g, const float* __restrict__ part_o,
                                                          const float* __restrict__ part_ml, int nsplit,
                                                          float* __restrict__ out, float* __restrict__ lse) {
    const int unit = blockIdx.x, gi = blockIdx.y, c = threadIdx.x;
    const int b = unit / g.n_kv_heads, h = unit % g.n_kv_heads;
    float M = -INFINITY;
    for (int s = 0; s < nsplit; ++s) M = fmaxf(M, part_ml[2 * (((size_t)unit * nsplit + s) * g.group + gi)]);
    float L = 0.f, O = 0.f;
    for (int s = 0; s < nsplit; ++s) {
        const size_t p = ((size_t)unit * nsplit + s) * g.group + gi;
        const float ms = part_ml[2 * p];
        const float wgt = (ms == -INFINITY) ? 0.f : exp2f(ms - M);
        L = fmaf(part_ml[2 * p + 1], wgt, L);
        O = fmaf(part_o[p * kD + c], wgt, O);
    }
    const size_t row = (size_t)b * g.n_q_heads + (size_t)h * g.group + gi;
    out[row * kD + c] = (L > 0.f) ? O / L : 0.f;
    if (lse != nullptr && c == 0) lse[row] = (L > 0.f) ? (M + log2f(L)) * kLn2 : -INFINITY;
}

}  // namespace

cudaError_t launch_attention(const CacheGeom& g, const LayerView& lv, const uint16_t* q, const int32_t* sel,
                             const int32_t* sel_count, int k_max, float scale, float* out, float* lse,
                             const AttnScratch& scr, int sm_count, cudaStream_t s, int* n_kernels) {
    int nsplit = (4 * sm_count + g.n_units - 1) / g.n_units;
    nsplit = max(1, min(nsplit, scr.max_splits));
    dim3 grid(nsplit, g.n_units);
    const float scale_log2 = scale * kLog2e;
    if (g.group <= 4)
        mkv_packed_attention_kernel<4><<<grid, 128, 0, s>>>(g, lv, q, sel, sel_count, k_max, scale_log2,
                                                            scr.part_o, scr.part_ml, nsplit);
    else
        mkv_packed_attention_kernel<8><<<grid, 128, 0, s>>>(g, lv, q, sel, sel_count, k_max, scale_log2,
                                                            scr.part_o, scr.part_ml, nsplit);
    cudaError_t err = cudaGetLastError();
    if (err != cudaSuccess) return err;
    dim3 cgrid(g.n_units, g.group);
    mkv_combine_kernel<<<cgrid, 128, 0, s>>>(g, scr.part_o, scr.part_ml, nsplit, out, lse);
    if (n_kernels) *n_kernels = 2;
    return cudaGetLastError();
}

}  // namespace mkv
