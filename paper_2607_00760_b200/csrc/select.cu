// select.cu — step 2 of the hot path: block scores on the packed block keys (PAPER.md:182,
// 214-216) and top-k block selection by token budget.  sm_100a.
#include "mkv_internal.cuh"

namespace mkv {

namespace {

constexpr unsigned kFull = 0xffffffffu;

__device__ __forceinline__ unsigned lanemask_lt() {
    unsigned m;
    asm("mov.u32 %0, %%lanemask_lt;" : "=r"(m));
    return m;
}

// order-preserving map fp32 -> u32 (larger float <=> larger key); -0 is folded onto +0
__device__ __forceinline__ uint32_t score_key(float s) {
    const uint32_t u = __float_as_uint(s + 0.0f);
    return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}

// ------------------------------------------------------------------------------------------
// score (v0): one thread per block key; packed vector product by walking the set bits of the
// position bitmap.  q of the unit's G heads sits in shared memory as fp32.
// ------------------------------------------------------------------------------------------
template <int GP>
__global__ void __launch_bounds__(256) mkv_score_kernel(CacheGeom g, LayerView lv, const uint16_t* __restrict__ q,
                                                        int reduce, float* __restrict__ scores) {
    const int unit = blockIdx.y;
    const int b = unit / g.n_kv_heads, h = unit % g.n_kv_heads;
    __shared__ float qs[kD][GP];  // [channel][head]: one channel's heads are contiguous
    for (int i = threadIdx.x; i < kD * GP; i += 256) {
        const int c = i / GP, gi = i % GP;
        qs[c][gi] = (gi < g.group)
                        ? bf16_bits_to_f32(q[((size_t)b * g.n_q_heads + (size_t)h * g.group + gi) * kD + c])
                        : 0.f;
    }
    __syncthreads();
    const int nseg = lv.unit_nseg[unit];
    const int blk = blockIdx.x * 256 + threadIdx.x;
    const int seg = blk / g.blocks_per_seg, i = blk % g.blocks_per_seg;
    if (seg >= nseg) return;
    const size_t e = (size_t)unit * lv.S_max + seg;
    const StratRec rec = lv.strat[e];
    const int nblk = (rec.n_tok + kB - 1) / kB;
    if (i >= nblk) return;
    const int r = rec.r_k;
    const uint8_t* base = lv.slice + ((size_t)lv.bk_off[e] << 4);
    float acc[GP];
#pragma unroll
    for (int gi = 0; gi < GP; ++gi) acc[gi] = 0.f;
    if (r < kD) {
        const uint4 bm = *reinterpret_cast<const uint4*>(base + 16 * i);
        const uint16_t* val = reinterpret_cast<const uint16_t*>(base + 16 * nblk + (size_t)i * 2 * r);
        const uint32_t words[4] = {bm.x, bm.y, bm.z, bm.w};
        int n = 0;
#pragma unroll
        for (int w = 0; w < 4; ++w) {
            uint32_t word = words[w];
            while (word) {
                const int c = 32 * w + __ffs(word) - 1;
                word &= word - 1;
                const float x = bf16_bits_to_f32(val[n++]);
#pragma unroll
                for (int gi = 0; gi < GP; ++gi) acc[gi] = fmaf(qs[c][gi], x, acc[gi]);
            }
        }
    } else {
        const uint16_t* val = reinterpret_cast<const uint16_t*>(base + (size_t)i * 2 * kD);
        for (int c = 0; c < kD; ++c) {
            const float x = bf16_bits_to_f32(val[c]);
#pragma unroll
            for (int gi = 0; gi < GP; ++gi) acc[gi] = fmaf(qs[c][gi], x, acc[gi]);
        }
    }
    float s = acc[0];
    if (reduce == 1) {
        for (int gi = 1; gi < g.group; ++gi) s += acc[gi];
    } else {
        for (int gi = 1; gi < g.group; ++gi) s = fmaxf(s, acc[gi]);
    }
    scores[(size_t)unit * g.score_stride + blk] = s + 0.0f;
}

// ------------------------------------------------------------------------------------------
// top-k: one CTA per unit.  MSB-first radix select (4 x 8 bits) on the order-preserving score
// keys finds the k-th best score; ties at that score go to the lower block index; the chosen
// blocks are emitted in ascending index order by a block-wide compaction.
// Budget rule (R8 = the oracle's walk): with uniform blocks of 8 tokens and at most
// one short block (the unit's last), the walk takes the k0 = budget/8 best blocks, plus one
// more iff the short block is among the k0+1 best and fits the remainder.
// ------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(1024) mkv_topk_kernel(CacheGeom g, LayerView lv, const float* __restrict__ scores,
                                                        int budget, int32_t* __restrict__ sel,
                                                        int32_t* __restrict__ sel_count, int k_max) {
    const int unit = blockIdx.x;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int ntok = lv.unit_ntok[unit];
    const int nblk = (ntok + kB - 1) / kB;
    const float* s = scores + (size_t)unit * g.score_stride;
    int32_t* out = sel + (size_t)unit * k_max;

    __shared__ unsigned hist[256];
    __shared__ uint32_t s_prefix;
    __shared__ int s_krem, s_neq;
    __shared__ int s_warp[32], s_warp2[32];

    const bool all = (ntok <= budget);
    const int k0 = budget / kB, rem = budget % kB, nbR = ntok % kB;
    const bool ragged_try = !all && nbR != 0 && nbR <= rem;
    int kq = all ? nblk : (ragged_try ? k0 + 1 : k0);  // rank whose key we look for
    uint32_t Ts = 0;
    int take_eq = 0;
    if (!all && kq > 0) {
        uint32_t prefix = 0;
        int krem = kq;
        for (int pass = 0; pass < 4; ++pass) {
            const int shift = 24 - 8 * pass;
            if (tid < 256) hist[tid] = 0;
            __syncthreads();
            const uint32_t hi_mask = pass == 0 ? 0u : (0xffffffffu << (shift + 8));
            for (int i = tid; i < nblk; i += 1024) {
                const uint32_t u = score_key(s[i]);
                if ((u & hi_mask) == prefix) atomicAdd(&hist[(u >> shift) & 255u], 1u);
            }
            __syncthreads();
            if (warp == 0) {
                unsigned mine[8], tot = 0;
#pragma unroll
                for (int j = 0; j < 8; ++j) { mine[j] = hist[8 * lane + j]; tot += mine[j]; }
                // suffix-exclusive sum over lanes: counts in bins above this lane's bins
                unsigned incl = tot;
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) {
                    const unsigned v = __shfl_down_sync(kFull, incl, o);
                    if (lane + o < 32) incl += v;
                }
                unsigned cum = incl - tot;
#pragma unroll
                for (int j = 7; j >= 0; --j) {
                    if (cum < (unsigned)krem && (unsigned)krem <= cum + mine[j]) {
                        s_prefix = prefix | ((uint32_t)(8 * lane + j) << shift);
                        s_krem = krem - (int)cum;
                        s_neq = (int)mine[j];
                    }
                    cum += mine[j];
                }
            }
            __syncthreads();
            prefix = s_prefix;
            krem = s_krem;
        }
        Ts = prefix;
        take_eq = krem;            // equals (by ascending index) inside the kq best
        const int n_eq = s_neq;    // all blocks whose score equals the threshold score
        if (ragged_try) {
            // the short block is the highest index: it is inside the k0+1 best iff it beats Ts or
            // ties with it and every tie is taken
            const uint32_t uR = score_key(s[nblk - 1]);
            const bool inside = (uR > Ts) || (uR == Ts && take_eq == n_eq);
            if (!inside) { take_eq -= 1; kq = k0; }
        }
    }

    // emission in ascending block index
    int carry_eq = 0, carry_out = 0;
    if (kq > 0) {
        for (int i0 = 0; i0 < nblk; i0 += 1024) {
            const int i = i0 + tid;
            bool gt = false, eq = false;
            if (i < nblk) {
                if (all) gt = true;
                else {
                    const uint32_t u = score_key(s[i]);
                    gt = u > Ts;
                    eq = u == Ts;
                }
            }
            const unsigned be = __ballot_sync(kFull, eq);
            if (lane == 0) s_warp[warp] = __popc(be);
            __syncthreads();
            int eq_before = carry_eq + __popc(be & lanemask_lt()), eq_total = 0;
            for (int w = 0; w < 32; ++w) {
                const int c = s_warp[w];
                if (w < warp) eq_before += c;
                eq_total += c;
            }
            const bool take = gt || (eq && eq_before < take_eq);
            const unsigned bt = __ballot_sync(kFull, take);
            if (lane == 0) s_warp2[warp] = __popc(bt);
            __syncthreads();
            int pos = carry_out + __popc(bt & lanemask_lt()), out_total = 0;
            for (int w = 0; w < 32; ++w) {
                const int c = s_warp2[w];
                if (w < warp) pos += c;
                out_total += c;
            }
            if (take && pos < k_max) out[pos] = i * kB;
            carry_eq += eq_total;
            carry_out += out_total;
            __syncthreads();
        }
    }
    const int count = min(carry_out, k_max);
    for (int p = count + tid; p < k_max; p += 1024) out[p] = -1;
    if (tid == 0) sel_count[unit] = count;
}

}  // namespace

cudaError_t launch_select(const CacheGeom& g, const LayerView& lv, const uint16_t* q, int budget, int reduce,
                          int32_t* sel, int32_t* sel_count, int k_max, float* scores, cudaStream_t s,
                          int* n_kernels) {
    dim3 grid((g.score_stride + 255) / 256, g.n_units);
    if (g.group <= 4) mkv_score_kernel<4><<<grid, 256, 0, s>>>(g, lv, q, reduce, scores);
    else mkv_score_kernel<8><<<grid, 256, 0, s>>>(g, lv, q, reduce, scores);
    cudaError_t err = cudaGetLastError();
    if (err != cudaSuccess) return err;
    mkv_topk_kernel<<<g.n_units, 1024, 0, s>>>(g, lv, scores, budget, sel, sel_count, k_max);
    if (n_kernels) *n_kernels = 2;
    return cudaGetLastError();
}

}  // namespace mkv
