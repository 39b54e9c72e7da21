// select.cu — step 2b of the hot path: top-k block selection by token budget
// on the scores of score.cu (step 2a).  sm_100a.
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
                          int32_t* sel, int32_t* sel_count, int k_max, float* scores, int sm_count,
                          cudaStream_t s, int* n_kernels) {
    cudaError_t err = launch_score(g, lv, q, reduce, scores, sm_count, s);
    if (err != cudaSuccess) return err;
    mkv_topk_kernel<<<g.n_units, 1024, 0, s>>>(g, lv, scores, budget, sel, sel_count, k_max);
    if (n_kernels) *n_kernels = 2;
    return cudaGetLastError();
}

}  // namespace mkv
