// select.cu — step 2b of the hot path: top-k block selection by token budget
// on the scores of score.cu (step 2a).  sm_100a.
#include <mutex>

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
// The keys of a CTA are cached in registers when they fit (kKeyCap = 16 per thread, blocked: thread t
// holds elements [16 t, 16 t + 16)), so the radix passes and the emission read global memory once.  Histogram updates are aggregated per warp with match.any (scores cluster in a
// few bins of the first pass); the emission gives every thread a run of consecutive blocks, so one
// block-wide scan of packed (greater, equal) counts orders the whole output.
constexpr int kKeyCap = 16384;  // 64 KB of keys
static_assert(kKeyCap == kTopkSlice, "the candidate scratch of mkv_api.cu is sized in slices of kKeyCap blocks");

// MODE 0: the whole unit in one CTA (nblk <= kKeyCap, or any size with uncached keys).
// Long units (score_stride > kKeyCap, e.g. 1M tokens) are selected in two stages so that every
// key is read from global memory once and all SMs take part:
// MODE 1: CTA (unit, p) keeps the kq_cap best blocks of slice p (kKeyCap blocks) as candidates
//         (order-preserving key + block index, ascending index, padded with key 0);
// MODE 2: one CTA per unit runs the same selection over the concatenated candidates.  The kq best
//         of the unit are among the kq best of their slices, and positions stay in index order.
template <int MODE>
__global__ void __launch_bounds__(1024) mkv_topk_kernel(CacheGeom g, LayerView lv, const float* __restrict__ scores,
                                                        int budget, int32_t* __restrict__ sel,
                                                        int32_t* __restrict__ sel_count, int k_max,
                                                        uint32_t* __restrict__ cand_key, int32_t* __restrict__ cand_idx,
                                                        int n_slices, int cand_cap, PlanRec* __restrict__ plan,
                                                        int plan_stride, uint32_t tag) {
    const int unit = MODE == 1 ? blockIdx.x / n_slices : blockIdx.x;
    const int slice = MODE == 1 ? blockIdx.x % n_slices : 0;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    pdl_wait();  // the scores (MODE 0, 1) / the candidates (MODE 2) are complete
    pdl_launch_dependents();
    const int ntok = lv.unit_ntok[unit];
    const int kB = g.B;                           // tokens per block (the cache's token-block size)
    const int nblk = (ntok + kB - 1) / kB;        // blocks of the unit
    const float* s = scores + (size_t)unit * g.score_stride;
    // the elements this CTA selects from: n of them; element i has key keyat(i) and block index idxat(i)
    const int base = MODE == 1 ? slice * kKeyCap : 0;
    const int n = MODE == 0 ? nblk : (MODE == 1 ? max(0, min(kKeyCap, nblk - base)) : n_slices * cand_cap);
    const uint32_t* ck = MODE == 2 ? cand_key + (size_t)unit * n_slices * cand_cap : nullptr;
    const int32_t* ci = MODE == 2 ? cand_idx + (size_t)unit * n_slices * cand_cap : nullptr;
    auto keyat = [&](int i) -> uint32_t { return MODE == 2 ? ck[i] : score_key(s[base + i]); };
    auto idxat = [&](int i) -> int { return MODE == 2 ? ci[i] : base + i; };
    int32_t* out = MODE == 1 ? nullptr : sel + (size_t)unit * k_max;
    uint32_t* okey = MODE == 1 ? cand_key + ((size_t)unit * n_slices + slice) * cand_cap : nullptr;
    int32_t* oidx = MODE == 1 ? cand_idx + ((size_t)unit * n_slices + slice) * cand_cap : nullptr;
    const int cap = MODE == 1 ? cand_cap : k_max;
    const bool cached = n <= kKeyCap;

    __shared__ unsigned hist[2 * 4096];
    __shared__ int s_krem;
    __shared__ unsigned long long s_warp[32];
    __shared__ unsigned long long s_scan[32];  // the emission's scan (its own array: a warp may still be reading s_warp)

    const int k0 = budget / kB, rem = budget % kB, nbR = ntok % kB;
    // MODE 1 keeps k0 + 1 per slice (the most the final stage can ask for); every element if fewer
    const bool all = MODE == 1 ? (n <= k0 + 1) : (ntok <= budget);
    const bool ragged_try = MODE != 1 && !all && nbR != 0 && nbR <= rem;
    int kq = MODE == 1 ? min(n, k0 + 1) : (all ? nblk : (ragged_try ? k0 + 1 : k0));  // rank whose key we look for
    uint32_t Ts = 0;
    int take_eq = 0;
    constexpr int kPerThread = kKeyCap / 1024;
    uint32_t kv[kPerThread];  // this thread's keys when the CTA's elements fit (cached)
#pragma unroll
    for (int j = 0; j < kPerThread; ++j) kv[j] = 0u;
    if (!all && kq > 0) {
        if (cached) {  // n <= kKeyCap = 16 x 1024: thread t keeps elements [16 t, 16 t + 16) in registers
            const int i0 = kPerThread * tid;
            if (MODE != 2 && (reinterpret_cast<uintptr_t>(s + base) & 15) == 0 && i0 + kPerThread <= n) {
                const float4* s4 = reinterpret_cast<const float4*>(s + base + i0);
#pragma unroll
                for (int j = 0; j < kPerThread / 4; ++j) {
                    const float4 f = s4[j];
                    kv[4 * j] = score_key(f.x); kv[4 * j + 1] = score_key(f.y);
                    kv[4 * j + 2] = score_key(f.z); kv[4 * j + 3] = score_key(f.w);
                }
            } else {
#pragma unroll
                for (int j = 0; j < kPerThread; ++j) kv[j] = i0 + j < n ? keyat(i0 + j) : 0u;
            }
        }
        uint32_t prefix = 0;
        int krem = kq;
        // MSB-first radix select in three passes of 12 + 12 + 8 bits: with 4096 bins the scores spread
        // over enough bins for plain shared-memory atomics, and later passes touch few elements.
        // Two barriers per pass: the histograms alternate between two buffers (a buffer is cleared one pass ahead, between
        // the barriers of the pass in between), and once the warps' totals are known every warp finds the bin of the
        // wanted key on its own -- from the totals the warp that holds it, from that warp's bins the bin -- so nothing has
        // to be broadcast.
        for (int i = tid; i < 2 * 4096; i += 1024) hist[i] = 0;
        __syncthreads();
        int n_eq = 0;
        bool all_of_bin = false;
        for (int pass = 0; pass < 3; ++pass) {
            const int shift = pass == 0 ? 20 : (pass == 1 ? 8 : 0);
            const int nbins = pass == 2 ? 256 : 4096;
            unsigned* cur = hist + (pass & 1) * 4096;
            const uint32_t hi_mask = pass == 0 ? 0u : (0xffffffffu << (pass == 1 ? 20 : 8));
            if (cached) {
#pragma unroll
                for (int j = 0; j < kPerThread; ++j) {
                    const uint32_t u = kv[j];
                    if (kPerThread * tid + j < n && (u & hi_mask) == prefix)
                        atomicAdd(&cur[(u >> shift) & (uint32_t)(nbins - 1)], 1u);
                }
            } else {
                for (int i = tid; i < n; i += 1024) {
                    const uint32_t u = keyat(i);
                    if ((u & hi_mask) == prefix) atomicAdd(&cur[(u >> shift) & (uint32_t)(nbins - 1)], 1u);
                }
            }
            __syncthreads();
            if (pass == 1 && tid < 256) hist[tid] = 0;  // buffer 0 is free since this barrier: cleared for the last pass
            // thread t owns bins [t bpt, (t+1) bpt); suffix scan inside the warp (higher lanes hold higher bins)
            const int bpt = nbins >> 10;  // 4 or 0 (256 bins: one bin for each of the first 256 threads)
            unsigned tot = 0;
            if (bpt) {
#pragma unroll
                for (int j = 0; j < 4; ++j) tot += cur[4 * tid + j];
            } else if (tid < 256) {
                tot = cur[tid];
            }
#pragma unroll
            for (int o = 16; o >= 1; o >>= 1) tot += __shfl_xor_sync(kFull, tot, o);
            if (lane == 0) s_warp[warp] = tot;
            __syncthreads();
            // every warp: the warp W whose bins hold the krem-th key from the top, and the count above W
            const unsigned wt = (unsigned)s_warp[lane];
            unsigned wincl = wt;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const unsigned v = __shfl_down_sync(kFull, wincl, o);
                if (lane + o < 32) wincl += v;
            }
            const unsigned hitw = __ballot_sync(kFull, wincl - wt < (unsigned)krem && (unsigned)krem <= wincl);
            const int W = __ffs(hitw) - 1;
            const unsigned aboveW = __shfl_sync(kFull, wincl - wt, W);
            // the bins of W's threads, one thread's worth per lane
            const int tW = 32 * W + lane;
            unsigned b4[4] = {0u, 0u, 0u, 0u}, bt = 0;
            if (bpt) {
#pragma unroll
                for (int j = 0; j < 4; ++j) { b4[j] = cur[4 * tW + j]; bt += b4[j]; }
            } else if (tW < 256) {
                b4[0] = cur[tW]; bt = b4[0];
            }
            unsigned bincl = bt;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const unsigned v = __shfl_down_sync(kFull, bincl, o);
                if (lane + o < 32) bincl += v;
            }
            unsigned cum = aboveW + bincl - bt;
            const int nb_mine = bpt ? 4 : 1, bin0 = bpt ? 4 * tW : tW;
            int f_bin = -1;
            unsigned f_cum = 0u, f_cnt = 0u;
#pragma unroll
            for (int j = 3; j >= 0; --j) {
                if (j < nb_mine) {
                    if (cum < (unsigned)krem && (unsigned)krem <= cum + b4[j]) { f_bin = bin0 + j; f_cum = cum; f_cnt = b4[j]; }
                    cum += b4[j];
                }
            }
            const int src = __ffs(__ballot_sync(kFull, f_bin >= 0)) - 1;
            prefix |= (uint32_t)__shfl_sync(kFull, f_bin, src) << shift;
            krem -= (int)__shfl_sync(kFull, f_cum, src);
            n_eq = (int)__shfl_sync(kFull, f_cnt, src);
            // Every key of the bin is wanted (the usual case after 24 bits: the bin holds one key): the selection is
            // "every key >= prefix", and the remaining bits need not be resolved.  (Uniform over the CTA: every warp
            // derives krem and n_eq from the same histogram.  Not with a short last block: its rule needs the exact
            // threshold key and the number of keys equal to it.)
            if (pass < 2 && krem == n_eq && !ragged_try) { all_of_bin = true; break; }
        }
        Ts = prefix;
        take_eq = all_of_bin ? 0x7fffffff : krem;  // equals (by ascending index) inside the kq best
        // (n_eq: all elements whose key equals the threshold key)
        if (ragged_try) {
            // the short block is the highest index: it is inside the k0+1 best iff it beats Ts or
            // ties with it and every tie is taken (MODE 2: and it survived as a candidate, i.e. it is
            // the last real candidate of the last slice)
            const uint32_t uR = score_key(s[nblk - 1]);
            bool is_elem = true;
            if (MODE == 2) {
                const int ls = (nblk - 1) / kKeyCap;  // its slice; real candidates come first in a slice
                int lo = 0, hi = cand_cap;            // first padding entry of the slice, by bisection
                while (lo < hi) {
                    const int mid = (lo + hi) >> 1;
                    if (ci[ls * cand_cap + mid] >= 0) lo = mid + 1; else hi = mid;
                }
                is_elem = lo > 0 && ci[ls * cand_cap + lo - 1] == nblk - 1;
            }
            const bool inside = (uR > Ts) || (uR == Ts && take_eq == n_eq && is_elem);
            if (!inside) { take_eq -= 1; kq = k0; }
        }
    }

    // emission in ascending position (= ascending block index): thread t owns elements [t E, (t+1) E)
    int count = 0;
    if (kq > 0) {
        const int E = cached ? kPerThread : (n + 1023) / 1024;
        const int i0 = min(n, tid * E), i1 = min(n, i0 + E);
        unsigned long long mine = 0;  // greater | equal << 32 among this thread's elements
        if (all) {
            if (MODE == 2) { for (int i = i0; i < i1; ++i) mine += ci[i] >= 0 ? 1ull : 0ull; }
            else mine = (unsigned long long)(i1 - i0);
        } else
            if (cached) {
#pragma unroll
                for (int j = 0; j < kPerThread; ++j)
                    if (i0 + j < i1) mine += (kv[j] > Ts ? 1ull : 0ull) + (kv[j] == Ts ? (1ull << 32) : 0ull);
            } else {
                for (int i = i0; i < i1; ++i) {
                    const uint32_t u = keyat(i);
                    mine += (u > Ts ? 1ull : 0ull) + (u == Ts ? (1ull << 32) : 0ull);
                }
            }
        // block-wide exclusive scan of the packed counts
        unsigned long long incl = mine;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const unsigned long long v = __shfl_up_sync(kFull, incl, o);
            if (lane >= o) incl += v;
        }
        if (lane == 31) s_scan[warp] = incl;
        __syncthreads();
        if (warp == 0) {
            const unsigned long long w = s_scan[lane];
            unsigned long long wi = w;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const unsigned long long v = __shfl_up_sync(kFull, wi, o);
                if (lane >= o) wi += v;
            }
            s_scan[lane] = wi - w;
            if (lane == 31) s_krem = (int)((uint32_t)wi + min((uint32_t)take_eq, (uint32_t)(wi >> 32)));
        }
        __syncthreads();
        const unsigned long long before = s_scan[warp] + incl - mine;
        int gt_before = (int)(uint32_t)before, eq_before = (int)(before >> 32);
        count = s_krem;
        auto emit = [&](int i, uint32_t u) {
            bool gt = all, eq = false;
            if (all) {
                if (MODE == 2) gt = ci[i] >= 0;
            } else {
                gt = u > Ts;
                eq = u == Ts;
            }
            const bool take = gt || (eq && eq_before < take_eq);
            const int pos = gt_before + min(eq_before, take_eq);
            if (take && pos < cap) {
                if (MODE == 1) { okey[pos] = all ? keyat(i) : u; oidx[pos] = idxat(i); }
                else out[pos] = idxat(i) * kB;
            }
            gt_before += gt ? 1 : 0;
            eq_before += eq ? 1 : 0;
        };
        if (cached && !all) {
#pragma unroll
            for (int j = 0; j < kPerThread; ++j)
                if (i0 + j < i1) emit(i0 + j, kv[j]);
        } else {
            for (int i = i0; i < i1; ++i) emit(i, all ? 0u : keyat(i));
        }
    }
    count = min(count, cap);
    if (MODE != 1 && plan != nullptr) {
        // what mkv_packed_attention needs to know about every selected block (payload offset, tokens, r_k, r_v): one
        // record per block, looked up by all threads at once (one round of table reads for the whole unit)
        __syncthreads();  // the CTA's writes to `out` are visible to its own threads
        // (a block of 16 tokens is two device blocks: two records, at 2 p and 2 p + 1)
        for (int p = tid; p < count * g.ppb && p < plan_stride; p += 1024) {
            PlanRec pr;
            pr.t0 = out[p >> (g.ppb - 1)] + kPhys * (p & (g.ppb - 1)); pr.tag = tag;  // ppb is 1 or 2
            plan_lookup(g, lv, unit, pr.t0, pr.off16, pr.meta);
            plan[(size_t)unit * plan_stride + p] = pr;
        }
    }
    if (MODE == 1) {
        for (int p = count + tid; p < cap; p += 1024) { okey[p] = 0u; oidx[p] = -1; }  // padding: below every real key
    } else {
        for (int p = count + tid; p < k_max; p += 1024) out[p] = -1;
        if (tid == 0) sel_count[unit] = count;
    }
}

}  // namespace

cudaError_t launch_select(const CacheGeom& g, const LayerView& lv, const uint16_t* q, int budget, int reduce,
                          int32_t* sel, int32_t* sel_count, int k_max, float* scores, uint32_t* cand_key,
                          int32_t* cand_idx, PlanRec* plan, int plan_stride, uint32_t tag, int sm_count, cudaStream_t s,
                          int* n_kernels) {
    cudaError_t err = launch_score(g, lv, q, reduce, scores, sm_count, s);
    if (err != cudaSuccess) return err;
    const int n_slices = (g.score_stride + kKeyCap - 1) / kKeyCap;
    const int cand_cap = budget / g.B + 1 < kKeyCap ? budget / g.B + 1 : kKeyCap;  // candidates kept per slice
    if (n_slices == 1) {
        err = launch_pdl(mkv_topk_kernel<0>, dim3(g.n_units), dim3(1024), 0, s, g, lv, (const float*)scores, budget, sel,
                         sel_count, k_max, (uint32_t*)nullptr, (int32_t*)nullptr, 1, 0, plan, plan_stride, tag);
        if (err != cudaSuccess) return err;
        if (n_kernels) *n_kernels = 2;
    } else {
        err = launch_pdl(mkv_topk_kernel<1>, dim3(g.n_units * n_slices), dim3(1024), 0, s, g, lv, (const float*)scores, budget,
                         sel, sel_count, k_max, cand_key, cand_idx, n_slices, cand_cap, (PlanRec*)nullptr, 0, 0u);
        if (err != cudaSuccess) return err;
        err = launch_pdl(mkv_topk_kernel<2>, dim3(g.n_units), dim3(1024), 0, s, g, lv, (const float*)scores, budget, sel,
                         sel_count, k_max, cand_key, cand_idx, n_slices, cand_cap, plan, plan_stride, tag);
        if (err != cudaSuccess) return err;
        if (n_kernels) *n_kernels = 3;
    }
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------
// mkv_topk_static — the budgeted top-k for callers that may not allocate device memory.
//
// Everything else in this library works on an mkv_cache, and mkv_cache_create obtains its arenas and
// scratch with some two dozen cudaMalloc calls.  Some users can do neither that nor an allocation of
// their own at the point where they need a selection: a decode loop running inside a serving engine
// whose pool allocator was given all of the GPU's memory at start-up (a raw cudaMalloc there fails
// for lack of memory, and one that succeeds stalls every stream of the device while it runs), a
// plug-in that is handed device pointers by its host program and has no allocator to ask, or code
// that is only ever called between the launches of someone else's latency-critical step.  Such a
// caller already has block scores of its own (or took them from mkv_select's scores_opt earlier)
// and needs step 2b alone.
//
// The one piece of scratch the selection needs -- the candidate lists that the first stage of the
// two-stage selection (units of more than kKeyCap blocks) hands to the second -- therefore lives in
// the library image itself: a file-scope __device__ array of kStaticCand entries (key + index,
// 8 bytes each = 4 MB) that every GPU which loads this library holds until the process exits.
// Host code cannot use the array's name as an address (on the host the symbol is only a handle), so the
// device address is looked up once per device with cudaGetSymbolAddress, with that device current,
// and kept; the kernels receive that pointer like any other buffer.
//
// All calls on one device share the array.  Nothing in it has to start at zero: the first stage
// writes every entry of every (unit, slice) list it then reads, real candidates first and padding
// after them, so what an earlier call left behind is never read.  Two calls whose kernels can run
// at the same time on one device (different streams, or threads) would overwrite each other's
// candidates: order them.
// ------------------------------------------------------------------------------------------
namespace {

constexpr int kStaticCand = MKV_TOPK_STATIC_MAX_CANDIDATES;
static __device__ __align__(256) unsigned char g_static_cand[(size_t)kStaticCand * 8];  // [keys: kStaticCand x u32][indices: kStaticCand x i32]

constexpr int kStaticMaxDevices = 64;
std::mutex g_static_mutex;
void* g_static_addr[kStaticMaxDevices] = {};  // device address of g_static_cand on each device, once looked up

// device address of the static scratch on `device` (which must be the current device)
cudaError_t static_scratch(int device, unsigned char** p) {
    std::lock_guard<std::mutex> lock(g_static_mutex);
    if (!g_static_addr[device]) {
        void* a = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&a, g_static_cand);
        if (e != cudaSuccess) return e;
        g_static_addr[device] = a;
    }
    *p = (unsigned char*)g_static_addr[device];
    return cudaSuccess;
}

}  // namespace

}  // namespace mkv

extern "C" int mkv_topk_static(int32_t device, const float* scores, const int32_t* n_tokens, int32_t n_units,
                               int32_t score_stride, int32_t token_block, int32_t token_budget, int32_t* sel,
                               int32_t* sel_count, int32_t k_max, void* stream) {
    using namespace mkv;
    if (!scores || !n_tokens || !sel || !sel_count) return set_error(MKV_E_ARG, "mkv_topk_static: NULL argument");
    if (n_units < 1 || score_stride < 1 || token_budget < 0) return set_error(MKV_E_ARG, "mkv_topk_static: bad sizes");
    if (token_block != 4 && token_block != 8 && token_block != 16)
        return set_error(MKV_E_ARG, "mkv_topk_static: token_block %d: must be 4, 8 or 16", token_block);
    const long long need = (long long)token_budget / token_block + 1;
    if (k_max < 1 || k_max < (need < score_stride ? need : score_stride))
        return set_error(MKV_E_ARG, "mkv_topk_static: k_max %d too small for budget %d", k_max, token_budget);
    if (device < 0 || device >= kStaticMaxDevices) return set_error(MKV_E_ARG, "mkv_topk_static: device %d out of range", device);
    const int n_slices = (score_stride + kKeyCap - 1) / kKeyCap;
    const int cand_cap = (int)(need < kKeyCap ? need : kKeyCap);  // candidates kept per slice
    const long long entries = n_slices > 1 ? (long long)n_units * n_slices * cand_cap : 0;
    if (entries > kStaticCand)
        return set_error(MKV_E_ARG,
                         "mkv_topk_static: %d units x %d slices x %d candidates = %lld entries of scratch; the static "
                         "array holds MKV_TOPK_STATIC_MAX_CANDIDATES = %d (lower the budget or split the units over calls)",
                         n_units, n_slices, cand_cap, entries, kStaticCand);
    cudaError_t e = cudaSetDevice(device);
    unsigned char* scratch = nullptr;
    if (e == cudaSuccess) e = static_scratch(device, &scratch);
    if (e != cudaSuccess) return set_error(MKV_E_CUDA, "mkv_topk_static: %s", cudaGetErrorString(e));
    // the kernels of mkv_select, given a geometry that holds only what they read: B, the score stride and the token counts
    CacheGeom g{};
    g.n_units = n_units; g.B = token_block; g.pb = token_block < kPhys ? token_block : kPhys; g.ppb = token_block / g.pb;
    g.score_stride = score_stride;
    LayerView lv{};
    lv.unit_ntok = const_cast<int32_t*>(n_tokens);
    cudaStream_t s = (cudaStream_t)stream;
    if (n_slices == 1) {  // one stage: no scratch at all
        e = launch_pdl(mkv_topk_kernel<0>, dim3(n_units), dim3(1024), 0, s, g, lv, scores, (int)token_budget, sel, sel_count,
                       (int)k_max, (uint32_t*)nullptr, (int32_t*)nullptr, 1, 0, (PlanRec*)nullptr, 0, 0u);
    } else {
        uint32_t* cand_key = reinterpret_cast<uint32_t*>(scratch);
        int32_t* cand_idx = reinterpret_cast<int32_t*>(scratch + (size_t)kStaticCand * 4);
        e = launch_pdl(mkv_topk_kernel<1>, dim3(n_units * n_slices), dim3(1024), 0, s, g, lv, scores, (int)token_budget, sel,
                       sel_count, (int)k_max, cand_key, cand_idx, n_slices, cand_cap, (PlanRec*)nullptr, 0, 0u);
        if (e == cudaSuccess)
            e = launch_pdl(mkv_topk_kernel<2>, dim3(n_units), dim3(1024), 0, s, g, lv, scores, (int)token_budget, sel,
                           sel_count, (int)k_max, cand_key, cand_idx, n_slices, cand_cap, (PlanRec*)nullptr, 0, 0u);
    }
    if (e == cudaSuccess) e = cudaGetLastError();
    if (e != cudaSuccess) return set_error(MKV_E_CUDA, "mkv_topk_static: %s", cudaGetErrorString(e));
    return MKV_OK;
}
