// mkv_internal.cuh — shared declarations of libmkv's CUDA translation units (sm_100a).
// Nothing here is used by, or derived from, the CPU oracle under oracle/.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include "mkv.h"

namespace mkv {

constexpr int kD = 128;          // head_dim supported on the GPU
constexpr int kPhys = 8;         // tokens of a device token block at most (one half of an mma M tile)
constexpr int kMaxGroup = 8;     // GQA group size limit
constexpr int kBitmapBytes = 16; // D/g/8 at g = 1

// strategy record as stored in the per-unit table and in the canonical blob (8 bytes)
struct __align__(8) StratRec {
    uint8_t r_k, r_v, g, B;
    uint16_t n_tok, flags;
};
static_assert(sizeof(StratRec) == 8, "strategy record is 8 bytes");

// Device-resident tables of one layer.  Offsets are in 16-byte units from `slice`.
struct LayerView {
    uint8_t* slice;               // packed payload slice of this layer (256-B aligned)
    uint64_t slice_bytes;
    StratRec* strat;              // [n_units][S_max]
    uint32_t* tok_off;            // [n_units][S_max]  token-block payloads of a segment
    uint32_t* bk_off;             // [n_units][S_max]  block-key payload of a segment
    int32_t* unit_nseg;           // [n_units]
    int32_t* unit_ntok;           // [n_units]
    unsigned long long* bump;     // bytes of `slice` in use
    unsigned long long* used_tok; // token-payload bytes in use (statistics)
    unsigned long long* used_bk;  // block-key payload bytes in use (statistics)
    int32_t S_max;
};

struct CacheGeom {
    int32_t n_layers, batch, n_kv_heads, n_q_heads, group, max_tokens, L, S_max, n_units;
    int32_t blocks_per_seg;   // L / B
    int32_t score_stride;     // ceil(max_tokens / B): blocks per unit capacity
    int32_t B;                // token-block size of the cache (4, 8 or 16): unit of selection, one block key each
    int32_t pb;               // tokens of a DEVICE token block: min(B, 8); a block of 16 tokens is stored as two of them
    int32_t ppb;              // device blocks per token block: B / pb (1 or 2)
};

// bytes of payloads (canonical sizes)
__host__ __device__ inline uint32_t pad16u(uint32_t x) { return (x + 15u) & ~15u; }
__host__ __device__ inline uint32_t vec_bytes(int r) { return (r == kD ? 0u : (uint32_t)kBitmapBytes) + 2u * (uint32_t)r; }
__host__ __device__ inline uint32_t tokblock_bytes(int r_k, int r_v, int nb) {
    return pad16u((uint32_t)nb * (vec_bytes(r_k) + vec_bytes(r_v)));
}
// device token blocks hold pb tokens, a segment's block keys one vector per B tokens
__host__ __device__ inline uint32_t seg_tok_bytes(int r_k, int r_v, int n_tok, int pb) {
    int full = n_tok / pb, rem = n_tok % pb;
    return (uint32_t)full * tokblock_bytes(r_k, r_v, pb) + (rem ? tokblock_bytes(r_k, r_v, rem) : 0u);
}
__host__ __device__ inline uint32_t seg_bk_bytes(int r_k, int n_tok, int B) {
    int nblk = (n_tok + B - 1) / B;
    return pad16u((uint32_t)nblk * vec_bytes(r_k));
}

// records the message mkv_last_error() returns on the calling thread and hands `code` back (mkv_api.cu): for entry
// points that live beside their kernels instead of in mkv_api.cu
int set_error(int code, const char* fmt, ...);

// ---- launchers (each enqueues on `stream`; returns cudaError) -----------------------------
struct CompressArgs {
    const uint16_t* k;
    const uint16_t* v;
    int64_t stride_b, stride_h, stride_t;
    int32_t b0, nb, seg0, nseg, n_tok;
    // top-r masks of the last mkv_segment_loss call, [unit][token][K, V] x 128 bits (or nullptr): mkv_compress_segment
    // takes a mask from here after checking it against the vector itself, so a stale entry is only a missed shortcut
    uint4* masks;
    int64_t mask_stride;  // tokens per unit in `masks` (= max_tokens)
};

cudaError_t launch_segment_loss(const CacheGeom& g, const CompressArgs& a, mkv_strategy cand,
                                double* loss_k, double* loss_v, cudaStream_t s);
cudaError_t launch_strategy_quantile(const double* loss_k, const double* loss_v, int n_units,
                                     int nseg, int n_dense, mkv_strategy sparse,
                                     mkv_strategy* out, cudaStream_t s);
cudaError_t launch_strategy_threshold(const double* loss_k, const double* loss_v, int ncand,
                                      long long n, const mkv_strategy* cands_host, double tau,
                                      mkv_strategy* out, cudaStream_t s);
cudaError_t launch_compress(const CacheGeom& g, const LayerView& lv, const CompressArgs& a,
                            const mkv_strategy* strat, unsigned long long* call_base,
                            uint32_t* dev_flags, cudaStream_t s, int* n_kernels);

cudaError_t launch_score(const CacheGeom& g, const LayerView& lv, const uint16_t* q, int reduce,
                         float* scores, int sm_count, cudaStream_t s);
struct PlanRec;
cudaError_t launch_select(const CacheGeom& g, const LayerView& lv, const uint16_t* q, int budget,
                          int reduce, int32_t* sel, int32_t* sel_count, int k_max, float* scores,
                          uint32_t* cand_key, int32_t* cand_idx, PlanRec* plan, int plan_stride, uint32_t tag,
                          int sm_count, cudaStream_t s, int* n_kernels);
constexpr int kTopkSlice = 16384;  // blocks per top-k slice (select.cu); longer units are selected in two stages

// One selected token block as the attention kernel needs it: a cache of the table lookups
// (strategy record + offset table) keyed by (layer, unit, position, first token).  mkv_select's top-k
// writes one record per selected block next to `sel`; mkv_packed_attention uses a record only if its
// tag and first token match the `sel` entry it reads (the packed arena is append-only, so a matching
// record is valid whatever call wrote it) and falls back to the tables otherwise.
struct __align__(16) PlanRec {
    int32_t t0;      // first token of the block
    uint32_t off16;  // payload offset in the layer slice, 16-B units
    uint32_t meta;   // r_k | r_v << 8 | nb << 16 | (g >= 2) << 24   (nb = tokens in the device block, 1..8; bit 24: the
                     // K values are stored pair-major, see mkv_walk.cuh)
    uint32_t tag;    // plan_tag(generation, layer); 0 = never written
};
// bit 31: written at all; bits 16-30: generation (15 bits); bits 0-15: layer.  The generation alone would let a record
// survive 32768 resets, so mkv_cache_reset also clears the records of the layers it resets (mkv_api.cu): a tag never
// has to tell two fillings of a layer apart on its own, and a captured launch that still carries an older tag finds
// no record of its own after a reset and falls back to the tables.
__host__ __device__ inline uint32_t plan_tag(uint32_t generation, int layer) {
    return ((generation & 0x7fffu) << 16) | ((uint32_t)layer & 0xffffu) | 0x80000000u;
}
#ifdef __CUDACC__
// table lookup of the DEVICE block that starts at token t0 of `unit`; meta = 0 if t0 is not a device-block start of the unit
__device__ __forceinline__ void plan_lookup(const CacheGeom& g, const LayerView& lv, int unit, int t0, uint32_t& off16,
                                            uint32_t& meta) {
    off16 = 0u; meta = 0u;
    if (t0 < 0 || t0 >= lv.unit_ntok[unit] || (t0 % g.pb) != 0) return;
    const int seg = t0 / g.L, in_seg = t0 - seg * g.L;
    const size_t e = (size_t)unit * lv.S_max + seg;
    const StratRec rec = lv.strat[e];
    if ((int)rec.n_tok <= in_seg) return;
    const uint32_t nb = (uint32_t)min(g.pb, (int)rec.n_tok - in_seg);
    off16 = lv.tok_off[e] + (uint32_t)(in_seg / g.pb) * (tokblock_bytes(rec.r_k, rec.r_v, g.pb) >> 4);
    meta = (uint32_t)rec.r_k | ((uint32_t)rec.r_v << 8) | (nb << 16) | (rec.g >= 2 && rec.r_k != kD ? 1u << 24 : 0u);
}
#endif

struct AttnScratch {
    float* zbuf;          // [n_units][z_unit_stride][8 G]  logits of blocks that do not fit a warp's shared-memory cache
    size_t z_unit_stride; // positions per unit in zbuf
    unsigned long long* stats;  // [8]       counters of mkv_attention_stats
    PlanRec* plan;        // [n_units][plan_stride] of this layer (may be nullptr)
    int32_t plan_stride;
    uint32_t plan_tag;
};
size_t attention_z_unit_stride(const CacheGeom& g);
size_t attention_zbuf_floats(const CacheGeom& g);
cudaError_t attention_prepare(const CacheGeom& g, int sm_count, int* cluster_cache);
// cluster_cache: two ints owned by the cache (cluster size chosen for the attention / the gather-only kernel; 0 = not yet)
cudaError_t launch_attention(const CacheGeom& g, const LayerView& lv, const uint16_t* q,
                             const int32_t* sel, const int32_t* sel_count, int k_max, float scale,
                             float* out, float* lse, const AttnScratch& scr, const uint16_t* upd_k,
                             const uint16_t* upd_v, const int32_t* upd_count, int sm_count, int* cluster_cache,
                             cudaStream_t s, int* n_kernels, bool gather_only = false);
cudaError_t launch_stream_read(const uint8_t* base, unsigned long long bytes, int sm_count, unsigned long long* sink,
                               cudaStream_t s);
cudaError_t launch_walk_probe(const CacheGeom& g, const LayerView& lv, const uint16_t* q, const int32_t* sel,
                              const int32_t* sel_count, int k_max, int reps, int sm_count, unsigned long long* sink,
                              cudaStream_t s);
// KV update buffer: copy n_new raw tokens of every unit into rows [n_have, n_have + n_new)
// and set the layer's device-side count to n_have + n_new
cudaError_t launch_update_copy(const CacheGeom& g, const CompressArgs& a, uint16_t* upd_k, uint16_t* upd_v,
                               int32_t* upd_count, int n_have, cudaStream_t s);

// rotation fold: q' = q R_k^T (bf16, fp32 FMA chain) and out = o' R_v (fp32, in place); R: [Hkv][D][D] fp32
cudaError_t launch_rotate_query(const CacheGeom& g, const uint16_t* q, const float* Rk, uint16_t* q_out, cudaStream_t s);
cudaError_t launch_rotate_output(const CacheGeom& g, float* out, const float* Rv, cudaStream_t s);

// ---- programmatic dependent launch (PDL) ----------------------------------------------------
// The decode kernels are launched with programmatic stream serialisation: kernel N+1 may be scheduled
// while kernel N drains, runs its global-memory-free preamble, and blocks in pdl_wait() until kernel N
// has completed and flushed.  Inside a captured CUDA graph this removes the launch gap between the
// three kernels of a decode step.  Everything a kernel reads or writes in global memory comes after
// pdl_wait(); pdl_launch_dependents() right after it lets the next kernel start as SMs free up.
#ifdef __CUDACC__
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

template <typename... KArgs, typename... Args>
inline cudaError_t launch_pdl(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t s,
                              Args... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = s;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr; cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kernel, KArgs(args)...);
}
#endif

// ---- small device helpers -----------------------------------------------------------------
__device__ __forceinline__ float bf16_bits_to_f32(uint32_t h) { return __uint_as_float(h << 16); }

// round-to-nearest-even fp32 -> bf16 bits (finite inputs)
__device__ __forceinline__ uint32_t f32_to_bf16_bits_rne(float f) {
    uint32_t u = __float_as_uint(f);
    u += 0x7FFFu + ((u >> 16) & 1u);
    return u >> 16;
}

}  // namespace mkv
