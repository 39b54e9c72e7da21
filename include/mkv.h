/*
 * mkv.h — C ABI of libmkv: decode-time attention over a dynamically two-D-compressed KV cache
 * (MosaicKV, arxiv/paper_2607_00760), hand-written CUDA for NVIDIA B200 (sm_100a).
 *
 * The hot path has three steps (§4.2, §5.1-5.3):
 *   1. compress  — per K/V vector keep the top-r elements by |x|, compute the
 *                  per-block mean keys, choose a strategy per segment
 *                   and pack kept elements behind a position bitmap
 *                  (PAPER.md:194-196);
 *   2. select    — score every token block with the current query on the packed block keys and
 *                  keep the top-k blocks;
 *   3. attention — PackedAttention: QK, softmax and PV over the selected packed tokens only
 *                  (PAPER.md:214-222), with a split-K combine.
 *
 * Conventions
 *   - Plain C, no torch types.  Every pointer is a DEVICE pointer unless its name ends in
 *     `_host`.  bf16 tensors are passed as `const void*` to uint16 bit patterns.
 *   - Every function returns MKV_OK (0) or a negative mkv_status; nothing throws or aborts.
 *     `mkv_last_error()` returns a thread-local message for the last failing call.
 *   - Argument errors are detected on the host before anything is enqueued.  Errors only a
 *     kernel can see (arena overflow, an invalid strategy record in device memory) set a sticky
 *     device flag that `mkv_cache_status()` reads (it synchronises).
 *   - `stream` is a cudaStream_t passed as void* (NULL = legacy default stream).  Except for
 *     create / free / export / bytes / status, calls only enqueue work and return immediately;
 *     they are CUDA-graph capturable (no allocation, no synchronisation).
 *   - Ownership: the caller owns every buffer it passes; the cache owns the packed arenas, its
 *     tables and its scratch.  A cache is not thread-safe; distinct caches are independent.  All
 *     calls on one cache must be ordered on one stream (or by events).
 *   - A *unit* is one (layer, request b, KV head h); units never interact.  Query head hq uses
 *     KV head hq / (n_q_heads / n_kv_heads).
 *   - Supported on the GPU today: head_dim = 128, token blocks B = 4, 8, 16 (one B per cache, mkv_cache_desc.token_block),
 *     element groups g = 1, 2, 4 (kept elements a multiple of g), segment_len a multiple of 8 and of B in [8, 4096], group G = n_q_heads/n_kv_heads <= 8.  Anything
 *     else is MKV_E_UNSUPPORTED / MKV_E_ARG (host-visible) or MKV_DEV_BAD_STRATEGY (device-visible).
 *   - Inputs must be finite; behaviour on NaN/Inf is unspecified.
 *
 * Canonical packed format (what mkv_cache_export returns; byte-identical to the CPU oracle):
 * see DESIGN.md "Canonical packed format".  In short, per unit:
 *   packed vector   = [bitmap D/g bits, LSB-first little-endian][kept bf16, ascending channel];
 *                     the bitmap is omitted when r == D
 *   token block     = [K bitmaps nb][K values nb*r_k][V bitmaps nb][V values nb*r_v], pad to 16 B
 *   segment         = its token blocks in order; block keys of the segment (separate arena) =
 *                     [bitmaps nblk][values nblk*r_k], pad to 16 B
 *   blob            = header(48 B) | strategy[S] (8 B) | tok_off[S] u32 | bk_off[S] u32 | pad16 |
 *                     token arena | block-key arena          (offsets in 16-B units)
 */
#ifndef MKV_H
#define MKV_H

#include <stdint.h>

#if defined(__GNUC__)
#define MKV_API __attribute__((visibility("default")))
#else
#define MKV_API
#endif

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    MKV_OK = 0,
    MKV_E_ARG = -1,          /* NULL / out-of-range / inconsistent argument */
    MKV_E_UNSUPPORTED = -2,  /* valid in the format, not built on the GPU yet (see Conventions) */
    MKV_E_NOMEM = -3,        /* device or host allocation failed */
    MKV_E_CUDA = -4,         /* a CUDA runtime call failed; message in mkv_last_error() */
    MKV_E_STATE = -5,        /* append-order violation (segments must arrive in ascending order) */
    MKV_E_DEVICE = -6        /* sticky device-side flag set; see mkv_cache_status */
} mkv_status;

/* device-side sticky flags reported by mkv_cache_status */
#define MKV_DEV_ARENA_OVERFLOW 1u /* a compress call needed more arena than the layer slice holds */
#define MKV_DEV_BAD_STRATEGY 2u   /* a strategy record in device memory was invalid/unsupported */

typedef struct mkv_cache mkv_cache; /* opaque: packed arenas + tables + scratch of one model */

typedef struct {
    int32_t n_layers;     /* >= 1 */
    int32_t batch;        /* requests */
    int32_t n_kv_heads;
    int32_t n_q_heads;    /* multiple of n_kv_heads, group <= 8 */
    int32_t head_dim;     /* D, must be 128 */
    int32_t max_tokens;   /* capacity per request */
    int32_t segment_len;  /* L: tokens per segment = granularity of the strategy */
    int32_t device;       /* CUDA device ordinal */
    uint64_t arena_bytes; /* packed payload bytes for ALL layers (split evenly per layer);
                             0 = size for the dense worst case */
    int32_t token_block;  /* B: tokens per token block = unit of selection, one block key each (4, 8 or 16;
                             0 = 8).  Every strategy of the cache must carry this B; segment_len must be a multiple of it */
    int32_t reserved;     /* must be 0 (anything else: MKV_E_ARG) */
} mkv_cache_desc;

/* Per-segment compression strategy: kept elements per K / V vector (multiples of
 * g, 1..D; r == D means "not channel-compressed"), element-group size, token-block size. */
typedef struct {
    uint8_t r_k, r_v, g, B;
} mkv_strategy;

/* Create / destroy.  `desc_host` is read during the call only.  Both calls synchronise. */
MKV_API int mkv_cache_create(const mkv_cache_desc* desc_host, mkv_cache** out);
MKV_API int mkv_cache_free(mkv_cache* cache); /* NULL is a no-op */

/* Forget every segment of `layer` (-1 = all layers) so it can be compressed again. */
MKV_API int mkv_cache_reset(mkv_cache* cache, int32_t layer, void* stream);

/*
 * Step 1c: compression loss of ONE candidate strategy.
 * k, v: bf16, element [b][h][t][c] at base + (b-b0)*stride_b + h*stride_h + t*stride_t + c
 * (strides in elements, channels contiguous), holding tokens [seg0*L, seg0*L + n_tok) of requests
 * [b0, b0+nb); nseg = ceil(n_tok / L), only the last segment may be short.
 * loss_k, loss_v: double [nb][n_kv_heads][nseg]:  sum of squares of the dropped elements /
 * sum of squares of all elements of the segment (0 if the segment is all zeros), fp64.
 */
MKV_API int mkv_segment_loss(const mkv_cache* cache, const void* k, const void* v, int64_t stride_b,
                     int64_t stride_h, int64_t stride_t, int32_t b0, int32_t nb, int32_t seg0,
                     int32_t nseg, int32_t n_tok, mkv_strategy cand, double* loss_k,
                     double* loss_v, void* stream);

/*
 * Step 1c, strategy choice.  Both write strat_out [n_units][nseg] (device).
 * quantile  (BASELINE.json config policy): per unit, the ceil(nseg*dense_num/dense_den) segments
 *           with the largest importance I = (loss_k+loss_v)/2 (ties -> lower segment index) get
 *           r_k = r_v = D; all others get `sparse`.
 * threshold: loss_k/loss_v are [ncand][n_units*nseg]; candidates are ordered most
 *           -> least aggressive; the first with I <= tau wins, none -> dense (g = 1).
 */
MKV_API int mkv_strategy_quantile(const mkv_cache* cache, const double* loss_k, const double* loss_v,
                          int32_t n_units, int32_t nseg, int32_t dense_num, int32_t dense_den,
                          mkv_strategy sparse, mkv_strategy* strat_out, void* stream);
MKV_API int mkv_strategy_threshold(const mkv_cache* cache, const double* loss_k, const double* loss_v,
                           int32_t ncand, int32_t n_units, int32_t nseg,
                           const mkv_strategy* cands_host, double tau, mkv_strategy* strat_out,
                           void* stream);

/*
 * Steps 1a, 1b, 1d: compress and pack segments [seg0, seg0+nseg) of
 * requests [b0, b0+nb) of `layer`; nseg = 1 is the literal "compress one segment".
 * k, v as in mkv_segment_loss.  strat: device, [nb][n_kv_heads][nseg].
 * Append-only: seg0 must equal the number of segments the request already holds in this layer
 * and its last segment must be full, else MKV_E_STATE.
 */
MKV_API int mkv_compress_segment(mkv_cache* cache, int32_t layer, const void* k, const void* v,
                         int64_t stride_b, int64_t stride_h, int64_t stride_t, int32_t b0,
                         int32_t nb, int32_t seg0, int32_t nseg, int32_t n_tok,
                         const mkv_strategy* strat, void* stream);

/*
 * Step 2: score every token block of every unit of `layer` with q on
 * the packed block keys (no 1/sqrt(D)), reduce over the GQA group (0 = max, 1 = sum) and select
 * blocks by (score descending, index ascending) while they fit in `token_budget` tokens.
 * q: bf16 [batch][n_q_heads][D].  sel: int32 [batch][n_kv_heads][k_max], first-token index of each
 * chosen block, ascending; unused tail = -1.  sel_count: int32 [batch][n_kv_heads].
 * k_max must be >= min(token_budget / B + 1, blocks per unit).  scores_opt: float
 * [batch][n_kv_heads][score_stride] or NULL, score_stride = ceil(max_tokens / B).
 */
MKV_API int mkv_select(const mkv_cache* cache, int32_t layer, const void* q, int32_t token_budget,
               int32_t reduce, int32_t* sel, int32_t* sel_count, int32_t k_max, float* scores_opt,
               void* stream);

/*
 * Step 3: PackedAttention over the tokens of the selected blocks, plus the
 * tokens of the layer's KV update buffer if it holds any (see mkv_update_append).
 * sel / sel_count as written by mkv_select (any order of blocks is accepted; entries the caller changed after
 * mkv_select are honoured: the per-block records mkv_select leaves for this call are verified against `sel`).
 * At most ceil(max_tokens / B) + 1 entries per unit are attended (one more than the unit has blocks); a caller-built
 * list that is longer (k_max and sel_count beyond that, which takes duplicates) is cut there.
 * One launch: one thread-block cluster per unit (one CTA per SM); the CTAs of a cluster exchange their maxima and partial
 * results through each other's shared memory (counted asynchronous stores, cluster barriers for clusters larger than two),
 * nothing else is shared between CTAs.
 * out: float [batch][n_q_heads][D].  lse_opt: float [batch][n_q_heads] or NULL (log-sum-exp of the
 * scaled logits; -inf and out = 0 for an empty selection).
 */
MKV_API int mkv_packed_attention(const mkv_cache* cache, int32_t layer, const void* q, const int32_t* sel,
                         const int32_t* sel_count, int32_t k_max, float softmax_scale, float* out,
                         float* lse_opt, void* stream);

/*
 * KV update buffer: the newest tokens of every unit are held uncompressed until a
 * whole segment can be compressed.  mkv_packed_attention attends the buffered tokens of `layer`
 * densely, after the selected packed blocks, and merges the two by the log-sum-exp rule; mkv_select
 * does not see them (they are always attended).
 *   append: k_new, v_new bf16, element [b][h][t][c] at base + b*stride_b + h*stride_h + t*stride_t + c
 *           for ALL requests b of the cache, t in [0, n_new): the next n_new tokens of every unit.
 *           The buffer holds at most segment_len tokens: MKV_E_STATE if they do not fit.
 *   flush:  compress the buffered tokens as the next segment of every unit (steps 1a, 1b, 1d; strat:
 *           device, [batch][n_kv_heads][1]) and empty the buffer.  Every request must hold the same
 *           number of full segments, else MKV_E_STATE.  Flushing fewer than segment_len tokens
 *           leaves a short last segment, after which nothing can be appended to the packed cache.
 *   count:  tokens currently buffered per unit (host value; no synchronisation).
 * A layer with an installed rotation (mkv_rotation_set) holds K R_k^T and V R_v^T, and so must its buffer: pass tokens
 * that are rotated the same way.  The buffer is attended with the folded query and its result goes through the output
 * fold like the packed part, so raw K / V in the buffer of a rotated layer give wrong results without any error.
 * mkv_cache_reset also empties the buffer.  The count lives in device memory and is updated on the stream, so a
 * captured CUDA graph of mkv_packed_attention stays valid across appends and flushes.
 */
MKV_API int mkv_update_append(mkv_cache* cache, int32_t layer, const void* k_new, const void* v_new,
                      int64_t stride_b, int64_t stride_h, int64_t stride_t, int32_t n_new,
                      void* stream);
MKV_API int mkv_update_flush(mkv_cache* cache, int32_t layer, const mkv_strategy* strat, void* stream);
MKV_API int mkv_update_count(const mkv_cache* cache, int32_t layer, int32_t* n_host);

/*
 * Per-head rotation fold.  The paper stores SVD-rotated K' = K R_k^T and V' = V R_v^T and
 * "merges the rotation into the single query vector" instead of rotating the matrices back.  The rotation itself is
 * the caller's (CPU-side management): compress K', V'; install the matrices with mkv_rotation_set; then
 *   rotate_query:  q_out = bf16(q R_k^T), q_out[i] = sum_j q[j] R_k[h][i][j], fp32, one FMA per j in ascending j
 *                  (q, q_out: bf16 [batch][n_q_heads][D], distinct buffers); feed q_out to mkv_select / mkv_packed_attention;
 *   rotate_output: out[j] = sum_i out[i] R_v[h][i][j] in place (float [batch][n_q_heads][D]), h = the head's KV head.
 * r_k, r_v: device, float [n_kv_heads][D][D] row-major, copied into the cache on `stream` (the first call of a cache
 * allocates: not capturable); both NULL removes the layer's rotation.  mkv_decode_host applies both folds on its own
 * when the layer has a rotation.  rotate_* on a layer without one is MKV_E_STATE.
 * Channel truncation is not built: a bitmap of 96 bits would break the 16-byte rows of the format.
 */
MKV_API int mkv_rotation_set(mkv_cache* cache, int32_t layer, const float* r_k, const float* r_v, void* stream);
MKV_API int mkv_rotate_query(const mkv_cache* cache, int32_t layer, const void* q, void* q_out, void* stream);
MKV_API int mkv_rotate_output(const mkv_cache* cache, int32_t layer, float* out, void* stream);

/*
 * One decode step of a layer on DEVICE buffers (steps 2 and 3 as one chain): [query fold] ->
 * block scores -> top-k -> PackedAttention -> [output fold], enqueued back to back on `stream` with programmatic
 * dependent launch, so each kernel's prologue overlaps its predecessor's tail and the chain captures into one CUDA
 * graph.  q: bf16 [batch][n_q_heads][D]; out: float [batch][n_q_heads][D]; lse_opt: float [batch][n_q_heads] or NULL.
 * sel_opt / sel_count_opt (both or neither): int32 [batch][n_kv_heads][k_max] / [batch][n_kv_heads] receive the
 * selection; with NULL the cache's own buffers are used and k_max is ignored.  A layer with an installed rotation
 * (mkv_rotation_set) gets both folds.  Results are those of mkv_select followed by mkv_packed_attention, bit for bit.
 */
MKV_API int mkv_decode_step(mkv_cache* cache, int32_t layer, const void* q, int32_t token_budget, int32_t reduce,
                    float softmax_scale, float* out, float* lse_opt, int32_t* sel_opt, int32_t* sel_count_opt,
                    int32_t k_max, void* stream);

/*
 * Steps 2+3 with HOST buffers (the end-to-end call): brings q_host (bf16 [batch][n_q_heads][D]) to the device, runs
 * mkv_decode_step, delivers out_host (float [batch][n_q_heads][D]).  Pinned (page-locked) buffers are read and written
 * by kernels of the chain itself (a 64-KB fetch kernel in front; the attention kernel stores straight into out_host, or
 * a store kernel behind the output fold), so the step never leaves the compute engine; pageable buffers, and pinned
 * ones that are not 16-byte aligned, fall back to cudaMemcpyAsync.  Everything is enqueued on `stream`; the caller synchronises the stream before reading out_host.  sel_host_opt [batch][n_kv_heads][token_budget/B + 1] and
 * sel_count_host_opt [batch][n_kv_heads] may be NULL.
 */
MKV_API int mkv_decode_host(mkv_cache* cache, int32_t layer, const void* q_host, int32_t token_budget,
                    int32_t reduce, float softmax_scale, float* out_host, int32_t* sel_host_opt,
                    int32_t* sel_count_host_opt, void* stream);

/*
 * Measurement aids (SURVEY 8(d) calibration rows).
 * gather: the PackedAttention kernel in the same launch configuration with all arithmetic removed — the K part and
 *         the V part of every selected token block are staged into shared memory exactly as mkv_packed_attention
 *         stages them (nothing is skipped), one word per lane is read back, nothing is written.  Its time is the
 *         ceiling the memory side sets for this access pattern.
 * stream: a plain streaming read of the first `bytes` bytes of the layer's packed arena (clamped to its size) in
 *         the same launch shape (one 512-thread CTA per SM, 16-byte loads): launch + pure-bandwidth floor.
 * walk:   the expansion of packed keys into tensor-core fragments alone: every warp of a one-CTA-
 *         per-SM grid copies the K parts of ONE group of the given selection (two consecutive selected token blocks)
 *         into shared memory once and runs the QK step on it `reps` times.  No staging, softmax, PV or output.  The
 *         difference of two calls with different `reps` is the time the shared-memory side needs per group: the
 *         floor of phase 1 of mkv_packed_attention and of the score kernel of mkv_select.  q: device bf16
 *         [batch][n_q_heads][128].
 * stats:  counters accumulated by mkv_packed_attention since the last reset: token blocks attended, token blocks
 *         whose V part was fetched (phase 2 skips a block whose probabilities are all < 2^-40 of the unit's
 *         largest), bytes of those V copies.  Synchronises.
 */
MKV_API int mkv_calibrate_gather(const mkv_cache* cache, int32_t layer, const int32_t* sel,
                         const int32_t* sel_count, int32_t k_max, void* stream);
MKV_API int mkv_calibrate_stream(const mkv_cache* cache, int32_t layer, uint64_t bytes, void* stream);
MKV_API int mkv_calibrate_walk(const mkv_cache* cache, int32_t layer, const void* q, const int32_t* sel,
                       const int32_t* sel_count, int32_t k_max, int32_t reps, void* stream);
MKV_API int mkv_attention_stats(const mkv_cache* cache, uint64_t* blocks_host, uint64_t* v_blocks_host,
                        uint64_t* v_bytes_host, int32_t reset);

/*
 * Step 2b alone, for callers that cannot allocate device memory (keep the best-scored token blocks
 * that fit the token budget).
 *
 * Who this is for.  Every other call works on an mkv_cache, and mkv_cache_create gets its arenas and scratch from
 * cudaMalloc.  That is not open to everyone: a decode loop inside a serving engine whose pool allocator took the whole
 * GPU at start-up (cudaMalloc finds no memory left, and where it succeeds it holds up every stream of the device while
 * it runs); a plug-in that is handed device pointers by its host program and owns no allocator; code that runs only
 * between the launches of somebody else's latency-critical step.  Such a caller brings block scores of its own (or the
 * ones mkv_select returned in scores_opt) and gets the selection without this library allocating or freeing anything:
 * no cudaMalloc, no cudaFree, no library routine that allocates, no mkv_cache.
 *
 * What it computes: exactly what mkv_select does after scoring.  Unit u has ceil(n_tokens[u] / token_block) blocks;
 * block i has score scores[u * score_stride + i] and token_block tokens (the last block of a unit may be shorter).
 * Blocks are taken by (score descending, index ascending) while they fit in token_budget tokens.
 *   scores:    device, float [n_units][score_stride], finite
 *   n_tokens:  device, int32 [n_units], 0 <= n_tokens[u] <= score_stride * token_block (NOT checked: a larger value
 *              reads past the unit's scores)
 *   sel:       device, int32 [n_units][k_max]: first-token index of every chosen block, ascending; unused tail = -1
 *   sel_count: device, int32 [n_units]
 *   k_max >= min(token_budget / token_block + 1, score_stride); token_block is 4, 8 or 16
 *   device:    ordinal of the GPU all four buffers live on; the call makes it the current device
 * The caller owns all four buffers; they are read / written on `stream` and the call returns without waiting.
 *
 * Scratch and its limit.  Units of more than 16384 blocks are selected in two stages (every 16384-block slice keeps
 * its token_budget / token_block + 1 best as candidates, then one pass picks among the candidates); the candidate
 * lists are the only scratch, and they live in an array compiled into the library: MKV_TOPK_STATIC_MAX_CANDIDATES
 * entries of 8 bytes = 4 MB, held by every GPU that loads libmkv until the process ends.  A call needs
 * n_units * ceil(score_stride / 16384) * min(token_budget / token_block + 1, 16384) entries; one that needs more is
 * refused with MKV_E_ARG and a message that names the three factors (nothing is enqueued) -- lower the budget or pass
 * the units in several calls.  Calls with score_stride <= 16384 use no scratch and have no such limit.
 *
 * The first call on a device looks up the array's device address (cudaGetSymbolAddress, which may also load the
 * library's device code on that GPU); make that first call before any stream capture begins.  All calls on a device
 * share the one array.  It needs no clearing -- every call overwrites all entries it later reads, so the previous
 * call's contents never matter -- but two calls that can run on the GPU at the same time (different streams without
 * an event between them, or two host threads) overwrite each other's candidates and return garbage: order them.
 */
#define MKV_TOPK_STATIC_MAX_CANDIDATES (1 << 19)
MKV_API int mkv_topk_static(int32_t device, const float* scores, const int32_t* n_tokens, int32_t n_units,
                    int32_t score_stride, int32_t token_block, int32_t token_budget, int32_t* sel,
                    int32_t* sel_count, int32_t k_max, void* stream);

/* Parity / dump: canonical blob of unit (layer, b, h) into host memory.  *need_host receives the
 * blob size; if cap < need nothing is copied and MKV_E_ARG is returned.  Synchronises. */
MKV_API int mkv_cache_export(const mkv_cache* cache, int32_t layer, int32_t b, int32_t h, void* buf_host,
                     uint64_t cap, uint64_t* need_host);

/* Bytes held for `layer`: token payloads, block-key payloads, tables in use.  Synchronises. */
MKV_API int mkv_cache_bytes(const mkv_cache* cache, int32_t layer, uint64_t* packed_host,
                    uint64_t* block_keys_host, uint64_t* tables_host);

/* Reads (and keeps) the sticky device flags; returns MKV_E_DEVICE if any is set.  Synchronises. */
MKV_API int mkv_cache_status(const mkv_cache* cache, uint32_t* flags_host);

/* Launch geometry of the last mkv_packed_attention / mkv_select call (for the bench's
 * gpu_launches count): number of kernels enqueued by that call. */
MKV_API int mkv_last_launch_count(const mkv_cache* cache, int32_t* select_kernels_host,
                          int32_t* attention_kernels_host, int32_t* compress_kernels_host);

MKV_API const char* mkv_last_error(void); /* thread-local, never NULL */
MKV_API int mkv_version(void);            /* ABI version, currently 2 (mkv_cache_desc gained token_block) */

#ifdef __cplusplus
}
#endif
#endif /* MKV_H */
