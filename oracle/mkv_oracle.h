/*
 * mkv_oracle.h — CPU oracle for the MosaicKV decode hot path (arxiv/paper_2607_00760).
 *
 * TEST INFRASTRUCTURE ONLY.  Plain, slow, obviously-correct C; fp64 arithmetic except
 * where a rounding to a storage type is part of the definition (block-key mean -> bf16,
 * element-group energy in fp32).  It shares NO code, header, table or helper with the
 * CUDA path under paper_2607_00760_b200/csrc/.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may load this library.
 *
 * Every function cites the PAPER.md passage it follows and the DESIGN.md reading
 * ("R#") it takes where the paper is silent.
 *
 * Pins: see tests/test_oracle_*.py (P1..P12 in DESIGN.md).  Unpinned: a worked numeric
 * example from the paper (the paper prints none; Figs. 5-6 were not extracted) —
 * "parity unpinned" for that item only.
 */
#ifndef MKV_ORACLE_H
#define MKV_ORACLE_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* Per-segment compression strategy record, 8 bytes (§4.3). */
typedef struct {
    uint8_t  r_k;    /* kept elements per K vector and per block key (multiple of g) */
    uint8_t  r_v;    /* kept elements per V vector */
    uint8_t  g;      /* element-group size 1/2/4 */
    uint8_t  B;      /* token-block size 4/8/16 */
    uint16_t n_tok;  /* tokens in this segment */
    uint16_t flags;  /* bit0: K dense (r_k == D), bit1: V dense (r_v == D) */
} orc_strat;

#define ORC_MAGIC 0x31564B4Du /* "MKV1" */
#define ORC_HEADER_BYTES 48

/* O1  top-r element(-group) selection, PAPER.md:180 / 196.  keep[D/g] <- 0/1 */
void orc_topr(const uint16_t* x, int D, int g, int r, uint8_t* keep);

/* O2  block key = mean of the block's uncompressed keys. out[D] bf16 */
void orc_block_key(const uint16_t* k, int nb, int D, uint16_t* out);

/* O3  relative squared Frobenius loss of one candidate, per segment.
 * k, v: [N][D] bf16 of ONE unit.  loss_k, loss_v: [S], S = ceil(N/L). */
int orc_segment_loss(const uint16_t* k, const uint16_t* v, int N, int D, int L,
                     int r_k, int r_v, int g, double* loss_k, double* loss_v);

/* O4a quantile rule (BASELINE config policy): the ceil(S*num/den) segments with the largest
 * importance I = (loss_k + loss_v)/2 (ties -> lower segment index) are kept dense. */
int orc_strategy_quantile(const double* loss_k, const double* loss_v, int S, int num, int den,
                          int D, int r_k, int r_v, int g, int B, uint8_t* strat4 /*[S][4]*/);

/* O4b threshold rule: first candidate (most -> least aggressive) with
 * I <= tau, else dense.  loss_*: [ncand][S]; cand4: [ncand][4] = r_k, r_v, g, B. */
int orc_strategy_threshold(const double* loss_k, const double* loss_v, int ncand, int S,
                           const uint8_t* cand4, double tau, int D, uint8_t* strat4);

/* O5  canonical export blob of one unit. */
uint64_t orc_blob_size(int N, int D, int L, const uint8_t* strat4 /*[S][4]*/);
int orc_compress_unit(const uint16_t* k, const uint16_t* v, int N, int D, int L,
                      const uint8_t* strat4, uint8_t* blob, uint64_t cap);
/* Unpack every vector of the blob back to dense bf16 with its 0/1 element mask.
 * k_out, v_out: [N][D]; bk_out: [nblk][D]; masks same shapes (uint8).  Any may be NULL. */
int orc_unpack_unit(const uint8_t* blob, uint16_t* k_out, uint8_t* k_mask, uint16_t* v_out,
                    uint8_t* v_mask, uint16_t* bk_out, uint8_t* bk_mask);
/* number of token blocks, and per block: first token + token count. Arrays may be NULL. */
int orc_blob_blocks(const uint8_t* blob, int32_t* first_tok, int32_t* n_tok);

/* O6  block scores on the packed block keys.
 * q: [G][D] bf16.  mode 0 = max over the group, 1 = sum.  s: [nblk] */
int orc_scores(const uint8_t* blob, const uint16_t* q, int G, int mode, double* s);

/* O7  top-k by token budget.  Returns count; sel ascending first-token. */
int orc_topk(const double* s, const int32_t* first_tok, const int32_t* n_tok, int nblk,
             int budget, int32_t* sel);

/* O8  attention over the selected packed tokens.
 * out: [G][D] double, lse: [G].  Empty selection -> out = 0, lse = -inf. */
int orc_attention(const uint8_t* blob, const uint16_t* q, int G, const int32_t* sel, int nsel,
                  double scale, double* out, double* lse);
/* same, but also returns the softmax weights p [G][ntok_selected] and the token ids. */
int orc_attention_weights(const uint8_t* blob, const uint16_t* q, int G, const int32_t* sel,
                          int nsel, double scale, double* out, double* lse, double* p,
                          int32_t* tok_ids, int cap_tok);
/* LSE merge of two partial results (the split-K combine rule, pinned by P10). */
void orc_merge(int G, int D, const double* o1, const double* lse1, const double* o2,
               const double* lse2, double* out, double* lse);

/* Batched drivers, OpenMP over independent units (used for timing and by tests). */
int orc_compress_units(const uint16_t* k, const uint16_t* v, int n_units, int N, int D, int L,
                       const uint8_t* strat4 /*[n_units][S][4]*/, uint8_t** blobs,
                       const uint64_t* caps);
int orc_decode_units(uint8_t* const* blobs, int n_units, const uint16_t* q /*[n_units][G][D]*/,
                     int G, int mode, int budget, double scale, int32_t* sel /*[n_units][k_max]*/,
                     int32_t* sel_count, int k_max, double* out /*[n_units][G][D]*/,
                     double* lse /*[n_units][G]*/);
int orc_attention_units(uint8_t* const* blobs, int n_units, const uint16_t* q, int G,
                        const int32_t* sel, const int32_t* sel_count, int k_max, double scale,
                        double* out, double* lse);
int orc_num_threads(void);

/* Rotation fold: q' = q R_k^T (fp32 FMA chain in ascending j, RNE to bf16) and
 * out = o' R_v (fp64).  R: [D][D] fp32 row-major. */
void orc_rotate_query(const uint16_t* q, int n, int D, const float* R, uint16_t* out);
void orc_rotate_output(double* o, int n, int D, const float* R);

#ifdef __cplusplus
}
#endif
#endif
