/*
 * mkv_oracle.c — CPU oracle for the MosaicKV decode hot path (arxiv/paper_2607_00760).
 *
 * TEST INFRASTRUCTURE ONLY — see mkv_oracle.h.  Nothing here is shared with, generated
 * for, or included by the CUDA path.  Written from PAPER.md; every function names the
 * passage it follows.  Deliberately unoptimised: sorts where a selection would do,
 * unpacks every vector to a dense double array before using it, one loop per formula.
 *
 * Build: gcc -O2 -std=c11 -ffp-contract=off -fopenmp -shared -fPIC (see oracle/build.py).
 * -ffp-contract=off matters: O1 (g>1) and O2 define fp32 results by IEEE add/mul/div in a
 * stated order, so no FMA contraction may be applied.
 */
#include "mkv_oracle.h"

#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* ---------------------------------------------------------------- bf16 <-> float */

static float bf16_to_f32(uint16_t h) {
    uint32_t u = (uint32_t)h << 16;
    float f;
    memcpy(&f, &u, 4);
    return f;
}
static double bf16_to_f64(uint16_t h) { return (double)bf16_to_f32(h); }

/* round-to-nearest-even fp32 -> bf16 (inputs are finite by contract) */
static uint16_t f32_to_bf16_rne(float f) {
    uint32_t u;
    memcpy(&u, &f, 4);
    uint32_t lsb = (u >> 16) & 1u;
    u += 0x7FFFu + lsb;
    return (uint16_t)(u >> 16);
}

/* ---------------------------------------------------------------- O1: top-r */

typedef struct {
    double key;
    int idx;
} rank_item;

/* order: key descending, ties -> lower index first (R1 / BASELINE north_star) */
static int rank_cmp(const void* a, const void* b) {
    const rank_item* x = (const rank_item*)a;
    const rank_item* y = (const rank_item*)b;
    if (x->key > y->key) return -1;
    if (x->key < y->key) return 1;
    return (x->idx > y->idx) - (x->idx < y->idx);
}

/*
 * PAPER.md:180 (§4.2 Stage-1): "For each KV vector, the top-r elements with the largest
 * absolute values are selected and all remaining elements are discarded."
 * PAPER.md:196 (§5.1): "selects groups of adjacent elements together ... one bit per
 * element group" (group size 1, 2 or 4).
 * Rank key (R4): g == 1 -> |x| compared exactly (15-bit magnitude of the bf16
 * pattern); g > 1 -> group energy sum_i x_i^2 evaluated in fp32, left to right.
 */
void orc_topr(const uint16_t* x, int D, int g, int r, uint8_t* keep) {
    int ng = D / g, nk = r / g;
    rank_item* it = (rank_item*)malloc(sizeof(rank_item) * (size_t)ng);
    for (int j = 0; j < ng; ++j) {
        it[j].idx = j;
        if (g == 1) {
            it[j].key = (double)(x[j] & 0x7FFFu);
        } else {
            float e = 0.0f;
            for (int i = 0; i < g; ++i) {
                float xi = bf16_to_f32(x[j * g + i]);
                float sq = xi * xi; /* exact in fp32 unless it over/underflows */
                e = e + sq;
            }
            it[j].key = (double)e;
        }
    }
    qsort(it, (size_t)ng, sizeof(rank_item), rank_cmp);
    for (int j = 0; j < ng; ++j) keep[j] = 0;
    for (int j = 0; j < nk && j < ng; ++j) keep[it[j].idx] = 1;
    free(it);
}

/* ---------------------------------------------------------------- O2: block key */

/*
 * "computes a per-block key vector as the mean of the key vectors within
 * each block"; the average is taken first, "then performs channel compression
 * on the K, V, and per-block key matrices" -> mean of the UNCOMPRESSED keys (R5).
 * Precision (R5): fp32 sum in ascending token order, IEEE fp32 division by nb, RNE to bf16.
 */
void orc_block_key(const uint16_t* k, int nb, int D, uint16_t* out) {
    for (int c = 0; c < D; ++c) {
        float s = 0.0f;
        for (int t = 0; t < nb; ++t) s = s + bf16_to_f32(k[(size_t)t * D + c]);
        float m = s / (float)nb;
        out[c] = f32_to_bf16_rne(m);
    }
}

/* ---------------------------------------------------------------- O3: loss */

/*
 * PAPER.md:238 (§5.5): "computes the compression loss for each token's KV vectors by
 * comparing the channel-compressed vectors with the original ones, and maintains an
 * accumulated total loss."  Reading R9: relative squared Frobenius error per segment,
 * L_X = sum_{t,c dropped} x^2 / sum_{t,c} x^2 (0 when the denominator is 0), fp64.
 */
int orc_segment_loss(const uint16_t* k, const uint16_t* v, int N, int D, int L, int r_k,
                     int r_v, int g, double* loss_k, double* loss_v) {
    if (D % g || r_k % g || r_v % g || r_k < g || r_v < g || r_k > D || r_v > D) return -1;
    int S = (N + L - 1) / L;
    uint8_t* keep = (uint8_t*)malloc((size_t)(D / g));
    for (int s = 0; s < S; ++s) {
        int t0 = s * L, t1 = (t0 + L < N) ? t0 + L : N;
        for (int which = 0; which < 2; ++which) {
            const uint16_t* x = which ? v : k;
            int r = which ? r_v : r_k;
            double dropped = 0.0, total = 0.0;
            for (int t = t0; t < t1; ++t) {
                const uint16_t* row = x + (size_t)t * D;
                orc_topr(row, D, g, r, keep);
                for (int c = 0; c < D; ++c) {
                    double xv = bf16_to_f64(row[c]);
                    total += xv * xv;
                    if (!keep[c / g]) dropped += xv * xv;
                }
            }
            double l = (total > 0.0) ? dropped / total : 0.0;
            if (which) loss_v[s] = l; else loss_k[s] = l;
        }
    }
    free(keep);
    return S;
}

/* ---------------------------------------------------------------- O4: strategy */

/*
 * BASELINE.json config policy ("0% on the top 10% of segments by importance") with
 * reading R10: importance I = (L_K + L_V)/2 at the aggressive candidate; the
 * ceil(S*num/den) segments of the unit with the largest I (ties -> lower index) stay
 * dense, the others take the candidate.
 */
int orc_strategy_quantile(const double* loss_k, const double* loss_v, int S, int num, int den,
                          int D, int r_k, int r_v, int g, int B, uint8_t* strat4) {
    if (den <= 0 || num < 0) return -1;
    int n_dense = (int)(((long long)S * num + den - 1) / den);
    if (n_dense > S) n_dense = S;
    rank_item* it = (rank_item*)malloc(sizeof(rank_item) * (size_t)S);
    for (int s = 0; s < S; ++s) {
        it[s].idx = s;
        it[s].key = 0.5 * (loss_k[s] + loss_v[s]);
    }
    qsort(it, (size_t)S, sizeof(rank_item), rank_cmp);
    for (int s = 0; s < S; ++s) {
        strat4[4 * s + 0] = (uint8_t)r_k;
        strat4[4 * s + 1] = (uint8_t)r_v;
        strat4[4 * s + 2] = (uint8_t)g;
        strat4[4 * s + 3] = (uint8_t)B;
    }
    for (int j = 0; j < n_dense; ++j) {
        int s = it[j].idx;
        strat4[4 * s + 0] = (uint8_t)D;
        strat4[4 * s + 1] = (uint8_t)D;
    }
    free(it);
    return n_dense;
}

/*
 * "evaluates the compression loss for each candidate compression rate ...
 * and element group size ... The highest compression rate and largest group size whose
 * loss remains below a threshold are selected."  Candidates arrive ordered most -> least
 * aggressive; the first with I <= tau wins; none -> dense (g = 1, B of the last candidate).
 */
int orc_strategy_threshold(const double* loss_k, const double* loss_v, int ncand, int S,
                           const uint8_t* cand4, double tau, int D, uint8_t* strat4) {
    if (ncand <= 0) return -1;
    for (int s = 0; s < S; ++s) {
        int chosen = -1;
        for (int c = 0; c < ncand; ++c) {
            double I = 0.5 * (loss_k[(size_t)c * S + s] + loss_v[(size_t)c * S + s]);
            if (I <= tau) { chosen = c; break; }
        }
        if (chosen >= 0) {
            memcpy(strat4 + 4 * s, cand4 + 4 * chosen, 4);
        } else {
            strat4[4 * s + 0] = (uint8_t)D;
            strat4[4 * s + 1] = (uint8_t)D;
            strat4[4 * s + 2] = 1;
            strat4[4 * s + 3] = cand4[4 * (ncand - 1) + 3];
        }
    }
    return 0;
}

/* ---------------------------------------------------------------- O5: packed format */

/*
 * PAPER.md:194 (§5.1): "packs all retained elements contiguously for each sparse vector
 * and employs a D-bit position bitmap, where each bit indicates whether the corresponding
 * element is retained"; one bit per element group.
 * Canonical layout (bit/value order = reading R16):
 *   packed vector  = [bitmap: ceil(D/g/8) bytes, bit j = byte j>>3, bit j&7 (LSB first)]
 *                    [kept elements, bf16, ascending channel order]; bitmap omitted if r==D
 *   token block    = [K bitmaps nb][K values nb][V bitmaps nb][V values nb], pad to 16 B
 *   segment        = its token blocks in order
 *   segment's block keys = [bitmaps nblk][values nblk], pad to 16 B   (separate arena)
 *   blob           = header(48) strat[S] tok_off[S] bk_off[S] pad16 | token arena | bk arena
 */
static int bm_bytes(int D, int g, int r) { return (r == D) ? 0 : (D / g + 7) / 8; }
static uint64_t pad16(uint64_t x) { return (x + 15u) & ~(uint64_t)15u; }

static uint64_t tokblock_bytes(int D, int r_k, int r_v, int g, int nb) {
    uint64_t b = (uint64_t)nb * (uint64_t)(bm_bytes(D, g, r_k) + 2 * r_k) +
                 (uint64_t)nb * (uint64_t)(bm_bytes(D, g, r_v) + 2 * r_v);
    return pad16(b);
}
static uint64_t seg_tok_bytes(int D, int r_k, int r_v, int g, int B, int n_tok) {
    uint64_t tot = 0;
    for (int t = 0; t < n_tok; t += B) {
        int nb = (n_tok - t < B) ? n_tok - t : B;
        tot += tokblock_bytes(D, r_k, r_v, g, nb);
    }
    return tot;
}
static uint64_t seg_bk_bytes(int D, int r_k, int g, int B, int n_tok) {
    int nblk = (n_tok + B - 1) / B;
    return pad16((uint64_t)nblk * (uint64_t)(bm_bytes(D, g, r_k) + 2 * r_k));
}
static uint64_t tables_bytes(int S) {
    return pad16((uint64_t)ORC_HEADER_BYTES + (uint64_t)S * 16u);
}

static int strat_ok(int D, int r_k, int r_v, int g, int B) {
    if (!(g == 1 || g == 2 || g == 4)) return 0;
    if (B < 1 || B > 64) return 0;
    if (D % g || r_k % g || r_v % g) return 0;
    if (r_k < g || r_v < g || r_k > D || r_v > D) return 0;
    return 1;
}

uint64_t orc_blob_size(int N, int D, int L, const uint8_t* strat4) {
    int S = (N + L - 1) / L;
    uint64_t tok = 0, bk = 0;
    for (int s = 0; s < S; ++s) {
        int r_k = strat4[4 * s], r_v = strat4[4 * s + 1], g = strat4[4 * s + 2], B = strat4[4 * s + 3];
        if (!strat_ok(D, r_k, r_v, g, B)) return 0;
        int n_tok = (s * L + L <= N) ? L : N - s * L;
        tok += seg_tok_bytes(D, r_k, r_v, g, B, n_tok);
        bk += seg_bk_bytes(D, r_k, g, B, n_tok);
    }
    return tables_bytes(S) + tok + bk;
}

/* write one packed vector: bitmap at bm (unless dense), values at val */
static void pack_vec(const uint16_t* x, int D, int g, int r, uint8_t* bm, uint8_t* val) {
    if (r == D) {
        memcpy(val, x, (size_t)D * 2);
        return;
    }
    uint8_t* keep = (uint8_t*)malloc((size_t)(D / g));
    orc_topr(x, D, g, r, keep);
    int nbm = bm_bytes(D, g, r);
    memset(bm, 0, (size_t)nbm);
    int n = 0;
    for (int j = 0; j < D / g; ++j) {
        if (!keep[j]) continue;
        bm[j >> 3] |= (uint8_t)(1u << (j & 7));
        for (int i = 0; i < g; ++i) {
            uint16_t e = x[j * g + i];
            memcpy(val + 2 * n, &e, 2);
            ++n;
        }
    }
    free(keep);
}

/* inverse of pack_vec: dense bf16 (zeros where dropped) and per-element 0/1 mask */
static void unpack_vec(const uint8_t* bm, const uint8_t* val, int D, int g, int r, uint16_t* x,
                       uint8_t* mask) {
    int n = 0;
    for (int c = 0; c < D; ++c) {
        int kept = 1;
        if (r != D) {
            int j = c / g;
            kept = (bm[j >> 3] >> (j & 7)) & 1;
        }
        uint16_t e = 0;
        if (kept) {
            memcpy(&e, val + 2 * n, 2);
            ++n;
        }
        if (x) x[c] = e;
        if (mask) mask[c] = (uint8_t)kept;
    }
}

static void put_u32(uint8_t* p, uint32_t v) { memcpy(p, &v, 4); }
static void put_u64(uint8_t* p, uint64_t v) { memcpy(p, &v, 8); }
static uint32_t get_u32(const uint8_t* p) { uint32_t v; memcpy(&v, p, 4); return v; }
static uint64_t get_u64(const uint8_t* p) { uint64_t v; memcpy(&v, p, 8); return v; }

/*
 * PAPER.md:200 (§5.2 Compressed KV Encoding): "all tokens are divided into multiple token
 * blocks ... A per-block key is computed as the average of the key vectors within each
 * block. MosaicKV then performs channel compression on the K, V, and per-block key
 * matrices, and stores the results in the packed KV format".  Rotation = identity (R18).
 */
int orc_compress_unit(const uint16_t* k, const uint16_t* v, int N, int D, int L,
                      const uint8_t* strat4, uint8_t* blob, uint64_t cap) {
    uint64_t need = orc_blob_size(N, D, L, strat4);
    if (need == 0 || need > cap) return -1;
    int S = (N + L - 1) / L;
    memset(blob, 0, (size_t)need);
    uint8_t* p_strat = blob + ORC_HEADER_BYTES;
    uint8_t* p_tokoff = p_strat + (size_t)S * 8;
    uint8_t* p_bkoff = p_tokoff + (size_t)S * 4;
    uint8_t* tok_arena = blob + tables_bytes(S);
    uint64_t tok_pos = 0, bk_pos = 0, tok_total = 0;
    for (int s = 0; s < S; ++s) {
        int n_tok = (s * L + L <= N) ? L : N - s * L;
        tok_total += seg_tok_bytes(D, strat4[4 * s], strat4[4 * s + 1], strat4[4 * s + 2],
                                   strat4[4 * s + 3], n_tok);
    }
    uint8_t* bk_arena = tok_arena + tok_total;
    uint16_t* bkey = (uint16_t*)malloc((size_t)D * 2);
    for (int s = 0; s < S; ++s) {
        int r_k = strat4[4 * s], r_v = strat4[4 * s + 1], g = strat4[4 * s + 2], B = strat4[4 * s + 3];
        int t0 = s * L;
        int n_tok = (t0 + L <= N) ? L : N - t0;
        orc_strat rec;
        rec.r_k = (uint8_t)r_k; rec.r_v = (uint8_t)r_v; rec.g = (uint8_t)g; rec.B = (uint8_t)B;
        rec.n_tok = (uint16_t)n_tok;
        rec.flags = (uint16_t)((r_k == D ? 1 : 0) | (r_v == D ? 2 : 0));
        memcpy(p_strat + (size_t)s * 8, &rec, 8);
        put_u32(p_tokoff + (size_t)s * 4, (uint32_t)(tok_pos / 16));
        put_u32(p_bkoff + (size_t)s * 4, (uint32_t)(bk_pos / 16));

        int nblk = (n_tok + B - 1) / B;
        int bmk = bm_bytes(D, g, r_k), bmv = bm_bytes(D, g, r_v);
        uint8_t* bk_bm = bk_arena + bk_pos;
        uint8_t* bk_val = bk_bm + (size_t)nblk * bmk;
        for (int b = 0; b < nblk; ++b) {
            int bt0 = t0 + b * B;
            int nb = (n_tok - b * B < B) ? n_tok - b * B : B;
            uint8_t* base = tok_arena + tok_pos;
            uint8_t* k_bm = base;
            uint8_t* k_val = k_bm + (size_t)nb * bmk;
            uint8_t* v_bm = k_val + (size_t)nb * r_k * 2;
            uint8_t* v_val = v_bm + (size_t)nb * bmv;
            for (int t = 0; t < nb; ++t) {
                pack_vec(k + (size_t)(bt0 + t) * D, D, g, r_k, k_bm + (size_t)t * bmk,
                         k_val + (size_t)t * r_k * 2);
                pack_vec(v + (size_t)(bt0 + t) * D, D, g, r_v, v_bm + (size_t)t * bmv,
                         v_val + (size_t)t * r_v * 2);
            }
            tok_pos += tokblock_bytes(D, r_k, r_v, g, nb);
            /* block key: mean of the uncompressed keys, then the same top-r_k (R6, R7) */
            orc_block_key(k + (size_t)bt0 * D, nb, D, bkey);
            pack_vec(bkey, D, g, r_k, bk_bm + (size_t)b * bmk, bk_val + (size_t)b * r_k * 2);
        }
        bk_pos += seg_bk_bytes(D, r_k, g, B, n_tok);
    }
    free(bkey);
    put_u32(blob + 0, ORC_MAGIC);
    put_u32(blob + 4, (uint32_t)D);
    put_u32(blob + 8, (uint32_t)N);
    put_u32(blob + 12, (uint32_t)L);
    put_u32(blob + 16, (uint32_t)S);
    put_u32(blob + 20, 0);
    put_u64(blob + 24, tok_pos);
    put_u64(blob + 32, bk_pos);
    put_u64(blob + 40, 0);
    return 0;
}

/* blob accessors */
typedef struct {
    int D, N, L, S;
    const uint8_t *strat, *tokoff, *bkoff, *tok, *bk;
} blob_view;

static int view_blob(const uint8_t* blob, blob_view* bv) {
    if (get_u32(blob) != ORC_MAGIC) return -1;
    bv->D = (int)get_u32(blob + 4);
    bv->N = (int)get_u32(blob + 8);
    bv->L = (int)get_u32(blob + 12);
    bv->S = (int)get_u32(blob + 16);
    bv->strat = blob + ORC_HEADER_BYTES;
    bv->tokoff = bv->strat + (size_t)bv->S * 8;
    bv->bkoff = bv->tokoff + (size_t)bv->S * 4;
    bv->tok = blob + tables_bytes(bv->S);
    bv->bk = bv->tok + get_u64(blob + 24);
    return 0;
}
static orc_strat seg_strat(const blob_view* bv, int s) {
    orc_strat r;
    memcpy(&r, bv->strat + (size_t)s * 8, 8);
    return r;
}

int orc_blob_blocks(const uint8_t* blob, int32_t* first_tok, int32_t* n_tok) {
    blob_view bv;
    if (view_blob(blob, &bv)) return -1;
    int n = 0;
    for (int s = 0; s < bv.S; ++s) {
        orc_strat st = seg_strat(&bv, s);
        for (int t = 0; t < st.n_tok; t += st.B) {
            if (first_tok) first_tok[n] = s * bv.L + t;
            if (n_tok) n_tok[n] = (st.n_tok - t < st.B) ? st.n_tok - t : st.B;
            ++n;
        }
    }
    return n;
}

int orc_unpack_unit(const uint8_t* blob, uint16_t* k_out, uint8_t* k_mask, uint16_t* v_out,
                    uint8_t* v_mask, uint16_t* bk_out, uint8_t* bk_mask) {
    blob_view bv;
    if (view_blob(blob, &bv)) return -1;
    int D = bv.D, blk_index = 0;
    for (int s = 0; s < bv.S; ++s) {
        orc_strat st = seg_strat(&bv, s);
        int g = st.g, B = st.B, r_k = st.r_k, r_v = st.r_v;
        int bmk = bm_bytes(D, g, r_k), bmv = bm_bytes(D, g, r_v);
        const uint8_t* seg = bv.tok + (uint64_t)get_u32(bv.tokoff + (size_t)s * 4) * 16;
        const uint8_t* bks = bv.bk + (uint64_t)get_u32(bv.bkoff + (size_t)s * 4) * 16;
        int nblk = (st.n_tok + B - 1) / B;
        uint64_t pos = 0;
        for (int b = 0; b < nblk; ++b) {
            int nb = (st.n_tok - b * B < B) ? st.n_tok - b * B : B;
            const uint8_t* k_bm = seg + pos;
            const uint8_t* k_val = k_bm + (size_t)nb * bmk;
            const uint8_t* v_bm = k_val + (size_t)nb * r_k * 2;
            const uint8_t* v_val = v_bm + (size_t)nb * bmv;
            for (int t = 0; t < nb; ++t) {
                size_t tok = (size_t)s * bv.L + (size_t)b * B + t;
                unpack_vec(k_bm + (size_t)t * bmk, k_val + (size_t)t * r_k * 2, D, g, r_k,
                           k_out ? k_out + tok * D : NULL, k_mask ? k_mask + tok * D : NULL);
                unpack_vec(v_bm + (size_t)t * bmv, v_val + (size_t)t * r_v * 2, D, g, r_v,
                           v_out ? v_out + tok * D : NULL, v_mask ? v_mask + tok * D : NULL);
            }
            pos += tokblock_bytes(D, r_k, r_v, g, nb);
            unpack_vec(bks + (size_t)b * bmk, bks + (size_t)nblk * bmk + (size_t)b * r_k * 2, D, g,
                       r_k, bk_out ? bk_out + (size_t)blk_index * D : NULL,
                       bk_mask ? bk_mask + (size_t)blk_index * D : NULL);
            ++blk_index;
        }
    }
    return blk_index;
}

/* ---------------------------------------------------------------- O6: scores */

/*
 * "an attention score is computed for each block via the dot product between
 * the current query vector and the per-block key"; the packed vector product
 * multiplies only at the set bits of the position bitmap.  GQA reading R11: one score per KV
 * head, max (mode 0) or sum (mode 1) over the G query heads of the group.  No 1/sqrt(D).
 */
int orc_scores(const uint8_t* blob, const uint16_t* q, int G, int mode, double* s) {
    blob_view bv;
    if (view_blob(blob, &bv)) return -1;
    int D = bv.D;
    int nblk = orc_blob_blocks(blob, NULL, NULL);
    uint16_t* bk = (uint16_t*)malloc((size_t)nblk * D * 2);
    uint8_t* bm = (uint8_t*)malloc((size_t)nblk * D);
    orc_unpack_unit(blob, NULL, NULL, NULL, NULL, bk, bm);
    for (int b = 0; b < nblk; ++b) {
        double best = 0.0;
        for (int h = 0; h < G; ++h) {
            double d = 0.0;
            for (int c = 0; c < D; ++c)
                if (bm[(size_t)b * D + c])
                    d += bf16_to_f64(q[(size_t)h * D + c]) * bf16_to_f64(bk[(size_t)b * D + c]);
            if (mode == 1) best = (h == 0) ? d : best + d;
            else best = (h == 0 || d > best) ? d : best;
        }
        s[b] = best;
    }
    free(bk);
    free(bm);
    return nblk;
}

/* ---------------------------------------------------------------- O7: top-k */

/*
 * "the top-k blocks with the highest scores are selected".
 * Reading R8: global per unit, by token budget.  Sort by (score descending, index
 * ascending); walk the list adding blocks while tokens_so_far + n_tok(b) <= budget; stop at
 * the first block that does not fit.  Output ascending first-token indices.
 */
int orc_topk(const double* s, const int32_t* first_tok, const int32_t* n_tok, int nblk,
             int budget, int32_t* sel) {
    rank_item* it = (rank_item*)malloc(sizeof(rank_item) * (size_t)(nblk > 0 ? nblk : 1));
    for (int b = 0; b < nblk; ++b) {
        it[b].idx = b;
        it[b].key = s[b] + 0.0; /* -0.0 ranks equal to +0.0 under the comparison anyway */
    }
    qsort(it, (size_t)nblk, sizeof(rank_item), rank_cmp);
    uint8_t* chosen = (uint8_t*)calloc((size_t)(nblk > 0 ? nblk : 1), 1);
    long long used = 0;
    for (int j = 0; j < nblk; ++j) {
        int b = it[j].idx;
        if (used + n_tok[b] > budget) break;
        used += n_tok[b];
        chosen[b] = 1;
    }
    int n = 0;
    for (int b = 0; b < nblk; ++b)
        if (chosen[b]) sel[n++] = first_tok[b];
    free(chosen);
    free(it);
    return n;
}

/* ---------------------------------------------------------------- O8: attention */

/*
 * attention over the selected blocks only, the standard dot product
 * replaced by the packed vector product.  For query head h over selected tokens T:
 *   z_t = scale * sum_{c kept in K_t} q_c K_{t,c};  p = softmax(z);  o_c = sum_{t: c kept in
 *   V_t} p_t V_{t,c};  lse = max + log(sum exp(z - max)).  fp64, no intermediate rounding.
 */
int orc_attention_weights(const uint8_t* blob, const uint16_t* q, int G, const int32_t* sel,
                          int nsel, double scale, double* out, double* lse, double* p_out,
                          int32_t* tok_ids, int cap_tok) {
    blob_view bv;
    if (view_blob(blob, &bv)) return -1;
    int D = bv.D, N = bv.N;
    /* gather the token ids of the selected blocks */
    int ntok = 0;
    for (int i = 0; i < nsel; ++i) {
        int t0 = sel[i];
        if (t0 < 0 || t0 >= N) return -2;
        orc_strat st = seg_strat(&bv, t0 / bv.L);
        int in_seg = t0 % bv.L;
        if (in_seg % st.B) return -3;
        ntok += (st.n_tok - in_seg < st.B) ? st.n_tok - in_seg : st.B;
    }
    int32_t* toks = (int32_t*)malloc(sizeof(int32_t) * (size_t)(ntok > 0 ? ntok : 1));
    ntok = 0;
    for (int i = 0; i < nsel; ++i) {
        int t0 = sel[i];
        orc_strat st = seg_strat(&bv, t0 / bv.L);
        int in_seg = t0 % bv.L;
        int nb = (st.n_tok - in_seg < st.B) ? st.n_tok - in_seg : st.B;
        for (int t = 0; t < nb; ++t) toks[ntok++] = t0 + t;
    }
    if (tok_ids) {
        if (ntok > cap_tok) { free(toks); return -4; }
        memcpy(tok_ids, toks, sizeof(int32_t) * (size_t)ntok);
    }
    /* unpack everything (slow, plain) */
    uint16_t* kd = (uint16_t*)malloc((size_t)N * D * 2);
    uint16_t* vd = (uint16_t*)malloc((size_t)N * D * 2);
    uint8_t* km = (uint8_t*)malloc((size_t)N * D);
    uint8_t* vm = (uint8_t*)malloc((size_t)N * D);
    orc_unpack_unit(blob, kd, km, vd, vm, NULL, NULL);
    double* z = (double*)malloc(sizeof(double) * (size_t)(ntok > 0 ? ntok : 1));
    for (int h = 0; h < G; ++h) {
        for (int c = 0; c < D; ++c) out[(size_t)h * D + c] = 0.0;
        if (ntok == 0) {
            lse[h] = -INFINITY;
            continue;
        }
        double m = -INFINITY;
        for (int i = 0; i < ntok; ++i) {
            size_t t = (size_t)toks[i];
            double d = 0.0;
            for (int c = 0; c < D; ++c)
                if (km[t * D + c]) d += bf16_to_f64(q[(size_t)h * D + c]) * bf16_to_f64(kd[t * D + c]);
            z[i] = scale * d;
            if (z[i] > m) m = z[i];
        }
        double sum = 0.0;
        for (int i = 0; i < ntok; ++i) sum += exp(z[i] - m);
        for (int i = 0; i < ntok; ++i) {
            size_t t = (size_t)toks[i];
            double p = exp(z[i] - m) / sum;
            if (p_out) p_out[(size_t)h * ntok + i] = p;
            for (int c = 0; c < D; ++c)
                if (vm[t * D + c]) out[(size_t)h * D + c] += p * bf16_to_f64(vd[t * D + c]);
        }
        lse[h] = m + log(sum);
    }
    free(z); free(kd); free(vd); free(km); free(vm); free(toks);
    return ntok;
}

int orc_attention(const uint8_t* blob, const uint16_t* q, int G, const int32_t* sel, int nsel,
                  double scale, double* out, double* lse) {
    return orc_attention_weights(blob, q, G, sel, nsel, scale, out, lse, NULL, NULL, 0);
}

/*
 * Split-K merge (not in the paper; DESIGN.md step 3d): two partial softmax results over
 * disjoint token sets combine as  lse = log(e^lse1 + e^lse2),  o = w1 o1 + w2 o2 with
 * w_i = e^(lse_i - lse).  Pinned by P10 (merge of halves == single pass).
 */
void orc_merge(int G, int D, const double* o1, const double* lse1, const double* o2,
               const double* lse2, double* out, double* lse) {
    for (int h = 0; h < G; ++h) {
        double a = lse1[h], b = lse2[h];
        double m = (a > b) ? a : b;
        if (m == -INFINITY) {
            lse[h] = -INFINITY;
            for (int c = 0; c < D; ++c) out[(size_t)h * D + c] = 0.0;
            continue;
        }
        double l = m + log(exp(a - m) + exp(b - m));
        double w1 = exp(a - l), w2 = exp(b - l);
        lse[h] = l;
        for (int c = 0; c < D; ++c)
            out[(size_t)h * D + c] = w1 * o1[(size_t)h * D + c] + w2 * o2[(size_t)h * D + c];
    }
}

/* ---------------------------------------------------------------- batched drivers */

int orc_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

int orc_compress_units(const uint16_t* k, const uint16_t* v, int n_units, int N, int D, int L,
                       const uint8_t* strat4, uint8_t** blobs, const uint64_t* caps) {
    int S = (N + L - 1) / L, err = 0;
#pragma omp parallel for schedule(dynamic, 1)
    for (int u = 0; u < n_units; ++u) {
        int rc = orc_compress_unit(k + (size_t)u * N * D, v + (size_t)u * N * D, N, D, L,
                                   strat4 + (size_t)u * S * 4, blobs[u], caps[u]);
        if (rc) {
#pragma omp atomic write
            err = rc;
        }
    }
    return err;
}

/* one decode step of the layer for every unit: O6 -> O7 -> O8 */
int orc_decode_units(uint8_t* const* blobs, int n_units, const uint16_t* q, int G, int mode,
                     int budget, double scale, int32_t* sel, int32_t* sel_count, int k_max,
                     double* out, double* lse) {
    int err = 0;
#pragma omp parallel for schedule(dynamic, 1)
    for (int u = 0; u < n_units; ++u) {
        blob_view bv;
        if (view_blob(blobs[u], &bv)) {
#pragma omp atomic write
            err = -1;
            continue;
        }
        int nblk = orc_blob_blocks(blobs[u], NULL, NULL);
        int32_t* ft = (int32_t*)malloc(sizeof(int32_t) * (size_t)(nblk + 1));
        int32_t* nt = (int32_t*)malloc(sizeof(int32_t) * (size_t)(nblk + 1));
        double* s = (double*)malloc(sizeof(double) * (size_t)(nblk + 1));
        int32_t* tmp = (int32_t*)malloc(sizeof(int32_t) * (size_t)(nblk + 1));
        orc_blob_blocks(blobs[u], ft, nt);
        const uint16_t* qu = q + (size_t)u * G * bv.D;
        orc_scores(blobs[u], qu, G, mode, s);
        int n = orc_topk(s, ft, nt, nblk, budget, tmp);
        if (n > k_max) {
#pragma omp atomic write
            err = -5;
            n = k_max;
        }
        memcpy(sel + (size_t)u * k_max, tmp, sizeof(int32_t) * (size_t)n);
        sel_count[u] = n;
        orc_attention(blobs[u], qu, G, tmp, n, scale, out + (size_t)u * G * bv.D,
                      lse + (size_t)u * G);
        free(ft); free(nt); free(s); free(tmp);
    }
    return err;
}

/* attention only (O8) for every unit with a given selection, OpenMP over units */
int orc_attention_units(uint8_t* const* blobs, int n_units, const uint16_t* q, int G,
                        const int32_t* sel, const int32_t* sel_count, int k_max, double scale,
                        double* out, double* lse) {
    int err = 0;
#pragma omp parallel for schedule(dynamic, 1)
    for (int u = 0; u < n_units; ++u) {
        blob_view bv;
        if (view_blob(blobs[u], &bv)) {
#pragma omp atomic write
            err = -1;
            continue;
        }
        int rc = orc_attention(blobs[u], q + (size_t)u * G * bv.D, G, sel + (size_t)u * k_max,
                               sel_count[u], scale, out + (size_t)u * G * bv.D, lse + (size_t)u * G);
        if (rc < 0) {
#pragma omp atomic write
            err = rc;
        }
    }
    return err;
}

/* ---------------------------------------------------------------- rotation fold */

/*
 * PAPER.md:114 (§2.3): "Given a matrix K, SVD decomposes it as K = K' R ... applies the rotations (K R_k^T and
 * V R_v^T)"; PAPER.md:218-220 (§5.3): "Instead of rotating the large matrix, MosaicKV merges the rotation into the
 * single query vector and uses the rotated query to compute the attention scores.  This approach is mathematically
 * equivalent".  With K' = K R_k^T stored, q K^T = (q R_k^T) K'^T, so the folded query is q' = q R_k^T:
 *   q'[i] = sum_j q[j] * R_k[i][j].
 * Reading (R18): q' is an INPUT of the bf16 kernels, so its rounding is part of the definition: the sum is
 * accumulated in fp32 with one fused multiply-add per j in ascending j, then rounded to bf16 (RNE).
 * q: [n][D] bf16, R: [D][D] fp32 row-major, out: [n][D] bf16.
 */
void orc_rotate_query(const uint16_t* q, int n, int D, const float* R, uint16_t* out) {
    for (int v = 0; v < n; ++v)
        for (int i = 0; i < D; ++i) {
            float acc = 0.0f;
            for (int j = 0; j < D; ++j) acc = fmaf(bf16_to_f32(q[(size_t)v * D + j]), R[(size_t)i * D + j], acc);
            out[(size_t)v * D + i] = f32_to_bf16_rne(acc);
        }
}

/*
 * The attention output of the rotated cache lives in the rotated space of V' = V R_v^T: O = P V = (P V') R_v, so
 *   out[j] = sum_i o'[i] * R_v[i][j]          (fp64).
 * o: [n][D] double (in place allowed: a temporary row is used), R: [D][D] fp32 row-major.
 */
void orc_rotate_output(double* o, int n, int D, const float* R) {
    double* tmp = (double*)malloc(sizeof(double) * (size_t)D);
    for (int v = 0; v < n; ++v) {
        for (int j = 0; j < D; ++j) {
            double acc = 0.0;
            for (int i = 0; i < D; ++i) acc += o[(size_t)v * D + i] * (double)R[(size_t)i * D + j];
            tmp[j] = acc;
        }
        for (int j = 0; j < D; ++j) o[(size_t)v * D + j] = tmp[j];
    }
    free(tmp);
}
