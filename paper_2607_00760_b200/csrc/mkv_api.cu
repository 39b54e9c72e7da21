// mkv_api.cu — the C ABI of libmkv (include/mkv.h): cache lifetime, host-side argument checks,
// export of the canonical blob, and dispatch to the kernels.  No CPU fallback exists: every
// step of the path runs in the CUDA kernels of this library.
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <new>
#include <algorithm>
#include <vector>

#include "mkv_internal.cuh"

using namespace mkv;

namespace {

thread_local char g_err[512] = "";

int fail(int code, const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
    return code;
}

#define MKV_CUDA(expr)                                                                          \
    do {                                                                                        \
        cudaError_t e_ = (expr);                                                                \
        if (e_ != cudaSuccess)                                                                  \
            return fail(e_ == cudaErrorMemoryAllocation ? MKV_E_NOMEM : MKV_E_CUDA, "%s: %s", #expr, \
                        cudaGetErrorString(e_));                                                \
    } while (0)

uint64_t align_up(uint64_t x, uint64_t a) { return (x + a - 1) / a * a; }

}  // namespace

int mkv::set_error(int code, const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
    return code;
}

struct mkv_cache {
    mkv_cache_desc desc{};
    CacheGeom geom{};
    int sm_count = 0;
    // device
    uint8_t* arena = nullptr;
    uint64_t slice_bytes = 0;
    StratRec* strat = nullptr;
    uint32_t* tok_off = nullptr;
    uint32_t* bk_off = nullptr;
    int32_t* unit_nseg = nullptr;
    int32_t* unit_ntok = nullptr;
    unsigned long long* counters = nullptr;  // [n_layers][4]: bump, used_tok, used_bk, pad
    uint32_t* dev_flags = nullptr;
    unsigned long long* call_base = nullptr;  // [n_units]
    float* scores = nullptr;                  // [n_units][score_stride]
    uint32_t* cand_key = nullptr;             // [n_units][slices * kTopkSlice]  top-k candidates of long units
    int32_t* cand_idx = nullptr;
    uint16_t* upd_k = nullptr;                // KV update buffer, raw bf16 [n_layers][n_units][L][D]
    uint16_t* upd_v = nullptr;
    int32_t* upd_cnt = nullptr;               // [n_layers] tokens buffered per unit (read by the attention kernel)
    std::vector<int32_t> upd_n;               // host mirror (every unit of a layer holds the same number)
    AttnScratch attn{};
    int attn_cluster[2] = {0, 0};             // cluster size of the attention / gather-only kernel for this cache (0 = not chosen yet)
    PlanRec* plan = nullptr;                  // [n_layers][n_units][sel_cap]: what top-k tells attention about each selected block
    uint32_t generation = 1;                  // bumped by mkv_cache_reset: invalidates every plan record
    unsigned long long* sink = nullptr;
    float* rot_k = nullptr;                   // [n_layers][n_kv_heads][D][D] rotation matrices (allocated by the first mkv_rotation_set)
    float* rot_v = nullptr;
    std::vector<uint8_t> rot_set;             // per layer: a rotation is installed
    uint16_t* q_rot = nullptr;                // [batch][n_q_heads][D] folded query of mkv_decode_host
    uint16_t* q_dev = nullptr;
    uint4* masks = nullptr;                   // [n_units][max_tokens][2]: top-r masks found by mkv_segment_loss (compress.cu)
    int32_t* sel_dev = nullptr;
    int32_t* selcnt_dev = nullptr;
    float* out_dev = nullptr;
    int sel_cap = 0;
    // host mirrors of the append state, [n_layers][batch]
    std::vector<int32_t> host_nseg, host_ntok;
    int last_select = 0, last_attn = 0, last_compress = 0;

    AttnScratch attn_scratch(int layer) const {
        AttnScratch a = attn;
        a.plan = plan + (size_t)layer * geom.n_units * sel_cap * geom.ppb;
        a.plan_stride = sel_cap * geom.ppb;
        a.plan_tag = plan_tag(generation, layer);
        return a;
    }
    LayerView view(int layer) const {
        LayerView v;
        const size_t tu = (size_t)layer * geom.n_units;
        v.slice = arena + (size_t)layer * slice_bytes;
        v.slice_bytes = slice_bytes;
        v.strat = strat + tu * geom.S_max;
        v.tok_off = tok_off + tu * geom.S_max;
        v.bk_off = bk_off + tu * geom.S_max;
        v.unit_nseg = unit_nseg + tu;
        v.unit_ntok = unit_ntok + tu;
        v.bump = counters + (size_t)layer * 4;
        v.used_tok = v.bump + 1;
        v.used_bk = v.bump + 2;
        v.S_max = geom.S_max;
        return v;
    }
};

extern "C" {

const char* mkv_last_error(void) { return g_err; }
int mkv_version(void) { return 2; }

int mkv_cache_free(mkv_cache* c) {
    if (!c) return MKV_OK;
    cudaSetDevice(c->desc.device);
    cudaDeviceSynchronize();
    void* ptrs[] = {c->arena, c->strat, c->tok_off, c->bk_off, c->unit_nseg, c->unit_ntok, c->counters,
                    c->dev_flags, c->call_base, c->scores, c->cand_key, c->cand_idx, c->upd_k, c->upd_v, c->upd_cnt, c->attn.zbuf, c->attn.stats, c->plan, c->sink, c->rot_k, c->rot_v, c->q_rot, c->q_dev,
                    c->sel_dev, c->selcnt_dev, c->out_dev, c->masks};
    for (void* p : ptrs)
        if (p) cudaFree(p);
    delete c;
    return MKV_OK;
}

int mkv_cache_create(const mkv_cache_desc* d, mkv_cache** out) {
    if (!d || !out) return fail(MKV_E_ARG, "mkv_cache_create: NULL argument");
    *out = nullptr;
    if (d->n_layers < 1 || d->batch < 1 || d->n_kv_heads < 1 || d->n_q_heads < 1 || d->max_tokens < 1)
        return fail(MKV_E_ARG, "mkv_cache_create: non-positive size");
    if (d->n_q_heads % d->n_kv_heads) return fail(MKV_E_ARG, "n_q_heads must be a multiple of n_kv_heads");
    if (d->reserved != 0) return fail(MKV_E_ARG, "mkv_cache_create: reserved = %d, must be 0", d->reserved);
    if (d->head_dim != kD) return fail(MKV_E_UNSUPPORTED, "head_dim %d: only 128 is built", d->head_dim);
    if (d->n_q_heads / d->n_kv_heads > kMaxGroup)
        return fail(MKV_E_UNSUPPORTED, "GQA group %d > %d", d->n_q_heads / d->n_kv_heads, kMaxGroup);
    if ((long long)d->batch * d->n_kv_heads > 2048)
        return fail(MKV_E_UNSUPPORTED, "batch * n_kv_heads = %lld units: at most 2048 are built", (long long)d->batch * d->n_kv_heads);
    const int B = d->token_block ? d->token_block : 8;
    if (B != 4 && B != 8 && B != 16) return fail(MKV_E_ARG, "token_block %d: must be 4, 8 or 16 (0 = 8)", d->token_block);
    if (d->segment_len < 8 || d->segment_len % 8 || d->segment_len % B || d->segment_len > 4096)
        return fail(MKV_E_UNSUPPORTED, "segment_len %d: need a multiple of 8 and of the token block in [8, 4096]", d->segment_len);
    int ndev = 0;
    MKV_CUDA(cudaGetDeviceCount(&ndev));
    if (d->device < 0 || d->device >= ndev) return fail(MKV_E_ARG, "device %d of %d", d->device, ndev);
    MKV_CUDA(cudaSetDevice(d->device));

    mkv_cache* c = new (std::nothrow) mkv_cache();
    if (!c) return fail(MKV_E_NOMEM, "host allocation failed");
    c->desc = *d;
    CacheGeom& g = c->geom;
    g.n_layers = d->n_layers; g.batch = d->batch; g.n_kv_heads = d->n_kv_heads; g.n_q_heads = d->n_q_heads;
    g.group = d->n_q_heads / d->n_kv_heads; g.max_tokens = d->max_tokens; g.L = d->segment_len;
    g.S_max = (d->max_tokens + g.L - 1) / g.L; g.n_units = d->batch * d->n_kv_heads;
    g.B = B; g.pb = B < kPhys ? B : kPhys; g.ppb = B / g.pb;
    g.blocks_per_seg = g.L / B; g.score_stride = (d->max_tokens + B - 1) / B;
    MKV_CUDA(cudaDeviceGetAttribute(&c->sm_count, cudaDevAttrMultiProcessorCount, d->device));

    // largest payloads: r = 127 on both sides (bitmap + 254 B per vector): 2 * 270 B per token (+ 16 B of padding per device
    // block), 270 B (+ padding) per block key
    const uint64_t worst = (uint64_t)g.n_units * ((uint64_t)d->max_tokens * 540 + ((uint64_t)d->max_tokens / g.pb + 1) * 16 +
                                                  (uint64_t)g.score_stride * 272 + 64 + 32ull * g.S_max) + 4096;
    uint64_t per_layer = d->arena_bytes ? d->arena_bytes / (uint64_t)d->n_layers : worst;
    per_layer = per_layer / 256 * 256;
    if (per_layer < 256) { delete c; return fail(MKV_E_ARG, "arena_bytes too small"); }
    c->slice_bytes = per_layer;

    const size_t tu = (size_t)g.n_layers * g.n_units;
    c->attn.z_unit_stride = attention_z_unit_stride(g);
    c->sel_cap = g.score_stride + 1;
    const size_t upd_bytes = (size_t)g.n_layers * g.n_units * g.L * kD * 2;
    c->upd_n.assign(g.n_layers, 0);
    c->rot_set.assign(g.n_layers, 0);
    const int topk_slices = (g.score_stride + kTopkSlice - 1) / kTopkSlice;
    const size_t cand_bytes = topk_slices > 1 ? (size_t)g.n_units * topk_slices * kTopkSlice * 4 : 256;
    struct { void** p; size_t bytes; } allocs[] = {
        {(void**)&c->arena, (size_t)per_layer * g.n_layers},
        {(void**)&c->strat, tu * g.S_max * sizeof(StratRec)},
        {(void**)&c->tok_off, tu * g.S_max * 4},
        {(void**)&c->bk_off, tu * g.S_max * 4},
        {(void**)&c->unit_nseg, tu * 4},
        {(void**)&c->unit_ntok, tu * 4},
        {(void**)&c->counters, (size_t)g.n_layers * 4 * 8},
        {(void**)&c->dev_flags, 256},
        {(void**)&c->call_base, (size_t)g.n_units * 8},
        {(void**)&c->scores, (size_t)g.n_units * g.score_stride * 4},
        {(void**)&c->cand_key, cand_bytes},
        {(void**)&c->cand_idx, cand_bytes},
        {(void**)&c->upd_k, upd_bytes},
        {(void**)&c->upd_v, upd_bytes},
        {(void**)&c->upd_cnt, (size_t)g.n_layers * 4 + 252},
        {(void**)&c->attn.zbuf, attention_zbuf_floats(g) * 4},
        {(void**)&c->attn.stats, 64},
        {(void**)&c->plan, tu * (size_t)c->sel_cap * g.ppb * sizeof(PlanRec)},
        {(void**)&c->sink, 64},
        {(void**)&c->q_dev, (size_t)g.batch * g.n_q_heads * kD * 2},
        {(void**)&c->q_rot, (size_t)g.batch * g.n_q_heads * kD * 2},
        {(void**)&c->sel_dev, (size_t)g.n_units * c->sel_cap * 4},
        {(void**)&c->selcnt_dev, (size_t)g.n_units * 4},
        {(void**)&c->out_dev, (size_t)g.batch * g.n_q_heads * kD * 4},
        {(void**)&c->masks, (size_t)g.n_units * (size_t)d->max_tokens * 32},
    };
    for (auto& a : allocs) {
        cudaError_t e = cudaMalloc(a.p, a.bytes);
        if (e != cudaSuccess) {
            cudaGetLastError();
            mkv_cache_free(c);
            return fail(MKV_E_NOMEM, "cudaMalloc(%zu bytes): %s", a.bytes, cudaGetErrorString(e));
        }
    }
    cudaMemset(c->unit_nseg, 0, tu * 4);
    cudaMemset(c->unit_ntok, 0, tu * 4);
    cudaMemset(c->counters, 0, (size_t)g.n_layers * 4 * 8);
    cudaMemset(c->dev_flags, 0, 256);
    cudaMemset(c->upd_cnt, 0, (size_t)g.n_layers * 4);
    cudaMemset(c->attn.stats, 0, 64);
    cudaMemset(c->plan, 0, tu * (size_t)c->sel_cap * g.ppb * sizeof(PlanRec));
    cudaMemset(c->strat, 0, tu * g.S_max * sizeof(StratRec));
    cudaMemset(c->masks, 0, (size_t)g.n_units * (size_t)d->max_tokens * 32);
    c->host_nseg.assign((size_t)g.n_layers * g.batch, 0);
    c->host_ntok.assign((size_t)g.n_layers * g.batch, 0);
    cudaError_t e = attention_prepare(g, c->sm_count, c->attn_cluster);
    if (e == cudaSuccess) e = cudaDeviceSynchronize();
    if (e != cudaSuccess) {
        mkv_cache_free(c);
        return fail(MKV_E_CUDA, "create: %s", cudaGetErrorString(e));
    }
    *out = c;
    return MKV_OK;
}

int mkv_cache_reset(mkv_cache* c, int32_t layer, void* stream) {
    if (!c) return fail(MKV_E_ARG, "NULL cache");
    const CacheGeom& g = c->geom;
    if (layer < -1 || layer >= g.n_layers) return fail(MKV_E_ARG, "layer %d out of range", layer);
    cudaStream_t s = (cudaStream_t)stream;
    const int l0 = layer < 0 ? 0 : layer, l1 = layer < 0 ? g.n_layers : layer + 1;
    ++c->generation;  // plan records written before the reset no longer match
    for (int l = l0; l < l1; ++l) {
        MKV_CUDA(cudaMemsetAsync(c->unit_nseg + (size_t)l * g.n_units, 0, (size_t)g.n_units * 4, s));
        MKV_CUDA(cudaMemsetAsync(c->unit_ntok + (size_t)l * g.n_units, 0, (size_t)g.n_units * 4, s));
        MKV_CUDA(cudaMemsetAsync(c->counters + (size_t)l * 4, 0, 32, s));
        for (int b = 0; b < g.batch; ++b) c->host_nseg[(size_t)l * g.batch + b] = c->host_ntok[(size_t)l * g.batch + b] = 0;
        MKV_CUDA(cudaMemsetAsync(c->upd_cnt + l, 0, 4, s));
        c->upd_n[l] = 0;
        // the layer's plan records describe payloads that are gone: cleared on the stream, so that also a launch
        // captured before the reset (its tag is a kernel argument) finds none of them when it is replayed afterwards
        const size_t per_layer = (size_t)g.n_units * c->sel_cap * g.ppb;
        MKV_CUDA(cudaMemsetAsync(c->plan + (size_t)l * per_layer, 0, per_layer * sizeof(PlanRec), s));
    }
    return MKV_OK;
}

static int check_kv_args(const mkv_cache* c, const char* fn, const void* k, const void* v, int64_t sb, int64_t sh,
                         int64_t st, int32_t b0, int32_t nb, int32_t seg0, int32_t nseg, int32_t n_tok) {
    if (!c || !k || !v) return fail(MKV_E_ARG, "%s: NULL argument", fn);
    const CacheGeom& g = c->geom;
    if (b0 < 0 || nb < 1 || b0 + nb > g.batch) return fail(MKV_E_ARG, "%s: requests [%d, %d) of %d", fn, b0, b0 + nb, g.batch);
    if (n_tok < 1 || nseg < 1 || seg0 < 0) return fail(MKV_E_ARG, "%s: empty range", fn);
    if (nseg != (n_tok + g.L - 1) / g.L) return fail(MKV_E_ARG, "%s: nseg %d != ceil(n_tok %d / L %d)", fn, nseg, n_tok, g.L);
    if ((int64_t)seg0 * g.L + n_tok > g.max_tokens) return fail(MKV_E_ARG, "%s: tokens exceed max_tokens %d", fn, g.max_tokens);
    if (st < kD || sh < 0 || sb < 0) return fail(MKV_E_ARG, "%s: bad strides", fn);
    return MKV_OK;
}

int mkv_segment_loss(const mkv_cache* c, const void* k, const void* v, int64_t sb, int64_t sh, int64_t st, int32_t b0,
                     int32_t nb, int32_t seg0, int32_t nseg, int32_t n_tok, mkv_strategy cand, double* loss_k,
                     double* loss_v, void* stream) {
    int rc = check_kv_args(c, "mkv_segment_loss", k, v, sb, sh, st, b0, nb, seg0, nseg, n_tok);
    if (rc) return rc;
    if (!loss_k || !loss_v) return fail(MKV_E_ARG, "mkv_segment_loss: NULL output");
    if (cand.r_k < 1 || cand.r_k > kD || cand.r_v < 1 || cand.r_v > kD) return fail(MKV_E_ARG, "candidate r out of range");
    if (cand.g != 1 && cand.g != 2 && cand.g != 4) return fail(MKV_E_ARG, "element group %d: must be 1, 2 or 4", cand.g);
    if (cand.r_k % cand.g || cand.r_v % cand.g) return fail(MKV_E_ARG, "kept elements must be multiples of the element group");
    CompressArgs a{(const uint16_t*)k, (const uint16_t*)v, sb, sh, st, b0, nb, seg0, nseg, n_tok, c->masks, c->geom.max_tokens};
    MKV_CUDA(cudaSetDevice(c->desc.device));
    MKV_CUDA(launch_segment_loss(c->geom, a, cand, loss_k, loss_v, (cudaStream_t)stream));
    return MKV_OK;
}

int mkv_strategy_quantile(const mkv_cache* c, const double* loss_k, const double* loss_v, int32_t n_units, int32_t nseg,
                          int32_t dense_num, int32_t dense_den, mkv_strategy sparse, mkv_strategy* out, void* stream) {
    if (!c || !loss_k || !loss_v || !out) return fail(MKV_E_ARG, "mkv_strategy_quantile: NULL argument");
    if (n_units < 1 || nseg < 1 || dense_den < 1 || dense_num < 0 || dense_num > dense_den)
        return fail(MKV_E_ARG, "mkv_strategy_quantile: bad sizes");
    long long nd = ((long long)nseg * dense_num + dense_den - 1) / dense_den;
    MKV_CUDA(cudaSetDevice(c->desc.device));
    MKV_CUDA(launch_strategy_quantile(loss_k, loss_v, n_units, nseg, (int)nd, sparse, out, (cudaStream_t)stream));
    return MKV_OK;
}

int mkv_strategy_threshold(const mkv_cache* c, const double* loss_k, const double* loss_v, int32_t ncand,
                           int32_t n_units, int32_t nseg, const mkv_strategy* cands_host, double tau,
                           mkv_strategy* out, void* stream) {
    if (!c || !loss_k || !loss_v || !out || !cands_host) return fail(MKV_E_ARG, "mkv_strategy_threshold: NULL argument");
    if (ncand < 1 || ncand > 64 || n_units < 1 || nseg < 1) return fail(MKV_E_ARG, "mkv_strategy_threshold: bad sizes");
    MKV_CUDA(cudaSetDevice(c->desc.device));
    // the candidates travel as a kernel argument (read during this call only: capturable, no staging buffer)
    MKV_CUDA(launch_strategy_threshold(loss_k, loss_v, ncand, (long long)n_units * nseg, cands_host, tau, out,
                                       (cudaStream_t)stream));
    return MKV_OK;
}

int mkv_compress_segment(mkv_cache* c, int32_t layer, const void* k, const void* v, int64_t sb, int64_t sh, int64_t st,
                         int32_t b0, int32_t nb, int32_t seg0, int32_t nseg, int32_t n_tok, const mkv_strategy* strat,
                         void* stream) {
    int rc = check_kv_args(c, "mkv_compress_segment", k, v, sb, sh, st, b0, nb, seg0, nseg, n_tok);
    if (rc) return rc;
    if (!strat) return fail(MKV_E_ARG, "mkv_compress_segment: NULL strategy");
    const CacheGeom& g = c->geom;
    if (layer < 0 || layer >= g.n_layers) return fail(MKV_E_ARG, "layer %d out of range", layer);
    for (int b = b0; b < b0 + nb; ++b) {
        const int have = c->host_nseg[(size_t)layer * g.batch + b];
        const int tok = c->host_ntok[(size_t)layer * g.batch + b];
        if (seg0 != have) return fail(MKV_E_STATE, "request %d holds %d segments; seg0 = %d (append-only)", b, have, seg0);
        if (tok != have * g.L) return fail(MKV_E_STATE, "request %d ends in a short segment; cannot append", b);
    }
    CompressArgs a{(const uint16_t*)k, (const uint16_t*)v, sb, sh, st, b0, nb, seg0, nseg, n_tok, c->masks, c->geom.max_tokens};
    MKV_CUDA(cudaSetDevice(c->desc.device));
    MKV_CUDA(launch_compress(g, c->view(layer), a, strat, c->call_base, c->dev_flags, (cudaStream_t)stream,
                             &c->last_compress));
    for (int b = b0; b < b0 + nb; ++b) {
        c->host_nseg[(size_t)layer * g.batch + b] = seg0 + nseg;
        c->host_ntok[(size_t)layer * g.batch + b] = seg0 * g.L + n_tok;
    }
    return MKV_OK;
}

int mkv_select(const mkv_cache* cc, int32_t layer, const void* q, int32_t budget, int32_t reduce, int32_t* sel,
               int32_t* sel_count, int32_t k_max, float* scores_opt, void* stream) {
    if (!cc || !q || !sel || !sel_count) return fail(MKV_E_ARG, "mkv_select: NULL argument");
    mkv_cache* c = const_cast<mkv_cache*>(cc);
    const CacheGeom& g = c->geom;
    if (layer < 0 || layer >= g.n_layers) return fail(MKV_E_ARG, "layer %d out of range", layer);
    if (budget < 0 || (reduce != 0 && reduce != 1)) return fail(MKV_E_ARG, "mkv_select: bad budget/reduce");
    const long long need = (long long)budget / g.B + 1;
    if (k_max < 1 || k_max < (need < g.score_stride ? need : g.score_stride))
        return fail(MKV_E_ARG, "mkv_select: k_max %d too small for budget %d", k_max, budget);
    MKV_CUDA(cudaSetDevice(c->desc.device));
    MKV_CUDA(launch_select(g, c->view(layer), (const uint16_t*)q, budget, reduce, sel, sel_count, k_max,
                           scores_opt ? scores_opt : c->scores, c->cand_key, c->cand_idx,
                           c->plan + (size_t)layer * g.n_units * c->sel_cap * g.ppb, c->sel_cap * g.ppb, plan_tag(c->generation, layer),
                           c->sm_count, (cudaStream_t)stream, &c->last_select));
    return MKV_OK;
}

int mkv_packed_attention(const mkv_cache* cc, int32_t layer, const void* q, const int32_t* sel,
                         const int32_t* sel_count, int32_t k_max, float scale, float* out, float* lse_opt,
                         void* stream) {
    if (!cc || !q || !sel || !sel_count || !out) return fail(MKV_E_ARG, "mkv_packed_attention: NULL argument");
    mkv_cache* c = const_cast<mkv_cache*>(cc);
    const CacheGeom& g = c->geom;
    if (layer < 0 || layer >= g.n_layers) return fail(MKV_E_ARG, "layer %d out of range", layer);
    if (k_max < 1) return fail(MKV_E_ARG, "mkv_packed_attention: k_max < 1");
    MKV_CUDA(cudaSetDevice(c->desc.device));
    const size_t upd_off = (size_t)layer * g.n_units * g.L * kD;
    MKV_CUDA(launch_attention(g, c->view(layer), (const uint16_t*)q, sel, sel_count, k_max, scale, out, lse_opt,
                              c->attn_scratch(layer), c->upd_k + upd_off, c->upd_v + upd_off, c->upd_cnt + layer,
                              c->sm_count, c->attn_cluster, (cudaStream_t)stream, &c->last_attn));
    return MKV_OK;
}

int mkv_calibrate_gather(const mkv_cache* cc, int32_t layer, const int32_t* sel, const int32_t* sel_count, int32_t k_max,
                         void* stream) {
    if (!cc || !sel || !sel_count) return fail(MKV_E_ARG, "mkv_calibrate_gather: NULL argument");
    mkv_cache* c = const_cast<mkv_cache*>(cc);
    const CacheGeom& g = c->geom;
    if (layer < 0 || layer >= g.n_layers) return fail(MKV_E_ARG, "layer %d out of range", layer);
    if (k_max < 1) return fail(MKV_E_ARG, "mkv_calibrate_gather: k_max < 1");
    MKV_CUDA(cudaSetDevice(c->desc.device));
    const size_t upd_off = (size_t)layer * g.n_units * g.L * kD;
    int n = 0;
    MKV_CUDA(launch_attention(g, c->view(layer), c->q_dev, sel, sel_count, k_max, 1.f, c->out_dev, nullptr,
                              c->attn_scratch(layer), c->upd_k + upd_off, c->upd_v + upd_off, c->upd_cnt + layer,
                              c->sm_count, c->attn_cluster, (cudaStream_t)stream, &n, true));
    return MKV_OK;
}

int mkv_calibrate_walk(const mkv_cache* cc, int32_t layer, const void* q, const int32_t* sel, const int32_t* sel_count,
                       int32_t k_max, int32_t reps, void* stream) {
    if (!cc || !q || !sel || !sel_count) return fail(MKV_E_ARG, "mkv_calibrate_walk: NULL argument");
    mkv_cache* c = const_cast<mkv_cache*>(cc);
    const CacheGeom& g = c->geom;
    if (layer < 0 || layer >= g.n_layers) return fail(MKV_E_ARG, "layer %d out of range", layer);
    if (k_max < 1 || reps < 1) return fail(MKV_E_ARG, "mkv_calibrate_walk: k_max < 1 or reps < 1");
    MKV_CUDA(cudaSetDevice(c->desc.device));
    MKV_CUDA(launch_walk_probe(g, c->view(layer), (const uint16_t*)q, sel, sel_count, k_max, reps, c->sm_count, c->sink,
                               (cudaStream_t)stream));
    return MKV_OK;
}

int mkv_calibrate_stream(const mkv_cache* cc, int32_t layer, uint64_t bytes, void* stream) {
    if (!cc) return fail(MKV_E_ARG, "mkv_calibrate_stream: NULL argument");
    mkv_cache* c = const_cast<mkv_cache*>(cc);
    const CacheGeom& g = c->geom;
    if (layer < 0 || layer >= g.n_layers) return fail(MKV_E_ARG, "layer %d out of range", layer);
    if (bytes > c->slice_bytes) bytes = c->slice_bytes;
    MKV_CUDA(cudaSetDevice(c->desc.device));
    MKV_CUDA(launch_stream_read(c->arena + (size_t)layer * c->slice_bytes, bytes, c->sm_count, c->sink, (cudaStream_t)stream));
    return MKV_OK;
}

int mkv_attention_stats(const mkv_cache* c, uint64_t* blocks_host, uint64_t* v_blocks_host, uint64_t* v_bytes_host,
                        int32_t reset) {
    if (!c) return fail(MKV_E_ARG, "NULL cache");
    MKV_CUDA(cudaSetDevice(c->desc.device));
    MKV_CUDA(cudaDeviceSynchronize());
    unsigned long long st[8];
    MKV_CUDA(cudaMemcpy(st, c->attn.stats, 64, cudaMemcpyDeviceToHost));
    if (blocks_host) *blocks_host = st[0];
    if (v_blocks_host) *v_blocks_host = st[1];
    if (v_bytes_host) *v_bytes_host = st[2];
    if (reset) MKV_CUDA(cudaMemset(c->attn.stats, 0, 64));
    return MKV_OK;
}

int mkv_rotation_set(mkv_cache* c, int32_t layer, const float* r_k, const float* r_v, void* stream) {
    if (!c) return fail(MKV_E_ARG, "NULL cache");
    const CacheGeom& g = c->geom;
    if (layer < 0 || layer >= g.n_layers) return fail(MKV_E_ARG, "layer %d out of range", layer);
    if ((r_k == nullptr) != (r_v == nullptr)) return fail(MKV_E_ARG, "mkv_rotation_set: pass both matrices or neither");
    MKV_CUDA(cudaSetDevice(c->desc.device));
    if (!r_k) { c->rot_set[layer] = 0; return MKV_OK; }
    const size_t per_layer = (size_t)g.n_kv_heads * kD * kD;
    if (!c->rot_k) {  // first use: this call allocates (it is the only non-capturable path of the call)
        cudaError_t e1 = cudaMalloc((void**)&c->rot_k, per_layer * g.n_layers * 4);
        cudaError_t e2 = e1 == cudaSuccess ? cudaMalloc((void**)&c->rot_v, per_layer * g.n_layers * 4) : e1;
        if (e2 != cudaSuccess) {
            cudaGetLastError();
            if (c->rot_k) { cudaFree(c->rot_k); c->rot_k = nullptr; }
            return fail(MKV_E_NOMEM, "mkv_rotation_set: cudaMalloc: %s", cudaGetErrorString(e2));
        }
    }
    MKV_CUDA(cudaMemcpyAsync(c->rot_k + per_layer * layer, r_k, per_layer * 4, cudaMemcpyDeviceToDevice, (cudaStream_t)stream));
    MKV_CUDA(cudaMemcpyAsync(c->rot_v + per_layer * layer, r_v, per_layer * 4, cudaMemcpyDeviceToDevice, (cudaStream_t)stream));
    c->rot_set[layer] = 1;
    return MKV_OK;
}

int mkv_rotate_query(const mkv_cache* c, int32_t layer, const void* q, void* q_out, void* stream) {
    if (!c || !q || !q_out) return fail(MKV_E_ARG, "mkv_rotate_query: NULL argument");
    const CacheGeom& g = c->geom;
    if (layer < 0 || layer >= g.n_layers) return fail(MKV_E_ARG, "layer %d out of range", layer);
    if (!c->rot_set[layer]) return fail(MKV_E_STATE, "mkv_rotate_query: layer %d has no rotation (mkv_rotation_set)", layer);
    if (q == q_out) return fail(MKV_E_ARG, "mkv_rotate_query: q_out must not alias q");
    MKV_CUDA(cudaSetDevice(c->desc.device));
    MKV_CUDA(launch_rotate_query(g, (const uint16_t*)q, c->rot_k + (size_t)layer * g.n_kv_heads * kD * kD, (uint16_t*)q_out,
                                 (cudaStream_t)stream));
    return MKV_OK;
}

int mkv_rotate_output(const mkv_cache* c, int32_t layer, float* out, void* stream) {
    if (!c || !out) return fail(MKV_E_ARG, "mkv_rotate_output: NULL argument");
    const CacheGeom& g = c->geom;
    if (layer < 0 || layer >= g.n_layers) return fail(MKV_E_ARG, "layer %d out of range", layer);
    if (!c->rot_set[layer]) return fail(MKV_E_STATE, "mkv_rotate_output: layer %d has no rotation (mkv_rotation_set)", layer);
    MKV_CUDA(cudaSetDevice(c->desc.device));
    MKV_CUDA(launch_rotate_output(g, out, c->rot_v + (size_t)layer * g.n_kv_heads * kD * kD, (cudaStream_t)stream));
    return MKV_OK;
}

int mkv_update_append(mkv_cache* c, int32_t layer, const void* k_new, const void* v_new, int64_t sb, int64_t sh,
                      int64_t st, int32_t n_new, void* stream) {
    if (!c || !k_new || !v_new) return fail(MKV_E_ARG, "mkv_update_append: NULL argument");
    const CacheGeom& g = c->geom;
    if (layer < 0 || layer >= g.n_layers) return fail(MKV_E_ARG, "layer %d out of range", layer);
    if (n_new < 1 || st < kD || sh < 0 || sb < 0) return fail(MKV_E_ARG, "mkv_update_append: bad n_new / strides");
    const int have = c->upd_n[layer];
    if (have + n_new > g.L)
        return fail(MKV_E_STATE, "mkv_update_append: buffer holds %d of %d tokens; %d more do not fit (flush first)", have,
                    g.L, n_new);
    CompressArgs a{(const uint16_t*)k_new, (const uint16_t*)v_new, sb, sh, st, 0, g.batch, 0, 1, n_new, nullptr, 0};
    MKV_CUDA(cudaSetDevice(c->desc.device));
    const size_t off = (size_t)layer * g.n_units * g.L * kD;
    MKV_CUDA(launch_update_copy(g, a, c->upd_k + off, c->upd_v + off, c->upd_cnt + layer, have, (cudaStream_t)stream));
    c->upd_n[layer] = have + n_new;
    return MKV_OK;
}

int mkv_update_flush(mkv_cache* c, int32_t layer, const mkv_strategy* strat, void* stream) {
    if (!c || !strat) return fail(MKV_E_ARG, "mkv_update_flush: NULL argument");
    const CacheGeom& g = c->geom;
    if (layer < 0 || layer >= g.n_layers) return fail(MKV_E_ARG, "layer %d out of range", layer);
    const int n = c->upd_n[layer];
    if (n == 0) return MKV_OK;
    const int seg0 = c->host_nseg[(size_t)layer * g.batch];
    for (int b = 1; b < g.batch; ++b)
        if (c->host_nseg[(size_t)layer * g.batch + b] != seg0)
            return fail(MKV_E_STATE, "mkv_update_flush: requests hold different numbers of segments");
    // the buffer is the raw K/V of the next segment of every unit: [b][h][t][c] with dense strides
    const int64_t sh = (int64_t)g.L * kD, sb = sh * g.n_kv_heads;
    const size_t off = (size_t)layer * g.n_units * g.L * kD;
    const int rc = mkv_compress_segment(c, layer, c->upd_k + off, c->upd_v + off, sb, sh, kD, 0, g.batch, seg0, 1, n, strat,
                                        stream);
    if (rc) return rc;
    MKV_CUDA(cudaMemsetAsync(c->upd_cnt + layer, 0, 4, (cudaStream_t)stream));
    c->upd_n[layer] = 0;
    return MKV_OK;
}

int mkv_update_count(const mkv_cache* c, int32_t layer, int32_t* n_host) {
    if (!c || !n_host) return fail(MKV_E_ARG, "mkv_update_count: NULL argument");
    if (layer < 0 || layer >= c->geom.n_layers) return fail(MKV_E_ARG, "layer %d out of range", layer);
    *n_host = c->upd_n[layer];
    return MKV_OK;
}

int mkv_decode_step(mkv_cache* c, int32_t layer, const void* q, int32_t budget, int32_t reduce, float scale, float* out,
                    float* lse_opt, int32_t* sel_opt, int32_t* sel_count_opt, int32_t k_max, void* stream) {
    if (!c || !q || !out) return fail(MKV_E_ARG, "mkv_decode_step: NULL argument");
    const CacheGeom& g = c->geom;
    if (layer < 0 || layer >= g.n_layers) return fail(MKV_E_ARG, "layer %d out of range", layer);
    if ((sel_opt == nullptr) != (sel_count_opt == nullptr)) return fail(MKV_E_ARG, "mkv_decode_step: sel and sel_count go together");
    cudaStream_t s = (cudaStream_t)stream;
    int32_t* sel = sel_opt ? sel_opt : c->sel_dev;
    int32_t* cnt = sel_opt ? sel_count_opt : c->selcnt_dev;
    if (!sel_opt) {
        long long km = (long long)budget / g.B + 1;
        k_max = (int32_t)(km > c->sel_cap ? c->sel_cap : km);
    }
    MKV_CUDA(cudaSetDevice(c->desc.device));
    const uint16_t* qd = (const uint16_t*)q;
    if (c->rot_set[layer]) {  // rotation fold: the cache holds K R_k^T, V R_v^T; attend with q R_k^T
        MKV_CUDA(launch_rotate_query(g, qd, c->rot_k + (size_t)layer * g.n_kv_heads * kD * kD, c->q_rot, s));
        qd = c->q_rot;
    }
    int rc = mkv_select(c, layer, qd, budget, reduce, sel, cnt, k_max, nullptr, stream);
    if (rc) return rc;
    rc = mkv_packed_attention(c, layer, qd, sel, cnt, k_max, scale, out, lse_opt, stream);
    if (rc) return rc;
    if (c->rot_set[layer]) MKV_CUDA(launch_rotate_output(g, out, c->rot_v + (size_t)layer * g.n_kv_heads * kD * kD, s));
    return MKV_OK;
}

namespace {

// 16-byte copy between device memory and device-mapped (pinned) host memory: part of the decode chain (PDL), so a
// host-buffer step stays on the compute engine instead of bouncing to a copy engine and back twice per layer
__global__ void __launch_bounds__(256) mkv_copy16_kernel(const uint4* __restrict__ src, uint4* __restrict__ dst, size_t n16) {
    pdl_wait();
    pdl_launch_dependents();
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n16; i += (size_t)gridDim.x * blockDim.x) dst[i] = src[i];
}

// device address of a pinned / registered host buffer the GPU can access directly, else nullptr.  The kernels that use
// it move 16 bytes per access, so a buffer that is not 16-byte aligned (a view into a pinned block at an odd offset)
// counts as not mapped: it takes the cudaMemcpyAsync path like pageable memory.
void* mapped_host(const void* p) {
    cudaPointerAttributes a;
    if (cudaPointerGetAttributes(&a, p) != cudaSuccess) { cudaGetLastError(); return nullptr; }
    if (a.type != cudaMemoryTypeHost || (reinterpret_cast<uintptr_t>(a.devicePointer) & 15u) != 0) return nullptr;
    return a.devicePointer;
}

}  // namespace

int mkv_decode_host(mkv_cache* c, int32_t layer, const void* q_host, int32_t budget, int32_t reduce, float scale,
                    float* out_host, int32_t* sel_host_opt, int32_t* sel_count_host_opt, void* stream) {
    if (!c || !q_host || !out_host) return fail(MKV_E_ARG, "mkv_decode_host: NULL argument");
    const CacheGeom& g = c->geom;
    cudaStream_t s = (cudaStream_t)stream;
    long long k_max = (long long)budget / g.B + 1;
    if (k_max > c->sel_cap) k_max = c->sel_cap;
    if (layer < 0 || layer >= g.n_layers) return fail(MKV_E_ARG, "layer %d out of range", layer);
    MKV_CUDA(cudaSetDevice(c->desc.device));
    const size_t q_bytes = (size_t)g.batch * g.n_q_heads * kD * 2, out_bytes = (size_t)g.batch * g.n_q_heads * kD * 4;
    // Pinned host buffers are read and written by kernels of the chain itself (q: one small fetch kernel; out: the
    // attention kernel's own stores, or a store kernel behind the output fold); pageable buffers take the copy engine.
    void* q_map = mapped_host(q_host);
    void* out_map = mapped_host(out_host);
    const bool rotated = !c->rot_set.empty() && c->rot_set[layer];
    if (q_map)
        MKV_CUDA(launch_pdl(mkv_copy16_kernel, dim3(8), dim3(256), (size_t)0, s, (const uint4*)q_map, (uint4*)c->q_dev, q_bytes / 16));
    else
        MKV_CUDA(cudaMemcpyAsync(c->q_dev, q_host, q_bytes, cudaMemcpyHostToDevice, s));
    float* out_arg = out_map && !rotated ? (float*)out_map : c->out_dev;
    const int rc = mkv_decode_step(c, layer, c->q_dev, budget, reduce, scale, out_arg, nullptr, nullptr, nullptr, 0, stream);
    if (rc) return rc;
    if (out_arg == c->out_dev) {
        if (out_map)
            MKV_CUDA(launch_pdl(mkv_copy16_kernel, dim3(16), dim3(256), (size_t)0, s, (const uint4*)c->out_dev, (uint4*)out_map, out_bytes / 16));
        else
            MKV_CUDA(cudaMemcpyAsync(out_host, c->out_dev, out_bytes, cudaMemcpyDeviceToHost, s));
    }
    if (sel_host_opt)
        MKV_CUDA(cudaMemcpyAsync(sel_host_opt, c->sel_dev, (size_t)g.n_units * k_max * 4, cudaMemcpyDeviceToHost, s));
    if (sel_count_host_opt)
        MKV_CUDA(cudaMemcpyAsync(sel_count_host_opt, c->selcnt_dev, (size_t)g.n_units * 4, cudaMemcpyDeviceToHost, s));
    return MKV_OK;
}

int mkv_cache_export(const mkv_cache* c, int32_t layer, int32_t b, int32_t h, void* buf, uint64_t cap,
                     uint64_t* need_host) {
    if (!c || !need_host) return fail(MKV_E_ARG, "mkv_cache_export: NULL argument");
    const CacheGeom& g = c->geom;
    if (layer < 0 || layer >= g.n_layers || b < 0 || b >= g.batch || h < 0 || h >= g.n_kv_heads)
        return fail(MKV_E_ARG, "mkv_cache_export: unit out of range");
    MKV_CUDA(cudaSetDevice(c->desc.device));
    MKV_CUDA(cudaDeviceSynchronize());
    const int unit = b * g.n_kv_heads + h;
    const LayerView lv = c->view(layer);
    int32_t S = 0, N = 0;
    MKV_CUDA(cudaMemcpy(&S, lv.unit_nseg + unit, 4, cudaMemcpyDeviceToHost));
    MKV_CUDA(cudaMemcpy(&N, lv.unit_ntok + unit, 4, cudaMemcpyDeviceToHost));
    std::vector<StratRec> rec(S);
    std::vector<uint32_t> toff(S), koff(S);
    if (S) {
        MKV_CUDA(cudaMemcpy(rec.data(), lv.strat + (size_t)unit * lv.S_max, (size_t)S * 8, cudaMemcpyDeviceToHost));
        MKV_CUDA(cudaMemcpy(toff.data(), lv.tok_off + (size_t)unit * lv.S_max, (size_t)S * 4, cudaMemcpyDeviceToHost));
        MKV_CUDA(cudaMemcpy(koff.data(), lv.bk_off + (size_t)unit * lv.S_max, (size_t)S * 4, cudaMemcpyDeviceToHost));
    }
    // canonical sizes (DESIGN.md format): the bitmap of a packed vector has D / g bits; the device keeps 128 bits for
    // every g (the decode kernels read one layout), so sizes and offsets are recomputed here
    auto vbc = [](int r, int gg) -> uint32_t { return 2u * (uint32_t)r + (r == kD ? 0u : (uint32_t)(kD / (8 * gg))); };
    auto tokc = [&](const StratRec& r, int nb) -> uint32_t { return pad16u((uint32_t)nb * (vbc(r.r_k, r.g) + vbc(r.r_v, r.g))); };
    const int B = g.B, pb = g.pb;
    auto segtokc = [&](const StratRec& r) -> uint64_t {
        const int full = r.n_tok / B, rem = r.n_tok % B;
        return (uint64_t)full * tokc(r, B) + (rem ? tokc(r, rem) : 0u);
    };
    auto segbkc = [&](const StratRec& r) -> uint64_t { return pad16u((uint32_t)((r.n_tok + B - 1) / B) * vbc(r.r_k, r.g)); };
    uint64_t tok_bytes = 0, bk_bytes = 0, ptok_bytes = 0, pbk_bytes = 0;
    for (int s = 0; s < S; ++s) {
        tok_bytes += segtokc(rec[s]);
        bk_bytes += segbkc(rec[s]);
        ptok_bytes += seg_tok_bytes(rec[s].r_k, rec[s].r_v, rec[s].n_tok, pb);
        pbk_bytes += seg_bk_bytes(rec[s].r_k, rec[s].n_tok, B);
    }
    const uint64_t tables = align_up(48 + (uint64_t)S * 16, 16);
    const uint64_t need = tables + tok_bytes + bk_bytes;
    *need_host = need;
    if (!buf) return MKV_OK;
    if (cap < need) return fail(MKV_E_ARG, "mkv_cache_export: need %llu bytes, cap %llu", (unsigned long long)need,
                                (unsigned long long)cap);
    uint8_t* p = (uint8_t*)buf;
    memset(p, 0, need);
    const uint32_t hdr[6] = {0x31564B4Du, (uint32_t)kD, (uint32_t)N, (uint32_t)g.L, (uint32_t)S, 0u};
    memcpy(p, hdr, 24);
    memcpy(p + 24, &tok_bytes, 8);
    memcpy(p + 32, &bk_bytes, 8);
    uint8_t* p_strat = p + 48;
    uint8_t* p_toff = p_strat + (size_t)S * 8;
    uint8_t* p_koff = p_toff + (size_t)S * 4;
    uint8_t* tok_arena = p + tables;
    uint8_t* bk_arena = tok_arena + tok_bytes;
    // the unit's device payloads, segment after segment (physical runs that are contiguous are copied at once)
    std::vector<uint8_t> ptok(ptok_bytes), pbk(pbk_bytes);
    {
        uint64_t tpos = 0, kpos = 0;
        int s = 0;
        while (s < S) {
            int e = s;
            uint64_t trun = 0, krun = 0;
            while (e < S) {
                const uint64_t tb = seg_tok_bytes(rec[e].r_k, rec[e].r_v, rec[e].n_tok, pb), kb = seg_bk_bytes(rec[e].r_k, rec[e].n_tok, B);
                if (e > s && ((uint64_t)toff[e] * 16 != (uint64_t)toff[s] * 16 + trun || (uint64_t)koff[e] * 16 != (uint64_t)koff[s] * 16 + krun))
                    break;
                trun += tb;
                krun += kb;
                ++e;
            }
            if (trun) MKV_CUDA(cudaMemcpy(ptok.data() + tpos, lv.slice + (uint64_t)toff[s] * 16, trun, cudaMemcpyDeviceToHost));
            if (krun) MKV_CUDA(cudaMemcpy(pbk.data() + kpos, lv.slice + (uint64_t)koff[s] * 16, krun, cudaMemcpyDeviceToHost));
            tpos += trun;
            kpos += krun;
            s = e;
        }
    }
    // One canonical group of n = n0 + n1 packed vectors from (up to) two device groups of n0 and n1 <= 8 vectors (a token
    // block of 16 tokens is stored as two device blocks).  Device group: its vectors' bitmaps of 128 bits (one bit per
    // channel, every channel of a kept element group set), then the kept values RANK-major (compress.cu).  Canonical: n
    // bitmaps of D / g bits (one per element group), then the values vector-major.  Dense vectors (r = D): values only.
    // pairs: K vectors and block keys with g >= 2 hold their values pair-major (compress.cu: pack_vector).
    auto repack = [](const uint8_t* src0, int n0, const uint8_t* src1, int n1, uint8_t* dst, int r, int gg, bool pairs) {
        const int n = n0 + n1;
        if (r == kD) {
            memcpy(dst, src0, (size_t)n0 * kD * 2);
            if (n1) memcpy(dst + (size_t)n0 * kD * 2, src1, (size_t)n1 * kD * 2);
            return;
        }
        const int bmc = kD / (8 * gg);
        uint8_t* o = dst + (size_t)n * bmc;
        for (int t = 0; t < n; ++t) {
            const uint8_t* src = t < n0 ? src0 : src1;
            const int tt = t < n0 ? t : t - n0, nn = t < n0 ? n0 : n1;
            for (int m = 0; m < kD / gg; ++m) {
                const int c = m * gg;
                if ((src[tt * kBitmapBytes + (c >> 3)] >> (c & 7)) & 1) dst[t * bmc + (m >> 3)] |= (uint8_t)(1u << (m & 7));
            }
            const uint8_t* v = src + (size_t)nn * kBitmapBytes;  // rank-major values of the device group
            for (int rho = 0; rho < r; ++rho) {
                const size_t at = pairs ? ((size_t)(rho >> 1) * nn + tt) * 2 + (rho & 1) : (size_t)rho * nn + tt;
                memcpy(o + 2 * ((size_t)t * r + rho), v + 2 * at, 2);
            }
        }
    };
    uint64_t tpos = 0, kpos = 0;            // canonical positions
    const uint8_t* tp = ptok.data();
    const uint8_t* kp = pbk.data();
    for (int sg = 0; sg < S; ++sg) {
        const StratRec& r = rec[sg];
        const int r_k = r.r_k, r_v = r.r_v, gg = r.g ? r.g : 1, n_tok = r.n_tok, nblk = (n_tok + B - 1) / B;
        const uint32_t ct = (uint32_t)(tpos / 16), ck = (uint32_t)(kpos / 16);
        memcpy(p_strat + (size_t)sg * 8, &r, 8);
        memcpy(p_toff + (size_t)sg * 4, &ct, 4);
        memcpy(p_koff + (size_t)sg * 4, &ck, 4);
        const uint32_t bmk = r_k == kD ? 0u : (uint32_t)kBitmapBytes;
        for (int blk = 0; blk < nblk; ++blk) {  // token blocks of B tokens = one or two device blocks of <= pb tokens
            const int nbt = std::min(B, n_tok - blk * B);
            const int n0 = std::min(pb, nbt), n1 = nbt - n0;
            const uint8_t* s0 = tp;
            const uint8_t* s1 = tp + tokblock_bytes(r_k, r_v, n0);
            uint8_t* d = tok_arena + tpos;
            repack(s0, n0, s1, n1, d, r_k, gg, gg >= 2);                                                            // K vectors
            repack(s0 + (size_t)n0 * (bmk + 2 * r_k), n0, s1 + (size_t)n1 * (bmk + 2 * r_k), n1,
                   d + (size_t)nbt * vbc(r_k, gg), r_v, gg, false);                                                 // V vectors
            tp += tokblock_bytes(r_k, r_v, n0) + (n1 ? tokblock_bytes(r_k, r_v, n1) : 0u);
            tpos += tokc(r, nbt);
        }
        // block keys of the segment: device [bitmaps nblk x 16][values, groups of 8 keys rank-major]; canonical
        // [bitmaps nblk x D/(8g)][values nblk x r_k vector-major]
        {
            uint8_t* d = bk_arena + kpos;
            const int bmc = r_k == kD ? 0 : kD / (8 * gg);
            for (int grp = 0; grp * 8 < nblk; ++grp) {
                const int n = std::min(8, nblk - 8 * grp);
                if (r_k == kD) { memcpy(d + (size_t)grp * 8 * kD * 2, kp + (size_t)grp * 8 * kD * 2, (size_t)n * kD * 2); continue; }
                // gather the group's bitmaps and values into one contiguous device-format group, then repack
                std::vector<uint8_t> tmp((size_t)n * kBitmapBytes + (size_t)n * r_k * 2), outg((size_t)n * bmc + (size_t)n * r_k * 2);
                memcpy(tmp.data(), kp + (size_t)grp * 8 * kBitmapBytes, (size_t)n * kBitmapBytes);
                memcpy(tmp.data() + (size_t)n * kBitmapBytes, kp + (size_t)nblk * kBitmapBytes + (size_t)grp * 8 * r_k * 2, (size_t)n * r_k * 2);
                repack(tmp.data(), n, nullptr, 0, outg.data(), r_k, gg, gg >= 2);
                memcpy(d + (size_t)grp * 8 * bmc, outg.data(), (size_t)n * bmc);
                memcpy(d + (size_t)nblk * bmc + (size_t)grp * 8 * r_k * 2, outg.data() + (size_t)n * bmc, (size_t)n * r_k * 2);
            }
            kp += seg_bk_bytes(r_k, n_tok, B);
            kpos += segbkc(r);
        }
    }
    return MKV_OK;
}

int mkv_cache_bytes(const mkv_cache* c, int32_t layer, uint64_t* packed, uint64_t* block_keys, uint64_t* tables) {
    if (!c) return fail(MKV_E_ARG, "NULL cache");
    const CacheGeom& g = c->geom;
    if (layer < 0 || layer >= g.n_layers) return fail(MKV_E_ARG, "layer %d out of range", layer);
    MKV_CUDA(cudaSetDevice(c->desc.device));
    MKV_CUDA(cudaDeviceSynchronize());
    unsigned long long cnt[4];
    MKV_CUDA(cudaMemcpy(cnt, c->counters + (size_t)layer * 4, 32, cudaMemcpyDeviceToHost));
    std::vector<int32_t> nseg(g.n_units);
    MKV_CUDA(cudaMemcpy(nseg.data(), c->unit_nseg + (size_t)layer * g.n_units, (size_t)g.n_units * 4, cudaMemcpyDeviceToHost));
    uint64_t segs = 0;
    for (int v : nseg) segs += (uint64_t)v;
    if (packed) *packed = cnt[1];
    if (block_keys) *block_keys = cnt[2];
    if (tables) *tables = segs * 16;
    return MKV_OK;
}

int mkv_cache_status(const mkv_cache* c, uint32_t* flags_host) {
    if (!c) return fail(MKV_E_ARG, "NULL cache");
    MKV_CUDA(cudaSetDevice(c->desc.device));
    MKV_CUDA(cudaDeviceSynchronize());
    uint32_t f = 0;
    MKV_CUDA(cudaMemcpy(&f, c->dev_flags, 4, cudaMemcpyDeviceToHost));
    if (flags_host) *flags_host = f;
    if (f) return fail(MKV_E_DEVICE, "device flags 0x%x (%s%s)", f, (f & MKV_DEV_ARENA_OVERFLOW) ? "arena overflow " : "",
                       (f & MKV_DEV_BAD_STRATEGY) ? "bad strategy" : "");
    return MKV_OK;
}

int mkv_last_launch_count(const mkv_cache* c, int32_t* sel_k, int32_t* attn_k, int32_t* comp_k) {
    if (!c) return fail(MKV_E_ARG, "NULL cache");
    if (sel_k) *sel_k = c->last_select;
    if (attn_k) *attn_k = c->last_attn;
    if (comp_k) *comp_k = c->last_compress;
    return MKV_OK;
}

}  // extern "C"
