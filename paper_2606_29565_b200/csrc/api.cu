// api.cu -- the C ABI of libprepos (include/prepos.h): argument checking, the context and its
// workspace carve-up, the host-side attention plan (Alg. 1 l.2-3 budget check lives here), and
// dispatch to the kernels.  No CPU fallback exists: without an sm_100 device every compute entry
// point fails with PREPOS_E_NO_DEVICE.
#include <math.h>
#include <stdio.h>
#include <string.h>

#include <new>

#include "common.cuh"

namespace {

thread_local char g_last_cuda_error[512] = "";

size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }
bool aligned16(const void *p) { return (reinterpret_cast<uintptr_t>(p) & 15) == 0; }

struct WsLayout {
    size_t rd_partials, rd_counter, attn_units, attn_partials, attn_counters, attn_yield, total;
    int max_units;
    size_t attn_counters_n;
};

// units per session we provision for: row chunks of <= 256 rows (tcgen05 path) or <= 16 rows (generic).
// 64 chunks of the generic path cover L <= 64 * 16 / G entry tokens for G <= 16; larger calls fail with
// PREPOS_E_WORKSPACE rather than overrun.
constexpr int kUnitsPerSession = 64;

WsLayout ws_layout(const prepos_model_shape &s, int max_sessions)
{
    WsLayout w;
    size_t off = 0;
    w.rd_partials = off;
    off = align_up(off + sizeof(RdPartial) * kRdMaxRows * kMaxRdPartials, 256);
    w.rd_counter = off;
    off = align_up(off + sizeof(unsigned int) * (kRdMaxRows + 1), 256);
    w.max_units = max_sessions * kUnitsPerSession;
    w.attn_units = off;
    off = align_up(off + sizeof(AttnUnit) * w.max_units, 256);
    w.attn_partials = off;
    off = align_up(off + sizeof(float) * 2 * kAttnMaxCtas * kAttnMaxRows * (static_cast<size_t>(s.head_dim) + 2), 256);
    w.attn_counters_n = static_cast<size_t>(s.layers) * s.n_kv_heads * w.max_units;
    w.attn_counters = off;
    off = align_up(off + sizeof(unsigned int) * w.attn_counters_n, 256);
    w.attn_yield = off;   // yield flag, pass state, per-CTA progress
    off = align_up(off + 256 + sizeof(int) * kAttnMaxCtas, 256);
    w.total = off;
    return w;
}

int check_shape(const prepos_model_shape *s)
{
    if (!s) return PREPOS_E_INVALID_ARG;
    if (s->layers <= 0 || s->n_q_heads <= 0 || s->n_kv_heads <= 0 || s->head_dim <= 0 || s->hidden <= 0 ||
        s->vocab < 2 || s->page_size <= 0)
        return PREPOS_E_SHAPE;
    if (s->n_q_heads % s->n_kv_heads != 0) return PREPOS_E_SHAPE;
    if (s->n_q_heads / s->n_kv_heads > 64) return PREPOS_E_SHAPE;
    if (s->head_dim % 8 != 0 || s->head_dim > 256) return PREPOS_E_SHAPE;
    if (s->hidden % 128 != 0) return PREPOS_E_SHAPE;
    if ((s->page_size & (s->page_size - 1)) != 0 || s->page_size > 128) return PREPOS_E_SHAPE;
    return PREPOS_OK;
}

}  // namespace

void prepos_note_cuda_error(cudaError_t e, const char *what, const char *file, int line)
{
    snprintf(g_last_cuda_error, sizeof g_last_cuda_error, "%s: %s (%s:%d)", cudaGetErrorName(e), what, file, line);
    fprintf(stderr, "libprepos: CUDA error %s\n", g_last_cuda_error);
}

void *prepos_get_encode_tiled()
{
    static void *fn = nullptr;
    if (!fn) {
        cudaDriverEntryPointQueryResult qres;
        void *f = nullptr;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &f, cudaEnableDefault, &qres) == cudaSuccess &&
            qres == cudaDriverEntryPointSuccess)
            fn = f;
    }
    return fn;
}

extern "C" {

const char *prepos_strerror(int status)
{
    switch (status) {
        case PREPOS_OK: return "ok";
        case PREPOS_SKIPPED_BUDGET: return "skipped: entry exceeds the session's cell-budget headroom";
        case PREPOS_E_INVALID_ARG: return "invalid argument";
        case PREPOS_E_SHAPE: return "unsupported shape";
        case PREPOS_E_ALIGN: return "pointer or stride not 16-byte aligned";
        case PREPOS_E_CUDA: return g_last_cuda_error[0] ? g_last_cuda_error : "CUDA error";
        case PREPOS_E_WORKSPACE: return "workspace too small";
        case PREPOS_E_NO_DEVICE: return "no sm_100 CUDA device available (libprepos has no CPU fallback)";
        case PREPOS_E_FIXED_SCRATCH:
            return "request exceeds the built-in scratch of the no-allocation entry point (prepos_scan_logits_noalloc: "
                   "n <= 32 rows, vocab <= 2^24; use prepos_scan_logits for more)";
        default: return "unknown status";
    }
}

int prepos_version(void) { return PREPOS_VERSION; }

size_t prepos_workspace_bytes(const prepos_model_shape *shape, int max_sessions)
{
    if (check_shape(shape) != PREPOS_OK || max_sessions <= 0) return 0;
    return ws_layout(*shape, max_sessions).total;
}

int prepos_ctx_create(prepos_ctx **out, const prepos_model_shape *shape, int max_sessions, void *workspace,
                      size_t workspace_bytes)
{
    if (!out) return PREPOS_E_INVALID_ARG;
    *out = nullptr;
    int st = check_shape(shape);
    if (st != PREPOS_OK) return st;
    if (max_sessions <= 0) return PREPOS_E_INVALID_ARG;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
        cudaGetLastError();
        return PREPOS_E_NO_DEVICE;
    }
    int dev = 0;
    PREPOS_CUDA_TRY(cudaGetDevice(&dev));
    cudaDeviceProp prop;
    PREPOS_CUDA_TRY(cudaGetDeviceProperties(&prop, dev));
    if (prop.major != 10) return PREPOS_E_NO_DEVICE;  // built for sm_100a only
    const WsLayout w = ws_layout(*shape, max_sessions);
    if (!workspace || workspace_bytes < w.total) return PREPOS_E_WORKSPACE;
    if ((reinterpret_cast<uintptr_t>(workspace) & 255) != 0) return PREPOS_E_ALIGN;

    prepos_ctx *c = new (std::nothrow) prepos_ctx();
    if (!c) return PREPOS_E_INVALID_ARG;
    c->shape = *shape;
    c->max_sessions = max_sessions;
    c->device = dev;
    c->num_sms = prop.multiProcessorCount;
    c->cc_major = prop.major;
    c->cc_minor = prop.minor;
    c->ws = static_cast<char *>(workspace);
    c->ws_bytes = workspace_bytes;
    c->launches = 0;
    c->attn_path = 0;
    c->rd_partials = reinterpret_cast<RdPartial *>(c->ws + w.rd_partials);
    c->rd_counter = reinterpret_cast<unsigned int *>(c->ws + w.rd_counter);
    c->attn_units = reinterpret_cast<AttnUnit *>(c->ws + w.attn_units);
    c->max_units = w.max_units;
    c->attn_partials = reinterpret_cast<float *>(c->ws + w.attn_partials);
    c->attn_counters = reinterpret_cast<unsigned int *>(c->ws + w.attn_counters);
    c->attn_counters_n = w.attn_counters_n;
    c->attn_yield_flag = reinterpret_cast<unsigned int *>(c->ws + w.attn_yield);
    c->attn_pass_state = c->attn_yield_flag + 1;
    c->attn_progress = reinterpret_cast<int *>(c->ws + w.attn_yield + 256);
    c->yield_host = nullptr;
    c->attn_launch_seq = 0;
    c->attn_slice = 0;
    c->attn_kv_prefetch = 0;
    c->yield_dirty = false;
    c->pass_open = false;
    c->pass_sliced = false;
    c->tm_pool_kind = 0;
    c->pass_grid = c->pass_merge_grid = c->pass_head_dim = 0;
    c->pass_smem = 0;
    c->plan_staging = nullptr;
    c->plan_inflight = false;
    c->tm_k_ptr = c->tm_v_ptr = nullptr;
    c->tm_layer_stride = c->tm_n_pages = 0;
    c->tm_kn_ptr = c->tm_vn_ptr = nullptr;
    c->tm_new_layer_stride = c->tm_new_rows = 0;
    c->tm_q_ptr = nullptr;
    c->tm_q_layer_stride = c->tm_q_rows = 0;
    // arrival counters start at zero and are reset by their last arriver
    cudaError_t e = cudaMemset(c->rd_counter, 0, sizeof(unsigned int) * (kRdMaxRows + 1));
    if (e == cudaSuccess) e = cudaMemset(c->attn_counters, 0, sizeof(unsigned int) * c->attn_counters_n);
    if (e == cudaSuccess) e = cudaMemset(c->ws + w.attn_yield, 0, 256 + sizeof(int) * kAttnMaxCtas);
    if (e == cudaSuccess) e = cudaMallocHost(reinterpret_cast<void **>(&c->yield_host), 2 * sizeof(unsigned int));
    if (e == cudaSuccess) {
        c->yield_host[0] = 0u;
        c->yield_host[1] = 0u;
    }
    if (e == cudaSuccess) e = cudaMallocHost(reinterpret_cast<void **>(&c->plan_staging), sizeof(AttnUnit) * c->max_units);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&c->plan_copied, cudaEventDisableTiming);
    if (e != cudaSuccess) {
        prepos_note_cuda_error(e, "ctx setup", __FILE__, __LINE__);
        if (c->plan_staging) cudaFreeHost(c->plan_staging);
        if (c->yield_host) cudaFreeHost(c->yield_host);
        delete c;
        return PREPOS_E_CUDA;
    }
    *out = c;
    return PREPOS_OK;
}

int prepos_ctx_destroy(prepos_ctx *ctx)
{
    if (!ctx) return PREPOS_E_INVALID_ARG;
    if (ctx->plan_inflight) cudaEventSynchronize(ctx->plan_copied);
    cudaEventDestroy(ctx->plan_copied);
    cudaFreeHost(ctx->plan_staging);
    cudaFreeHost(ctx->yield_host);
    delete ctx;
    return PREPOS_OK;
}

int prepos_ctx_sync(prepos_ctx *ctx, void *stream)
{
    if (!ctx) return PREPOS_E_INVALID_ARG;
    PREPOS_CUDA_TRY(cudaStreamSynchronize(static_cast<cudaStream_t>(stream)));
    PREPOS_CUDA_TRY(cudaGetLastError());
    return PREPOS_OK;
}

int64_t prepos_ctx_launch_count(const prepos_ctx *ctx) { return ctx ? ctx->launches : -1; }

int prepos_ctx_set_attn_path(prepos_ctx *ctx, int path)
{
    if (!ctx || path < 0 || path > 2) return PREPOS_E_INVALID_ARG;
    if (path == 2 && !prepos_attn_umma_supported(ctx) && !prepos_attn_umma_fp8_supported(ctx)) return PREPOS_E_SHAPE;
    ctx->attn_path = path;
    ctx->plan_key.clear();
    return PREPOS_OK;
}

}  // extern "C" (reopened below: the attention entry points share a host-side planner)

namespace {

// Host-side attention plan shared by the bf16 and the FP8 entry points: argument checks, Alg. 1 l.2-3 budget check
// (PAPER.md:145-146), one AttnUnit per (session, row chunk of `chunk_tok` entry tokens), cached on the batch
// geometry and uploaded to the ctx workspace when it changes.  `mode` separates plans of different kernels.
// `entries_in_cache`: the entry tokens are read from the session's pages like cached ones (the FP8 path appends
// their codes first), so a unit's tiles cover n_s + tok0 + ntok tokens and it has no entry tiles.
int plan_attn(prepos_ctx *ctx, int mode, int chunk_tok, bool entries_in_cache, int n_sessions, int page_table_stride,
              const int32_t *n_s, const int32_t *l_entry, const int32_t *capacity_tokens, int32_t *status_per_session,
              cudaStream_t stream)
{
    const prepos_model_shape &s = ctx->shape;
    std::vector<int32_t> key;
    key.reserve(3 * n_sessions + 3);
    key.push_back(mode);
    key.push_back(n_sessions);
    key.push_back(page_table_stride);   // the plan was checked against this stride
    for (int i = 0; i < n_sessions; ++i) {
        if (n_s[i] < 0 || l_entry[i] < 0 || capacity_tokens[i] < 0) return PREPOS_E_INVALID_ARG;
        key.push_back(n_s[i]);
        key.push_back(l_entry[i]);
        key.push_back(capacity_tokens[i]);
    }
    const bool reuse = (key == ctx->plan_key);
    if (!reuse) {
        std::vector<AttnUnit> units;
        int row0 = 0, prefix = 0;
        for (int i = 0; i < n_sessions; ++i) {
            const int L = l_entry[i];
            // Alg. 1 l.2-3: skip when the entry does not fit the cell-budget headroom
            const bool skip = L > capacity_tokens[i] - n_s[i];
            if (!skip && L > 0) {
                const int64_t need_pages = (static_cast<int64_t>(n_s[i]) + L + s.page_size - 1) / s.page_size;
                if (need_pages > page_table_stride) return PREPOS_E_INVALID_ARG;
                for (int tok0 = 0; tok0 < L; tok0 += chunk_tok) {
                    AttnUnit u;
                    memset(&u, 0, sizeof u);
                    u.session = i;
                    u.n_s = n_s[i];
                    u.l_entry = L;
                    u.tok0 = tok0;
                    u.ntok = (L - tok0 < chunk_tok) ? L - tok0 : chunk_tok;
                    u.row0 = row0;
                    if (entries_in_cache) {
                        u.n_load = n_s[i] + tok0 + u.ntok;
                        u.n_cached_tiles = (u.n_load + kAttnTileTokens - 1) / kAttnTileTokens;
                        u.n_tiles = u.n_cached_tiles;
                    } else {
                        u.n_load = n_s[i];
                        u.n_cached_tiles = (n_s[i] + kAttnTileTokens - 1) / kAttnTileTokens;
                        u.n_tiles = u.n_cached_tiles + (tok0 + u.ntok + kAttnTileTokens - 1) / kAttnTileTokens;
                    }
                    u.tile_prefix = prefix;
                    prefix += u.n_tiles;
                    units.push_back(u);
                }
            }
            row0 += L;
        }
        if (static_cast<int>(units.size()) > ctx->max_units) return PREPOS_E_WORKSPACE;
        if (ctx->plan_inflight) {
            PREPOS_CUDA_TRY(cudaEventSynchronize(ctx->plan_copied));
            ctx->plan_inflight = false;
        }
        ctx->plan_units.swap(units);
        ctx->plan_key.swap(key);
        if (!ctx->plan_units.empty()) {
            memcpy(ctx->plan_staging, ctx->plan_units.data(), sizeof(AttnUnit) * ctx->plan_units.size());
            PREPOS_CUDA_TRY(cudaMemcpyAsync(ctx->attn_units, ctx->plan_staging, sizeof(AttnUnit) * ctx->plan_units.size(),
                                            cudaMemcpyHostToDevice, stream));
            PREPOS_CUDA_TRY(cudaEventRecord(ctx->plan_copied, stream));
            ctx->plan_inflight = true;
        }
    }
    if (status_per_session)
        for (int i = 0; i < n_sessions; ++i)
            status_per_session[i] = (l_entry[i] > capacity_tokens[i] - n_s[i]) ? PREPOS_SKIPPED_BUDGET : PREPOS_OK;
    // The previous tcgen05 pass may have been stopped (a yield request, or a segment limit) and never resumed to its
    // end: this call abandons it, and its half-counted arrival counters must not reach the new pass's last-arriver
    // merge.  (The yield flag itself needs no clearing: it names the launch it stops, see prepos_ctx_request_yield.)
    if (ctx->yield_dirty || (ctx->pass_open && ctx->pass_sliced)) {
        PREPOS_CUDA_TRY(cudaMemsetAsync(ctx->attn_counters, 0, sizeof(unsigned int) * ctx->attn_counters_n, stream));
        ctx->yield_dirty = false;
    }
    ctx->pass_open = false;
    return PREPOS_OK;
}

}  // namespace

extern "C" {

int prepos_entry_attn(prepos_ctx *ctx, int layer_begin, int layer_end, int n_sessions, const void *q,
                      int64_t q_layer_stride, const void *k_new, const void *v_new, int64_t kv_new_layer_stride,
                      void *k_pool, void *v_pool, int64_t pool_layer_stride, int64_t n_pages,
                      const int32_t *page_table, int page_table_stride, const int32_t *n_s, const int32_t *l_entry,
                      const int32_t *capacity_tokens, void *out, int64_t out_layer_stride,
                      int32_t *status_per_session, float softmax_scale, void *stream)
{
    if (!ctx) return PREPOS_E_INVALID_ARG;
    const prepos_model_shape &s = ctx->shape;
    if (layer_begin < 0 || layer_end > s.layers || layer_begin > layer_end || n_sessions < 0) return PREPOS_E_INVALID_ARG;
    if (n_sessions > ctx->max_sessions) return PREPOS_E_WORKSPACE;
    if (n_sessions == 0 || layer_begin == layer_end) return PREPOS_OK;
    if (!q || !k_new || !v_new || !k_pool || !v_pool || !page_table || !n_s || !l_entry || !capacity_tokens || !out)
        return PREPOS_E_INVALID_ARG;
    if (!aligned16(q) || !aligned16(k_new) || !aligned16(v_new) || !aligned16(k_pool) || !aligned16(v_pool) ||
        !aligned16(out) || !aligned16(page_table))
        return PREPOS_E_ALIGN;
    if ((q_layer_stride | kv_new_layer_stride | pool_layer_stride | out_layer_stride) & 7) return PREPOS_E_ALIGN;
    if (n_pages <= 0 || page_table_stride <= 0) return PREPOS_E_INVALID_ARG;

    const int G = s.n_q_heads / s.n_kv_heads;
    const bool use_umma = (ctx->attn_path == 2) || (ctx->attn_path == 0 && prepos_attn_umma_supported(ctx));
    // row chunk: entry tokens whose G rows share one unit
    const int chunk_tok = use_umma ? (kAttnMaxRows / G > 0 ? kAttnMaxRows / G : 1) : (G > 16 ? 1 : 16 / G);
    const int st = plan_attn(ctx, use_umma ? 2 : 1, chunk_tok, false, n_sessions, page_table_stride, n_s, l_entry,
                             capacity_tokens, status_per_session, static_cast<cudaStream_t>(stream));
    if (st != PREPOS_OK) return st;
    if (ctx->plan_units.empty()) return PREPOS_OK;

    AttnArgs a;
    memset(&a, 0, sizeof a);
    a.layer_begin = layer_begin;
    a.layer_end = layer_end;
    a.n_units = static_cast<int>(ctx->plan_units.size());
    a.sum_rows = 0;
    for (int i = 0; i < n_sessions; ++i) a.sum_rows += l_entry[i];
    a.q = static_cast<const __nv_bfloat16 *>(q);
    a.k_new = static_cast<const __nv_bfloat16 *>(k_new);
    a.v_new = static_cast<const __nv_bfloat16 *>(v_new);
    a.k_pool = static_cast<__nv_bfloat16 *>(k_pool);
    a.v_pool = static_cast<__nv_bfloat16 *>(v_pool);
    a.out = static_cast<__nv_bfloat16 *>(out);
    a.q_layer_stride = q_layer_stride;
    a.kv_new_layer_stride = kv_new_layer_stride;
    a.pool_layer_stride = pool_layer_stride;
    a.out_layer_stride = out_layer_stride;
    a.n_pages = n_pages;
    a.page_table = page_table;
    a.page_table_stride = page_table_stride;
    a.scale = softmax_scale > 0.f ? softmax_scale : 1.0f / sqrtf(static_cast<float>(s.head_dim));
    if (use_umma) {
        const AttnUnit &last = ctx->plan_units.back();
        return prepos_launch_attn_umma(ctx, a, last.tile_prefix + last.n_tiles, static_cast<cudaStream_t>(stream));
    }
    return prepos_launch_attn_generic(ctx, a, static_cast<cudaStream_t>(stream));
}

int prepos_entry_attn_fp8(prepos_ctx *ctx, int layer_begin, int layer_end, int n_sessions, const void *q,
                          int64_t q_layer_stride, const void *k_new, const void *v_new, int64_t kv_new_layer_stride,
                          void *k_pool8, void *v_pool8, int64_t pool_layer_stride, int64_t n_pages,
                          const float *k_scale, const float *v_scale, int64_t scale_layer_stride,
                          const int32_t *page_table, int page_table_stride, const int32_t *n_s,
                          const int32_t *l_entry, const int32_t *capacity_tokens, void *out, int64_t out_layer_stride,
                          int32_t *status_per_session, float softmax_scale, void *stream)
{
    if (!ctx) return PREPOS_E_INVALID_ARG;
    const prepos_model_shape &s = ctx->shape;
    if (layer_begin < 0 || layer_end > s.layers || layer_begin > layer_end || n_sessions < 0) return PREPOS_E_INVALID_ARG;
    if (n_sessions > ctx->max_sessions) return PREPOS_E_WORKSPACE;
    if (n_sessions == 0 || layer_begin == layer_end) return PREPOS_OK;
    if (!q || !k_new || !v_new || !k_pool8 || !v_pool8 || !k_scale || !v_scale || !page_table || !n_s || !l_entry ||
        !capacity_tokens || !out)
        return PREPOS_E_INVALID_ARG;
    if (!aligned16(q) || !aligned16(k_new) || !aligned16(v_new) || !aligned16(k_pool8) || !aligned16(v_pool8) ||
        !aligned16(out) || !aligned16(page_table) || (reinterpret_cast<uintptr_t>(k_scale) & 3) ||
        (reinterpret_cast<uintptr_t>(v_scale) & 3))
        return PREPOS_E_ALIGN;
    if ((q_layer_stride | kv_new_layer_stride | out_layer_stride) & 7) return PREPOS_E_ALIGN;
    if (pool_layer_stride & 15) return PREPOS_E_ALIGN;
    if (s.head_dim % 16 != 0) return PREPOS_E_SHAPE;
    if (n_pages <= 0 || page_table_stride <= 0) return PREPOS_E_INVALID_ARG;

    const int G = s.n_q_heads / s.n_kv_heads;
    if (ctx->attn_path == 2 && !prepos_attn_umma_fp8_supported(ctx)) return PREPOS_E_SHAPE;
    const bool use_umma = (ctx->attn_path != 1) && prepos_attn_umma_fp8_supported(ctx);
    const int chunk_tok = use_umma ? (kAttnMaxRows / G > 0 ? kAttnMaxRows / G : 1) : (G > 16 ? 1 : 16 / G);
    const int st = plan_attn(ctx, use_umma ? 4 : 3, chunk_tok, true, n_sessions, page_table_stride, n_s, l_entry,
                             capacity_tokens, status_per_session, static_cast<cudaStream_t>(stream));
    if (st != PREPOS_OK) return st;
    if (ctx->plan_units.empty()) return PREPOS_OK;

    AttnArgs a;
    memset(&a, 0, sizeof a);
    a.layer_begin = layer_begin;
    a.layer_end = layer_end;
    a.n_units = static_cast<int>(ctx->plan_units.size());
    a.sum_rows = 0;
    for (int i = 0; i < n_sessions; ++i) a.sum_rows += l_entry[i];
    a.q = static_cast<const __nv_bfloat16 *>(q);
    a.k_new = static_cast<const __nv_bfloat16 *>(k_new);
    a.v_new = static_cast<const __nv_bfloat16 *>(v_new);
    a.k_pool8 = static_cast<uint8_t *>(k_pool8);
    a.v_pool8 = static_cast<uint8_t *>(v_pool8);
    a.k_scale = k_scale;
    a.v_scale = v_scale;
    a.scale_layer_stride = scale_layer_stride;
    a.out = static_cast<__nv_bfloat16 *>(out);
    a.q_layer_stride = q_layer_stride;
    a.kv_new_layer_stride = kv_new_layer_stride;
    a.pool_layer_stride = pool_layer_stride;
    a.out_layer_stride = out_layer_stride;
    a.n_pages = n_pages;
    a.page_table = page_table;
    a.page_table_stride = page_table_stride;
    a.scale = softmax_scale > 0.f ? softmax_scale : 1.0f / sqrtf(static_cast<float>(s.head_dim));
    const AttnUnit &last = ctx->plan_units.back();
    return prepos_launch_attn_fp8(ctx, a, use_umma, last.tile_prefix + last.n_tiles, static_cast<cudaStream_t>(stream));
}

int prepos_ctx_set_attn_slice(prepos_ctx *ctx, int max_segments_per_launch)
{
    if (!ctx || max_segments_per_launch < 0) return PREPOS_E_INVALID_ARG;
    ctx->attn_slice = max_segments_per_launch;
    return PREPOS_OK;
}

int prepos_ctx_set_kv_prefetch(prepos_ctx *ctx, int on)
{
    if (!ctx) return PREPOS_E_INVALID_ARG;
    ctx->attn_kv_prefetch = on ? 1 : 0;
    return PREPOS_OK;
}

int prepos_ctx_request_yield(prepos_ctx *ctx, void *stream)
{
    if (!ctx) return PREPOS_E_INVALID_ARG;
    if (!ctx->pass_open) return PREPOS_OK;   // no tcgen05 pass was issued on this ctx: nothing to stop
    ctx->yield_dirty = true;
    // The flag carries the sequence number of the launch it is meant for (the ctx's latest): the kernel stops only
    // when the flag equals its own number.  A copy that lands late -- after that launch has ended, because the
    // request's stream was backlogged -- therefore cannot stop a later pass or a resume, and nothing ever has to clear
    // the flag (a clear could itself race with a fresh request).  The pinned source word is read when the copy
    // executes; a newer request may have raised it by then, which only retargets the copy at the newer launch.
    ctx->yield_host[0] = ctx->attn_launch_seq;
    PREPOS_CUDA_TRY(cudaMemcpyAsync(ctx->attn_yield_flag, ctx->yield_host, sizeof(unsigned int), cudaMemcpyHostToDevice,
                                    static_cast<cudaStream_t>(stream)));
    return PREPOS_OK;
}

int prepos_entry_attn_pending(prepos_ctx *ctx, void *stream, int32_t *pending_out)
{
    if (!ctx || !pending_out) return PREPOS_E_INVALID_ARG;
    *pending_out = 0;
    if (!ctx->pass_open) return PREPOS_OK;
    PREPOS_CUDA_TRY(cudaMemcpyAsync(ctx->yield_host + 1, ctx->attn_pass_state, sizeof(unsigned int),
                                    cudaMemcpyDeviceToHost, static_cast<cudaStream_t>(stream)));
    PREPOS_CUDA_TRY(cudaStreamSynchronize(static_cast<cudaStream_t>(stream)));
    *pending_out = (ctx->yield_host[1] == ctx->attn_launch_seq) ? 1 : 0;
    return PREPOS_OK;
}

int prepos_entry_attn_resume(prepos_ctx *ctx, void *stream)
{
    if (!ctx) return PREPOS_E_INVALID_ARG;
    if (!ctx->pass_open) return PREPOS_OK;   // nothing to resume (no tcgen05 pass is open on this ctx)
    // the resume is a new launch with a new sequence number: the request that stopped its predecessor does not match it
    return prepos_resume_attn_umma(ctx, static_cast<cudaStream_t>(stream));
}

int prepos_ready_dist(prepos_ctx *ctx, int n, const int32_t *session_ids, const void *hidden, const void *w_vocab,
                      const int64_t *position_p, const uint64_t *entry_hash, const int32_t *skip_mask,
                      prepos_record *records, const uint64_t *session_version, const uint64_t *expected_version,
                      float *logits_out, void *stream)
{
    if (!ctx || n < 0) return PREPOS_E_INVALID_ARG;
    if (n == 0) return PREPOS_OK;
    if (!session_ids || !hidden || !w_vocab || !records || !session_version) return PREPOS_E_INVALID_ARG;
    if (!aligned16(hidden) || !aligned16(w_vocab) || !aligned16(records)) return PREPOS_E_ALIGN;
    return prepos_launch_ready_dist(ctx, n, session_ids, static_cast<const __nv_bfloat16 *>(hidden),
                                    static_cast<const __nv_bfloat16 *>(w_vocab), position_p, entry_hash, skip_mask,
                                    records, session_version, expected_version, logits_out,
                                    static_cast<cudaStream_t>(stream));
}

int prepos_ready_dist_w4(prepos_ctx *ctx, int n, const int32_t *session_ids, const void *hidden, const void *w4,
                         const void *w_scale, const int64_t *position_p, const uint64_t *entry_hash,
                         const int32_t *skip_mask, prepos_record *records, const uint64_t *session_version,
                         const uint64_t *expected_version, float *logits_out, void *stream)
{
    if (!ctx || n < 0) return PREPOS_E_INVALID_ARG;
    if (n == 0) return PREPOS_OK;
    if (!session_ids || !hidden || !w4 || !w_scale || !records || !session_version) return PREPOS_E_INVALID_ARG;
    if (!aligned16(hidden) || !aligned16(w4) || !aligned16(records) || (reinterpret_cast<uintptr_t>(w_scale) & 1))
        return PREPOS_E_ALIGN;
    return prepos_launch_ready_dist_w4(ctx, n, session_ids, static_cast<const __nv_bfloat16 *>(hidden),
                                       static_cast<const uint8_t *>(w4), static_cast<const __nv_bfloat16 *>(w_scale),
                                       position_p, entry_hash, skip_mask, records, session_version, expected_version,
                                       logits_out, static_cast<cudaStream_t>(stream));
}

int prepos_scan_logits(prepos_ctx *ctx, int n, const float *logits, prepos_record *out, void *stream)
{
    if (!ctx || n < 0) return PREPOS_E_INVALID_ARG;
    if (n == 0) return PREPOS_OK;
    if (!logits || !out) return PREPOS_E_INVALID_ARG;
    if (!aligned16(out)) return PREPOS_E_ALIGN;
    return prepos_launch_scan_logits(ctx, n, logits, out, static_cast<cudaStream_t>(stream));
}

int prepos_gate_serve(prepos_ctx *ctx, int n_requests, const int32_t *session_ids, const uint64_t *request_entry_hash,
                      const prepos_record *records, const uint64_t *session_version, const uint32_t *fast_set_bitmap,
                      float tau, int strict_gt, int32_t *decision_out, int32_t *token_out, void *stream)
{
    if (!ctx || n_requests < 0) return PREPOS_E_INVALID_ARG;
    if (n_requests == 0) return PREPOS_OK;
    if (!session_ids || !records || !session_version || !fast_set_bitmap || !decision_out || !token_out)
        return PREPOS_E_INVALID_ARG;
    if (!aligned16(records)) return PREPOS_E_ALIGN;
    return prepos_launch_gate_serve(ctx, n_requests, session_ids, request_entry_hash, records, session_version,
                                    fast_set_bitmap, tau, strict_gt, decision_out, token_out,
                                    static_cast<cudaStream_t>(stream));
}

int prepos_invalidate(prepos_ctx *ctx, int n, const int32_t *session_ids, uint64_t *session_version,
                      prepos_record *records, void *stream)
{
    if (!ctx || n < 0) return PREPOS_E_INVALID_ARG;
    if (n == 0) return PREPOS_OK;
    if (!session_ids || !session_version || !records) return PREPOS_E_INVALID_ARG;
    return prepos_launch_invalidate(ctx, n, session_ids, session_version, records, static_cast<cudaStream_t>(stream));
}

int prepos_gate_sweep(prepos_ctx *ctx, int n, const prepos_record *records, const uint64_t *session_version,
                      const uint32_t *fast_set_bitmap, const int32_t *full_path_token, int n_tau, const float *taus,
                      int strict_gt, prepos_sweep_point *out, void *stream)
{
    if (!ctx || n < 0 || n_tau < 0) return PREPOS_E_INVALID_ARG;
    if (n_tau == 0) return PREPOS_OK;
    if (!taus || !out || (n > 0 && (!records || !session_version || !fast_set_bitmap || !full_path_token)))
        return PREPOS_E_INVALID_ARG;
    if (!aligned16(records) || (reinterpret_cast<uintptr_t>(out) & 7)) return PREPOS_E_ALIGN;
    return prepos_launch_gate_sweep(ctx, n, records, session_version, fast_set_bitmap, full_path_token, n_tau, taus,
                                    strict_gt, out, static_cast<cudaStream_t>(stream));
}

int prepos_fastset_build(const int32_t *ids, int n, int V, uint32_t *bitmap_host)
{
    if (!bitmap_host || V <= 0 || n < 0 || (n > 0 && !ids)) return PREPOS_E_INVALID_ARG;
    const int words = (V + 31) / 32;
    memset(bitmap_host, 0, sizeof(uint32_t) * words);
    for (int i = 0; i < n; ++i) {
        if (ids[i] < 0 || ids[i] >= V) return PREPOS_E_INVALID_ARG;
        bitmap_host[ids[i] >> 5] |= 1u << (ids[i] & 31);
    }
    return PREPOS_OK;
}

}  // extern "C"
