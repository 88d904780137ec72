// common.cuh -- shared declarations of libprepos' translation units (CUDA side only; the CPU oracle
// under oracle/ shares nothing with this tree).
#pragma once

#include <cuda.h>
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include <vector>

#include "../../include/prepos.h"

static_assert(sizeof(prepos_record) == 48, "prepos_record must be 48 bytes");

#define PREPOS_CUDA_TRY(expr)                                  \
    do {                                                       \
        cudaError_t e_ = (expr);                               \
        if (e_ != cudaSuccess) {                               \
            prepos_note_cuda_error(e_, #expr, __FILE__, __LINE__); \
            return PREPOS_E_CUDA;                              \
        }                                                      \
    } while (0)

void prepos_note_cuda_error(cudaError_t e, const char *what, const char *file, int line);
void *prepos_get_encode_tiled();  // cuTensorMapEncodeTiled through the runtime's driver entry point (api.cu)

// Every libprepos kernel is launched with programmatic stream serialization: its prologue (barrier init, TMEM
// allocation, tensor-map prefetch, and -- for the LM head -- the first W_vocab stages, which no libprepos kernel
// writes) may overlap the tail of the previous libprepos kernel in the stream; each kernel executes
// griddepcontrol.wait before it touches anything a predecessor can have written.  After a kernel that never
// triggers early (anything that is not ours) the launch behaves exactly like an ordinary one.
template <typename... KArgs, typename... Args>
inline cudaError_t prepos_launch_pdl(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t stream,
                                     Args &&...args)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid;
    cfg.blockDim = block;
    cfg.dynamicSmemBytes = smem;
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kernel, static_cast<KArgs>(args)...);
}

constexpr int kMaxRdPartials = 1024;  // CTAs of a ready-dist launch (upper bound on its grid)
constexpr int kRdMaxRows = 128;       // hidden rows reduced by one ready-dist launch
constexpr int kAttnTileTokens = 128;  // KV tokens per tile of the tcgen05 attention kernel
constexpr int kAttnMaxRows = 256;     // query rows (G * entry tokens) per attention unit
constexpr int kAttnMaxCtas = 256;     // upper bound on the persistent attention grid (one CTA per SM: 148 on B200)

// per-CTA partial of the vocabulary reduction (a4): merged under the order (logit desc, id asc)
struct RdPartial {
    float m;   // running max
    float s;   // sum exp(l - m)
    float v1;  // best logit
    float v2;  // second best
    int32_t i1;
    int32_t i2;
    int32_t nonfinite;
    int32_t pad;
};
static_assert(sizeof(RdPartial) == 32, "RdPartial");

// one (session, row-chunk) of an attention call; (layer, kv head) are grid dimensions on top of it
struct AttnUnit {
    int32_t session;      // index in the call's batch
    int32_t n_s;          // cached tokens
    int32_t l_entry;      // entry tokens of the session
    int32_t tok0;         // first entry token of this row chunk
    int32_t ntok;         // entry tokens in this chunk (rows = ntok * G)
    int32_t row0;         // session's first row in the packed sum_L axis
    int32_t n_cached_tiles;  // ceil(n_s / tile)
    int32_t n_tiles;      // cached tiles + new-token tiles visible to this chunk
    int32_t tile_prefix;  // sum of n_tiles of the units before this one (within one (layer, head))
    int32_t n_load;       // tokens read from the session's pages: n_s, or n_s + tok0 + ntok when the entry tokens are
                          // read back from the cache they were appended to (FP8 path)
    int32_t pad[2];
};
static_assert(sizeof(AttnUnit) == 48, "AttnUnit");

struct prepos_ctx {
    prepos_model_shape shape;
    int max_sessions;
    int device;
    int num_sms;
    int cc_major, cc_minor;
    char *ws;
    size_t ws_bytes;
    int64_t launches;
    int attn_path;
    // workspace carve-up (device pointers into ws)
    RdPartial *rd_partials;    // [kRdMaxRows][kMaxRdPartials]
    unsigned int *rd_counter;  // arrival counter of the cross-CTA pass (self-resetting)
    AttnUnit *attn_units;      // device copy of the plan
    int max_units;
    float *attn_partials;      // [2 * kAttnMaxCtas] slots of kAttnMaxRows * (d + 2) floats
    unsigned int *attn_counters;  // [layers * Hkv * max_units] arrival counters (self-resetting)
    size_t attn_counters_n;
    // yield / resume of the tcgen05 attention pass (prepos_ctx_request_yield, prepos_entry_attn_resume)
    unsigned int *attn_yield_flag;   // device word polled by the persistent CTAs: the launch_seq of the launch to stop
    unsigned int *attn_pass_state;   // device word: launch_seq of the last launch that stopped early
    int *attn_progress;              // device [kAttnMaxCtas]: segments completed per CTA
    unsigned int *yield_host;        // pinned: [0] = source of the flag copy (a launch_seq), [1] = read-back of pass_state
    unsigned int attn_launch_seq;
    int attn_slice;                  // > 0: at most this many segments per CTA and launch
    int attn_kv_prefetch;            // 1: cached K/V tiles may be requested before the previous kernel has ended
    bool yield_dirty;                // a yield was requested since the arrival counters were last cleared
    bool pass_sliced;                // the last tcgen05 launch ran with a segment limit (it may have stopped early)
    bool pass_open;                  // the last attention call was a tcgen05 launch that can be resumed
    std::vector<unsigned char> pass_params;   // its kernel parameters
    int pass_grid, pass_merge_grid, pass_head_dim;
    bool pass_fp8;
    size_t pass_smem;
    // host-side plan cache
    std::vector<AttnUnit> plan_units;
    std::vector<int32_t> plan_key;
    AttnUnit *plan_staging;  // pinned host staging for the H2D plan copy
    cudaEvent_t plan_copied;
    bool plan_inflight;
    // TMA descriptor cache for the KV pools
    void *tm_k_ptr, *tm_v_ptr;
    int tm_pool_kind;                // 0 none, 1 bf16 pools (5-D map), 2 e4m3 pools (3-D byte map)
    int64_t tm_layer_stride, tm_n_pages;
    CUtensorMap tm_k, tm_v;
    // ... and for the call's entry K/V
    const void *tm_kn_ptr, *tm_vn_ptr;
    int64_t tm_new_layer_stride, tm_new_rows;
    CUtensorMap tm_kn, tm_vn;
    // ... and for the call's Q
    const void *tm_q_ptr;
    int64_t tm_q_layer_stride, tm_q_rows;
    CUtensorMap tm_q;
};

// ---- per-file launchers (all return a PREPOS_* status) -------------------------------------------
int prepos_launch_ready_dist(prepos_ctx *ctx, int n, const int32_t *session_ids, const __nv_bfloat16 *hidden,
                             const __nv_bfloat16 *w, const int64_t *position_p, const uint64_t *entry_hash,
                             const int32_t *skip_mask, prepos_record *records, const uint64_t *session_version,
                             const uint64_t *expected_version, float *logits_out, cudaStream_t stream);
int prepos_launch_ready_dist_w4(prepos_ctx *ctx, int n, const int32_t *session_ids, const __nv_bfloat16 *hidden,
                                const uint8_t *w4, const __nv_bfloat16 *w_scale, const int64_t *position_p,
                                const uint64_t *entry_hash, const int32_t *skip_mask, prepos_record *records,
                                const uint64_t *session_version, const uint64_t *expected_version, float *logits_out,
                                cudaStream_t stream);
int prepos_launch_scan_logits(prepos_ctx *ctx, int n, const float *logits, prepos_record *out, cudaStream_t stream);
int prepos_launch_gate_serve(prepos_ctx *ctx, int n, const int32_t *session_ids, const uint64_t *req_hash,
                             const prepos_record *records, const uint64_t *session_version,
                             const uint32_t *bitmap, float tau, int strict_gt, int32_t *decision, int32_t *token,
                             cudaStream_t stream);
int prepos_launch_gate_sweep(prepos_ctx *ctx, int n, const prepos_record *records, const uint64_t *session_version,
                             const uint32_t *bitmap, const int32_t *full_path_token, int n_tau, const float *taus,
                             int strict_gt, prepos_sweep_point *out, cudaStream_t stream);
int prepos_launch_invalidate(prepos_ctx *ctx, int n, const int32_t *session_ids, uint64_t *session_version,
                             prepos_record *records, cudaStream_t stream);

struct AttnArgs {
    int layer_begin, layer_end, n_units;
    int sum_rows;  // rows of the packed sum_L axis of q / k_new / v_new / out
    const __nv_bfloat16 *q, *k_new, *v_new;
    __nv_bfloat16 *k_pool, *v_pool, *out;
    int64_t q_layer_stride, kv_new_layer_stride, pool_layer_stride, out_layer_stride, n_pages;
    const int32_t *page_table;
    int page_table_stride;
    float scale;
    // FP8 (e4m3) KV cache, reading Q20: code pools [layer][n_pages][Hkv][page][d] uint8 (layer stride in
    // bytes = pool_layer_stride) and one fp32 scale per (layer, page, kv head) for K and for V
    uint8_t *k_pool8, *v_pool8;
    const float *k_scale, *v_scale;
    int64_t scale_layer_stride;
};
int prepos_launch_attn_fp8(prepos_ctx *ctx, const AttnArgs &a, bool use_umma, int total_tiles_per_lh, cudaStream_t stream);
int prepos_launch_attn_generic(prepos_ctx *ctx, const AttnArgs &a, cudaStream_t stream);
int prepos_launch_attn_umma(prepos_ctx *ctx, const AttnArgs &a, int total_tiles_per_lh, cudaStream_t stream);
int prepos_resume_attn_umma(prepos_ctx *ctx, cudaStream_t stream);
bool prepos_attn_umma_fp8_supported(const prepos_ctx *ctx);
int prepos_launch_attn_umma_fp8(prepos_ctx *ctx, const AttnArgs &a, int total_tiles_per_lh, cudaStream_t stream);
bool prepos_attn_umma_supported(const prepos_ctx *ctx);
