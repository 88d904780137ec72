/*
 * prepos.h -- C ABI of libprepos: the data-parallel hot path of speculative pre-positioning
 * (arxiv/paper_2606_29565; citations are PAPER.md:<line> of the paper text) on one B200 (sm_100a).
 *
 * The calls follow the paper's problem statement (Alg. 1 PAPER.md:140-164,
 * Alg. 2, Sec. 3.6):
 *
 *   prepos_entry_attn   Alg. 1 l.2-6: budget check, Append(E), attention part of Forward(E)
 *   prepos_ready_dist   Alg. 1 l.6 (LM head at the last entry position) + l.10-12 (record)
 *                       + Alg. 2 l.3-4 (Top2, gamma, argmax) moved to pre-position time
 *   prepos_scan_logits  Alg. 2 l.3-4 on a stored logit vector: the serve-time T_scan(V), Eq. 3
 *   prepos_gate_serve   Alg. 2, batched: validity/eligibility, Eq. 12 gate, serve or fall through
 *   prepos_invalidate   Sec. 3.6: version bump + valid clear in the step that mutates the state
 *
 * Conventions
 *   - Every call returns an int status: 0 = PREPOS_OK, > 0 informational, < 0 error.  No exceptions,
 *     no exit(), no memory handed to the caller.  prepos_strerror() names a status.
 *   - Pointers marked DEVICE are device pointers owned by the caller (16-byte aligned); pointers marked
 *     HOST are ordinary host memory, read (or written) before the call returns.  The library never
 *     allocates, frees, evicts or resizes caller memory ("skips the pre-position rather
 *     than evicting live state").  It owns only the opaque prepos_ctx, whose device scratch is the
 *     caller-supplied workspace.
 *   - Launches are asynchronous on `stream` (a cudaStream_t passed as void*; NULL = the legacy default
 *     stream) and stream-ordered with each other.  An asynchronous CUDA fault surfaces as PREPOS_E_CUDA
 *     on a later call or on prepos_ctx_sync().
 *   - Kernels are launched with programmatic dependent launch: a kernel's prologue may overlap the tail of the
 *     previous libprepos kernel in the stream, and prepos_ready_dist starts fetching w_vocab before its
 *     predecessor has finished.  Everything a libprepos call can write (pools, out, records, versions,
 *     decisions) is read only after the predecessor has completed; w_vocab, fast_set_bitmap and page_table are
 *     inputs no libprepos call writes, and must not be written by a caller's kernel that itself triggers
 *     dependent launches early and is still running when the call is issued.  After any ordinary kernel, copy
 *     or event the calls behave as plain stream-ordered launches.
 *   - The persistent kernels leave registers and shared memory for one small block per SM, so that a
 *     prepos_gate_serve issued on a higher-priority stream runs beside a pre-position pass instead of behind it
 *     (PAPER.md:132, 144).
 *   - Record publication (Sec. 3.6: a cached distribution is never served after the state
 *     changed).  A record may be re-published (prepos_ready_dist) or invalidated (prepos_invalidate) on one stream
 *     while prepos_gate_serve reads it on another.  Writer: flags <- next sequence number with VALID clear; fence;
 *     payload incl. the version stamp; fence; flags <- sequence | VALID.  Reader: word 1 (gap, flags, version); fence;
 *     words 0 and 2; fence; word 1 again -- any difference means a publication was in progress and the request falls
 *     through (PREPOS_STALE_OR_INVALID); then the live session version is read and compared with the stamp.  A serve
 *     therefore returns top1 and gap of ONE publication, stamped with the version that was live when the serve read
 *     it.  One writer per record at a time: two prepos_ready_dist calls for the same session must be stream-ordered.
 *     Pass expected_version to prepos_ready_dist whenever a mutation can commit (on any stream) while the
 *     pre-position is running: the record is stamped with the version its inputs were computed at, never with a
 *     later one.
 *   - bf16 tensors are raw 16-bit patterns (void*).  All accumulation and every record field is fp32.
 *   - A ctx is not thread-safe; use one ctx per host thread / stream.
 */
#ifndef PREPOS_H_
#define PREPOS_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define PREPOS_VERSION 101 /* 0.1.1: bumped whenever a signature, a struct or a status code changes; the Python
                              * binding refuses a library whose prepos_version() differs from the one it was written for */

/* status codes */
enum {
    PREPOS_OK = 0,
    PREPOS_SKIPPED_BUDGET = 1, /* Alg. 1 l.2-3: L_entry > headroom; nothing was touched */
    PREPOS_E_INVALID_ARG = -1,
    PREPOS_E_SHAPE = -2,     /* shape outside what the kernels support (see prepos_ctx_create) */
    PREPOS_E_ALIGN = -3,     /* a device pointer or stride is not 16-byte aligned */
    PREPOS_E_CUDA = -4,      /* a CUDA runtime/driver call or an earlier kernel failed */
    PREPOS_E_WORKSPACE = -5, /* the workspace given to prepos_ctx_create is too small for this call */
    PREPOS_E_NO_DEVICE = -6, /* no sm_100 device / driver: there is no CPU fallback */
    PREPOS_E_FIXED_SCRATCH = -7 /* the request exceeds the built-in scratch of a no-allocation entry point */
};

/* serve decisions written by prepos_gate_serve (Alg. 2) */
enum {
    PREPOS_SERVED = 0,           /* l.6: one cached token returned, scheduler bypassed */
    PREPOS_GAP_BELOW_TAU = 1,    /* l.9: gamma < tau (or <= tau when strict) */
    PREPOS_NOT_IN_FAST_SET = 2,  /* l.9: argmax not in A */
    PREPOS_STALE_OR_INVALID = 3, /* l.1-2: no valid record for the live state version */
    PREPOS_INELIGIBLE = 4        /* l.1-2: realised entry != pre-positioned entry */
};

/* record flag bits; bits 2..31 of `flags` hold the publication sequence number (see "Record publication") */
#define PREPOS_FLAG_VALID 1u     /* Alg. 1 l.12 decoded/valid */
#define PREPOS_FLAG_NONFINITE 2u /* a logit was NaN/Inf: never served */
#define PREPOS_FLAG_MASK 3u

typedef struct prepos_ctx prepos_ctx;

typedef struct {
    int32_t layers;     /* KV layers */
    int32_t n_q_heads;  /* Hq */
    int32_t n_kv_heads; /* Hkv, divides Hq; query head h reads kv head h / (Hq/Hkv) */
    int32_t head_dim;   /* d: multiple of 8, <= 256.  d in {64,128} with page_size 16 takes the tcgen05 path */
    int32_t hidden;     /* H: multiple of 128 */
    int32_t vocab;      /* V >= 2 */
    int32_t page_size;  /* tokens per KV page (power of two, <= 128) */
} prepos_model_shape;

/*
 * The ready-distribution record kept on the session ("or only
 * (argmax, gamma) under the gate").  48 bytes, 16-byte aligned, one per session id.
 */
typedef struct {
    float max_logit;     /* l^(1) */
    float lse;           /* log sum_v exp(l_v), natural log */
    int32_t top1;        /* argmax(l_ready): ties -> lowest id */
    int32_t top2;        /* id of l^(2) under the order (logit desc, id asc) */
    float gap;           /* gamma = l^(1) - l^(2), Eq. 11 */
    uint32_t flags;      /* PREPOS_FLAG_* in bits 0-1, publication sequence number in bits 2-31 */
    uint64_t version;    /* session state version the record was computed at */
    uint64_t entry_hash; /* caller's hash of the pre-positioned entry tokens; 0 = relaxed match */
    int64_t position;    /* decision point p = n_s + L_entry, Eq. 1 */
} prepos_record;

const char *prepos_strerror(int status);
int prepos_version(void);

/* Bytes of device workspace a ctx needs to serve calls of up to max_sessions sessions per call. */
size_t prepos_workspace_bytes(const prepos_model_shape *shape, int max_sessions);

/*
 * Creates a context bound to the current CUDA device.  `workspace` (DEVICE, 256-byte aligned,
 * workspace_bytes >= prepos_workspace_bytes()) stays owned by the caller and must outlive the ctx.
 * Errors: PREPOS_E_NO_DEVICE, PREPOS_E_SHAPE, PREPOS_E_WORKSPACE, PREPOS_E_ALIGN, PREPOS_E_CUDA.
 */
int prepos_ctx_create(prepos_ctx **out, const prepos_model_shape *shape, int max_sessions,
                      void *workspace, size_t workspace_bytes);
int prepos_ctx_destroy(prepos_ctx *ctx);
/* cudaStreamSynchronize(stream) + report any pending asynchronous error. */
int prepos_ctx_sync(prepos_ctx *ctx, void *stream);
/* Number of libprepos kernels launched through this ctx since creation (for accounting). */
int64_t prepos_ctx_launch_count(const prepos_ctx *ctx);
/* Tuning knob: 0 = automatic; 1 = force the generic CUDA-core attention kernel; 2 = force tcgen05. */
int prepos_ctx_set_attn_path(prepos_ctx *ctx, int path);

/*
 * Alg. 1 l.2-6 for layers [layer_begin, layer_end) over a batch of sessions.
 *
 * For every session s, layer l, query head h and entry row i in [0, L_s): softmax over the cached
 * tokens j < n_s[s] (read through the page table) and the entry tokens j' <= i ("causal among
 * themselves") of (q_i . k_j) * scale, times V -- and the entry K/V are written into the session's
 * pages at positions n_s .. n_s+L_s-1 (Append(E), l.5).  The decision point is p = n_s + L_s (Eq. 1);
 * the caller advances its own n_s after the call.
 *
 * q, out     DEVICE bf16 [layer][sum_L][Hq][d]; rows of session s start at sum_{t<s} L_t; layer l at
 *            base + l * q_layer_stride elements (out: out_layer_stride)
 * k_new,v_new DEVICE bf16 [layer][sum_L][Hkv][d], layer stride kv_new_layer_stride elements
 * k_pool,v_pool DEVICE bf16 [layer][n_pages][Hkv][page_size][d], layer stride pool_layer_stride elements
 * page_table DEVICE int32 [n_sessions][page_table_stride]: physical page of logical page t of session s
 * n_s, l_entry, capacity_tokens  HOST int32 [n_sessions]: cached tokens, entry tokens, tokens the
 *            session's pages can hold (cell budget: headroom B = capacity - n_s)
 * status_per_session HOST int32 [n_sessions] (nullable): PREPOS_OK or PREPOS_SKIPPED_BUDGET.  A skipped
 *            session has no side effect at all: its pages and its rows of `out` are untouched.
 * softmax_scale  <= 0 means 1/sqrt(d)
 *
 * Returns PREPOS_OK (also when some sessions were skipped) or an error; on error nothing was launched.
 */
int prepos_entry_attn(prepos_ctx *ctx, int layer_begin, int layer_end, int n_sessions,
                      const void *q, int64_t q_layer_stride,
                      const void *k_new, const void *v_new, int64_t kv_new_layer_stride,
                      void *k_pool, void *v_pool, int64_t pool_layer_stride, int64_t n_pages,
                      const int32_t *page_table, int page_table_stride,
                      const int32_t *n_s, const int32_t *l_entry, const int32_t *capacity_tokens,
                      void *out, int64_t out_layer_stride,
                      int32_t *status_per_session, float softmax_scale, void *stream);

/*
 * Early KV streaming for the one-launch-per-layer schedule.  By default every access of a prepos_entry_attn launch
 * waits for the previous kernel in the stream to end (programmatic dependent launch).  With on = 1 the launch may
 * request the CACHED K/V tiles (positions < n_s of the call's layers) as soon as its CTAs are resident -- while the
 * previous layer's merge is still running -- and only Q, the entry K/V, the appends and the outputs wait.  The
 * caller guarantees that no kernel still running when the call is issued writes those cached tokens or the page
 * table: true between the layers of one pass (layer l's launch appends to layer l's pages only), NOT true for a call
 * that reads what the call right before it appended (a delta resume on the same layers: leave it off or put any
 * ordinary operation in between).  Applies to the bf16 tcgen05 path.
 */
int prepos_ctx_set_kv_prefetch(prepos_ctx *ctx, int on);

/*
 * prepos_entry_attn over an FP8 KV cache (the paper's headline model "runs at 4-bit
 * precision", without naming a storage format: DESIGN.md reading Q20).  Same call, same budget
 * check, same outputs; the session's pages hold OCP e4m3 codes (1-4-3, bias 7, no infinities, max 448):
 *   k_pool8, v_pool8  DEVICE uint8 [layer][n_pages][Hkv][page_size][d], layer stride pool_layer_stride BYTES (a
 *                     multiple of 16); d a multiple of 16
 *   k_scale, v_scale  DEVICE fp32 [layer][n_pages][Hkv], layer stride scale_layer_stride elements: one positive scale
 *                     per (layer, page, kv head), caller-owned, for EVERY page of the session including the ones the
 *                     entry is appended to; cached value = decode(code) * scale
 * Append(E) (Alg. 1 l.5) stores code = e4m3(fp32(x) / scale), division and conversion round-to-nearest-even,
 * saturating at +-448, for every entry token; Forward(E) (l.6) runs after it, so entry row i sees the entry tokens
 * j' <= i through their stored codes (pre-positioning L1 then L2 tokens equals pre-positioning L1 + L2).  q, k_new,
 * v_new and out stay bf16; softmax and accumulation are fp32 as in prepos_entry_attn.
 */
int prepos_entry_attn_fp8(prepos_ctx *ctx, int layer_begin, int layer_end, int n_sessions,
                          const void *q, int64_t q_layer_stride,
                          const void *k_new, const void *v_new, int64_t kv_new_layer_stride,
                          void *k_pool8, void *v_pool8, int64_t pool_layer_stride, int64_t n_pages,
                          const float *k_scale, const float *v_scale, int64_t scale_layer_stride,
                          const int32_t *page_table, int page_table_stride,
                          const int32_t *n_s, const int32_t *l_entry, const int32_t *capacity_tokens,
                          void *out, int64_t out_layer_stride,
                          int32_t *status_per_session, float softmax_scale, void *stream);

/*
 * Yield and resume ("runs at the lowest scheduling priority and yields
 * immediately", Alg. 1 l.1, Eq. 7).  The tcgen05 attention pass is a persistent kernel that
 * holds every SM; a request that needs whole SMs (the fall-through decode step, Eq. 5) would wait for it to end.
 * Its CTAs therefore have a yield point at every segment boundary (a segment = the CTA's part of one
 * (layer, kv head, session row chunk), at most n_s / 128 + 1 KV tiles):
 *
 *   prepos_ctx_request_yield   asks the ctx's LATEST tcgen05 attention launch to stop: a 4-byte copy on `stream` (use
 *                              the request's high-priority stream; the copy engine does not wait for the running
 *                              kernel) writes that launch's sequence number into the ctx's device yield word.  Every
 *                              CTA of that launch re-reads the word at least every 8 KV tiles, finishes its current
 *                              segment, records how many segments it has completed, and exits; the SMs go to whatever
 *                              is queued at higher priority.  Outputs of finished segments are final, partials of cut
 *                              units stay in the ctx workspace.  A request only ever stops the launch it names: one
 *                              that lands after that launch has ended is inert (it cannot stop a later call or a
 *                              resume).  PREPOS_OK without a copy when the ctx has no tcgen05 launch to stop.
 *   prepos_entry_attn_resume   re-issues the SAME launch on `stream` under a new sequence number: every CTA skips the
 *                              segments it completed and carries on.  The result is the one an uninterrupted call
 *                              gives, bit for bit (same plan, same split, same merge order).  A no-op launch when
 *                              the pass had already finished; PREPOS_OK without a launch when nothing is open.
 *   prepos_entry_attn_pending  synchronises `stream` and tells whether the ctx's last attention launch stopped at a
 *                              yield point (1) or ran to completion (0).
 *   prepos_ctx_set_attn_slice  n > 0: every launch (the first and each resume) runs at most n segments per CTA --
 *                              a bounded-residency pass for callers that prefer time slices to a flag; 0 = off.
 *
 * Between a yield and its resume the ctx must not be given another prepos_entry_attn call (it would reuse the
 * workspace the stopped pass still needs; doing so abandons the stopped pass -- whether it was stopped by a request or
 * by a segment limit -- and the new call starts from clean arrival counters), and nothing queued behind the
 * stopped launch on its stream may read `out`.  Request a yield only while no further attention call of this ctx is
 * queued behind the running one.  The generic CUDA-core path has no yield point (its CTAs are short-lived).
 */
int prepos_ctx_request_yield(prepos_ctx *ctx, void *stream);
int prepos_entry_attn_resume(prepos_ctx *ctx, void *stream);
int prepos_entry_attn_pending(prepos_ctx *ctx, void *stream, int32_t *pending_out /* HOST */);
int prepos_ctx_set_attn_slice(prepos_ctx *ctx, int max_segments_per_launch);

/*
 * Alg. 1 l.6 (LM head) + l.10-12 and Alg. 2 l.3-4 (Eq. 11):
 * logits l_v = sum_k W[v][k] x_r[k] for each of n hidden rows, reduced in the same pass to the
 * record {max, lse, top1, top2, gap} under the order (logit desc, id asc).  records[session_ids[r]]
 * is overwritten: version = expected_version[r], the state version the caller computed hidden row r at,
 * and the record is VALID only if that still equals session_version[session_ids[r]] when the pass ends (a
 * mutation that committed meanwhile, on any stream, leaves it invalid: Sec. 3.6).  With expected_version
 * NULL the live version at the end of the pass is stamped, which is right only when every mutation of the
 * session is stream-ordered with this call.  flags = VALID (| NONFINITE) plus the publication sequence,
 * position = position_p[r] (0 if NULL), entry_hash likewise.
 * skip_mask (DEVICE int32 [n], nullable): rows with a non-zero entry are left untouched (sessions
 * whose pre-position was skipped on budget; their record is NOT made valid).
 *
 * hidden DEVICE bf16 [n][H]; w_vocab DEVICE bf16 [V][H] row-major; session_ids DEVICE int32 [n];
 * position_p DEVICE int64 [n] nullable; entry_hash DEVICE uint64 [n] nullable;
 * records DEVICE (indexed by session id); session_version DEVICE uint64 (indexed by session id);
 * expected_version DEVICE uint64 [n] nullable;
 * logits_out DEVICE fp32 [n][V] nullable (the full ready distribution).
 */
int prepos_ready_dist(prepos_ctx *ctx, int n, const int32_t *session_ids,
                      const void *hidden, const void *w_vocab,
                      const int64_t *position_p, const uint64_t *entry_hash, const int32_t *skip_mask,
                      prepos_record *records, const uint64_t *session_version,
                      const uint64_t *expected_version, float *logits_out, void *stream);

/*
 * prepos_ready_dist over a 4-bit W_vocab (the paper's headline model "runs at 4-bit
 * precision", without naming a format: DESIGN.md reading Q21).  Same record, same stamping and
 * publication, same optional logits_out as prepos_ready_dist; only the weights differ:
 *   w4      DEVICE uint8 [V][H/2]: two's-complement int4 codes in -8..7, two per byte, the element with even k in the
 *           low nibble
 *   w_scale DEVICE bf16 [V][H/128]: one scale per (vocabulary row, group of 128 consecutive k)
 *   W[v][k] = code[v][k] * w_scale[v][k / 128]; l_v = sum_k W[v][k] x[k].  The kernel widens the codes exactly,
 *   accumulates each group in fp32 and multiplies the group sum by its scale: no weight is ever rounded.
 * The pass reads V*H/2 + V*H/64 bytes per 8 hidden rows (a batch of n rows takes ceil(n / 8) passes).
 */
int prepos_ready_dist_w4(prepos_ctx *ctx, int n, const int32_t *session_ids,
                         const void *hidden, const void *w4, const void *w_scale,
                         const int64_t *position_p, const uint64_t *entry_hash, const int32_t *skip_mask,
                         prepos_record *records, const uint64_t *session_version,
                         const uint64_t *expected_version, float *logits_out, void *stream);

/*
 * Alg. 2 l.3-4 on stored logits (the paper's serve-time vocabulary scan, Eq. 3):
 * out[r] gets max_logit, lse, top1, top2, gap and the NONFINITE flag from logits[r][0..V); the other
 * fields of out[r] (version, entry_hash, position, VALID bit) are left as they are.
 * logits DEVICE fp32 [n][V]; out DEVICE [n].
 */
int prepos_scan_logits(prepos_ctx *ctx, int n, const float *logits, prepos_record *out, void *stream);

/*
 * prepos_scan_logits for callers that cannot allocate device memory.
 *
 * Who that is.  The scan is the serve-time fast path (Alg. 2 l.3-4; T_scan(V), Eq. 3):
 * it runs inside a serving engine's request handler.  Such an engine has normally handed all of the GPU's memory to
 * its own pool (weights + KV cache) at start-up, so a cudaMalloc from a plug-in either fails or, when it succeeds,
 * stalls every stream of the device while the driver maps the memory -- on the one path the paper wants at ~1 ms.
 * The same holds for a component that is loaded into a process it does not own and has no say over that process's
 * allocator.  Every other libprepos call needs a prepos_ctx, and a ctx needs a caller-allocated device workspace (and
 * creates pinned host buffers); this call needs neither.
 *
 * What it does instead.  The kernel's scratch -- one 32-byte partial per (row, CTA) and one arrival counter per row
 * for its single cross-CTA pass -- is a fixed array inside the library image:
 * PREPOS_SCAN_NOALLOC_SCRATCH_BYTES (65 792) bytes of device memory on every GPU that loads libprepos, held until the
 * process exits whether or not this call is ever made.  The call itself issues one 4*n-byte cudaMemsetAsync and one
 * kernel on `stream`; it calls no cudaMalloc / cudaFree / cudaMallocHost and no library routine that allocates.
 *
 * Limits (the price of a fixed array): n <= PREPOS_SCAN_NOALLOC_MAX_ROWS and vocab <= PREPOS_SCAN_NOALLOC_MAX_VOCAB,
 * otherwise PREPOS_E_FIXED_SCRATCH and nothing is launched; larger batches belong to prepos_scan_logits.
 *
 * Result: exactly what prepos_scan_logits writes -- out[r] gets max_logit, lse, top1, top2, gap and the NONFINITE
 * flag of logits[r][0..vocab), the other fields of out[r] are left as they are.
 *
 * First call on a device.  The first call made while a given device is current looks up the array's device address
 * (cudaGetSymbolAddress, which also makes the CUDA runtime load the library's kernels onto that device) and checks
 * that the device is sm_100; the address is kept for later calls.  Make that first call during start-up, on every
 * device you will use, before any stream capture begins.  Later calls do no set-up.
 *
 * Sharing.  There is ONE array per GPU and process, every call uses it, and it keeps the previous call's contents
 * (the call re-zeroes the counters it needs; the partials are overwritten before they are read).  Two calls that can
 * run on the same GPU at the same time -- different streams, different host threads -- race on it and may write wrong
 * records: order them (same stream, or an event between them).  Calls on different GPUs do not interact.
 *
 * logits DEVICE fp32 [n][vocab], 4-byte aligned; out DEVICE [n], 16-byte aligned; the current device must be the one
 * that owns them.  Errors: PREPOS_E_INVALID_ARG (n < 0, vocab < 2, null pointer), PREPOS_E_FIXED_SCRATCH,
 * PREPOS_E_ALIGN, PREPOS_E_NO_DEVICE, PREPOS_E_CUDA.
 */
#define PREPOS_SCAN_NOALLOC_MAX_ROWS 32
#define PREPOS_SCAN_NOALLOC_MAX_VOCAB (1 << 24)
#define PREPOS_SCAN_NOALLOC_SCRATCH_BYTES (256 + 32 * 64 * PREPOS_SCAN_NOALLOC_MAX_ROWS)
int prepos_scan_logits_noalloc(int n, int vocab, const float *logits, prepos_record *out, void *stream);

/*
 * Alg. 2, batched.  For request r on session sid = session_ids[r]:
 *   records[sid] not VALID, NONFINITE, or records[sid].version != session_version[sid] -> STALE_OR_INVALID
 *   both hashes non-zero and different                                               -> INELIGIBLE
 *   top1 not in A                                                                    -> NOT_IN_FAST_SET
 *   gap < tau (strict_gt: gap <= tau, the paper's Eq. 12 form)                        -> GAP_BELOW_TAU
 *   otherwise SERVED with token_out[r] = top1.  token_out[r] = -1 unless SERVED.
 * All arrays DEVICE (decision_out / token_out may be pinned host memory, which the device addresses directly: a lone
 * serve is then one launch and one sync, no copy).  request_entry_hash nullable (= all relaxed).  fast_set_bitmap: ceil(V/32) words,
 * bit (id & 31) of word (id >> 5).  The version compare is the authority (Sec. 3.6): a record whose
 * session was invalidated earlier in stream order is never served.
 */
int prepos_gate_serve(prepos_ctx *ctx, int n_requests, const int32_t *session_ids,
                      const uint64_t *request_entry_hash,
                      const prepos_record *records, const uint64_t *session_version,
                      const uint32_t *fast_set_bitmap, float tau, int strict_gt,
                      int32_t *decision_out, int32_t *token_out, void *stream);

/*
 * Sec. 3.6: for every listed session (ids may repeat; each occurrence is one
 * mutation) session_version[sid] += 1 and records[sid].flags &= ~VALID.  Call it on the stream, and
 * in the step, that performs the mutation; later serves on that stream see the bump.
 * session_ids DEVICE int32 [n]; session_version, records DEVICE.
 */
int prepos_invalidate(prepos_ctx *ctx, int n, const int32_t *session_ids,
                      uint64_t *session_version, prepos_record *records, void *stream);

/*
 * Risk-coverage sweep of the gate (Sec. 2.4, Eq. 13-14; the calibration measurement of
 * PAPER.md:254): for each threshold taus[t], over the n decision points records[0..n):
 *   accepted       = #{ i : records[i] VALID, finite, fresh (version == session_version[i]), top1 in A,
 *                        gap >= tau (strict_gt: gap > tau) }                       -- the numerator of c(tau), Eq. 13
 *   false_accepts  = #{ accepted i : records[i].top1 != full_path_token[i] }       -- the numerator of r(tau), Eq. 14
 *   coverage = accepted / n, far = false_accepts / accepted (0 when nothing is accepted), and the Wilson 95%
 *   score intervals of both ((0, 1) for an empty denominator), all in fp64.
 * "Calibration selects the smallest tau such that r(tau) <= r_max" is one pass of the caller over
 * out[].  records, session_version, fast_set_bitmap, full_path_token [n] int32, taus [n_tau] float and
 * out [n_tau] are DEVICE pointers; out is fully overwritten.  One CTA per threshold.
 */
typedef struct {
    float tau;
    int32_t n;
    int32_t accepted;
    int32_t false_accepts;
    double coverage, far;
    double cov_lo, cov_hi;
    double far_lo, far_hi;
} prepos_sweep_point; /* 64 bytes */

int prepos_gate_sweep(prepos_ctx *ctx, int n, const prepos_record *records, const uint64_t *session_version,
                      const uint32_t *fast_set_bitmap, const int32_t *full_path_token, int n_tau,
                      const float *taus, int strict_gt, prepos_sweep_point *out, void *stream);

/* HOST helper: A as a bitmap.  ids HOST int32 [n]; bitmap_host HOST uint32 [ceil(V/32)] (overwritten). */
int prepos_fastset_build(const int32_t *ids, int n, int V, uint32_t *bitmap_host);

#ifdef __cplusplus
}
#endif
#endif /* PREPOS_H_ */
