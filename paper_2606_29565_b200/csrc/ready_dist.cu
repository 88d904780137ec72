// ready_dist.cu -- a3 + a4: the last-position LM head fused with the vocabulary reduction into the
// ready-distribution record (Alg. 1 l.6, l.10-12; Top2/gamma/argmax of Alg. 2
// l.3-4, Eq. 11), plus a4' the standalone scan of stored logits
// (Eq. 3).
//
// The pass is a pure HBM stream of W_vocab [V][H] bf16 (1.05 GB at V=128256, H=4096).  Design:
//   * persistent CTAs, one per SM; CTA c owns the 128-row vocabulary tiles c, c+grid, ...
//   * one producer warp streams [128 rows x 128 cols] stages of W through a ring of shared-memory
//     buffers with TMA (cp.async.bulk.tensor, 128B swizzle) completing on mbarriers;
//   * eight consumer warps (16 rows each) read the swizzled tiles with ldmatrix and multiply them
//     with up to 8 hidden rows held in shared memory using warp-level bf16 MMA with fp32
//     accumulation.  The work is HBM-bound (2 flop/byte per hidden row): the tensor instruction is
//     used only to keep the instruction count per byte far below the issue limit, so that the
//     stream is never stalled by ALU work; it is not a tcgen05-class contraction.
//   * every lane keeps a running (top1, top2, max, sum-exp) state for the logits it produces, warp
//     shuffles reduce it, and a single cross-CTA pass by the last-arriving CTA merges the per-CTA
//     partials in CTA order under the total order (logit desc, id asc), so ids are independent of
//     the reduction tree.
#include <math_constants.h>

#include <mutex>

#include "common.cuh"
#include "ptx.cuh"

namespace {

constexpr int kTileRows = 128;
constexpr int kBoxCols = 64;                                  // 128 B of bf16: one swizzle span
constexpr int kStageCols = 128;                               // two TMA boxes per stage
constexpr int kBoxBytes = kTileRows * kBoxCols * 2;           // 16 KB
constexpr int kStageBytes = kTileRows * kStageCols * 2;       // 32 KB
constexpr int kConsumerWarps = 8;
constexpr int kThreads = (kConsumerWarps + 1) * 32;
constexpr int kNB = 8;       // hidden rows per pass (the n8 of m16n8k16)
constexpr int kXPad = 8;     // bf16 elements of row padding of the hidden rows in smem (bank spread)
constexpr int kMaxStages = 6;

struct Top2Lse {
    float v1, v2, m, s;
    int i1, i2;
    int nonfinite;
};

__device__ __forceinline__ Top2Lse t2_init()
{
    Top2Lse t;
    t.v1 = t.v2 = -CUDART_INF_F;
    t.i1 = t.i2 = 0x7fffffff;
    t.m = -CUDART_INF_F;
    t.s = 0.f;
    t.nonfinite = 0;
    return t;
}
// (logit desc, id asc): the one order used everywhere (reading Q8)
__device__ __forceinline__ bool t2_better(float va, int ia, float vb, int ib)
{
    return va > vb || (va == vb && ia < ib);
}
__device__ __forceinline__ void t2_insert(Top2Lse &t, float v, int i)
{
    if (t2_better(v, i, t.v1, t.i1)) {
        t.v2 = t.v1;
        t.i2 = t.i1;
        t.v1 = v;
        t.i1 = i;
    } else if (t2_better(v, i, t.v2, t.i2)) {
        t.v2 = v;
        t.i2 = i;
    }
}
__device__ __forceinline__ void t2_push(Top2Lse &t, float v, int i)
{
    if (!(fabsf(v) <= 3.0e38f)) t.nonfinite = 1;  // NaN or Inf
    t2_insert(t, v, i);
    if (v > t.m) {
        t.s = t.s * __expf(t.m - v) + 1.f;
        t.m = v;
    } else {
        t.s += __expf(v - t.m);
    }
}
__device__ __forceinline__ void t2_merge(Top2Lse &a, const Top2Lse &b)
{
    t2_insert(a, b.v1, b.i1);
    t2_insert(a, b.v2, b.i2);
    const float m = fmaxf(a.m, b.m);
    if (m > -CUDART_INF_F) {
        a.s = a.s * __expf(a.m - m) + b.s * __expf(b.m - m);
        a.m = m;
    }
    a.nonfinite |= b.nonfinite;
}
__device__ __forceinline__ Top2Lse t2_shfl_xor(const Top2Lse &t, int mask)
{
    Top2Lse o;
    o.v1 = __shfl_xor_sync(0xffffffffu, t.v1, mask);
    o.v2 = __shfl_xor_sync(0xffffffffu, t.v2, mask);
    o.m = __shfl_xor_sync(0xffffffffu, t.m, mask);
    o.s = __shfl_xor_sync(0xffffffffu, t.s, mask);
    o.i1 = __shfl_xor_sync(0xffffffffu, t.i1, mask);
    o.i2 = __shfl_xor_sync(0xffffffffu, t.i2, mask);
    o.nonfinite = __shfl_xor_sync(0xffffffffu, t.nonfinite, mask);
    return o;
}
__device__ __forceinline__ void t2_store(RdPartial *p, const Top2Lse &t)
{
    RdPartial r;
    r.m = t.m;
    r.s = t.s;
    r.v1 = t.v1;
    r.v2 = t.v2;
    r.i1 = t.i1;
    r.i2 = t.i2;
    r.nonfinite = t.nonfinite;
    r.pad = 0;
    *reinterpret_cast<uint4 *>(p) = *reinterpret_cast<uint4 *>(&r);
    *(reinterpret_cast<uint4 *>(p) + 1) = *(reinterpret_cast<uint4 *>(&r) + 1);
}
__device__ __forceinline__ Top2Lse t2_load(const RdPartial *p)
{
    // written by another CTA in this launch: read through L2
    const uint4 a = __ldcg(reinterpret_cast<const uint4 *>(p));
    const uint4 b = __ldcg(reinterpret_cast<const uint4 *>(p) + 1);
    Top2Lse t;
    t.m = __uint_as_float(a.x);
    t.s = __uint_as_float(a.y);
    t.v1 = __uint_as_float(a.z);
    t.v2 = __uint_as_float(a.w);
    t.i1 = static_cast<int>(b.x);
    t.i2 = static_cast<int>(b.y);
    t.nonfinite = static_cast<int>(b.z);
    return t;
}

// the record's reduction fields; version/hash/position/VALID are the caller's business
__device__ __forceinline__ void write_record_fields(prepos_record *rec, const Top2Lse &t)
{
    rec->max_logit = t.v1;
    rec->lse = t.m + __logf(t.s);
    rec->top1 = t.i1;
    rec->top2 = (t.i2 == 0x7fffffff) ? -1 : t.i2;
    rec->gap = (t.i2 == 0x7fffffff) ? CUDART_INF_F : t.v1 - t.v2;
}

struct RdParams {
    int n;  // hidden rows in this pass (<= kNB)
    int H, V;
    int n_stages;
    int x_rows;  // rows of the smem hidden block (n+1 with a trailing zero row, or 8)
    const __nv_bfloat16 *hidden;  // [n][H]
    const int32_t *session_ids;   // [n]
    const int64_t *position_p;
    const uint64_t *entry_hash;
    const int32_t *skip_mask;
    prepos_record *records;
    const uint64_t *session_version;
    const uint64_t *expected_version;  // [n] or null
    float *logits_out;  // [n][V] or null
    RdPartial *partials;
    unsigned int *counter;
};

// Alg. 1 l.10-12 for one session: publishes the record so that a gate serve on ANOTHER stream never pairs fields of
// two different publications (protocol in include/prepos.h "Record publication"): the upper 30 bits of `flags` are a
// sequence number.  (1) flags <- new sequence, VALID clear; fence; (2) payload incl. the version stamp; fence;
// (3) flags <- sequence | VALID.  The stamp is the version the caller computed the hidden row at (`expected`), and
// the record is made VALID only if that still is the live version (Sec. 3.6: a state mutation that commits while the
// pre-position is running must win); without `expected` the live version at this moment is stamped (same-stream use).
__device__ __forceinline__ void publish_record(const RdParams &p, int row, const Top2Lse &t)
{
    const int sid = p.session_ids[row];
    prepos_record *rec = p.records + sid;
    volatile uint32_t *fl = &rec->flags;
    const uint32_t seq = ((*fl >> 2) + 1u) << 2;
    *fl = seq;
    __threadfence();
    const uint64_t live = *reinterpret_cast<const volatile uint64_t *>(p.session_version + sid);
    const uint64_t stamp = p.expected_version ? p.expected_version[row] : live;
    write_record_fields(rec, t);
    rec->entry_hash = p.entry_hash ? p.entry_hash[row] : 0ull;
    rec->position = p.position_p ? p.position_p[row] : 0ll;
    rec->version = stamp;
    __threadfence();
    *fl = seq | (stamp == live ? PREPOS_FLAG_VALID : 0u) | (t.nonfinite ? PREPOS_FLAG_NONFINITE : 0u);
}

// Merge `n_parts` per-CTA partials of row `row` (partials[row * kMaxRdPartials + c]) in CTA order with one
// warp; result valid in lane 0.
__device__ __forceinline__ Top2Lse merge_partials_warp(const RdPartial *partials, int row, int n_parts, int lane)
{
    Top2Lse acc = t2_init();
    constexpr int kBatch = 5;  // 148 CTAs = 5 partials per lane: loaded together, merged in CTA order
    for (int c0 = lane; c0 < n_parts; c0 += 32 * kBatch) {
        Top2Lse part[kBatch];
#pragma unroll
        for (int j = 0; j < kBatch; ++j)
            if (c0 + 32 * j < n_parts) part[j] = t2_load(partials + static_cast<size_t>(row) * kMaxRdPartials + c0 + 32 * j);
#pragma unroll
        for (int j = 0; j < kBatch; ++j)
            if (c0 + 32 * j < n_parts) t2_merge(acc, part[j]);
    }
#pragma unroll
    for (int mask = 1; mask < 32; mask <<= 1) {
        const Top2Lse o = t2_shfl_xor(acc, mask);
        t2_merge(acc, o);
    }
    return acc;
}


// The single cross-CTA pass: the last CTA to arrive merges the per-CTA partials of every hidden row in CTA order
// and writes the records (Alg. 1 l.10-12: position, dist (here: argmax, gamma, max, lse), decoded/valid).
// Called by all threads of the CTA after their partials are stored (and fenced).
__device__ __forceinline__ void finalize_records(const RdParams &p, int warp, int lane, int n_warps)
{
    __shared__ int s_is_last;
    if (threadIdx.x == 0) {
        const unsigned int prev = atomicAdd(p.counter, 1u);
        s_is_last = (prev == gridDim.x - 1);
    }
    __syncthreads();
    if (!s_is_last) return;
    __threadfence();
    for (int row = warp; row < p.n; row += n_warps) {
        const Top2Lse t = merge_partials_warp(p.partials, row, gridDim.x, lane);
        if (lane == 0 && !(p.skip_mask && p.skip_mask[row])) publish_record(p, row, t);
    }
    if (threadIdx.x == 0) *p.counter = 0u;  // self-reset for the next launch on this stream
}

__global__ void __launch_bounds__(kThreads, 1)
ready_dist_kernel(const __grid_constant__ CUtensorMap tm_w, const RdParams p)
{
    extern __shared__ __align__(1024) uint8_t smem_raw[];
    // carve: [stages][32 KB] | x block | barriers | per-warp partials
    uint8_t *smem = reinterpret_cast<uint8_t *>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
    uint8_t *stage_base = smem;
    const int x_stride = p.H + kXPad;  // elements
    __nv_bfloat16 *xs = reinterpret_cast<__nv_bfloat16 *>(smem + static_cast<size_t>(p.n_stages) * kStageBytes);
    uint64_t *bars = reinterpret_cast<uint64_t *>(reinterpret_cast<uint8_t *>(xs) +
                                                  ((static_cast<size_t>(p.x_rows) * x_stride * 2 + 15) & ~size_t(15)));
    uint64_t *full_bar = bars;
    uint64_t *empty_bar = bars + kMaxStages;
    RdPartial *warp_part = reinterpret_cast<RdPartial *>(bars + 2 * kMaxStages);  // [kConsumerWarps][kNB]
    const int warp = threadIdx.x >> 5;
    const int lane = threadIdx.x & 31;
    const int n_tiles = (p.V + kTileRows - 1) / kTileRows;
    const int n_kc = p.H / kStageCols;

    if (threadIdx.x == 0) {
        for (int s = 0; s < p.n_stages; ++s) {
            ptx::mbar_init(ptx::smem_u32(&full_bar[s]), 1);
            ptx::mbar_init(ptx::smem_u32(&empty_bar[s]), kConsumerWarps);
        }
        ptx::fence_mbar_init();
    }
    __syncthreads();
    ptx::griddep_launch();

    if (warp == kConsumerWarps) {
        // ===== TMA producer =====  W_vocab is never written by a libprepos kernel: its first stages are fetched
        // while the previous kernel in the stream (the entry attention) is still draining
        if (lane == 0) {
            ptx::prefetch_tmap(&tm_w);
            const uint64_t pol = ptx::policy_evict_first();  // W is read once per pass
            int stage = 0;
            uint32_t phase = 0;
            for (int tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
                for (int kc = 0; kc < n_kc; ++kc) {
                    ptx::mbar_wait(ptx::smem_u32(&empty_bar[stage]), phase ^ 1);
                    const uint32_t fb = ptx::smem_u32(&full_bar[stage]);
                    ptx::mbar_arrive_expect_tx(fb, kStageBytes);
                    const uint32_t dst = ptx::smem_u32(stage_base + static_cast<size_t>(stage) * kStageBytes);
                    ptx::tma_load_2d(dst, &tm_w, fb, kc * kStageCols, tile * kTileRows, pol);
                    ptx::tma_load_2d(dst + kBoxBytes, &tm_w, fb, kc * kStageCols + kBoxCols, tile * kTileRows, pol);
                    if (++stage == p.n_stages) {
                        stage = 0;
                        phase ^= 1;
                    }
                }
            }
        }
        ptx::griddep_wait();  // the cross-CTA pass below reads and writes what earlier kernels own
    } else {
        // ===== consumers: 16 vocabulary rows per warp =====
        // hidden rows -> smem (row x_rows-1 is zero when n < 8; lanes of absent rows read it): the first access
        // to memory an earlier kernel may have written
        ptx::griddep_wait();
        {
            const int chunks_per_row = p.H / 8;
            for (int idx = threadIdx.x; idx < p.x_rows * chunks_per_row; idx += kConsumerWarps * 32) {
                const int r = idx / chunks_per_row, c = idx - r * chunks_per_row;
                uint4 v = make_uint4(0, 0, 0, 0);
                if (r < p.n) v = *reinterpret_cast<const uint4 *>(p.hidden + static_cast<size_t>(r) * p.H + c * 8);
                *reinterpret_cast<uint4 *>(xs + static_cast<size_t>(r) * x_stride + c * 8) = v;
            }
        }
        ptx::bar_sync(1, kConsumerWarps * 32);
        Top2Lse st[2];
        st[0] = t2_init();
        st[1] = t2_init();
        const int n0 = 2 * (lane & 3);  // this lane's two hidden rows (accumulator columns)
        // ldmatrix lane addressing.  A: matrices (r0-7,k0-7) (r8-15,k0-7) (r0-7,k8-15) (r8-15,k8-15)
        const int a_row = warp * 16 + (lane & 7) + ((lane >> 3) & 1) * 8;
        const int a_kc = lane >> 4;  // 16-byte chunk within the 32-byte k-step
        // B: matrices (k0-7) (k8-15) (k16-23) (k24-31), each 8 hidden rows x 16 B
        const int b_row = min(lane & 7, p.x_rows - 1);
        const uint32_t xs_lane = ptx::smem_u32(xs + static_cast<size_t>(b_row) * x_stride + (lane >> 3) * 8);

        int stage = 0;
        uint32_t phase = 0;
        for (int tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
            float acc[4] = {0.f, 0.f, 0.f, 0.f};
            for (int kc = 0; kc < n_kc; ++kc) {
                ptx::mbar_wait(ptx::smem_u32(&full_bar[stage]), phase);
                const uint32_t sbase = ptx::smem_u32(stage_base + static_cast<size_t>(stage) * kStageBytes);
#pragma unroll
                for (int box = 0; box < 2; ++box) {
                    const uint32_t abase = sbase + box * kBoxBytes + a_row * 128;
                    const uint32_t xk = xs_lane + (kc * kStageCols + box * kBoxCols) * 2;
#pragma unroll
                    for (int kk = 0; kk < 2; ++kk) {  // 32 columns = two k16 steps per B ldmatrix
                        uint32_t b0, b1, b2, b3;
                        ptx::ldmatrix_x4(xk + kk * 64, b0, b1, b2, b3);
#pragma unroll
                        for (int ks = 0; ks < 2; ++ks) {
                            const int chunk = (kk * 2 + ks) * 2 + a_kc;  // 16-byte chunk index in the 128-byte row
                            uint32_t a0, a1, a2, a3;
                            ptx::ldmatrix_x4(abase + ((chunk ^ (a_row & 7)) << 4), a0, a1, a2, a3);
                            ptx::mma_bf16_16816(acc, a0, a1, a2, a3, ks ? b2 : b0, ks ? b3 : b1);
                        }
                    }
                }
                __syncwarp();
                if (lane == 0) ptx::mbar_arrive(ptx::smem_u32(&empty_bar[stage]));
                if (++stage == p.n_stages) {
                    stage = 0;
                    phase ^= 1;
                }
            }
            // logits of rows v, v+8 for hidden rows n0, n0+1
            const int v = tile * kTileRows + warp * 16 + (lane >> 2);
#pragma unroll
            for (int j = 0; j < 2; ++j) {
                if (n0 + j < p.n) {
                    if (v < p.V) t2_push(st[j], acc[j], v);
                    if (v + 8 < p.V) t2_push(st[j], acc[2 + j], v + 8);
                    if (p.logits_out) {
                        float *lo = p.logits_out + static_cast<size_t>(n0 + j) * p.V;
                        if (v < p.V) lo[v] = acc[j];
                        if (v + 8 < p.V) lo[v + 8] = acc[2 + j];
                    }
                }
            }
        }
        // lanes sharing lane&3 hold the same hidden rows: reduce over lane bits 2..4
#pragma unroll
        for (int j = 0; j < 2; ++j) {
#pragma unroll
            for (int mask = 4; mask < 32; mask <<= 1) {
                const Top2Lse o = t2_shfl_xor(st[j], mask);
                t2_merge(st[j], o);
            }
        }
        if (lane < 4) {
            t2_store(&warp_part[warp * kNB + n0], st[0]);
            t2_store(&warp_part[warp * kNB + n0 + 1], st[1]);
        }
    }
    __syncthreads();
    // CTA partial per hidden row (fixed warp order), then the single cross-CTA pass
    if (threadIdx.x < p.n) {
        Top2Lse acc = t2_init();
        for (int w = 0; w < kConsumerWarps; ++w) {
            const RdPartial *q = &warp_part[w * kNB + threadIdx.x];
            Top2Lse t;
            t.m = q->m, t.s = q->s, t.v1 = q->v1, t.v2 = q->v2, t.i1 = q->i1, t.i2 = q->i2, t.nonfinite = q->nonfinite;
            t2_merge(acc, t);
        }
        t2_store(p.partials + static_cast<size_t>(threadIdx.x) * kMaxRdPartials + blockIdx.x, acc);
        __threadfence();
    }
    __syncthreads();
    finalize_records(p, warp, lane, kThreads / 32);
}

// ---- a3 + a4 over a 4-bit W_vocab (reading Q21) -----------
// w4 [V][H/2]: two's-complement int4 codes, two per byte (even k in the low nibble); w_scale [V][H/128] bf16, one
// per (vocabulary row, group of 128 consecutive k); W[v][k] = code * scale.  A quarter of the bytes of the bf16 pass
// (V*H/2 + V*H/64), so a quarter of its HBM time -- and four times the arithmetic per byte: the codes are widened
// to bf16 in registers (exact: |code| <= 8) and multiplied with the hidden rows by the same warp-level MMA, the
// fp32 sum of each 128-k group is scaled once (the scale never rounds a weight), and the record is reduced exactly
// as in ready_dist_kernel.
//   * one TMA box = one scale group of one vocabulary tile: [128 rows][64 B]; a stage = up to four boxes (512 k)
//   * thread (g, t) of a warp owns rows g, g+8 of the warp's 16 and the 16 bytes [16t, 16t+16) of each: word j of
//     them holds k = 32t + 8j + (0..7).  `(w >> 4i) & 0x000f000f` puts nibbles i and i+4 into the two halves of a
//     register, which is the A fragment (row g; MMA columns 2t, 2t+1) of one m16n8k16 -- so MMA column p stands for
//     k = 32t + 8j + {0,4 | 1,5} (first MMA of word j) or {2,6 | 3,7} (second).  The hidden rows are laid out in
//     shared memory in exactly that order when they are loaded, so one 16-byte read yields the B fragments of both.
constexpr int kW4BoxBytes = kTileRows * 64;               // 8 KB: 128 rows x 128 codes
constexpr int kW4BoxesPerStage = 4;
constexpr int kW4StageBytes = kW4BoxesPerStage * kW4BoxBytes;  // 32 KB
constexpr int kW4Group = 128;
constexpr int kW4XPad = 32;  // bf16 elements: the row stride of the hidden block is 64 B mod 128 B (bank spread)

// eight int4 codes (one 32-bit word) -> four bf16x2 registers holding (136 + code_i, 136 + code_{i+4}), exactly:
// ((w >> 4i) & 0x000f000f) ^ 0x43084308 flips the sign bit of each nibble (code + 8 in 0..15) and sets the bf16
// exponent of 128 around it -- one shift and one LOP3 per register.  The offset 136 is taken out of the group sum
// afterwards (sum_k (136 + c_k) x_k = sum_k c_k x_k + 136 sum_k x_k), which costs four FMAs per 128 k instead of a
// packed subtraction per register: the widening, not the stream, is what the issue slots are spent on.
__device__ __forceinline__ void w4_widen(uint32_t w, uint32_t (&r)[4], uint32_t mask, uint32_t magic)
{
    // mask = 0x000f000f and magic = 0x43084308 live in registers so that (x & mask) ^ magic is ONE three-input LOP3
#pragma unroll
    for (int i = 0; i < 4; ++i)
        asm("lop3.b32 %0, %1, %2, %3, 0x6a;" : "=r"(r[i]) : "r"(w >> (4 * i)), "r"(mask), "r"(magic));
}
constexpr float kW4Offset = 136.f;

__global__ void __launch_bounds__(kThreads, 1)
ready_dist_w4_kernel(const __grid_constant__ CUtensorMap tm_w4, const RdParams p, const __nv_bfloat16 *__restrict__ w_scale)
{
    extern __shared__ __align__(1024) uint8_t smem_raw[];
    uint8_t *smem = smem_raw;   // declared 1024-byte aligned; no integer round trip, so that loads stay LDS
    uint8_t *stage_base = smem;
    const int x_stride = p.H + kW4XPad;  // elements
    __nv_bfloat16 *xs = reinterpret_cast<__nv_bfloat16 *>(smem + static_cast<size_t>(p.n_stages) * kW4StageBytes);
    uint64_t *bars = reinterpret_cast<uint64_t *>(reinterpret_cast<uint8_t *>(xs) +
                                                  ((static_cast<size_t>(p.x_rows) * x_stride * 2 + 15) & ~size_t(15)));
    uint64_t *full_bar = bars;
    uint64_t *empty_bar = bars + kMaxStages;
    RdPartial *warp_part = reinterpret_cast<RdPartial *>(bars + 2 * kMaxStages);  // [kConsumerWarps][kNB]
    float *xsum = reinterpret_cast<float *>(warp_part + kConsumerWarps * kNB);    // [n_groups][kNB]: sum of x over a group
    const int warp = threadIdx.x >> 5;
    const int lane = threadIdx.x & 31;
    const int n_tiles = (p.V + kTileRows - 1) / kTileRows;
    const int n_groups = p.H / kW4Group;
    const int n_kc = (n_groups + kW4BoxesPerStage - 1) / kW4BoxesPerStage;

    if (threadIdx.x == 0) {
        for (int s = 0; s < p.n_stages; ++s) {
            ptx::mbar_init(ptx::smem_u32(&full_bar[s]), 1);
            ptx::mbar_init(ptx::smem_u32(&empty_bar[s]), kConsumerWarps);
        }
        ptx::fence_mbar_init();
    }
    __syncthreads();
    ptx::griddep_launch();

    if (warp == kConsumerWarps) {
        // ===== TMA producer (the weights are never written by a libprepos kernel: fetched before the wait) =====
        if (lane == 0) {
            ptx::prefetch_tmap(&tm_w4);
            const uint64_t pol = ptx::policy_evict_first();
            int stage = 0;
            uint32_t phase = 0;
            for (int tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
                for (int kc = 0; kc < n_kc; ++kc) {
                    const int nb = (n_groups - kc * kW4BoxesPerStage < kW4BoxesPerStage) ? n_groups - kc * kW4BoxesPerStage
                                                                                         : kW4BoxesPerStage;
                    ptx::mbar_wait(ptx::smem_u32(&empty_bar[stage]), phase ^ 1);
                    const uint32_t fb = ptx::smem_u32(&full_bar[stage]);
                    ptx::mbar_arrive_expect_tx(fb, nb * kW4BoxBytes);
                    const uint32_t dst = ptx::smem_u32(stage_base + static_cast<size_t>(stage) * kW4StageBytes);
                    for (int b = 0; b < nb; ++b)
                        ptx::tma_load_2d(dst + b * kW4BoxBytes, &tm_w4, fb, (kc * kW4BoxesPerStage + b) * 64,
                                         tile * kTileRows, pol);
                    if (++stage == p.n_stages) {
                        stage = 0;
                        phase ^= 1;
                    }
                }
            }
        }
        ptx::griddep_wait();
    } else {
        // ===== consumers: 16 vocabulary rows per warp =====
        ptx::griddep_wait();
        {
            // hidden rows -> smem in MMA order: the 8 elements k0..k0+7 of a word are stored (0,4,1,5,2,6,3,7), and the
            // words of a group as [j][t] (thread t's word j), so that a quarter-warp reads 64 contiguous bytes per row
            const int chunks_per_row = p.H / 8;
            for (int idx = threadIdx.x; idx < p.x_rows * chunks_per_row; idx += kConsumerWarps * 32) {
                const int r = idx / chunks_per_row, c = idx - r * chunks_per_row;
                uint4 v = make_uint4(0, 0, 0, 0);
                if (r < p.n) v = *reinterpret_cast<const uint4 *>(p.hidden + static_cast<size_t>(r) * p.H + c * 8);
                uint4 o;
                o.x = __byte_perm(v.x, v.z, 0x5410);  // (x0, x4)
                o.y = __byte_perm(v.x, v.z, 0x7632);  // (x1, x5)
                o.z = __byte_perm(v.y, v.w, 0x5410);  // (x2, x6)
                o.w = __byte_perm(v.y, v.w, 0x7632);  // (x3, x7)
                const int grp = c >> 4, within = c & 15, t = within >> 2, j = within & 3;
                *reinterpret_cast<uint4 *>(xs + static_cast<size_t>(r) * x_stride + grp * kW4Group + j * 32 + t * 8) = o;
            }
        }
        ptx::bar_sync(1, kConsumerWarps * 32);
        // per (group, hidden row) sums of x, in fp32 from the bf16 values the MMA multiplies (for the offset above)
        for (int idx = threadIdx.x; idx < n_groups * kNB; idx += kConsumerWarps * 32) {
            const int grp = idx / kNB, r = idx - grp * kNB;
            float acc = 0.f;
            if (r < p.n) {   // from the block just written (the order inside a group does not matter for a sum)
                const uint4 *xr = reinterpret_cast<const uint4 *>(xs + static_cast<size_t>(r) * x_stride + grp * kW4Group);
                for (int k = 0; k < kW4Group / 8; ++k) {
                    const uint4 u = xr[k];
                    const uint32_t w[4] = {u.x, u.y, u.z, u.w};
#pragma unroll
                    for (int i = 0; i < 4; ++i) acc += __uint_as_float(w[i] << 16) + __uint_as_float(w[i] & 0xffff0000u);
                }
            }
            xsum[idx] = acc;
        }
        ptx::bar_sync(1, kConsumerWarps * 32);
        Top2Lse st[2];
        st[0] = t2_init();
        st[1] = t2_init();
        const int g = lane >> 2, t = lane & 3;
        const int n0 = 2 * t;  // this lane's two hidden rows (accumulator columns)
        const int b_row = min(g, p.x_rows - 1);   // B fragment: hidden row g (absent rows read the zero row)
        const __nv_bfloat16 *xs_lane = xs + static_cast<size_t>(b_row) * x_stride + t * 8;
        const int w_off = (warp * 16 + g) * 64 + t * 16;   // this lane's 16 bytes of row g within a box
        uint32_t w4_mask, w4_magic;   // opaque to the compiler: kept in registers, not folded into immediates
        asm volatile("mov.b32 %0, 0x000f000f;\nmov.b32 %1, 0x43084308;" : "=r"(w4_mask), "=r"(w4_magic));

        int stage = 0;
        uint32_t phase = 0;
        for (int tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
            float tot[4] = {0.f, 0.f, 0.f, 0.f};
            const int v = tile * kTileRows + warp * 16 + g;
            const __nv_bfloat16 *sc_a = w_scale + static_cast<size_t>(v) * n_groups;
            const __nv_bfloat16 *sc_b = w_scale + static_cast<size_t>(v + 8) * n_groups;
            for (int kc = 0; kc < n_kc; ++kc) {
                const int g0 = kc * kW4BoxesPerStage;
                const int nb = (n_groups - g0 < kW4BoxesPerStage) ? n_groups - g0 : kW4BoxesPerStage;
                // the stage's group scales of this lane's two rows: issued before the wait for the codes
                float sa[kW4BoxesPerStage], sb[kW4BoxesPerStage];
                if (nb == kW4BoxesPerStage && (n_groups & 3) == 0 && (reinterpret_cast<uintptr_t>(w_scale) & 7) == 0) {
                    // four consecutive bf16 scales of a row: one 8-byte load (rows are n_groups * 2 bytes apart)
                    const uint2 ua = (v < p.V) ? __ldg(reinterpret_cast<const uint2 *>(sc_a + g0)) : make_uint2(0, 0);
                    const uint2 ub = (v + 8 < p.V) ? __ldg(reinterpret_cast<const uint2 *>(sc_b + g0)) : make_uint2(0, 0);
                    sa[0] = __uint_as_float(ua.x << 16), sa[1] = __uint_as_float(ua.x & 0xffff0000u);
                    sa[2] = __uint_as_float(ua.y << 16), sa[3] = __uint_as_float(ua.y & 0xffff0000u);
                    sb[0] = __uint_as_float(ub.x << 16), sb[1] = __uint_as_float(ub.x & 0xffff0000u);
                    sb[2] = __uint_as_float(ub.y << 16), sb[3] = __uint_as_float(ub.y & 0xffff0000u);
                } else {
#pragma unroll
                    for (int b = 0; b < kW4BoxesPerStage; ++b) {
                        sa[b] = (b < nb && v < p.V) ? __bfloat162float(sc_a[g0 + b]) : 0.f;
                        sb[b] = (b < nb && v + 8 < p.V) ? __bfloat162float(sc_b[g0 + b]) : 0.f;
                    }
                }
                ptx::mbar_wait(ptx::smem_u32(&full_bar[stage]), phase);
                const uint8_t *sbase = stage_base + static_cast<size_t>(stage) * kW4StageBytes;
#pragma unroll
                for (int b = 0; b < kW4BoxesPerStage; ++b) {
                    if (b < nb) {
                        const uint4 wa = *reinterpret_cast<const uint4 *>(sbase + b * kW4BoxBytes + w_off);
                        const uint4 wb = *reinterpret_cast<const uint4 *>(sbase + b * kW4BoxBytes + w_off + 8 * 64);
                        const uint32_t wav[4] = {wa.x, wa.y, wa.z, wa.w}, wbv[4] = {wb.x, wb.y, wb.z, wb.w};
                        const __nv_bfloat16 *xk = xs_lane + (g0 + b) * kW4Group;
                        float acc[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
                        for (int j = 0; j < 4; ++j) {
                            const uint4 xb = *reinterpret_cast<const uint4 *>(xk + j * 32);
                            uint32_t ra[4], rb[4];
                            w4_widen(wav[j], ra, w4_mask, w4_magic);
                            w4_widen(wbv[j], rb, w4_mask, w4_magic);
                            ptx::mma_bf16_16816(acc, ra[0], rb[0], ra[1], rb[1], xb.x, xb.y);
                            ptx::mma_bf16_16816(acc, ra[2], rb[2], ra[3], rb[3], xb.z, xb.w);
                        }
                        const float2 xs2 = *reinterpret_cast<const float2 *>(xsum + (g0 + b) * kNB + n0);
                        const float o0 = kW4Offset * xs2.x, o1 = kW4Offset * xs2.y;
                        tot[0] = fmaf(sa[b], acc[0] - o0, tot[0]);
                        tot[1] = fmaf(sa[b], acc[1] - o1, tot[1]);
                        tot[2] = fmaf(sb[b], acc[2] - o0, tot[2]);
                        tot[3] = fmaf(sb[b], acc[3] - o1, tot[3]);
                    }
                }
                __syncwarp();
                if (lane == 0) ptx::mbar_arrive(ptx::smem_u32(&empty_bar[stage]));
                if (++stage == p.n_stages) {
                    stage = 0;
                    phase ^= 1;
                }
            }
#pragma unroll
            for (int j = 0; j < 2; ++j) {
                if (n0 + j < p.n) {
                    if (v < p.V) t2_push(st[j], tot[j], v);
                    if (v + 8 < p.V) t2_push(st[j], tot[2 + j], v + 8);
                    if (p.logits_out) {
                        float *lo = p.logits_out + static_cast<size_t>(n0 + j) * p.V;
                        if (v < p.V) lo[v] = tot[j];
                        if (v + 8 < p.V) lo[v + 8] = tot[2 + j];
                    }
                }
            }
        }
#pragma unroll
        for (int j = 0; j < 2; ++j) {
#pragma unroll
            for (int mask = 4; mask < 32; mask <<= 1) {
                const Top2Lse o = t2_shfl_xor(st[j], mask);
                t2_merge(st[j], o);
            }
        }
        if (lane < 4) {
            t2_store(&warp_part[warp * kNB + n0], st[0]);
            t2_store(&warp_part[warp * kNB + n0 + 1], st[1]);
        }
    }
    __syncthreads();
    if (threadIdx.x < p.n) {
        Top2Lse acc = t2_init();
        for (int w = 0; w < kConsumerWarps; ++w) {
            const RdPartial *q = &warp_part[w * kNB + threadIdx.x];
            Top2Lse t;
            t.m = q->m, t.s = q->s, t.v1 = q->v1, t.v2 = q->v2, t.i1 = q->i1, t.i2 = q->i2, t.nonfinite = q->nonfinite;
            t2_merge(acc, t);
        }
        t2_store(p.partials + static_cast<size_t>(threadIdx.x) * kMaxRdPartials + blockIdx.x, acc);
        __threadfence();
    }
    __syncthreads();
    finalize_records(p, warp, lane, kThreads / 32);
}

// ---- a3 + a4 for a batch of sessions (9..128 hidden rows per launch): one pass over W for all of them ----------
// With more than a handful of hidden rows the LM head is a real contraction [n x H] . [H x V]: tcgen05.mma with the
// hidden rows as the M operand (rows past n are zero-filled by TMA or never read back), a 128-row vocabulary tile
// as the N operand, fp32 accumulators in TMEM.  D[session][vocab row]: TMEM lane = session, so one epilogue thread
// owns one session and scans its 128 new logits per tile into ONE (top1, top2, max, sum-exp) state -- no cross-lane
// reduction at all.  Still a pure HBM stream of W: the [x_rows x 128] slice of the hidden rows that rides along in
// each stage comes from L2.
constexpr int kBThreads = 192;  // warp 0: TMA, warp 1: MMA issue + TMEM, warps 2-5: epilogue (one TMEM quadrant each)
constexpr int kBMaxStages = 5;

__device__ __forceinline__ uint32_t rd_desc_lo(uint32_t saddr) { return ((saddr >> 4) & 0x3fffu) | (1u << 16); }
constexpr uint32_t kRdDescHi = (1024u >> 4) | (1u << 14) | (2u << 29);  // SBO 1024 B, version 1, SWIZZLE_128B
constexpr uint32_t kRdIdesc = (1u << 4) | (1u << 7) | (1u << 10) | ((128u >> 3) << 17) | ((128u >> 4) << 24);

__global__ void __launch_bounds__(kBThreads, 1)
ready_dist_batch_kernel(const __grid_constant__ CUtensorMap tm_w, const __grid_constant__ CUtensorMap tm_x,
                        const RdParams p)
{
    extern __shared__ __align__(1024) uint8_t smem_raw[];
    uint8_t *smem = reinterpret_cast<uint8_t *>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
    const int x_box_bytes = p.x_rows * kBoxCols * 2;          // one 64-column box of the hidden rows
    const int stage_bytes = kStageBytes + 2 * x_box_bytes;    // W [128 x 128] + X [x_rows x 128]
    // the M = 128 MMA reads 128 rows of the hidden-row boxes: with x_rows < 128 it runs past the last stage into
    // this pad (garbage rows of D that no thread reads back), which keeps the reads inside the CTA's allocation
    const int pad_bytes = kBoxBytes - x_box_bytes;
    uint64_t *bars = reinterpret_cast<uint64_t *>(smem + static_cast<size_t>(p.n_stages) * stage_bytes + pad_bytes);
    uint64_t *full_bar = bars, *empty_bar = bars + kBMaxStages;
    uint64_t *d_full = bars + 2 * kBMaxStages, *d_empty = d_full + 2;
    uint32_t *tmem_slot = reinterpret_cast<uint32_t *>(d_empty + 2);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int n_tiles = (p.V + kTileRows - 1) / kTileRows;
    const int n_kc = p.H / kStageCols;

    if (threadIdx.x == 0) {
        for (int s = 0; s < p.n_stages; ++s) {
            ptx::mbar_init(ptx::smem_u32(&full_bar[s]), 1);
            ptx::mbar_init(ptx::smem_u32(&empty_bar[s]), 1);
        }
        for (int b = 0; b < 2; ++b) {
            ptx::mbar_init(ptx::smem_u32(&d_full[b]), 1);
            ptx::mbar_init(ptx::smem_u32(&d_empty[b]), 128);
        }
        ptx::fence_mbar_init();
    }
    if (warp == 1) {
        ptx::tmem_alloc<256>(ptx::smem_u32(tmem_slot));
        ptx::tmem_relinquish();
    }
    ptx::tc_fence_before();
    __syncthreads();
    ptx::tc_fence_after();
    const uint32_t tmem = *tmem_slot;
    ptx::griddep_wait();  // the hidden rows ride in every stage: nothing useful to fetch before the predecessor ends
    ptx::griddep_launch();

    if (warp == 0) {
        // ===== TMA producer: W stage (two 64-column boxes) + the matching columns of the hidden rows =====
        if (lane == 0) {
            ptx::prefetch_tmap(&tm_w);
            ptx::prefetch_tmap(&tm_x);
            const uint64_t pol_w = ptx::policy_evict_first();  // W is read once per pass
            const uint64_t pol_x = ptx::policy_evict_last();   // the hidden rows are re-read by every tile
            int stage = 0;
            uint32_t phase = 0;
            for (int tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
                for (int kc = 0; kc < n_kc; ++kc) {
                    ptx::mbar_wait(ptx::smem_u32(&empty_bar[stage]), phase ^ 1);
                    const uint32_t fb = ptx::smem_u32(&full_bar[stage]);
                    ptx::mbar_arrive_expect_tx(fb, stage_bytes);
                    const uint32_t dst = ptx::smem_u32(smem + static_cast<size_t>(stage) * stage_bytes);
                    ptx::tma_load_2d(dst, &tm_w, fb, kc * kStageCols, tile * kTileRows, pol_w);
                    ptx::tma_load_2d(dst + kBoxBytes, &tm_w, fb, kc * kStageCols + kBoxCols, tile * kTileRows, pol_w);
                    ptx::tma_load_2d(dst + kStageBytes, &tm_x, fb, kc * kStageCols, 0, pol_x);
                    ptx::tma_load_2d(dst + kStageBytes + x_box_bytes, &tm_x, fb, kc * kStageCols + kBoxCols, 0, pol_x);
                    if (++stage == p.n_stages) {
                        stage = 0;
                        phase ^= 1;
                    }
                }
            }
        }
    } else if (warp == 1) {
        // ===== MMA issuer: D[buf] = X . W_tile^T over H, 8 x k16 per stage =====
        int stage = 0, it = 0;
        uint32_t phase = 0;
        for (int tile = blockIdx.x; tile < n_tiles; tile += gridDim.x, ++it) {
            const int buf = it & 1;
            ptx::mbar_wait(ptx::smem_u32(&d_empty[buf]), ((it >> 1) & 1) ^ 1);
            ptx::tc_fence_after();
            const uint32_t d = tmem + buf * 128;
            for (int kc = 0; kc < n_kc; ++kc) {
                ptx::mbar_wait(ptx::smem_u32(&full_bar[stage]), phase);
                ptx::tc_fence_after();
                const uint32_t sb = ptx::smem_u32(smem + static_cast<size_t>(stage) * stage_bytes);
                const uint32_t wlo = rd_desc_lo(sb), xlo = rd_desc_lo(sb + kStageBytes);
                const uint32_t xbox = static_cast<uint32_t>(x_box_bytes) >> 4;
                const uint32_t eb = ptx::smem_u32(&empty_bar[stage]), fb = ptx::smem_u32(&d_full[buf]);
                const uint32_t acc0 = (kc != 0);
                const bool last = (kc == n_kc - 1);
                if (ptx::elect_one()) {
#pragma unroll
                    for (int ks = 0; ks < 8; ++ks) {
                        const uint32_t koff = ((ks & 3) * 32) >> 4;
                        ptx::umma_ss2(d, xlo + (ks >> 2) * xbox + koff, wlo + (ks >> 2) * (kBoxBytes >> 4) + koff, kRdDescHi,
                                      kRdIdesc, ks == 0 ? acc0 : 1u);
                    }
                    ptx::umma_commit(eb);
                    if (last) ptx::umma_commit(fb);
                }
                __syncwarp();
                if (++stage == p.n_stages) {
                    stage = 0;
                    phase ^= 1;
                }
            }
        }
    } else {
        // ===== epilogue: thread = session (TMEM lane), scans the tile's 128 logits =====
        const int sess = ((warp & 3) << 5) | lane;
        const uint32_t lane_addr = static_cast<uint32_t>((warp & 3) << 5) << 16;
        const bool live = sess < p.n;
        Top2Lse st = t2_init();
        int it = 0;
        for (int tile = blockIdx.x; tile < n_tiles; tile += gridDim.x, ++it) {
            const int buf = it & 1;
            ptx::mbar_wait(ptx::smem_u32(&d_full[buf]), (it >> 1) & 1);
            ptx::tc_fence_after();
            const int v0 = tile * kTileRows;
            const int nv = (p.V - v0 < kTileRows) ? p.V - v0 : kTileRows;
#pragma unroll 1
            for (int cb = 0; cb < kTileRows; cb += 32) {
                uint32_t r[32];
                ptx::tmem_ld_32x32b_x32(tmem + lane_addr + buf * 128 + cb, r);
                ptx::tmem_ld_wait();
                if (live) {
#pragma unroll
                    for (int c = 0; c < 32; ++c)
                        if (cb + c < nv) t2_push(st, __uint_as_float(r[c]), v0 + cb + c);
                    if (p.logits_out) {
                        float *lo = p.logits_out + static_cast<size_t>(sess) * p.V + v0 + cb;
                        if (cb + 32 <= nv && ((reinterpret_cast<uintptr_t>(lo) & 15) == 0)) {
#pragma unroll
                            for (int c = 0; c < 32; c += 4)
                                *reinterpret_cast<uint4 *>(lo + c) = make_uint4(r[c], r[c + 1], r[c + 2], r[c + 3]);
                        } else {
#pragma unroll
                            for (int c = 0; c < 32; ++c)
                                if (cb + c < nv) lo[c] = __uint_as_float(r[c]);
                        }
                    }
                }
            }
            ptx::tc_fence_before();
            ptx::mbar_arrive(ptx::smem_u32(&d_empty[buf]));
        }
        if (live) {
            t2_store(p.partials + static_cast<size_t>(sess) * kMaxRdPartials + blockIdx.x, st);
            __threadfence();
        }
    }
    ptx::tc_fence_before();
    __syncthreads();
    if (warp == 1) ptx::tmem_dealloc<256>(tmem);
}

// The single cross-CTA pass of the batched kernel, as its own launch: one warp per hidden row merges that row's
// per-CTA partials in CTA order and writes the record.  (Done by the last-arriving CTA inside the kernel, the merge
// of 64 rows x 148 partials by six warps was a 60 us serial tail behind a 160 us stream of W.)
__global__ void __launch_bounds__(32) rd_finalize_kernel(const RdParams p, int n_parts)
{
    ptx::griddep_wait();
    ptx::griddep_launch();
    const int row = blockIdx.x, lane = threadIdx.x;
    const Top2Lse t = merge_partials_warp(p.partials, row, n_parts, lane);
    if (lane == 0 && !(p.skip_mask && p.skip_mask[row])) publish_record(p, row, t);
}

// ---- a4': scan of stored fp32 logits ---------------------------------------------------------------
constexpr int kScanThreads = 256;

__global__ void __launch_bounds__(kScanThreads)
scan_logits_kernel(int V, const float *__restrict__ logits, prepos_record *__restrict__ out, RdPartial *partials,
                   unsigned int *counters)
{
    const int row = blockIdx.y;
    const float *lg = logits + static_cast<size_t>(row) * V;
    Top2Lse st = t2_init();
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    // 128-bit loads where the row base allows it
    const bool vec_ok = ((reinterpret_cast<uintptr_t>(lg) & 15) == 0);
    const int v4 = vec_ok ? V / 4 : 0;
    for (int i = blockIdx.x * kScanThreads + threadIdx.x; i < v4; i += gridDim.x * kScanThreads) {
        const float4 x = __ldg(reinterpret_cast<const float4 *>(lg) + i);
        t2_push(st, x.x, 4 * i);
        t2_push(st, x.y, 4 * i + 1);
        t2_push(st, x.z, 4 * i + 2);
        t2_push(st, x.w, 4 * i + 3);
    }
    for (int i = v4 * 4 + blockIdx.x * kScanThreads + threadIdx.x; i < V; i += gridDim.x * kScanThreads)
        t2_push(st, __ldg(lg + i), i);
#pragma unroll
    for (int mask = 1; mask < 32; mask <<= 1) {
        const Top2Lse o = t2_shfl_xor(st, mask);
        t2_merge(st, o);
    }
    __shared__ RdPartial s_part[kScanThreads / 32];
    __shared__ int s_is_last;
    if (lane == 0) t2_store(&s_part[warp], st);
    __syncthreads();
    if (threadIdx.x == 0) {
        Top2Lse acc = t2_init();
        for (int w = 0; w < kScanThreads / 32; ++w) {
            const RdPartial *q = &s_part[w];
            Top2Lse t;
            t.m = q->m, t.s = q->s, t.v1 = q->v1, t.v2 = q->v2, t.i1 = q->i1, t.i2 = q->i2, t.nonfinite = q->nonfinite;
            t2_merge(acc, t);
        }
        t2_store(partials + static_cast<size_t>(row) * kMaxRdPartials + blockIdx.x, acc);
        __threadfence();
        const unsigned int prev = atomicAdd(&counters[row], 1u);
        s_is_last = (prev == gridDim.x - 1);
    }
    __syncthreads();
    if (!s_is_last) return;
    __threadfence();
    if (warp == 0) {
        const Top2Lse t = merge_partials_warp(partials, row, gridDim.x, lane);
        if (lane == 0) {
            prepos_record *rec = out + row;
            write_record_fields(rec, t);
            const uint32_t f = rec->flags & ~PREPOS_FLAG_NONFINITE;
            rec->flags = f | (t.nonfinite ? PREPOS_FLAG_NONFINITE : 0u);
            counters[row] = 0u;
        }
    }
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

}  // namespace

int prepos_launch_ready_dist(prepos_ctx *ctx, int n, const int32_t *session_ids, const __nv_bfloat16 *hidden,
                             const __nv_bfloat16 *w, const int64_t *position_p, const uint64_t *entry_hash,
                             const int32_t *skip_mask, prepos_record *records, const uint64_t *session_version,
                             const uint64_t *expected_version, float *logits_out, cudaStream_t stream)
{
    const int H = ctx->shape.hidden, V = ctx->shape.vocab;
    EncodeTiledFn encode = reinterpret_cast<EncodeTiledFn>(prepos_get_encode_tiled());
    if (!encode) return PREPOS_E_CUDA;
    CUtensorMap tm;
    const cuuint64_t dims[2] = {static_cast<cuuint64_t>(H), static_cast<cuuint64_t>(V)};
    const cuuint64_t strides[1] = {static_cast<cuuint64_t>(H) * 2};
    const cuuint32_t box[2] = {kBoxCols, kTileRows};
    const cuuint32_t estr[2] = {1, 1};
    if (encode(&tm, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<__nv_bfloat16 *>(w), dims, strides, box, estr,
               CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
               CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
        return PREPOS_E_CUDA;

    const int n_tiles = (V + kTileRows - 1) / kTileRows;
    const int grid = n_tiles < ctx->num_sms ? n_tiles : ctx->num_sms;
    if (n > kNB) {
        // a batch of sessions: one pass over W per 128 hidden rows on the tensor cores
        for (int r0 = 0; r0 < n; r0 += kRdMaxRows) {
            RdParams p;
            p.n = (n - r0 < kRdMaxRows) ? n - r0 : kRdMaxRows;
            p.H = H;
            p.V = V;
            p.x_rows = p.n <= 32 ? 32 : (p.n <= 64 ? 64 : 128);
            CUtensorMap tmx;
            const cuuint64_t xdims[2] = {static_cast<cuuint64_t>(H), static_cast<cuuint64_t>(p.n)};
            const cuuint32_t xbox[2] = {kBoxCols, static_cast<cuuint32_t>(p.x_rows)};
            if (encode(&tmx, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<__nv_bfloat16 *>(hidden + static_cast<size_t>(r0) * H),
                       xdims, strides, xbox, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                       CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
                return PREPOS_E_CUDA;
            const int stage_bytes = kStageBytes + 2 * p.x_rows * kBoxCols * 2;
            const size_t fixed = 1024 + (kBoxBytes - p.x_rows * kBoxCols * 2) + (2 * kBMaxStages + 4) * 8 + 16;
            int stages = static_cast<int>((232448 - fixed) / stage_bytes);
            if (stages > kBMaxStages) stages = kBMaxStages;
            p.n_stages = stages;
            p.hidden = hidden + static_cast<size_t>(r0) * H;
            p.session_ids = session_ids + r0;
            p.position_p = position_p ? position_p + r0 : nullptr;
            p.entry_hash = entry_hash ? entry_hash + r0 : nullptr;
            p.skip_mask = skip_mask ? skip_mask + r0 : nullptr;
            p.records = records;
            p.session_version = session_version;
            p.expected_version = expected_version ? expected_version + r0 : nullptr;
            p.logits_out = logits_out ? logits_out + static_cast<size_t>(r0) * V : nullptr;
            p.partials = ctx->rd_partials;
            p.counter = ctx->rd_counter;
            const size_t smem = fixed + static_cast<size_t>(stages) * stage_bytes;
            PREPOS_CUDA_TRY(cudaFuncSetAttribute(ready_dist_batch_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                                 static_cast<int>(smem)));
            PREPOS_CUDA_TRY(prepos_launch_pdl(ready_dist_batch_kernel, dim3(grid), dim3(kBThreads), smem, stream, tm, tmx, p));
            PREPOS_CUDA_TRY(prepos_launch_pdl(rd_finalize_kernel, dim3(p.n), dim3(32), 0, stream, p, grid));
            ctx->launches += 2;
        }
        return PREPOS_OK;
    }
    for (int r0 = 0; r0 < n; r0 += kNB) {
        RdParams p;
        p.n = (n - r0 < kNB) ? n - r0 : kNB;
        p.H = H;
        p.V = V;
        p.x_rows = (p.n < kNB) ? p.n + 1 : kNB;
        const size_t x_bytes = (static_cast<size_t>(p.x_rows) * (H + kXPad) * 2 + 15) & ~size_t(15);
        const size_t fixed = 1024 + x_bytes + 2 * kMaxStages * 8 + kConsumerWarps * kNB * sizeof(RdPartial);
        if (fixed + 2 * static_cast<size_t>(kStageBytes) > 232448) return PREPOS_E_SHAPE;   // H too large for two stages
        int stages = static_cast<int>((232448 - fixed) / kStageBytes);
        if (stages > kMaxStages) stages = kMaxStages;
        p.n_stages = stages;
        p.hidden = hidden + static_cast<size_t>(r0) * H;
        p.session_ids = session_ids + r0;
        p.position_p = position_p ? position_p + r0 : nullptr;
        p.entry_hash = entry_hash ? entry_hash + r0 : nullptr;
        p.skip_mask = skip_mask ? skip_mask + r0 : nullptr;
        p.records = records;
        p.session_version = session_version;
        p.expected_version = expected_version ? expected_version + r0 : nullptr;
        p.logits_out = logits_out ? logits_out + static_cast<size_t>(r0) * V : nullptr;
        p.partials = ctx->rd_partials;
        p.counter = ctx->rd_counter;
        const size_t smem = fixed + static_cast<size_t>(stages) * kStageBytes;
        PREPOS_CUDA_TRY(cudaFuncSetAttribute(ready_dist_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                             static_cast<int>(smem)));
        PREPOS_CUDA_TRY(prepos_launch_pdl(ready_dist_kernel, dim3(grid), dim3(kThreads), smem, stream, tm, p));
        ctx->launches += 1;
    }
    return PREPOS_OK;
}

int prepos_launch_ready_dist_w4(prepos_ctx *ctx, int n, const int32_t *session_ids, const __nv_bfloat16 *hidden,
                                const uint8_t *w4, const __nv_bfloat16 *w_scale, const int64_t *position_p,
                                const uint64_t *entry_hash, const int32_t *skip_mask, prepos_record *records,
                                const uint64_t *session_version, const uint64_t *expected_version, float *logits_out,
                                cudaStream_t stream)
{
    const int H = ctx->shape.hidden, V = ctx->shape.vocab;
    EncodeTiledFn encode = reinterpret_cast<EncodeTiledFn>(prepos_get_encode_tiled());
    if (!encode) return PREPOS_E_CUDA;
    CUtensorMap tm;
    const cuuint64_t dims[2] = {static_cast<cuuint64_t>(H / 2), static_cast<cuuint64_t>(V)};
    const cuuint64_t strides[1] = {static_cast<cuuint64_t>(H / 2)};
    const cuuint32_t box[2] = {64, kTileRows};
    const cuuint32_t estr[2] = {1, 1};
    if (encode(&tm, CU_TENSOR_MAP_DATA_TYPE_UINT8, 2, const_cast<uint8_t *>(w4), dims, strides, box, estr,
               CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
               CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
        return PREPOS_E_CUDA;
    const int n_tiles = (V + kTileRows - 1) / kTileRows;
    const int grid = n_tiles < ctx->num_sms ? n_tiles : ctx->num_sms;
    // up to 8 hidden rows per pass over the codes (a batch of more rows takes ceil(n / 8) passes)
    for (int r0 = 0; r0 < n; r0 += kNB) {
        RdParams p;
        p.n = (n - r0 < kNB) ? n - r0 : kNB;
        p.H = H;
        p.V = V;
        p.x_rows = (p.n < kNB) ? p.n + 1 : kNB;
        const size_t x_bytes = (static_cast<size_t>(p.x_rows) * (H + kW4XPad) * 2 + 15) & ~size_t(15);
        const size_t fixed = 1024 + x_bytes + 2 * kMaxStages * 8 + kConsumerWarps * kNB * sizeof(RdPartial) +
                             static_cast<size_t>(H / kW4Group) * kNB * sizeof(float);
        if (fixed + 2 * static_cast<size_t>(kW4StageBytes) > 232448) return PREPOS_E_SHAPE;   // H too large for two stages
        int stages = static_cast<int>((232448 - fixed) / kW4StageBytes);
        if (stages > kMaxStages) stages = kMaxStages;
        p.n_stages = stages;
        p.hidden = hidden + static_cast<size_t>(r0) * H;
        p.session_ids = session_ids + r0;
        p.position_p = position_p ? position_p + r0 : nullptr;
        p.entry_hash = entry_hash ? entry_hash + r0 : nullptr;
        p.skip_mask = skip_mask ? skip_mask + r0 : nullptr;
        p.records = records;
        p.session_version = session_version;
        p.expected_version = expected_version ? expected_version + r0 : nullptr;
        p.logits_out = logits_out ? logits_out + static_cast<size_t>(r0) * V : nullptr;
        p.partials = ctx->rd_partials;
        p.counter = ctx->rd_counter;
        const size_t smem = fixed + static_cast<size_t>(stages) * kW4StageBytes;
        PREPOS_CUDA_TRY(cudaFuncSetAttribute(ready_dist_w4_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                             static_cast<int>(smem)));
        PREPOS_CUDA_TRY(prepos_launch_pdl(ready_dist_w4_kernel, dim3(grid), dim3(kThreads), smem, stream, tm, p, w_scale));
        ctx->launches += 1;
    }
    return PREPOS_OK;
}

int prepos_launch_scan_logits(prepos_ctx *ctx, int n, const float *logits, prepos_record *out, cudaStream_t stream)
{
    const int V = ctx->shape.vocab;
    for (int r0 = 0; r0 < n; r0 += kRdMaxRows) {
        const int rows = (n - r0 < kRdMaxRows) ? n - r0 : kRdMaxRows;
        int gx = (V + kScanThreads * 16 - 1) / (kScanThreads * 16);  // >= 16 logits per thread
        if (gx > 64) gx = 64;
        if (gx < 1) gx = 1;
        scan_logits_kernel<<<dim3(gx, rows), kScanThreads, 0, stream>>>(V, logits + static_cast<size_t>(r0) * V,
                                                                        out + r0, ctx->rd_partials,
                                                                        ctx->rd_counter + 1);
        PREPOS_CUDA_TRY(cudaGetLastError());
        ctx->launches += 1;
    }
    return PREPOS_OK;
}

// ---- a4' for callers that cannot allocate: prepos_scan_logits_noalloc ------------------------------------------
// The serve-time vocabulary scan (Alg. 2 l.3-4; T_scan(V) of Eq. 3) needs a little
// scratch for its single cross-CTA pass: one 32-byte partial per (row, CTA) and one arrival counter per row.
// prepos_scan_logits takes it from the ctx workspace, which somebody had to allocate.  The variant below takes it
// from a fixed array that is part of the library image instead, so that the call needs neither a ctx nor a
// workspace nor any allocation of its own (who needs that, and the limits: include/prepos.h).
//
// g_scan_noalloc_scratch lives in the device memory of every GPU that loads libprepos, from module load until the
// process exits.  Layout: [0, 256) arrival counters (one uint32 per row), then [row][kNaMaxParts] RdPartial.
constexpr int kNaMaxRows = PREPOS_SCAN_NOALLOC_MAX_ROWS;
constexpr int kNaMaxParts = 64;          // CTAs per row (the grid's x extent is capped at this)
constexpr int kNaCounterBytes = 256;
constexpr size_t kNaScratchBytes = kNaCounterBytes + sizeof(RdPartial) * kNaMaxRows * kNaMaxParts;
static_assert(kNaMaxRows * sizeof(unsigned int) <= kNaCounterBytes, "counter block");
static_assert(kNaScratchBytes == PREPOS_SCAN_NOALLOC_SCRATCH_BYTES, "header and kernel disagree on the scratch size");

static __device__ __align__(256) unsigned char g_scan_noalloc_scratch[kNaScratchBytes];

namespace {

// scan_logits_kernel with the partials packed [row][kNaMaxParts] (gridDim.x <= kNaMaxParts): same per-thread scan,
// same warp / CTA reduction, same merge order in the last-arriving CTA (lane c takes partials c and c + 32 in that
// order, then the xor tree), so the records equal the ones prepos_scan_logits writes for the same grid.
__global__ void __launch_bounds__(kScanThreads)
scan_logits_noalloc_kernel(int V, const float *__restrict__ logits, prepos_record *__restrict__ out,
                           RdPartial *partials, unsigned int *counters)
{
    const int row = blockIdx.y;
    const float *lg = logits + static_cast<size_t>(row) * V;
    Top2Lse st = t2_init();
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const bool vec_ok = ((reinterpret_cast<uintptr_t>(lg) & 15) == 0);
    const int v4 = vec_ok ? V / 4 : 0;
    for (int i = blockIdx.x * kScanThreads + threadIdx.x; i < v4; i += gridDim.x * kScanThreads) {
        const float4 x = __ldg(reinterpret_cast<const float4 *>(lg) + i);
        t2_push(st, x.x, 4 * i);
        t2_push(st, x.y, 4 * i + 1);
        t2_push(st, x.z, 4 * i + 2);
        t2_push(st, x.w, 4 * i + 3);
    }
    for (int i = v4 * 4 + blockIdx.x * kScanThreads + threadIdx.x; i < V; i += gridDim.x * kScanThreads)
        t2_push(st, __ldg(lg + i), i);
#pragma unroll
    for (int mask = 1; mask < 32; mask <<= 1) {
        const Top2Lse o = t2_shfl_xor(st, mask);
        t2_merge(st, o);
    }
    __shared__ RdPartial s_part[kScanThreads / 32];
    __shared__ int s_is_last;
    if (lane == 0) t2_store(&s_part[warp], st);
    __syncthreads();
    RdPartial *row_parts = partials + static_cast<size_t>(row) * kNaMaxParts;
    if (threadIdx.x == 0) {
        Top2Lse acc = t2_init();
        for (int w = 0; w < kScanThreads / 32; ++w) {
            const RdPartial *q = &s_part[w];
            Top2Lse t;
            t.m = q->m, t.s = q->s, t.v1 = q->v1, t.v2 = q->v2, t.i1 = q->i1, t.i2 = q->i2, t.nonfinite = q->nonfinite;
            t2_merge(acc, t);
        }
        t2_store(row_parts + blockIdx.x, acc);
        __threadfence();
        const unsigned int prev = atomicAdd(&counters[row], 1u);
        s_is_last = (prev == gridDim.x - 1);
    }
    __syncthreads();
    if (!s_is_last) return;
    __threadfence();
    if (warp == 0) {
        Top2Lse acc = t2_init();
        const int n_parts = static_cast<int>(gridDim.x);
        Top2Lse part[kNaMaxParts / 32];
#pragma unroll
        for (int j = 0; j < kNaMaxParts / 32; ++j)
            if (lane + 32 * j < n_parts) part[j] = t2_load(row_parts + lane + 32 * j);
#pragma unroll
        for (int j = 0; j < kNaMaxParts / 32; ++j)
            if (lane + 32 * j < n_parts) t2_merge(acc, part[j]);
#pragma unroll
        for (int mask = 1; mask < 32; mask <<= 1) {
            const Top2Lse o = t2_shfl_xor(acc, mask);
            t2_merge(acc, o);
        }
        if (lane == 0) {
            prepos_record *rec = out + row;
            write_record_fields(rec, acc);
            const uint32_t f = rec->flags & ~PREPOS_FLAG_NONFINITE;
            rec->flags = f | (acc.nonfinite ? PREPOS_FLAG_NONFINITE : 0u);
        }
    }
}

// Device address of g_scan_noalloc_scratch, per device ordinal.  In host code the array's name only stands in for
// the symbol: it is not an address a kernel (or cudaMemsetAsync) can use.  The real address is asked for once per
// device, with that device current, and kept.
constexpr int kNaMaxDevices = 64;
std::mutex g_na_mutex;
unsigned char *g_na_scratch_addr[kNaMaxDevices] = {};

int scan_noalloc_scratch(unsigned char **addr)
{
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
        cudaGetLastError();
        return PREPOS_E_NO_DEVICE;
    }
    int dev = 0;
    PREPOS_CUDA_TRY(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kNaMaxDevices) return PREPOS_E_NO_DEVICE;
    std::lock_guard<std::mutex> lock(g_na_mutex);
    if (!g_na_scratch_addr[dev]) {
        int major = 0;
        PREPOS_CUDA_TRY(cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev));
        if (major != 10) return PREPOS_E_NO_DEVICE;  // built for sm_100a only
        unsigned char *p = nullptr;
        PREPOS_CUDA_TRY(cudaGetSymbolAddress(reinterpret_cast<void **>(&p), g_scan_noalloc_scratch));
        if (!p) return PREPOS_E_CUDA;
        g_na_scratch_addr[dev] = p;
    }
    *addr = g_na_scratch_addr[dev];
    return PREPOS_OK;
}

}  // namespace

extern "C" int prepos_scan_logits_noalloc(int n, int vocab, const float *logits, prepos_record *out, void *stream)
{
    if (n < 0 || vocab < 2) return PREPOS_E_INVALID_ARG;
    if (n > PREPOS_SCAN_NOALLOC_MAX_ROWS || vocab > PREPOS_SCAN_NOALLOC_MAX_VOCAB) return PREPOS_E_FIXED_SCRATCH;
    if (n == 0) return PREPOS_OK;
    if (!logits || !out) return PREPOS_E_INVALID_ARG;
    if ((reinterpret_cast<uintptr_t>(out) & 15) || (reinterpret_cast<uintptr_t>(logits) & 3)) return PREPOS_E_ALIGN;
    unsigned char *scratch = nullptr;
    const int st = scan_noalloc_scratch(&scratch);
    if (st != PREPOS_OK) return st;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    unsigned int *counters = reinterpret_cast<unsigned int *>(scratch);
    RdPartial *partials = reinterpret_cast<RdPartial *>(scratch + kNaCounterBytes);
    // the array keeps whatever the previous call left: the arrival counters must start at zero, the partials are
    // fully overwritten before they are read
    PREPOS_CUDA_TRY(cudaMemsetAsync(counters, 0, sizeof(unsigned int) * n, s));
    int gx = (vocab + kScanThreads * 16 - 1) / (kScanThreads * 16);  // as prepos_scan_logits: >= 16 logits per thread
    if (gx > kNaMaxParts) gx = kNaMaxParts;
    if (gx < 1) gx = 1;
    scan_logits_noalloc_kernel<<<dim3(gx, n), kScanThreads, 0, s>>>(vocab, logits, out, partials, counters);
    PREPOS_CUDA_TRY(cudaGetLastError());
    return PREPOS_OK;
}
