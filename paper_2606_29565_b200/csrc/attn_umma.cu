// attn_umma.cu -- a1 + a2 on the 5th-generation tensor cores: the entry tokens' G*L query rows attend the
// session's paged bf16 KV cache (Alg. 1 l.5-6; Eq. 1) as a dense contraction
// [G*L x d] . [d x n_s] -> softmax -> [G*L x n_s] . [n_s x d] per KV head.  Arithmetic intensity is G*L
// flop per KV byte (96..384 at the BASELINE configs), so the pass is HBM-bound up to the ridge and needs
// ~0.6-1 PFLOP/s to stay there: tcgen05.mma with TMEM accumulators, KV pages staged by TMA.
//
// Work decomposition (stream-K over KV tiles): the launch's work is the linear space
//   (layer, kv head) x units x 128-token tiles
// cut into one contiguous range per persistent CTA (1 CTA / SM).  A CTA walks its range as segments
// (= its part of one unit).  A unit covered by one segment is written directly; otherwise every
// covering CTA writes a normalised fp32 partial + log-sum-exp, bumps the unit's arrival counter, and the
// last CTA to arrive combines the partials in CTA order (the single cross-CTA pass; deterministic for a
// fixed plan whoever arrives last).  A CTA runs the cut head segment at the end of its range FIRST, so that both
// partials of a cut unit are delivered early and no merge sits in the kernel's tail.
//
// Inside a CTA (384 threads):
//   warp 0  K producer: TMA into a ring of K tiles -- cached tiles through a 5-D map over the pool (one
//           4 KB box per page), entry-token tiles through a 5-D map over K_new (one box per 8 tokens)
//   warp 3  V producer: same for V (plus a zero fill of the rows of an entry tile no box covers)
//   warp 2  TMEM allocator, Q loader (TMA, one box per 8-row group of the unit's (token, head) rows, issued as soon
//           as the previous segment's last QK has retired) and the Append(E) writer (Alg. 1 l.5): K_new/V_new ->
//           the session's pages
//   warp 1  MMA issuer: S = Q K^T (SS, K-major SW128) into TMEM, O += P V (A = P from TMEM, B = V MN-major);
//           warp-uniform descriptor words, only the tcgen05 instructions under elect.sync
//   warps 4-7 / 8-11  two softmax warpgroups, one TMEM lane (= query row) per thread: online softmax
//           with lazy rescaling, P written back to TMEM as bf16 over S.
// The CTA always runs two independent streams (S_w, O_w, own running max/sum): with >128 rows stream w
// owns M-tile w; with <=128 rows the streams take alternate KV tiles and are merged in the epilogue.
#include <math_constants.h>
#include <stdio.h>
#include <string.h>

#include <type_traits>

#include "common.cuh"
#include "ptx.cuh"

namespace {

constexpr int kThreads = 384;
constexpr int kTile = kAttnTileTokens;  // 128 tokens
constexpr int kNK = 3;                  // K ring slots
constexpr int kLastArriverMax = 4;        // partials of a cut unit that the last-arriving CTA combines on the spot
constexpr float kRescaleThreshold = 8.f;  // log2 units: lazy rescale (P <= 2^8)
// Register budget: the kernel is launched with kLaunchRegs per thread, NOT the whole register file, and uses 1 KB less
// than the shared-memory maximum, so that one small CTA of another kernel -- the gate serve of a request that
// arrives while the idle-window pass is running (the pass "yields to any request") -- fits
// beside it on every SM: 384 * 160 = 61440 registers leave 4096, a 128-thread gate_serve CTA takes 3072.
constexpr int kLaunchRegs = 160;
constexpr int kServiceRegs = 64;          // 128 * 64 + 256 * 208 = 384 * 160
constexpr int kSoftmaxRegs = 208;

struct UmmaParams {
    AttnArgs a;
    const AttnUnit *units;
    int Hq, Hkv, page, page_shift;
    int n_lh;           // (layer, kv head) pairs in this launch
    int tiles_per_lh;   // sum of n_tiles over units
    long long total_tiles;
    int q_tiles;        // resident Q M-tiles (1 or 2)
    int nv;             // V ring slots
    float scale_log2;
    int use_bnd;        // 1: CTA c's range is [bnd[c], bnd[c + 1]) (units fewer than CTAs: whole CTAs per unit)
    int bnd[kAttnMaxCtas + 1];
    float *partials;    // [2 * grid] slots of kAttnMaxRows * (D + 2) floats: O as float4 [D / 4][256 rows] (a warp's
                        // 32 rows of one float4 column are 512 contiguous bytes), lse2 [256], pad [256]
    unsigned int *counters;  // [n_lh][n_units] arrival counters of the cross-CTA pass (self-resetting)
    // ---- yield / resume (the idle-window pass "yields to any request")
    const unsigned int *yield_flag;  // device word: == launch_seq asks every CTA of THAT launch to stop at its next segment boundary
    int *progress;                   // [grid] segments CTA c has completed in this pass (over all its launches)
    unsigned int *pass_state;        // a CTA that stops early writes launch_seq here
    unsigned int launch_seq;
    int resume;                      // 1: CTA c skips its first progress[c] segments
    int slice;                       // > 0: stop after this many segments per launch (bounded residency)
    int early_kv;                    // 1: the cached K/V tiles may be requested before the previous kernel has ended
};

struct Seg {
    AttnUnit u;
    int unit_idx, layer, kvh, lh;
    int tb, te;      // tile range within the unit
    int slot;        // partial slot of this CTA used when the segment is cut: 0 = starts at the CTA's first tile
    int direct;      // segment covers the whole unit
};

// Walks the CTA's contiguous range [t0, t1) of the global tile space as segments (= the CTA's part of one
// unit).  Processing order: when the range ends inside a unit, that cut head segment goes FIRST, then the rest
// in natural order.  A cut unit's head (end of CTA c's range) and tail (start of CTA c+1's range) are then both
// delivered early in the kernel, so the cross-CTA merge never sits in the kernel's tail.
struct SegIter {
    long long t0, t, t_stop, t1;
    long long tl;     // start of the end-cut segment emitted first (or -1)
    int prev_unit;
    __device__ SegIter(const UmmaParams &p, long long t0_, long long t1_) : t0(t0_), t(t0_), t_stop(t1_), t1(t1_), tl(-1), prev_unit(-1)
    {
        if (t1 <= t0) return;
        const long long last = t1 - 1;
        const int lh = static_cast<int>(last / p.tiles_per_lh);
        const int off = static_cast<int>(last - static_cast<long long>(lh) * p.tiles_per_lh);
        const int ui = find_unit(p, off);
        const AttnUnit u = p.units[ui];
        const long long U0 = static_cast<long long>(lh) * p.tiles_per_lh + u.tile_prefix;
        if (U0 + u.n_tiles > t1 && U0 > t0) {  // cut at the end, and not the CTA's only segment
            tl = U0;
            t_stop = U0;
        }
    }
    __device__ static int find_unit(const UmmaParams &p, int off)
    {
        // the last unit with tile_prefix <= off
        int lo = 0, hi = p.a.n_units - 1;
        while (lo < hi) {
            const int mid = (lo + hi + 1) >> 1;
            if (p.units[mid].tile_prefix <= off) lo = mid;
            else hi = mid - 1;
        }
        return lo;
    }
    __device__ void fill(const UmmaParams &p, Seg &s, long long from, long long limit, int ui, int lh, int off)
    {
        s.unit_idx = ui;
        s.u = p.units[ui];
        s.lh = lh;
        s.layer = p.a.layer_begin + lh / p.Hkv;
        s.kvh = lh % p.Hkv;
        s.tb = off - s.u.tile_prefix;
        const long long unit_end = static_cast<long long>(lh) * p.tiles_per_lh + s.u.tile_prefix + s.u.n_tiles;
        const long long end = unit_end < limit ? unit_end : limit;
        s.te = s.tb + static_cast<int>(end - from);
        s.slot = (from == t0) ? 0 : 1;
        s.direct = (s.tb == 0 && s.te == s.u.n_tiles);
    }
    __device__ bool next(const UmmaParams &p, Seg &s)
    {
        if (tl >= 0) {
            const int lh = static_cast<int>(tl / p.tiles_per_lh);
            const int off = static_cast<int>(tl - static_cast<long long>(lh) * p.tiles_per_lh);
            fill(p, s, tl, t1, find_unit(p, off), lh, off);
            tl = -1;
            return true;
        }
        if (t >= t_stop) return false;
        const int lh = static_cast<int>(t / p.tiles_per_lh);
        const int off = static_cast<int>(t - static_cast<long long>(lh) * p.tiles_per_lh);
        int ui;
        if (prev_unit < 0) ui = find_unit(p, off);
        else ui = (prev_unit + 1 == p.a.n_units) ? 0 : prev_unit + 1;  // segments end on unit boundaries
        prev_unit = ui;
        fill(p, s, t, t_stop, ui, lh, off);
        t += s.te - s.tb;
        return true;
    }
};

// CTA c's range of the global tile space is [cta_begin(c), cta_begin(c + 1)): equal shares of the tile space
// (stream-K), or the host's table when the launch has fewer units than CTAs (then every unit gets whole CTAs).
__device__ __forceinline__ long long cta_begin(const UmmaParams &p, int grid, int c)
{
    if (p.use_bnd) return p.bnd[c];
    return p.total_tiles * c / grid;
}
// the CTA whose range holds tile t
__device__ __forceinline__ int cta_of(const UmmaParams &p, int grid, long long t)
{
    if (p.use_bnd) {
        int lo = 0, hi = grid - 1;   // the last c with bnd[c] <= t
        while (lo < hi) {
            const int mid = (lo + hi + 1) >> 1;
            if (p.bnd[mid] <= t) lo = mid;
            else hi = mid - 1;
        }
        return lo;
    }
    return static_cast<int>(((t + 1) * grid + p.total_tiles - 1) / p.total_tiles) - 1;
}

// 64-bit UMMA shared-memory descriptor, SWIZZLE_128B, version 1 (sm_100), as two words: low = start address and
// leading byte offset, high = stride byte offset, version and swizzle (the high word is one constant per tile layout)
__device__ __forceinline__ uint32_t desc_lo(uint32_t saddr, uint32_t lbo_bytes)
{
    return ((saddr >> 4) & 0x3fffu) | (((lbo_bytes >> 4) & 0x3fffu) << 16);
}
__host__ __device__ constexpr uint32_t desc_hi(uint32_t sbo_bytes)
{
    return ((sbo_bytes >> 4) & 0x3fffu) | (1u << 14) | (2u << 29);
}

// byte offset of (row r, 16-byte chunk c of a D-wide bf16 row) in a tile laid out
// [row group of 8][64-column half][8 rows][128 B] with the 128-byte swizzle (chunk ^= row % 8)
template <int D>
__device__ __forceinline__ uint32_t tile_offset(int r, int c)
{
    constexpr int kHalves = D / 64;
    const int hf = c >> 3, cc = c & 7;
    return static_cast<uint32_t>((r >> 3) * (kHalves * 1024) + hf * 1024 + (r & 7) * 128 + ((cc ^ (r & 7)) << 4));
}

__device__ __forceinline__ uint32_t pack_bf16(float lo, float hi)
{
    uint32_t r;
    asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(r) : "f"(hi), "f"(lo));
    return r;
}

// Append(E) for one (session, layer, kv head), by one warp
template <int D>
__device__ __forceinline__ void append_entry(const UmmaParams &p, const Seg &s, int lane)
{
    constexpr int kChunks = D / 8;  // 16-byte chunks per row
    constexpr int kBatch = 4;
    const size_t lo = static_cast<size_t>(s.layer);
    const int32_t *pt = p.a.page_table + static_cast<size_t>(s.u.session) * p.a.page_table_stride;
    const __nv_bfloat16 *ksrc = p.a.k_new + lo * p.a.kv_new_layer_stride;
    const __nv_bfloat16 *vsrc = p.a.v_new + lo * p.a.kv_new_layer_stride;
    __nv_bfloat16 *kpool = p.a.k_pool + lo * p.a.pool_layer_stride;
    __nv_bfloat16 *vpool = p.a.v_pool + lo * p.a.pool_layer_stride;
    const int total = s.u.l_entry * kChunks;
    for (int base = lane; base < total; base += 32 * kBatch) {
        uint4 kv[kBatch], vv[kBatch];
        int pg[kBatch];
#pragma unroll
        for (int u = 0; u < kBatch; ++u) {
            const int idx = base + u * 32;
            if (idx < total) {
                const int tok = idx / kChunks, c = idx - tok * kChunks;
                const size_t so = (static_cast<size_t>(s.u.row0 + tok) * p.Hkv + s.kvh) * D + c * 8;
                kv[u] = __ldg(reinterpret_cast<const uint4 *>(ksrc + so));
                vv[u] = __ldg(reinterpret_cast<const uint4 *>(vsrc + so));
                pg[u] = __ldg(pt + ((s.u.n_s + tok) >> p.page_shift));
            }
        }
#pragma unroll
        for (int u = 0; u < kBatch; ++u) {
            const int idx = base + u * 32;
            if (idx < total) {
                const int tok = idx / kChunks, c = idx - tok * kChunks;
                const int j = s.u.n_s + tok;
                const size_t po = ((static_cast<size_t>(pg[u]) * p.Hkv + s.kvh) * p.page + (j & (p.page - 1))) * D + c * 8;
                *reinterpret_cast<uint4 *>(kpool + po) = kv[u];
                *reinterpret_cast<uint4 *>(vpool + po) = vv[u];
            }
        }
    }
}

// kFp8 (reading Q20): the pools hold e4m3 codes with one fp32 scale per (page, kv
// head); a tile arrives as 128 x D BYTES (half the HBM traffic), [token][128 B] with the 128-byte swizzle -- which IS
// the K-major operand layout of an 8-bit MMA.
//   S = Q K^T runs on the FP8 tensor path (kind::f8f6f4, K = 32 per instruction) straight from the K slab as it
//     landed: no conversion of K at all, and a K ring of six 16 KB slots.  Q (bf16, 8 significant bits) is split
//     exactly into two e4m3 operands at the start of a segment by the softmax warps: per row a power-of-two scale
//     2^k brings max|q| into [128, 256), Qh = q with the mantissa truncated to 3 bits, Ql = q - Qh (both x 2^k);
//     S = (Qh + Ql) K^T is two accumulating passes, the same tensor time as one bf16 pass.  (Elements more than 2^10
//     below their row's maximum lose bits of Ql: an absolute error below 2^-17 of that maximum.)
//   O += P V stays f16 x f16: P is packed as fp16, the V slab lands in the upper half of its 32 KB slot and is widened
//     in place to the fp16 tile (cvt e4m3 -> f16 is exact) by warps 2 and 3, 64 token rows each.
//   The page scales never touch an operand: the K scale of a column's page (times 2^-k of the row) multiplies its
//   score inside the softmax's scale FMA, the V scale multiplies its probability before P is packed.
//   The entry tokens were appended (quantised) by fp8_append_kernel before this launch and are read back from the
//   pages like cached ones: a unit has no entry tiles, causality is a per-row column limit.
template <int D, bool kFp8>
__global__ void __maxnreg__(kLaunchRegs)
attn_umma_kernel(const __grid_constant__ CUtensorMap tm_k, const __grid_constant__ CUtensorMap tm_v,
                 const __grid_constant__ CUtensorMap tm_kn, const __grid_constant__ CUtensorMap tm_vn,
                 const __grid_constant__ CUtensorMap tm_q,
                 const UmmaParams p)
{
    static_assert(!kFp8 || D == 128, "the FP8 tiles are one 128-byte swizzle row per token");
    constexpr int kHalves = D / 64;
    constexpr int kTileBytes = kTile * D * 2;         // one K or V tile / one Q M-tile
    constexpr int kRawBytes = kTile * D;              // an e4m3 tile as it arrives (kFp8)
    constexpr int kNK8 = 2 * kNK;                     // kFp8: K slabs are used as they land, 16 KB a slot
    constexpr uint32_t kDescHi8 = desc_hi(1024);      // 8-bit K-major tile: 8 rows x 128 B per group
    constexpr uint32_t kIdescQK8 = (1u << 4) | ((kTile >> 3) << 17) | ((128u >> 4) << 24);   // e4m3 x e4m3 -> f32
    constexpr int kGroupStride = kHalves * 1024;      // bytes between 8-row groups
    constexpr uint32_t kFmt = kFp8 ? 0u : 1u;         // kind::f16 operand format: 0 = f16, 1 = bf16
    constexpr uint32_t kIdescQK = (1u << 4) | (kFmt << 7) | (kFmt << 10) | ((kTile >> 3) << 17) | ((128u >> 4) << 24);
    constexpr uint32_t kIdescPV = (1u << 4) | (kFmt << 7) | (kFmt << 10) | (1u << 16) | ((D >> 3) << 17) | ((128u >> 4) << 24);
    constexpr uint32_t kDescHi = desc_hi(kGroupStride);
    constexpr int kColS = 0;        // S_w at columns w * 128 (P_w aliases its first 64 columns)
    constexpr int kColO = 256;      // O_w at columns 256 + w * D

    extern __shared__ __align__(1024) uint8_t smem_raw[];
    if (ptx::smem_u32(smem_raw) & 1023u) __trap();  // the swizzled tiles rely on the 1024-byte base alignment
    uint8_t *q_s = smem_raw;
    uint8_t *k_s = q_s + p.q_tiles * kTileBytes;
    uint8_t *v_s = k_s + kNK * kTileBytes;
    uint8_t *tail = v_s + p.nv * kTileBytes;
    uint64_t *bars = reinterpret_cast<uint64_t *>(tail);
    uint64_t *k_full = bars, *k_empty = bars + 3, *v_full = bars + 6, *v_empty = bars + 9;
    uint64_t *s_full = bars + 12, *p_ready = bars + 14, *o_done = bars + 16, *q_full = bars + 18;
    uint64_t *q_empty = bars + 19;    // the segment's last QK has read Q: the loader may overwrite it
    // kFp8: V widened (two warps arrive), Q split, and the six-slot K ring
    uint64_t *v_conv = bars + 20, *q_conv = bars + 23, *k_full8 = bars + 24, *k_empty8 = bars + 30;
    float2 *ml_x = reinterpret_cast<float2 *>(bars + 36);  // [128] (m, l) of stream 1 / the row factors back
    uint32_t *tmem_slot = reinterpret_cast<uint32_t *>(ml_x + 128);
    int *merge_info = reinterpret_cast<int *>(tmem_slot + 1);  // [3]: c0 (or -1 = not last), c1, c0's slot
    // segment admission (yield / resume): [0] segments admitted in this launch, [1] the first one refused (or
    // INT_MAX), [2] segments completed in the pass when this launch ends.  Written by lane 0 of the K producer, the
    // role that reaches a segment first; every other role asks before it starts a segment.
    int *sched = merge_info + 3;
    // kFp8: page scales of the last 8 K tiles, [tile % 8][0..7 K scale of 16-column block b | 8..15 V scale]
    // (36 barriers + the 1 KB exchange + 4 + 12 + 12 bytes = 1340 -> 1344; plain pointer arithmetic on the shared array,
    // so that the loads stay shared-memory loads)
    float *sc_s = reinterpret_cast<float *>(tail + 1344);
    // kFp8: [128] 2^-k of the rows of M-tile 0 (both streams need it when they share the tile).  Lives in the (m, l)
    // exchange array, which is idle between a segment's epilogue and its successor's first tile.
    float *rowf_s = reinterpret_cast<float *>(ml_x);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

    if (threadIdx.x == 32) {
        for (int i = 0; i < 3; ++i) {
            ptx::mbar_init(ptx::smem_u32(&k_full[i]), 1);
            ptx::mbar_init(ptx::smem_u32(&k_empty[i]), 1);
            ptx::mbar_init(ptx::smem_u32(&v_full[i]), 1);
            ptx::mbar_init(ptx::smem_u32(&v_empty[i]), 1);
        }
        for (int i = 0; i < 2; ++i) {
            ptx::mbar_init(ptx::smem_u32(&s_full[i]), 1);
            ptx::mbar_init(ptx::smem_u32(&p_ready[i]), 128);
            ptx::mbar_init(ptx::smem_u32(&o_done[i]), 1);
        }
        ptx::mbar_init(ptx::smem_u32(q_full), 1);
        ptx::mbar_init(ptx::smem_u32(q_empty), 1);
        for (int i = 0; i < 3; ++i) ptx::mbar_init(ptx::smem_u32(&v_conv[i]), 2);
        for (int i = 0; i < 6; ++i) {
            ptx::mbar_init(ptx::smem_u32(&k_full8[i]), 1);
            ptx::mbar_init(ptx::smem_u32(&k_empty8[i]), 1);
        }
        ptx::mbar_init(ptx::smem_u32(q_conv), 1);
        ptx::fence_mbar_init();
        sched[0] = 0;
        sched[1] = 0x7fffffff;
        sched[2] = 0;
    }
    if (warp == 2) {
        ptx::tmem_alloc<512>(ptx::smem_u32(tmem_slot));
        ptx::tmem_relinquish();
    } else if (threadIdx.x == 0) {
        ptx::prefetch_tmap(&tm_k);
        ptx::prefetch_tmap(&tm_v);
        if constexpr (!kFp8) {
            ptx::prefetch_tmap(&tm_kn);
            ptx::prefetch_tmap(&tm_vn);
        }
        ptx::prefetch_tmap(&tm_q);
    }
    // rows of a Q M-tile that no TMA box covers are never written: clear the buffer once so they stay finite (part of
    // the prologue that overlaps the previous kernel's tail)
    for (int off = threadIdx.x * 16; off < p.q_tiles * kTileBytes; off += kThreads * 16)
        *reinterpret_cast<uint4 *>(q_s + off) = make_uint4(0, 0, 0, 0);
    ptx::fence_proxy_async_smem();
    ptx::tc_fence_before();
    __syncthreads();
    ptx::tc_fence_after();
    const uint32_t tmem = *tmem_slot;
    // everything above touched only this CTA's shared memory and TMEM; from here on the kernel reads what earlier
    // kernels in the stream wrote (the plan, the pools, Q).  With early_kv (prepos_ctx_set_kv_prefetch: the caller
    // guarantees that no kernel still running writes the CACHED tokens this call reads) the K / V producers start
    // streaming cached tiles right away -- the rings fill while the predecessor's merge is still running, which in the
    // one-launch-per-layer schedule hides the first-byte latency of every layer -- and every other access (Q, the
    // entry K/V, the appends, out, the partial slots) waits for the predecessor where it is first needed.
    const bool early = p.early_kv && !p.resume;
    if (!early) ptx::griddep_wait();
    ptx::griddep_launch();

    const long long t0 = cta_begin(p, gridDim.x, blockIdx.x);
    const long long t1 = cta_begin(p, gridDim.x, blockIdx.x + 1);
    const int skip = p.resume ? p.progress[blockIdx.x] : 0;   // segments this CTA completed before a yield
    // may the role start the n-th segment of this launch?  (the K producer has admitted it, or refused it)
    auto admitted = [&](int n) -> bool {
        while (true) {
            if (ptx::ld_acquire_cta_smem(&sched[0]) > n) return true;
            if (ptx::ld_acquire_cta_smem(&sched[1]) <= n) return false;
        }
    };
    const int G = p.Hq / p.Hkv;
    const int pages_per_tile = kTile >> p.page_shift;
    const int page_bytes = p.page * D * 2;
    const int page_groups = p.page >> 3;
    // the role's next segment of this launch (skipping what the pass already completed); false at the end or a yield
    auto next_seg = [&](SegIter &it, Seg &s, int &seg, int &kproc) -> bool {
        while (it.next(p, s)) {
            if (seg++ < skip) continue;
            if (!admitted(kproc)) return false;
            ++kproc;
            return true;
        }
        return false;
    };
    // kFp8: widen 64 token rows (two batches of 32: lane = row) of the e4m3 V tile in the upper half of `slot` to the
    // fp16 tile the MMA reads, in place.  Warp 2 takes rows 0-63, whose output (bytes 0-16 K) touches no raw byte;
    // warp 3 takes rows 64-127, whose output (bytes 16-32 K) covers the raw rows 0-63 and its own: it loads a batch
    // into registers first, and before its first store waits (named barrier 2) until warp 2 has loaded its last batch.
    // Rows from `zero_from` on are written as zeros (P is 0 there, but 0 x NaN would poison O).
    auto widen_tile = [&](uint8_t *slot, int zero_from, int upper) {
#pragma unroll 1
        for (int b = 2 * upper; b < 2 * upper + 2; ++b) {
            const int r = b * 32 + lane;
            const uint32_t r7s = static_cast<uint32_t>(r & 7) << 4;
            const uint8_t *src = slot + kRawBytes + r * D;
            uint8_t *dst = slot + (r >> 3) * kGroupStride + (r & 7) * 128;   // row r of half 0; half 1 is 1024 B on
            uint4 raw[D / 16];
#pragma unroll
            for (int c = 0; c < D / 16; ++c) raw[c] = *reinterpret_cast<const uint4 *>(src + ((c << 4) ^ r7s));
            __syncwarp();
            // warp 2 (b == 1): every raw row below 64 is now in registers or already widened; warp 3 (b == 2): so its
            // output may overwrite them.  (A sync on both sides: one rendezvous per tile, neither warp runs a tile ahead.)
            if (b == 1 || b == 2) ptx::bar_sync(2, 64);
            if (b * 32 + 32 <= zero_from) {   // warp-uniform: every row of the batch is a valid token
#pragma unroll
                for (int c = 0; c < D / 16; ++c) {
                    uint4 lo, hi;
                    ptx::e4m3x4_to_f16x4(raw[c].x, lo.x, lo.y);
                    ptx::e4m3x4_to_f16x4(raw[c].y, lo.z, lo.w);
                    ptx::e4m3x4_to_f16x4(raw[c].z, hi.x, hi.y);
                    ptx::e4m3x4_to_f16x4(raw[c].w, hi.z, hi.w);
                    uint8_t *d = dst + (c >> 2) * 1024;
                    *reinterpret_cast<uint4 *>(d + ((((2 * c) & 7) << 4) ^ r7s)) = lo;
                    *reinterpret_cast<uint4 *>(d + ((((2 * c + 1) & 7) << 4) ^ r7s)) = hi;
                }
            } else {
                const uint32_t keep = (r < zero_from) ? 0xffffffffu : 0u;
#pragma unroll
                for (int c = 0; c < D / 16; ++c) {
                    uint4 lo, hi;
                    ptx::e4m3x4_to_f16x4(raw[c].x, lo.x, lo.y);
                    ptx::e4m3x4_to_f16x4(raw[c].y, lo.z, lo.w);
                    ptx::e4m3x4_to_f16x4(raw[c].z, hi.x, hi.y);
                    ptx::e4m3x4_to_f16x4(raw[c].w, hi.z, hi.w);
                    lo.x &= keep, lo.y &= keep, lo.z &= keep, lo.w &= keep;
                    hi.x &= keep, hi.y &= keep, hi.z &= keep, hi.w &= keep;
                    uint8_t *d = dst + (c >> 2) * 1024;
                    *reinterpret_cast<uint4 *>(d + ((((2 * c) & 7) << 4) ^ r7s)) = lo;
                    *reinterpret_cast<uint4 *>(d + ((((2 * c + 1) & 7) << 4) ^ r7s)) = hi;
                }
            }
            __syncwarp();
        }
        ptx::fence_proxy_async_smem();
        __syncwarp();
    };

    // register budget: launch gives kLaunchRegs x 384 threads.  The four service warps (warpgroup 0) hand theirs
    // down to kServiceRegs; each softmax thread, which holds a 128-wide score row, grows to kSoftmaxRegs.
    if (warp < 4) {
    // (setmaxnreg is a warpgroup-wide instruction: the four service warps take the same count)
    ptx::setmaxnreg_dec<kServiceRegs>();
    if (kFp8 && warp == 3) {
        // ===================== kFp8: V widening (the V slabs are requested by warp 0, right behind the K slabs) ====
        SegIter it(p, t0, t1);
        Seg s;
        int seg = 0, kproc = 0, cslot = 0;
        uint32_t cph = 0;
        while (next_seg(it, s, seg, kproc)) {
            for (int t = s.tb; t < s.te; ++t) {
                ptx::mbar_wait(ptx::smem_u32(&v_full[cslot]), cph);
                widen_tile(v_s + cslot * kTileBytes, s.u.n_load - t * kTile, 1);
                if (lane == 0) ptx::mbar_arrive(ptx::smem_u32(&v_conv[cslot]));
                if (++cslot == p.nv) {
                    cslot = 0;
                    cph ^= 1;
                }
            }
        }
    } else if (kFp8 && warp == 0) {
        // ===================== kFp8: K and V slab requests, page scales =====================
        // One warp requests both streams (a slab is requested as soon as its slot is free, never behind the widening
        // of another tile): K slabs into the six 16 KB slots of the K ring, V slabs into the upper half of the V
        // slots.  Lanes 0-7 / 8-15 also fetch the K / V scale of the tile's eight 16-column blocks and put them into
        // the scale ring BEFORE the arrive on the K barrier, so that whoever sees the K tile sees its scales.
        if constexpr (kFp8) {
            const uint64_t pol = ptx::policy_evict_first();
            int kslot = 0, vslot = 0, seg = 0, kproc = 0, ktile = 0;
            uint32_t kph = 0, vph = 0;
            SegIter it(p, t0, t1);
            Seg s;
            unsigned int yflag = (lane == 0) ? ptx::ld_volatile_global(p.yield_flag) : 0u;
            int ypoll = 0;   // tiles since launch: the flag is re-read every 8 tiles, ACROSS segments
            while (it.next(p, s)) {
                if (seg++ < skip) continue;
                int stop = 0;
                if (lane == 0) {
                    stop = (yflag == p.launch_seq) || (p.slice > 0 && kproc >= p.slice);
                    if (stop) ptx::st_release_cta_smem(&sched[1], kproc);
                    else ptx::st_release_cta_smem(&sched[0], kproc + 1);
                }
                stop = __shfl_sync(0xffffffffu, stop, 0);
                if (stop) break;
                ++kproc;
                const int n_pages_valid = (s.u.n_load + p.page - 1) >> p.page_shift;
                const int32_t *pt = p.a.page_table + static_cast<size_t>(s.u.session) * p.a.page_table_stride;
                const float *scl = (lane < 8 ? p.a.k_scale : p.a.v_scale) + static_cast<size_t>(s.layer) * p.a.scale_layer_stride;
                auto page_of = [&](int t) -> int {   // the page this lane requests of tile t
                    const int idx = t * pages_per_tile + lane;
                    return (t < s.te && lane < pages_per_tile && idx < n_pages_valid) ? __ldg(pt + idx) : -1;
                };
                auto scale_page_of = [&](int t) -> int {   // the page of this lane's 16-column block of tile t
                    const int idx = t * pages_per_tile + (((lane & 7) * 16) >> p.page_shift);
                    return (t < s.te && lane < 16 && idx < n_pages_valid) ? __ldg(pt + idx) : -1;
                };
                auto scale_of = [&](int pg) -> float {
                    return pg >= 0 ? __ldg(scl + static_cast<size_t>(pg) * p.Hkv + s.kvh) : 0.f;
                };
                int pg_next = page_of(s.tb);
                int spg_next = scale_page_of(s.tb + 1);
                float sc_next = scale_of(scale_page_of(s.tb));
                for (int t = s.tb; t < s.te; ++t) {
                    if (lane == 0 && (++ypoll & 7) == 0) yflag = ptx::ld_volatile_global(p.yield_flag);
                    const int pg = pg_next;
                    const float sc_now = sc_next;
                    pg_next = page_of(t + 1);
                    sc_next = scale_of(spg_next);
                    spg_next = scale_page_of(t + 2);
                    int nvp = n_pages_valid - t * pages_per_tile;
                    nvp = nvp < pages_per_tile ? nvp : pages_per_tile;
                    const int coord = (pg * p.Hkv + s.kvh) * p.page;
                    // ---- K
                    if (lane == 0) ptx::mbar_wait(ptx::smem_u32(&k_empty8[kslot]), kph ^ 1);
                    __syncwarp();
                    if (lane < 16) sc_s[(ktile & 7) * 16 + lane] = sc_now;
                    __syncwarp();
                    const uint32_t kfb = ptx::smem_u32(&k_full8[kslot]);
                    if (lane == 0) ptx::mbar_arrive_expect_tx(kfb, nvp * p.page * D);
                    __syncwarp();
                    if (pg >= 0)
                        ptx::tma_load_3d(ptx::smem_u32(k_s + kslot * kRawBytes + lane * p.page * D), &tm_k, kfb, 0, coord,
                                         s.layer, pol);
                    ++ktile;
                    if (++kslot == kNK8) {
                        kslot = 0;
                        kph ^= 1;
                    }
                    // ---- V
                    if (lane == 0) ptx::mbar_wait(ptx::smem_u32(&v_empty[vslot]), vph ^ 1);
                    __syncwarp();
                    const uint32_t vfb = ptx::smem_u32(&v_full[vslot]);
                    if (lane == 0) ptx::mbar_arrive_expect_tx(vfb, nvp * p.page * D);
                    __syncwarp();
                    if (pg >= 0)
                        ptx::tma_load_3d(ptx::smem_u32(v_s + vslot * kTileBytes + kRawBytes + lane * p.page * D), &tm_v, vfb, 0,
                                         coord, s.layer, pol);
                    if (++vslot == p.nv) {
                        vslot = 0;
                        vph ^= 1;
                    }
                }
            }
            if (lane == 0) sched[2] = skip + kproc;   // read after the CTA-wide barrier at the end
        }
    } else if (warp == 0 || warp == 3) {
        // ===================== K (warp 0) / V (warp 3) TMA producers =====================
        const bool is_v = (warp == 3);
        const CUtensorMap *tm = is_v ? &tm_v : &tm_k;
        const CUtensorMap *tmn = is_v ? &tm_vn : &tm_kn;
        uint64_t *full = is_v ? v_full : k_full, *empty = is_v ? v_empty : k_empty;
        uint8_t *ring = is_v ? v_s : k_s;
        const int n_slots = is_v ? p.nv : kNK;
        const uint64_t pol = ptx::policy_evict_first();   // the cache is streamed once per pass
        const uint64_t pol_new = ptx::policy_evict_last();  // entry K/V: just produced, re-read by every row chunk
        int slot = 0;
        uint32_t ph = 0;
        bool dep_waited = false;
        SegIter it(p, t0, t1);
        Seg s;
        int seg = 0, kproc = 0;
        // the yield flag is read ahead of its use (at launch, then every 8 tiles of the CTA's stream -- the count
        // carries across segments, so a CTA whose segments are all shorter than 8 tiles still sees a request within
        // 8 tiles): never a load on the critical path.  The flag names the launch it stops (its launch_seq): a request
        // that lands late, after its pass has ended, cannot stop a later pass or a resume.
        unsigned int yflag = (!is_v && lane == 0) ? ptx::ld_volatile_global(p.yield_flag) : 0u;
        int ypoll = 0;
        while (it.next(p, s)) {
            if (seg++ < skip) continue;
            if (!is_v) {
                int stop = 0;
                if (lane == 0) {
                    stop = (yflag == p.launch_seq) || (p.slice > 0 && kproc >= p.slice);
                    if (stop) ptx::st_release_cta_smem(&sched[1], kproc);
                    else ptx::st_release_cta_smem(&sched[0], kproc + 1);
                }
                stop = __shfl_sync(0xffffffffu, stop, 0);
                if (stop) break;
            } else if (!admitted(kproc)) {
                break;
            }
            ++kproc;
            const int n_pages_valid = (s.u.n_load + p.page - 1) >> p.page_shift;
            const int32_t *pt = p.a.page_table + static_cast<size_t>(s.u.session) * p.a.page_table_stride;
            // this lane's page of tile t (page-table reads run one tile ahead of the TMA issue)
            auto page_of = [&](int t) -> int {
                const int idx = t * pages_per_tile + lane;
                return (t < s.u.n_cached_tiles && lane < pages_per_tile && idx < n_pages_valid) ? __ldg(pt + idx) : -1;
            };
            int pg_next = page_of(s.tb);
            for (int t = s.tb; t < s.te; ++t) {
                if (!is_v && lane == 0 && (++ypoll & 7) == 0) yflag = ptx::ld_volatile_global(p.yield_flag);
                const int pg = pg_next;
                if (t + 1 < s.te) pg_next = page_of(t + 1);
                if (lane == 0) ptx::mbar_wait(ptx::smem_u32(&empty[slot]), ph ^ 1);
                __syncwarp();
                uint8_t *dst = ring + slot * kTileBytes;
                const uint32_t fb = ptx::smem_u32(&full[slot]);
                if (t < s.u.n_cached_tiles) {
                    int nvp = n_pages_valid - t * pages_per_tile;
                    nvp = nvp < pages_per_tile ? nvp : pages_per_tile;
                    if (lane == 0) ptx::mbar_arrive_expect_tx(fb, nvp * page_bytes);
                    __syncwarp();
                    if (pg >= 0)
                        ptx::tma_load_5d(ptx::smem_u32(dst + lane * page_bytes), tm, fb, 0, 0, 0,
                                         (pg * p.Hkv + s.kvh) * page_groups, s.layer, pol);
                } else {
                    if (early && !dep_waited) {   // K_new / V_new are the predecessor's business
                        ptx::griddep_wait();
                        dep_waited = true;
                    }
                    // entry-token tile: one box per 8 tokens straight from K_new / V_new.  Tokens past the ones this
                    // unit can see (later tokens, the next session's, or out of bounds = zero) are finite and masked
                    // by the softmax; V rows that no box covers are zeroed so that P = 0 never meets stale NaNs.
                    const int nb = (t - s.u.n_cached_tiles) * kTile;  // first entry token of this tile
                    int nvis = s.u.tok0 + s.u.ntok - nb;              // entry tokens this unit can see here
                    nvis = nvis < kTile ? nvis : kTile;
                    const int ng = (nvis + 7) >> 3;
                    if (is_v) {
                        for (int off = ng * kGroupStride + lane * 16; off < kTileBytes; off += 32 * 16)
                            *reinterpret_cast<uint4 *>(dst + off) = make_uint4(0, 0, 0, 0);
                        ptx::fence_proxy_async_smem();
                        __syncwarp();
                    }
                    if (lane == 0) ptx::mbar_arrive_expect_tx(fb, ng * kGroupStride);
                    __syncwarp();
                    if (lane < ng)
                        ptx::tma_load_5d(ptx::smem_u32(dst + lane * kGroupStride), tmn, fb, 0, s.u.row0 + nb + lane * 8, 0,
                                         s.kvh, s.layer, pol_new);
                }
                if (++slot == n_slots) {
                    slot = 0;
                    ph ^= 1;
                }
            }
        }
        if (!is_v && lane == 0) sched[2] = skip + kproc;   // read after the CTA-wide barrier at the end
    } else if (warp == 2) {
        // ===================== service warp: Q loader, Append(E), cross-CTA merge =====================
        SegIter it(p, t0, t1);
        Seg s;
        const uint64_t pol_q = ptx::policy_evict_last();  // Q is re-read by every CTA that shares the unit
        if (early) ptx::griddep_wait();   // Q, the appends and (kFp8) nothing else of this warp precede the predecessor's end
        int k = 0, seg = 0;
        int cslot = 0;   // kFp8: ring slot of the V tile being widened
        uint32_t cph = 0;
        while (it.next(p, s)) {
            if (seg++ < skip) continue;
            if (!admitted(k)) break;
            // ---- Q rows -> smem (swizzled K-major tiles) by TMA, as soon as the previous segment's last QK has read
            // the buffer.  Row r of the unit is entry token tok0 + r / G, query
            // head kvh * G + r % G; rows past the unit hold other tokens' Q or zeros and are never written out.
            if (k > 0) ptx::mbar_wait(ptx::smem_u32(q_empty), (k - 1) & 1);
            {
                // one TMA box per 8-row group: gbox = min(G, 8) heads x 8 / gbox tokens x both 64-column halves
                const int rows = s.u.ntok * G;
                const int ng = (rows + 7) >> 3;
                if (lane == 0) ptx::mbar_arrive_expect_tx(ptx::smem_u32(q_full), ng * kGroupStride);
                __syncwarp();
                for (int g = lane; g < ng; g += 32) {
                    int tok, head;
                    if (G <= 8) {
                        tok = s.u.tok0 + g * (8 / G);
                        head = s.kvh * G;
                    } else {
                        const int gpt = G >> 3;
                        tok = s.u.tok0 + g / gpt;
                        head = s.kvh * G + (g % gpt) * 8;
                    }
                    ptx::tma_load_5d(ptx::smem_u32(q_s + (g >> 4) * kTileBytes + (g & 15) * kGroupStride), &tm_q,
                                     ptx::smem_u32(q_full), 0, head, s.u.row0 + tok, 0, s.layer, pol_q);
                }
            }
            ++k;
            if constexpr (kFp8) {
                // ---- widen token rows 0-63 of the segment's V tiles as they land (warp 3 takes rows 64-127)
                for (int t = s.tb; t < s.te; ++t) {
                    ptx::mbar_wait(ptx::smem_u32(&v_full[cslot]), cph);
                    widen_tile(v_s + cslot * kTileBytes, s.u.n_load - t * kTile, 0);
                    if (lane == 0) ptx::mbar_arrive(ptx::smem_u32(&v_conv[cslot]));
                    if (++cslot == p.nv) {
                        cslot = 0;
                        cph ^= 1;
                    }
                }
            } else {
                // ---- Append(E) (Alg. 1 l.5): K_new / V_new -> the session's pages.  Owned by the CTA that runs the
                // last tile of the session's last row chunk, once per (layer, kv head).  Nothing in this launch reads
                // cache positions >= n_s, so the copy needs no ordering with the tiles.
                if (s.u.tok0 + s.u.ntok == s.u.l_entry && s.te == s.u.n_tiles) append_entry<D>(p, s, lane);
            }
        }
    } else if (warp == 1) {
        // ===================== MMA issuer =====================
        int kslot = 0, vslot = 0;
        uint32_t kph = 0, vph = 0, qph = 0;
        uint32_t pph = 0;  // bit w = phase parity of p_ready[w]
        SegIter it(p, t0, t1);
        Seg s;
        int seg = 0, kproc = 0;
        while (it.next(p, s)) {
            if (seg++ < skip) continue;
            if (!admitted(kproc)) break;
            ++kproc;
            const int rows = s.u.ntok * G;
            const int n_mt = rows > 128 ? 2 : 1;
            const int n_tiles = s.te - s.tb;
            const int n_items = n_tiles * n_mt;
            ptx::mbar_wait(ptx::smem_u32(kFp8 ? q_conv : q_full), qph);
            qph ^= 1;
            ptx::tc_fence_after();

            auto issue_qk = [&](int i) {
                const int w = i & 1;
                const int mt = (n_mt == 2) ? w : 0;
                const bool first_use = (n_mt == 1) || w == 0;
                const bool last_use = (n_mt == 1) || w == 1;
                if (first_use) {
                    ptx::mbar_wait(ptx::smem_u32(kFp8 ? &k_full8[kslot] : &k_full[kslot]), kph);
                    ptx::tc_fence_after();
                }
                // descriptor words are warp-uniform and computed by the whole warp; only the tcgen05 instructions sit
                // under elect (a lane-0 branch would drag every operand through ELECT + R2UR per MMA)
                const uint32_t qlo = desc_lo(ptx::smem_u32(q_s + mt * kTileBytes), 16);
                const uint32_t klo = desc_lo(ptx::smem_u32(k_s + kslot * (kFp8 ? kRawBytes : kTileBytes)), 16);
                const uint32_t sd = tmem + kColS + w * 128;
                const uint32_t sfb = ptx::smem_u32(&s_full[w]);
                const uint32_t keb = ptx::smem_u32(kFp8 ? &k_empty8[kslot] : &k_empty[kslot]);
                const bool q_last = (i == n_items - 1);
                if (ptx::elect_one()) {
                    if constexpr (kFp8) {
                        // S = Qh K^T + Ql K^T on the 8-bit path: Qh in the first, Ql in the second 16 KB of the M-tile's
                        // buffer, each [row][128 B] like the K slab; 32 elements (32 bytes) per instruction
#pragma unroll
                        for (int part = 0; part < 2; ++part)
#pragma unroll
                            for (int ks = 0; ks < 4; ++ks) {
                                const uint32_t off = (ks * 32) >> 4;
                                ptx::umma_ss2_f8(sd, qlo + ((part * kRawBytes) >> 4) + off, klo + off, kDescHi8, kIdescQK8,
                                                 (part | ks) != 0);
                            }
                    } else {
#pragma unroll
                    for (int hf = 0; hf < kHalves; ++hf)
#pragma unroll
                        for (int ks = 0; ks < 4; ++ks) {
                            const uint32_t off = (hf * 1024 + ks * 32) >> 4;
                            ptx::umma_ss2(sd, qlo + off, klo + off, kDescHi, kIdescQK, (hf | ks) != 0);
                        }
                    }
                    ptx::umma_commit(sfb);
                    if (last_use) ptx::umma_commit(keb);
                    if (q_last) ptx::umma_commit(ptx::smem_u32(q_empty));  // Q may be overwritten
                }
                __syncwarp();
                if (last_use) {
                    if (++kslot == (kFp8 ? kNK8 : kNK)) {
                        kslot = 0;
                        kph ^= 1;
                    }
                }
            };

            issue_qk(0);
            if (n_items > 1) issue_qk(1);
            for (int i = 0; i < n_items; ++i) {
                const int w = i & 1;
                const int t = s.tb + (n_mt == 2 ? (i >> 1) : i);
                const bool first_use = (n_mt == 1) || w == 0;
                const bool last_use = (n_mt == 1) || w == 1;
                if (first_use && kFp8) {
                    ptx::mbar_wait(ptx::smem_u32(&v_conv[vslot]), vph);   // widened, rows past the valid tokens zeroed
                } else if (first_use) {
                    ptx::mbar_wait(ptx::smem_u32(&v_full[vslot]), vph);
                    // rows past the valid tokens of a ragged cached tile hold whatever the pool / the ring held, and the
                    // last 8-token box of an entry tile reaches into rows of later tokens or of the NEXT session (which
                    // the caller may never have initialised, e.g. a budget-skipped neighbour): P is exactly 0 there,
                    // but 0 * NaN would poison O, so zero them before the MMA reads them.
                    int valid, zero_to;
                    if (t < s.u.n_cached_tiles) {
                        valid = s.u.n_load - t * kTile;
                        zero_to = kTile;
                    } else {
                        valid = s.u.tok0 + s.u.ntok - (t - s.u.n_cached_tiles) * kTile;
                        zero_to = ((valid + 7) >> 3) << 3;   // the producer zeroed every row no box covers
                    }
                    zero_to = zero_to < kTile ? zero_to : kTile;
                    if (valid < zero_to) {
                        uint8_t *vb = v_s + vslot * kTileBytes;
                        for (int idx = valid * (D / 8) + lane; idx < zero_to * (D / 8); idx += 32) {
                            const int r = idx / (D / 8), c = idx - r * (D / 8);
                            *reinterpret_cast<uint4 *>(vb + tile_offset<D>(r, c)) = make_uint4(0, 0, 0, 0);
                        }
                        ptx::fence_proxy_async_smem();
                        __syncwarp();
                    }
                }
                ptx::mbar_wait(ptx::smem_u32(&p_ready[w]), (pph >> w) & 1u);
                pph ^= 1u << w;
                ptx::tc_fence_after();
                const uint32_t vlo = desc_lo(ptx::smem_u32(v_s + vslot * kTileBytes), 1024);
                const uint32_t od = tmem + kColO + w * D, pa = tmem + kColS + w * 128;
                const uint32_t veb = ptx::smem_u32(&v_empty[vslot]);
                const uint32_t first_pv = (i < 2) ? 0u : 1u;  // first PV of stream i & 1 in this segment overwrites O
                if (ptx::elect_one()) {
#pragma unroll
                    for (int ks = 0; ks < kTile / 16; ++ks)
                        ptx::umma_ts2(od, pa + ks * 8, vlo + ((ks * 2 * kGroupStride) >> 4), kDescHi, kIdescPV,
                                      ks == 0 ? first_pv : 1u);
                    if (last_use) ptx::umma_commit(veb);
                }
                __syncwarp();
                if (last_use) {
                    if (++vslot == p.nv) {
                        vslot = 0;
                        vph ^= 1;
                    }
                }
                if (i + 2 < n_items) issue_qk(i + 2);
            }
            if (ptx::elect_one()) {
                ptx::umma_commit(ptx::smem_u32(&o_done[0]));
                ptx::umma_commit(ptx::smem_u32(&o_done[1]));
            }
            __syncwarp();
        }
    }
    } else {
        ptx::setmaxnreg_inc<kSoftmaxRegs>();
        if (early) ptx::griddep_wait();   // out, the partial slots and the counters are shared with the predecessor
        // ===================== softmax warpgroups (warps 4-7: stream 0, warps 8-11: stream 1) =====================
        const int w = (warp - 4) >> 2;
        const int row = ((warp & 3) << 5) | lane;              // TMEM lane == row within the M-tile
        const uint32_t lane_addr = static_cast<uint32_t>((warp & 3) << 5) << 16;
        const int st = threadIdx.x - 128;                      // 0..255 among softmax threads
        uint32_t sph = 0, oph = 0;
        uint32_t qph = 0;      // kFp8: parity of q_full
        int ktile_base = 0;    // kFp8: K tiles of the segments before this one (index of the scale ring)
        SegIter it(p, t0, t1);
        Seg s;
        int seg = 0, kproc = 0;
        while (it.next(p, s)) {
            if (seg++ < skip) continue;
            if (!admitted(kproc)) break;
            ++kproc;
            const int rows = s.u.ntok * G;
            const int n_mt = rows > 128 ? 2 : 1;
            const int n_tiles = s.te - s.tb;
            const int n_items = n_tiles * n_mt;
            const int mt = (n_mt == 2) ? w : 0;
            const int urow = mt * 128 + row;                   // row within the unit
            const int my_tok = s.u.tok0 + urow / G;            // entry token of this row (if urow < rows)
            const bool row_valid = urow < rows;
            float srow = p.scale_log2;   // kFp8: softmax scale x log2(e) x 2^-k of this thread's row
            if constexpr (kFp8) {
                // Q arrived as bf16 (8 significant bits): split it exactly into two e4m3 operands, in place.  The thread
                // owns its query row: 2^k brings the row's max|q| into [128, 256); Qh = q with the mantissa truncated
                // to 3 bits, Ql = q - Qh (at most 4 significant bits), both x 2^k; 2^-k goes into the softmax scale.
                // Qh fills the first, Ql the second 16 KB of the M-tile's buffer, [row][128 B] with the 128-byte swizzle.
                ptx::mbar_wait(ptx::smem_u32(q_full), qph);
                qph ^= 1;
                const bool conv = (n_mt == 2) || (w == 0);
                uint8_t *qt = q_s + mt * kTileBytes;
                uint4 qr[D / 8];
                if (conv) {
#pragma unroll
                    for (int c = 0; c < D / 8; ++c) qr[c] = *reinterpret_cast<const uint4 *>(qt + tile_offset<D>(row, c));
                }
                ptx::bar_sync(1, 256);   // every row is in registers before the buffer is rewritten
                float rowf = 1.f;
                if (conv) {
                    uint32_t amax_bits = 0u;   // max over |x| as bf16 bit patterns (monotone in the magnitude)
#pragma unroll
                    for (int c = 0; c < D / 8; ++c) {
                        const uint32_t wds[4] = {qr[c].x, qr[c].y, qr[c].z, qr[c].w};
#pragma unroll
                        for (int i = 0; i < 4; ++i) {
                            amax_bits = max(amax_bits, (wds[i] << 16) & 0x7fff0000u);
                            amax_bits = max(amax_bits, wds[i] & 0x7fff0000u);
                        }
                    }
                    int k = amax_bits ? 7 + 127 - static_cast<int>(amax_bits >> 23) : 0;
                    k = k < -100 ? -100 : (k > 100 ? 100 : k);
                    const float up = __int_as_float((k + 127) << 23);
                    rowf = __int_as_float((127 - k) << 23);
                    uint8_t *qrow = qt + (row >> 3) * 1024 + (row & 7) * 128;
                    const uint32_t r7s = static_cast<uint32_t>(row & 7) << 4;
#pragma unroll
                    for (int c = 0; c < D / 16; ++c) {   // 16 elements = two bf16 chunks -> one 16-byte chunk of each part
                        const uint32_t wds[8] = {qr[2 * c].x, qr[2 * c].y, qr[2 * c].z, qr[2 * c].w,
                                                 qr[2 * c + 1].x, qr[2 * c + 1].y, qr[2 * c + 1].z, qr[2 * c + 1].w};
                        uint32_t ph[4], pl[4];
#pragma unroll
                        for (int i = 0; i < 4; ++i) {
                            uint32_t hh = 0u, ll = 0u;
#pragma unroll
                            for (int j = 0; j < 2; ++j) {
                                const uint32_t wd = wds[2 * i + j];
                                const float x0 = __uint_as_float(wd << 16), x1 = __uint_as_float(wd & 0xffff0000u);
                                const float h0 = __uint_as_float((wd << 16) & 0xfff00000u), h1 = __uint_as_float(wd & 0xfff00000u);
                                hh |= ptx::pack_e4m3x2(h0 * up, h1 * up) << (16 * j);
                                ll |= ptx::pack_e4m3x2((x0 - h0) * up, (x1 - h1) * up) << (16 * j);
                            }
                            ph[i] = hh;
                            pl[i] = ll;
                        }
                        *reinterpret_cast<uint4 *>(qrow + ((c << 4) ^ r7s)) = make_uint4(ph[0], ph[1], ph[2], ph[3]);
                        *reinterpret_cast<uint4 *>(qrow + kRawBytes + ((c << 4) ^ r7s)) = make_uint4(pl[0], pl[1], pl[2], pl[3]);
                    }
                    if (n_mt == 1) rowf_s[row] = rowf;
                }
                ptx::fence_proxy_async_smem();
                ptx::bar_sync(1, 256);
                if (st == 0) ptx::mbar_arrive(ptx::smem_u32(q_conv));
                if (n_mt == 1 && w == 1) rowf = rowf_s[row];
                srow = p.scale_log2 * rowf;
            }
            float m_used = -CUDART_INF_F, l_sum = 0.f;
            bool have = false;
            for (int i = w; i < n_items; i += 2) {
                const int t = s.tb + (n_mt == 2 ? (i >> 1) : i);
                // visible columns of this tile for this row
                int limit = kTile;
                if (t < s.u.n_cached_tiles) {
                    const int valid = s.u.n_load - t * kTile;
                    limit = valid < kTile ? valid : kTile;
                    if constexpr (kFp8) {
                        // the entry tokens sit in the cache: row i sees keys j <= n_s + i (reading Q5)
                        const int causal = (urow < rows) ? s.u.n_s + my_tok + 1 - t * kTile : kTile;
                        limit = causal < limit ? (causal < 0 ? 0 : causal) : limit;
                    }
                } else {
                    const int nb = (t - s.u.n_cached_tiles) * kTile;
                    limit = (urow < rows) ? my_tok - nb + 1 : 1;   // causal among the entry tokens (reading Q5)
                    limit = limit < 0 ? 0 : (limit > kTile ? kTile : limit);
                }
                ptx::mbar_wait(ptx::smem_u32(&s_full[w]), sph);
                sph ^= 1;
                ptx::tc_fence_after();
                // The tile body exists twice (all columns visible / masked at `limit`): one body with a branch
                // around the masking makes the compiler copy the whole 128-register score row at the join.
                auto tile_body = [&](auto masked_tag) {
                    constexpr bool kMasked = decltype(masked_tag)::value;
                    uint32_t sr[128];
                    {
                        const uint32_t sa = tmem + lane_addr + kColS + w * 128;
                        ptx::tmem_ld_32x32b_x32(sa, sr);
                        ptx::tmem_ld_32x32b_x32(sa + 32, sr + 32);
                        ptx::tmem_ld_32x32b_x32(sa + 64, sr + 64);
                        ptx::tmem_ld_32x32b_x32(sa + 96, sr + 96);
                        ptx::tmem_ld_wait();
                    }
                    float mx = -CUDART_INF_F;
                    if constexpr (kMasked) {
#pragma unroll
                        for (int c = 0; c < 128; ++c) {
                            const float v = (c < limit) ? __uint_as_float(sr[c]) : -CUDART_INF_F;
                            sr[c] = __float_as_uint(v);
                            mx = fmaxf(mx, v);
                        }
                    } else {
                        // four independent chains (one chain of 64 three-input maxima is ~300 cycles of latency)
                        float m1 = -CUDART_INF_F, m2 = -CUDART_INF_F, m3 = -CUDART_INF_F;
#pragma unroll
                        for (int c = 0; c < 128; c += 8) {
                            mx = fmaxf(fmaxf(mx, __uint_as_float(sr[c])), __uint_as_float(sr[c + 1]));
                            m1 = fmaxf(fmaxf(m1, __uint_as_float(sr[c + 2])), __uint_as_float(sr[c + 3]));
                            m2 = fmaxf(fmaxf(m2, __uint_as_float(sr[c + 4])), __uint_as_float(sr[c + 5]));
                            m3 = fmaxf(fmaxf(m3, __uint_as_float(sr[c + 6])), __uint_as_float(sr[c + 7]));
                        }
                        mx = fmaxf(fmaxf(mx, m1), fmaxf(m2, m3));
                    }
                    const float m_new = fmaxf(m_used, mx * p.scale_log2);
                    // lazy rescale, warp-uniform because the TMEM round trip of O is warp-collective.  Only rows of the
                    // unit vote: a row past them holds whatever the Q buffer held before (another segment's, or another
                    // launch's after a resume), and its maximum must not decide WHEN the valid rows of its warp rescale
                    // -- the result would stay within tolerance but depend on what ran on the SM before.
                    const bool need = row_valid && (m_new > m_used + kRescaleThreshold);
                    if (__any_sync(0xffffffffu, need)) {
                        const float alpha = (m_used == -CUDART_INF_F) ? 0.f : exp2f(m_used - m_new);
                        l_sum *= alpha;
                        if (have) {
                            const uint32_t oa = tmem + lane_addr + kColO + w * D;
#pragma unroll 1
                            for (int cb = 0; cb < D; cb += 32) {
                                uint32_t o[32];
                                ptx::tmem_ld_32x32b_x32(oa + cb, o);
                                ptx::tmem_ld_wait();
#pragma unroll
                                for (int c = 0; c < 32; ++c) o[c] = __float_as_uint(__uint_as_float(o[c]) * alpha);
                                ptx::tmem_st_32x32b_x32(oa + cb, o);
                            }
                        }
                        m_used = m_new;
                    }
                    const float m_eff = (m_used == -CUDART_INF_F) ? 0.f : m_used;  // fully masked so far: p = 0
                    const float neg_m = -m_eff;
                    const uint32_t pa = tmem + lane_addr + kColS + w * 128;
                    // packed fp32 pairs: one FFMA2 scales two scores, one FADD2 adds two probabilities to the row sum
                    const uint64_t sc2 = ptx::pack_f32x2(p.scale_log2, p.scale_log2), nm2 = ptx::pack_f32x2(neg_m, neg_m);
                    uint64_t acc_a = 0ull, acc_b = 0ull;
#pragma unroll
                    for (int cb = 0; cb < 128; cb += 32) {
                        uint32_t pk[16];
#pragma unroll
                        for (int c = 0; c < 32; c += 2) {
                            const uint64_t x2 = ptx::fma_f32x2(
                                ptx::pack_f32x2(__uint_as_float(sr[cb + c]), __uint_as_float(sr[cb + c + 1])), sc2, nm2);
                            float x0, x1;
                            ptx::unpack_f32x2(x2, x0, x1);
                            // every fourth pair of a fully visible tile takes its exp2 on the FMA pipe: the XU
                            // (MUFU.EX2, 4 lanes per scheduler) is a co-limit of the tensor-bound shapes
                            const bool poly = !kMasked && ((c >> 1) & 3) == 3;   // measured on config 5: 0% 2.10, 25% 1.83, 37.5% 1.86, 50% 2.05 Mcycles
                            float p0, p1;
                            if (poly) {
                                ptx::ex2_poly2(x0, x1, p0, p1);
                            } else {
                                p0 = ptx::ex2(x0);
                                p1 = ptx::ex2(x1);
                            }
                            if (c & 2) acc_b = ptx::add_f32x2(acc_b, ptx::pack_f32x2(p0, p1));
                            else acc_a = ptx::add_f32x2(acc_a, ptx::pack_f32x2(p0, p1));
                            pk[c >> 1] = pack_bf16(p0, p1);
                        }
                        ptx::tmem_st_32x32b_x16(pa + (cb >> 1), pk);
                    }
                    float a0, a1;
                    ptx::unpack_f32x2(ptx::add_f32x2(acc_a, acc_b), a0, a1);
                    l_sum += a0 + a1;
                };
                // kFp8: the same body with the K scale of each 16-column block in the scale FMA (and in the maximum,
                // block by block) and the V scale on the probabilities before they are packed (fp16)
                auto tile_body_q = [&](auto masked_tag) {
                    constexpr bool kMasked = decltype(masked_tag)::value;
                    // the tile's scales: [0..7] K (times the softmax scale and 2^-k of the row below), [8..15] V; read
                    // where they are used (broadcast shared-memory loads) rather than held in 16 registers
                    const float *scb = sc_s + ((ktile_base + (t - s.tb)) & 7) * 16;
                    uint32_t sr[128];
                    {
                        const uint32_t sa = tmem + lane_addr + kColS + w * 128;
                        ptx::tmem_ld_32x32b_x32(sa, sr);
                        ptx::tmem_ld_32x32b_x32(sa + 32, sr + 32);
                        ptx::tmem_ld_32x32b_x32(sa + 64, sr + 64);
                        ptx::tmem_ld_32x32b_x32(sa + 96, sr + 96);
                        ptx::tmem_ld_wait();
                    }
                    float mx = -CUDART_INF_F;
#pragma unroll
                    for (int b = 0; b < 8; ++b) {
                        float m0 = -CUDART_INF_F, m1 = -CUDART_INF_F;
#pragma unroll
                        for (int c = b * 16; c < b * 16 + 16; c += 2) {
                            if constexpr (kMasked) {
                                if (c >= limit) sr[c] = __float_as_uint(-CUDART_INF_F);
                                if (c + 1 >= limit) sr[c + 1] = __float_as_uint(-CUDART_INF_F);
                            }
                            m0 = fmaxf(m0, __uint_as_float(sr[c]));
                            m1 = fmaxf(m1, __uint_as_float(sr[c + 1]));
                        }
                        const float mb = fmaxf(m0, m1);
                        // a block with no visible column has max -inf (and, past the valid pages, scale 0)
                        if (mb != -CUDART_INF_F) mx = fmaxf(mx, mb * (scb[b] * srow));
                    }
                    const float m_new = fmaxf(m_used, mx);
                    const bool need = row_valid && (m_new > m_used + kRescaleThreshold);   // as in tile_body: valid rows vote
                    if (__any_sync(0xffffffffu, need)) {
                        const float alpha = (m_used == -CUDART_INF_F) ? 0.f : exp2f(m_used - m_new);
                        l_sum *= alpha;
                        if (have) {
                            const uint32_t oa = tmem + lane_addr + kColO + w * D;
#pragma unroll 1
                            for (int cb = 0; cb < D; cb += 32) {
                                uint32_t o[32];
                                ptx::tmem_ld_32x32b_x32(oa + cb, o);
                                ptx::tmem_ld_wait();
#pragma unroll
                                for (int c = 0; c < 32; ++c) o[c] = __float_as_uint(__uint_as_float(o[c]) * alpha);
                                ptx::tmem_st_32x32b_x32(oa + cb, o);
                            }
                        }
                        m_used = m_new;
                    }
                    const float m_eff = (m_used == -CUDART_INF_F) ? 0.f : m_used;
                    const float neg_m = -m_eff;
                    const uint32_t pa = tmem + lane_addr + kColS + w * 128;
                    const uint64_t nm2 = ptx::pack_f32x2(neg_m, neg_m);
                    uint64_t acc_a = 0ull, acc_b = 0ull;
#pragma unroll
                    for (int cb = 0; cb < 128; cb += 32) {
                        uint32_t pk[16];
#pragma unroll
                        for (int c = 0; c < 32; c += 2) {
                            const int b = (cb + c) >> 4;
                            const float ksb = scb[b] * srow, vsb = scb[8 + b];
                            float x0, x1;
                            if constexpr (kMasked) {
                                // a masked score is -inf and its block's scale may be 0: keep it -inf, not NaN
                                const float s0 = __uint_as_float(sr[cb + c]), s1 = __uint_as_float(sr[cb + c + 1]);
                                x0 = (s0 == -CUDART_INF_F) ? -CUDART_INF_F : fmaf(s0, ksb, neg_m);
                                x1 = (s1 == -CUDART_INF_F) ? -CUDART_INF_F : fmaf(s1, ksb, neg_m);
                            } else {
                                const uint64_t x2 = ptx::fma_f32x2(
                                    ptx::pack_f32x2(__uint_as_float(sr[cb + c]), __uint_as_float(sr[cb + c + 1])),
                                    ptx::pack_f32x2(ksb, ksb), nm2);
                                ptx::unpack_f32x2(x2, x0, x1);
                            }
                            const bool poly = !kMasked && ((c >> 1) & 3) == 3;   // every fourth pair on the FMA pipe, as above
                            float p0, p1;
                            if (poly) {
                                ptx::ex2_poly2(x0, x1, p0, p1);
                            } else {
                                p0 = ptx::ex2(x0);
                                p1 = ptx::ex2(x1);
                            }
                            if (c & 2) acc_b = ptx::add_f32x2(acc_b, ptx::pack_f32x2(p0, p1));
                            else acc_a = ptx::add_f32x2(acc_a, ptx::pack_f32x2(p0, p1));
                            pk[c >> 1] = ptx::pack_f16x2(p0 * vsb, p1 * vsb);
                        }
                        ptx::tmem_st_32x32b_x16(pa + (cb >> 1), pk);
                    }
                    float a0, a1;
                    ptx::unpack_f32x2(ptx::add_f32x2(acc_a, acc_b), a0, a1);
                    l_sum += a0 + a1;
                };
                // the choice must be warp-uniform (the bodies hold warp-collective TMEM accesses and votes), and the
                // causal limit is per row: a tile is "fully visible" only if it is so for all 32 rows of the warp
                const bool all_visible = __all_sync(0xffffffffu, limit >= kTile);
                // A warp whose 32 rows all lie past the unit's rows (64 or 96 query rows in a 128-row M-tile) has nothing to
                // compute: its P rows stay whatever S left there, and the O rows they produce are never read (a row of
                // O depends on its own row of P only).  It still keeps step with the tiles through the barriers.
                const bool warp_dead = (mt * 128 + (warp & 3) * 32) >= rows;
                if (warp_dead) {
                } else if constexpr (kFp8) {
                    if (all_visible) tile_body_q(std::false_type{});
                    else tile_body_q(std::true_type{});
                } else {
                    if (all_visible) tile_body(std::false_type{});
                    else tile_body(std::true_type{});
                }
                ptx::tmem_st_wait();
                ptx::tc_fence_before();
                ptx::mbar_arrive(ptx::smem_u32(&p_ready[w]));
                have = true;
            }
            if constexpr (kFp8) ktile_base += n_tiles;
            // ---- epilogue
            ptx::mbar_wait(ptx::smem_u32(&o_done[w]), oph);
            oph ^= 1;
            ptx::tc_fence_after();
            __nv_bfloat16 *ob = p.a.out + static_cast<size_t>(s.layer) * p.a.out_layer_stride;
            float *slot = p.partials + static_cast<size_t>(2 * blockIdx.x + s.slot) * (kAttnMaxRows * (D + 2));
            if (n_mt == 2) {
                // stream w owns M-tile w: rows urow, all D columns.  A row that saw no column in this segment (a cut
                // segment made only of a later entry tile: G = 1 units span two entry tiles) contributes a zero partial
                // with log-sum-exp -inf, which the merges weigh with 0.
                const bool seen = l_sum > 0.f;
                const float inv = seen ? 1.f / l_sum : 0.f;
                const bool live = urow < rows;
                const uint32_t oa = tmem + lane_addr + kColO + w * D;
                __nv_bfloat16 *orow = ob + (static_cast<size_t>(s.u.row0 + my_tok) * p.Hq + s.kvh * G + urow % G) * D;
#pragma unroll
                for (int cb = 0; cb < D; cb += 32) {
                    uint32_t o[32];
                    ptx::tmem_ld_32x32b_x32(oa + cb, o);
                    ptx::tmem_ld_wait();
                    if (!seen) {
#pragma unroll
                        for (int c = 0; c < 32; ++c) o[c] = 0u;
                    }
                    if (live) {
                        if (s.direct) {
#pragma unroll
                            for (int c = 0; c < 32; c += 8) {
                                uint4 v;
                                v.x = pack_bf16(__uint_as_float(o[c]) * inv, __uint_as_float(o[c + 1]) * inv);
                                v.y = pack_bf16(__uint_as_float(o[c + 2]) * inv, __uint_as_float(o[c + 3]) * inv);
                                v.z = pack_bf16(__uint_as_float(o[c + 4]) * inv, __uint_as_float(o[c + 5]) * inv);
                                v.w = pack_bf16(__uint_as_float(o[c + 6]) * inv, __uint_as_float(o[c + 7]) * inv);
                                *reinterpret_cast<uint4 *>(orow + cb + c) = v;
                            }
                        } else {
#pragma unroll
                            for (int c = 0; c < 32; c += 4)
                                reinterpret_cast<float4 *>(slot)[static_cast<size_t>((cb + c) >> 2) * kAttnMaxRows + urow] =
                                    make_float4(__uint_as_float(o[c]) * inv, __uint_as_float(o[c + 1]) * inv,
                                                __uint_as_float(o[c + 2]) * inv, __uint_as_float(o[c + 3]) * inv);
                        }
                    }
                }
                if (live && !s.direct) slot[kAttnMaxRows * D + urow] = seen ? m_used + log2f(l_sum) : -CUDART_INF_F;
            } else {
                // both streams hold partial sums of the same rows: exchange (m, l), then WG w finishes columns
                // [w * D/2, (w+1) * D/2) of the merged row
                // (one 1 KB array both ways: stream 1 hands (m, l) to stream 0, which hands back the two row factors)
                const bool two = n_items > 1;
                if (w == 1) ml_x[row] = make_float2(m_used, l_sum);
                ptx::bar_sync(1, 256);
                float fa, fb, lse2 = 0.f;
                if (w == 0) {
                    const float2 b = ml_x[row];
                    const float M = two ? fmaxf(m_used, b.x) : m_used;
                    if (M == -CUDART_INF_F) {   // the row saw no column in this segment: zero partial, lse -inf
                        fa = fb = 0.f;
                        lse2 = -CUDART_INF_F;
                    } else {
                        const float wa = exp2f(m_used - M), wb = two ? exp2f(b.x - M) : 0.f;
                        const float L = wa * l_sum + wb * b.y;
                        const float inv = 1.f / L;
                        fa = wa * inv;
                        fb = wb * inv;
                        lse2 = M + log2f(L);
                    }
                    ml_x[row] = make_float2(fa, fb);
                }
                ptx::bar_sync(1, 256);
                if (w == 1) {
                    const float2 f2 = ml_x[row];
                    fa = f2.x;
                    fb = f2.y;
                }
                const bool live = row < rows;
                constexpr int kHalfD = D / 2;
                const uint32_t oa0 = tmem + lane_addr + kColO + w * kHalfD;
                const uint32_t oa1 = tmem + lane_addr + kColO + D + w * kHalfD;
                const int tok = s.u.tok0 + row / G;
                __nv_bfloat16 *orow = ob + (static_cast<size_t>(s.u.row0 + tok) * p.Hq + s.kvh * G + row % G) * D + w * kHalfD;
#pragma unroll
                for (int cb = 0; cb < kHalfD; cb += 32) {
                    uint32_t o0[32], o1[32];
                    ptx::tmem_ld_32x32b_x32(oa0 + cb, o0);
                    if (two) ptx::tmem_ld_32x32b_x32(oa1 + cb, o1);
                    ptx::tmem_ld_wait();
                    float f[32];
#pragma unroll
                    for (int c = 0; c < 32; ++c)
                        f[c] = two ? fmaf(__uint_as_float(o0[c]), fa, __uint_as_float(o1[c]) * fb)
                                   : __uint_as_float(o0[c]) * fa;
                    if (live) {
                        if (s.direct) {
#pragma unroll
                            for (int c = 0; c < 32; c += 8) {
                                uint4 v;
                                v.x = pack_bf16(f[c], f[c + 1]);
                                v.y = pack_bf16(f[c + 2], f[c + 3]);
                                v.z = pack_bf16(f[c + 4], f[c + 5]);
                                v.w = pack_bf16(f[c + 6], f[c + 7]);
                                *reinterpret_cast<uint4 *>(orow + cb + c) = v;
                            }
                        } else {
#pragma unroll
                            for (int c = 0; c < 32; c += 4)
                                reinterpret_cast<float4 *>(slot)[static_cast<size_t>((w * kHalfD + cb + c) >> 2) * kAttnMaxRows + row] =
                                    make_float4(f[c], f[c + 1], f[c + 2], f[c + 3]);
                        }
                    }
                }
                if (live && !s.direct && w == 0) slot[kAttnMaxRows * D + row] = lse2;
                ptx::bar_sync(1, 256);  // ml_x is reused by the next segment
            }
            // ---- the single cross-CTA pass: the last CTA to deliver its partial of a cut unit combines them
            if (!s.direct) {
                const long long U0s = static_cast<long long>(s.lh) * p.tiles_per_lh + s.u.tile_prefix;
                const int c0s = cta_of(p, gridDim.x, U0s);
                const int c1s = cta_of(p, gridDim.x, U0s + s.u.n_tiles - 1);
                // up to kLastArriverMax partials: the last CTA to arrive combines them right here.  More (a unit spread
                // over many CTAs, e.g. one launch per layer): the partials are complete when this kernel ends and
                // attn_merge_kernel, launched right behind it, combines them -- no ticket, and no CTA ever waits for
                // another one.
                if (c1s - c0s >= kLastArriverMax) continue;
                // the barrier orders every thread's partial stores before thread 0's release fence + ticket
                ptx::bar_sync(1, 256);
                if (st == 0) {
                    unsigned int *cnt = p.counters + static_cast<size_t>(s.lh) * p.a.n_units + s.unit_idx;
                    ptx::fence_acq_rel_gpu();
                    const unsigned int prev = atomicAdd(cnt, 1u);
                    const bool last = (prev == static_cast<unsigned int>(c1s - c0s));
                    if (last) {
                        *cnt = 0u;  // self-reset for the next launch
                        ptx::fence_acq_rel_gpu();
                    }
                    merge_info[0] = last ? c0s : -1;
                    merge_info[1] = c1s;
                    merge_info[2] = (cta_begin(p, gridDim.x, c0s) < U0s) ? 1 : 0;  // c0's slot for this unit
                }
                ptx::bar_sync(1, 256);
                const int c0 = merge_info[0], c1 = merge_info[1], c0_slot = merge_info[2];
                if (c0 >= 0) {
                    constexpr int kVec = D / 4;  // float4 per row
                    constexpr int kMaxC = kLastArriverMax;  // partials combined with all loads in flight
                    constexpr size_t kSlotFloats = static_cast<size_t>(kAttnMaxRows) * (D + 2);
                    const float *base0 = p.partials + (2 * static_cast<size_t>(c0) + c0_slot) * kSlotFloats;
                    const int nc = c1 - c0 + 1;
                    constexpr int kU = 4;  // rows x float4 columns per thread and pass: kU * 2 * nc loads in flight
                    const int total = rows * kVec;
                    auto store_row = [&](int idx, const float4 &acc, float wsum) {
                        const int v = idx / rows, r = idx - v * rows;
                        const float inv = 1.f / wsum;
                        const int tok = s.u.tok0 + r / G, h = s.kvh * G + r % G;
                        uint2 pk;
                        pk.x = pack_bf16(acc.x * inv, acc.y * inv);
                        pk.y = pack_bf16(acc.z * inv, acc.w * inv);
                        *reinterpret_cast<uint2 *>(ob + (static_cast<size_t>(s.u.row0 + tok) * p.Hq + h) * D + v * 4) = pk;
                    };
                    // all loads of a pass are issued before the first use: one L2 round trip (~2 us under a full HBM
                    // stream) per pass.  Two partials (the common cut) take 12 rows per thread and pass, i.e. one pass
                    // for up to 96 rows; up to four partials take 4.
                    auto merge_pass = [&](auto ku_tag, auto kc_tag) {
                        constexpr int kU_ = decltype(ku_tag)::value, kC_ = decltype(kc_tag)::value;
                        for (int idx0 = st; idx0 < total; idx0 += 256 * kU_) {
                            float lse[kU_][kC_];
                            float4 o[kU_][kC_];
#pragma unroll
                            for (int u = 0; u < kU_; ++u) {
                                const int idx = idx0 + u * 256;
                                const int v = idx / rows, r = idx - v * rows;   // lanes run along the rows
#pragma unroll
                                for (int j = 0; j < kC_; ++j) {
                                    const float *sl = (j == 0) ? base0 : p.partials + 2 * static_cast<size_t>(c0 + j) * kSlotFloats;
                                    lse[u][j] = -CUDART_INF_F;
                                    o[u][j] = make_float4(0.f, 0.f, 0.f, 0.f);
                                    if (j < nc && idx < total) {
                                        lse[u][j] = __ldcg(sl + kAttnMaxRows * D + r);
                                        o[u][j] = __ldcg(reinterpret_cast<const float4 *>(sl) + static_cast<size_t>(v) * kAttnMaxRows + r);
                                    }
                                }
                            }
#pragma unroll
                            for (int u = 0; u < kU_; ++u) {
                                const int idx = idx0 + u * 256;
                                if (idx >= total) continue;
                                float M = lse[u][0];
#pragma unroll
                                for (int j = 1; j < kC_; ++j) M = fmaxf(M, lse[u][j]);
                                float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
                                float wsum = 0.f;
#pragma unroll
                                for (int j = 0; j < kC_; ++j) {  // CTA order
                                    const float wgt = (j < nc && lse[u][j] != -CUDART_INF_F) ? exp2f(lse[u][j] - M) : 0.f;
                                    acc.x = fmaf(wgt, o[u][j].x, acc.x);
                                    acc.y = fmaf(wgt, o[u][j].y, acc.y);
                                    acc.z = fmaf(wgt, o[u][j].z, acc.z);
                                    acc.w = fmaf(wgt, o[u][j].w, acc.w);
                                    wsum += wgt;
                                }
                                store_row(idx, acc, wsum);
                            }
                        }
                    };
                    if (nc <= 2) {
                        merge_pass(std::integral_constant<int, 12>{}, std::integral_constant<int, 2>{});
                    } else {  // nc <= kLastArriverMax == kMaxC: more partials are combined by attn_merge_kernel
                        merge_pass(std::integral_constant<int, kU>{}, std::integral_constant<int, kMaxC>{});
                    }
                }
                ptx::bar_sync(1, 256);  // merge_info is reused by the next segment
            }
        }
    }

    ptx::tc_fence_before();
    __syncthreads();
    if (warp == 2) ptx::tmem_dealloc<512>(tmem);
    if (threadIdx.x == 0) {
        p.progress[blockIdx.x] = sched[2];
        if (sched[1] != 0x7fffffff) *p.pass_state = p.launch_seq;   // this launch left segments for a resume
    }
}

// The cross-CTA pass of units spread over more than kLastArriverMax CTAs (a launch with few units and many CTAs: one
// launch per layer, a single long session), as its own launch right behind the attention kernel.  Its
// griddepcontrol.wait returns when that kernel has ended, so every partial is complete: no ticket, no CTA waiting for
// another one (the in-kernel form of this pass spun on co-residency that an ordinary launch does not guarantee).  One
// CTA = 32 rows x 4 float4 columns of one unit: a warp's lanes run along the rows of one float4 column (512
// contiguous bytes of a partial), partials are combined in CTA order with kCB loads in flight per thread.
template <int D>
__global__ void __launch_bounds__(128) attn_merge_kernel(const UmmaParams p, int attn_grid)
{
    ptx::griddep_launch();
    ptx::griddep_wait();
    // the attention launch stopped at a yield point: its partials are incomplete, the resume's merge does the work
    if (ptx::ld_volatile_global(p.pass_state) == p.launch_seq) return;
    constexpr int kVec = D / 4;
    constexpr int kRowBlks = kAttnMaxRows / 32, kColBlks = kVec / 4;
    constexpr int kCB = 8;
    constexpr size_t kSlotFloats = static_cast<size_t>(kAttnMaxRows) * (D + 2);
    const int G = p.Hq / p.Hkv;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const long long n_items = static_cast<long long>(p.n_lh) * p.a.n_units * (kRowBlks * kColBlks);
    for (long long item = blockIdx.x; item < n_items; item += gridDim.x) {
        const int sub = static_cast<int>(item % (kRowBlks * kColBlks));
        const long long lu = item / (kRowBlks * kColBlks);
        const int ui = static_cast<int>(lu % p.a.n_units), lh = static_cast<int>(lu / p.a.n_units);
        const int rb = sub / kColBlks, v = (sub % kColBlks) * 4 + warp;
        const AttnUnit u = p.units[ui];
        const int rows = u.ntok * G;
        if (rb * 32 >= rows) continue;
        const long long U0 = static_cast<long long>(lh) * p.tiles_per_lh + u.tile_prefix;
        const int c0 = cta_of(p, attn_grid, U0), c1 = cta_of(p, attn_grid, U0 + u.n_tiles - 1);
        const int nc = c1 - c0 + 1;
        if (nc <= kLastArriverMax) continue;   // combined inside the attention kernel
        const int r = rb * 32 + lane;
        if (r >= rows) continue;
        const int c0_slot = (cta_begin(p, attn_grid, c0) < U0) ? 1 : 0;
        float M = -CUDART_INF_F, wsum = 0.f;
        float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
        for (int cb = 0; cb < nc; cb += kCB) {
            float lse[kCB];
            float4 o[kCB];
#pragma unroll
            for (int q = 0; q < kCB; ++q) {
                lse[q] = -CUDART_INF_F;
                o[q] = make_float4(0.f, 0.f, 0.f, 0.f);
                if (cb + q < nc) {
                    const int c = c0 + cb + q;
                    const float *sl = p.partials + (2 * static_cast<size_t>(c) + (c == c0 ? c0_slot : 0)) * kSlotFloats;
                    lse[q] = __ldcg(sl + kAttnMaxRows * D + r);
                    o[q] = __ldcg(reinterpret_cast<const float4 *>(sl) + static_cast<size_t>(v) * kAttnMaxRows + r);
                }
            }
            float mc = lse[0];
#pragma unroll
            for (int q = 1; q < kCB; ++q) mc = fmaxf(mc, lse[q]);
            const float Mn = fmaxf(M, mc);
            if (Mn == -CUDART_INF_F) continue;   // nothing seen so far
            const float resc = (M == -CUDART_INF_F) ? 0.f : exp2f(M - Mn);
            acc.x *= resc;
            acc.y *= resc;
            acc.z *= resc;
            acc.w *= resc;
            wsum *= resc;
            M = Mn;
#pragma unroll
            for (int q = 0; q < kCB; ++q) {  // CTA order
                const float wgt = (lse[q] == -CUDART_INF_F) ? 0.f : exp2f(lse[q] - M);
                acc.x = fmaf(wgt, o[q].x, acc.x);
                acc.y = fmaf(wgt, o[q].y, acc.y);
                acc.z = fmaf(wgt, o[q].z, acc.z);
                acc.w = fmaf(wgt, o[q].w, acc.w);
                wsum += wgt;
            }
        }
        const float inv = 1.f / wsum;
        const int layer = p.a.layer_begin + lh / p.Hkv, kvh = lh % p.Hkv;
        const int tok = u.tok0 + r / G, h = kvh * G + r % G;
        __nv_bfloat16 *ob = p.a.out + static_cast<size_t>(layer) * p.a.out_layer_stride;
        uint2 pk;
        pk.x = pack_bf16(acc.x * inv, acc.y * inv);
        pk.y = pack_bf16(acc.z * inv, acc.w * inv);
        *reinterpret_cast<uint2 *>(ob + (static_cast<size_t>(u.row0 + tok) * p.Hq + h) * D + v * 4) = pk;
    }
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

int encode_pool_map(CUtensorMap *tm, void *pool, const prepos_model_shape &s, int64_t layer_stride, int64_t n_pages)
{
    EncodeTiledFn encode = reinterpret_cast<EncodeTiledFn>(prepos_get_encode_tiled());
    if (!encode) return PREPOS_E_CUDA;
    const int D = s.head_dim, halves = D / 64, groups = s.page_size / 8;
    const cuuint64_t dims[5] = {64, 8, static_cast<cuuint64_t>(halves),
                                static_cast<cuuint64_t>(n_pages) * s.n_kv_heads * groups,
                                static_cast<cuuint64_t>(s.layers)};
    const cuuint64_t strides[4] = {static_cast<cuuint64_t>(D) * 2, 128, static_cast<cuuint64_t>(8) * D * 2,
                                   static_cast<cuuint64_t>(layer_stride) * 2};
    const cuuint32_t box[5] = {64, 8, static_cast<cuuint32_t>(halves), static_cast<cuuint32_t>(groups), 1};
    const cuuint32_t estr[5] = {1, 1, 1, 1, 1};
    const CUresult r = encode(tm, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 5, pool, dims, strides, box, estr,
                              CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                              CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
        fprintf(stderr, "libprepos: cuTensorMapEncodeTiled(pool) failed: %d\n", static_cast<int>(r));
        return PREPOS_E_CUDA;
    }
    return PREPOS_OK;
}

// e4m3 pool [layer][n_pages][Hkv][page][d] bytes: a box is one (page, kv head) slab, [page tokens][d = 128 bytes],
// 128-byte swizzle (16-byte chunk c of token row r lands at chunk c ^ (r % 8))
int encode_pool8_map(CUtensorMap *tm, void *pool, const prepos_model_shape &s, int64_t layer_stride_bytes, int64_t n_pages)
{
    EncodeTiledFn encode = reinterpret_cast<EncodeTiledFn>(prepos_get_encode_tiled());
    if (!encode) return PREPOS_E_CUDA;
    const int D = s.head_dim;
    const cuuint64_t dims[3] = {static_cast<cuuint64_t>(D), static_cast<cuuint64_t>(n_pages) * s.n_kv_heads * s.page_size,
                                static_cast<cuuint64_t>(s.layers)};
    const cuuint64_t lstride = (s.layers > 1) ? static_cast<cuuint64_t>(layer_stride_bytes) : dims[0] * dims[1];
    const cuuint64_t strides[2] = {static_cast<cuuint64_t>(D), lstride};
    const cuuint32_t box[3] = {static_cast<cuuint32_t>(D), static_cast<cuuint32_t>(s.page_size), 1};
    const cuuint32_t estr[3] = {1, 1, 1};
    const CUresult r = encode(tm, CU_TENSOR_MAP_DATA_TYPE_UINT8, 3, pool, dims, strides, box, estr,
                              CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                              CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
        fprintf(stderr, "libprepos: cuTensorMapEncodeTiled(e4m3 pool) failed: %d\n", static_cast<int>(r));
        return PREPOS_E_CUDA;
    }
    return PREPOS_OK;
}

// K_new / V_new [layer][sum_L][Hkv][d]: a box is 8 consecutive tokens of one kv head, laid out like one 8-row group
// of a pool tile ([64-column half][8 rows][128 B], 128-byte swizzle); tokens past sum_L read as zero.
int encode_new_map(CUtensorMap *tm, const void *base, const prepos_model_shape &s, int64_t layer_stride, int64_t sum_rows)
{
    EncodeTiledFn encode = reinterpret_cast<EncodeTiledFn>(prepos_get_encode_tiled());
    if (!encode) return PREPOS_E_CUDA;
    const int D = s.head_dim, halves = D / 64;
    const cuuint64_t tok_stride = static_cast<cuuint64_t>(s.n_kv_heads) * D * 2;
    // a one-layer tensor may come with any layer stride: give the (unused) dimension a valid one
    const cuuint64_t lstride = (s.layers > 1) ? static_cast<cuuint64_t>(layer_stride) * 2 : tok_stride * static_cast<cuuint64_t>(sum_rows);
    const cuuint64_t dims[5] = {64, static_cast<cuuint64_t>(sum_rows), static_cast<cuuint64_t>(halves),
                                static_cast<cuuint64_t>(s.n_kv_heads), static_cast<cuuint64_t>(s.layers)};
    const cuuint64_t strides[4] = {tok_stride, 128, static_cast<cuuint64_t>(D) * 2, lstride};
    const cuuint32_t box[5] = {64, 8, static_cast<cuuint32_t>(halves), 1, 1};
    const cuuint32_t estr[5] = {1, 1, 1, 1, 1};
    const CUresult r = encode(tm, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 5, const_cast<void *>(base), dims, strides, box, estr,
                              CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                              CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
        fprintf(stderr, "libprepos: cuTensorMapEncodeTiled(entry K/V) failed: %d\n", static_cast<int>(r));
        return PREPOS_E_CUDA;
    }
    return PREPOS_OK;
}

// Q [layer][sum_L][Hq][d]: a box is one 8-row group of a unit's Q tile, rows ordered (token, head within the kv
// group): min(G, 8) heads x 8 / min(G, 8) tokens, laid out [64-column half][8 rows][128 B] with the 128-byte swizzle
int encode_q_map(CUtensorMap *tm, const void *base, const prepos_model_shape &s, int64_t layer_stride, int64_t sum_rows)
{
    EncodeTiledFn encode = reinterpret_cast<EncodeTiledFn>(prepos_get_encode_tiled());
    if (!encode) return PREPOS_E_CUDA;
    const int D = s.head_dim, halves = D / 64, G = s.n_q_heads / s.n_kv_heads;
    const int gbox = G < 8 ? G : 8, tbox = 8 / gbox;
    const cuuint64_t tok_stride = static_cast<cuuint64_t>(s.n_q_heads) * D * 2;
    const cuuint64_t lstride = (s.layers > 1) ? static_cast<cuuint64_t>(layer_stride) * 2 : tok_stride * static_cast<cuuint64_t>(sum_rows);
    const cuuint64_t dims[5] = {64, static_cast<cuuint64_t>(s.n_q_heads), static_cast<cuuint64_t>(sum_rows),
                                static_cast<cuuint64_t>(halves), static_cast<cuuint64_t>(s.layers)};
    const cuuint64_t strides[4] = {static_cast<cuuint64_t>(D) * 2, tok_stride, 128, lstride};
    const cuuint32_t box[5] = {64, static_cast<cuuint32_t>(gbox), static_cast<cuuint32_t>(tbox), static_cast<cuuint32_t>(halves), 1};
    const cuuint32_t estr[5] = {1, 1, 1, 1, 1};
    const CUresult r = encode(tm, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 5, const_cast<void *>(base), dims, strides, box, estr,
                              CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                              CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
        fprintf(stderr, "libprepos: cuTensorMapEncodeTiled(Q) failed: %d\n", static_cast<int>(r));
        return PREPOS_E_CUDA;
    }
    return PREPOS_OK;
}

template <int D, bool kFp8>
int issue(prepos_ctx *ctx, cudaStream_t stream, int resume);

template <int D, bool kFp8>
int launch(prepos_ctx *ctx, const AttnArgs &a, int tiles_per_lh, cudaStream_t stream)
{
    UmmaParams p;
    p.a = a;
    p.units = ctx->attn_units;
    p.Hq = ctx->shape.n_q_heads;
    p.Hkv = ctx->shape.n_kv_heads;
    p.page = ctx->shape.page_size;
    p.page_shift = 0;
    while ((1 << p.page_shift) < p.page) ++p.page_shift;
    p.n_lh = (a.layer_end - a.layer_begin) * p.Hkv;
    p.tiles_per_lh = tiles_per_lh;
    p.total_tiles = static_cast<long long>(p.n_lh) * tiles_per_lh;
    p.scale_log2 = a.scale * 1.4426950408889634f;
    p.partials = ctx->attn_partials;
    const int G = p.Hq / p.Hkv;
    bool two = false;
    for (const AttnUnit &u : ctx->plan_units) two |= (u.ntok * G > 128);
    p.q_tiles = two ? 2 : 1;
    p.nv = two ? 2 : 3;
    if (D == 64) p.nv = 3;
    constexpr int kTileBytes = kTile * D * 2;
    // tail: 36 barriers, the (m, l) exchange, TMEM slot + merge info + segment admission (+ kFp8: the scale ring)
    const size_t smem = static_cast<size_t>(p.q_tiles + kNK + p.nv) * kTileBytes + 36 * 8 + 128 * 8 + 40 + (kFp8 ? 8 * 16 * 4 + 16 : 0);
    // one CTA per SM; never more CTAs than tiles, never more than the partial slots provisioned
    long long grid = ctx->num_sms;
    if (grid > p.total_tiles) grid = p.total_tiles;
    if (grid > kAttnMaxCtas) grid = kAttnMaxCtas;
    // Short ranges of an HBM-bound launch: a cut segment costs its CTA ~8 us (partial store, ticket, merge), which is
    // a tenth of a 57-tile range.  When every unit has the same number of tiles and the units divide evenly over a
    // slightly smaller grid, use that grid: every CTA then runs whole units only (no partials, no merge), and 85% of
    // the SMs still saturate HBM (config 2: 256 units on 128 CTAs, 0.110 -> 0.102 ms).  Tensor-bound launches
    // (two M-tiles) need every SM, and long ranges (config 3) amortise their two cuts.
    if (!two && p.total_tiles / grid < 128) {
        bool uniform = true;
        for (const AttnUnit &u : ctx->plan_units) uniform &= (u.n_tiles == ctx->plan_units[0].n_tiles);
        const long long n_units_total = static_cast<long long>(p.n_lh) * a.n_units;
        if (uniform)
            for (long long g = grid; g * 100 >= static_cast<long long>(ctx->num_sms) * 85; --g)
                if (n_units_total % g == 0) {
                    grid = g;
                    break;
                }
    }
    // Fewer units than CTAs (one launch per layer: 8 kv heads for 148 CTAs): give every unit a whole number of CTAs,
    // in proportion to its tiles, and cut it evenly among them.  No CTA then straddles two units (one segment, one
    // epilogue per CTA) and the CTAs of a unit finish together.
    p.use_bnd = 0;
    long long n_wide_bnd = 0;   // units given more than kLastArriverMax CTAs by the table below
    {
        const long long n_units_total = static_cast<long long>(p.n_lh) * a.n_units;
        if (n_units_total < grid && p.total_tiles < (1ll << 30)) {
            std::vector<long long> start, tiles;
            for (int lh = 0; lh < p.n_lh; ++lh)
                for (const AttnUnit &u : ctx->plan_units) {
                    start.push_back(static_cast<long long>(lh) * tiles_per_lh + u.tile_prefix);
                    tiles.push_back(u.n_tiles);
                }
            const int n = static_cast<int>(tiles.size());
            std::vector<int> k(n);
            long long used = 0;
            for (int i = 0; i < n; ++i) {
                long long ki = tiles[i] * grid / p.total_tiles;
                ki = ki < 1 ? 1 : (ki > tiles[i] ? tiles[i] : ki);
                k[i] = static_cast<int>(ki);
                used += ki;
            }
            while (used < grid) {   // hand the remaining CTAs to the units with the most tiles per CTA
                int best = -1;
                for (int i = 0; i < n; ++i)
                    if (k[i] < tiles[i] && (best < 0 || tiles[i] * k[best] > tiles[best] * k[i])) best = i;
                if (best < 0) break;
                ++k[best];
                ++used;
            }
            if (used == grid) {
                int c = 0;
                for (int i = 0; i < n; ++i) {
                    for (int j = 0; j < k[i]; ++j) p.bnd[c++] = static_cast<int>(start[i] + tiles[i] * j / k[i]);
                    n_wide_bnd += (k[i] > kLastArriverMax);
                }
                p.bnd[c] = static_cast<int>(p.total_tiles);
                p.use_bnd = 1;
            }
        }
    }
    // (the bf16 pools take a 5-D map, the e4m3 pools a 3-D byte map: the kind is part of the cache key, since the same
    // base address, stride value and page count can describe either when a ctx alternates between the two)
    if (kFp8) {
        if (ctx->tm_pool_kind != 2 || ctx->tm_k_ptr != a.k_pool8 || ctx->tm_v_ptr != a.v_pool8 ||
            ctx->tm_layer_stride != a.pool_layer_stride || ctx->tm_n_pages != a.n_pages) {
            int st = encode_pool8_map(&ctx->tm_k, a.k_pool8, ctx->shape, a.pool_layer_stride, a.n_pages);
            if (st == PREPOS_OK) st = encode_pool8_map(&ctx->tm_v, a.v_pool8, ctx->shape, a.pool_layer_stride, a.n_pages);
            if (st != PREPOS_OK) return st;
            ctx->tm_k_ptr = a.k_pool8;
            ctx->tm_v_ptr = a.v_pool8;
            ctx->tm_layer_stride = a.pool_layer_stride;
            ctx->tm_n_pages = a.n_pages;
            ctx->tm_pool_kind = 2;
        }
    } else if (ctx->tm_pool_kind != 1 || ctx->tm_k_ptr != a.k_pool || ctx->tm_v_ptr != a.v_pool ||
               ctx->tm_layer_stride != a.pool_layer_stride || ctx->tm_n_pages != a.n_pages) {
        int st = encode_pool_map(&ctx->tm_k, a.k_pool, ctx->shape, a.pool_layer_stride, a.n_pages);
        if (st == PREPOS_OK) st = encode_pool_map(&ctx->tm_v, a.v_pool, ctx->shape, a.pool_layer_stride, a.n_pages);
        if (st != PREPOS_OK) return st;
        ctx->tm_k_ptr = a.k_pool;
        ctx->tm_v_ptr = a.v_pool;
        ctx->tm_layer_stride = a.pool_layer_stride;
        ctx->tm_n_pages = a.n_pages;
        ctx->tm_pool_kind = 1;
    }
    // entry K/V maps: they follow the call's K_new / V_new pointers (the FP8 path reads the entry from the cache)
    if (!kFp8 && (ctx->tm_kn_ptr != a.k_new || ctx->tm_vn_ptr != a.v_new || ctx->tm_new_layer_stride != a.kv_new_layer_stride ||
        ctx->tm_new_rows != a.sum_rows)) {
        int st = encode_new_map(&ctx->tm_kn, a.k_new, ctx->shape, a.kv_new_layer_stride, a.sum_rows);
        if (st == PREPOS_OK) st = encode_new_map(&ctx->tm_vn, a.v_new, ctx->shape, a.kv_new_layer_stride, a.sum_rows);
        if (st != PREPOS_OK) return st;
        ctx->tm_kn_ptr = a.k_new;
        ctx->tm_vn_ptr = a.v_new;
        ctx->tm_new_layer_stride = a.kv_new_layer_stride;
        ctx->tm_new_rows = a.sum_rows;
    }
    if (ctx->tm_q_ptr != a.q || ctx->tm_q_layer_stride != a.q_layer_stride || ctx->tm_q_rows != a.sum_rows) {
        const int st = encode_q_map(&ctx->tm_q, a.q, ctx->shape, a.q_layer_stride, a.sum_rows);
        if (st != PREPOS_OK) return st;
        ctx->tm_q_ptr = a.q;
        ctx->tm_q_layer_stride = a.q_layer_stride;
        ctx->tm_q_rows = a.sum_rows;
    }
    if (static_cast<size_t>(p.n_lh) * a.n_units > ctx->attn_counters_n) return PREPOS_E_WORKSPACE;
    p.counters = ctx->attn_counters;
    // units spread over more than kLastArriverMax CTAs are combined by attn_merge_kernel behind the attention kernel
    long long merge_units = 0;
    if (p.use_bnd) {
        merge_units = n_wide_bnd;
    } else {
        const long long m = p.total_tiles / grid;   // shortest CTA range
        long long max_n = 0;
        for (const AttnUnit &u : ctx->plan_units) max_n = u.n_tiles > max_n ? u.n_tiles : max_n;
        if ((max_n - 1 + m - 1) / m + 1 > kLastArriverMax) {
            auto cta_of_h = [&](long long t) { return ((t + 1) * grid + p.total_tiles - 1) / p.total_tiles - 1; };
            for (int lh = 0; lh < p.n_lh; ++lh)
                for (const AttnUnit &u : ctx->plan_units) {
                    const long long U0 = static_cast<long long>(lh) * tiles_per_lh + u.tile_prefix;
                    merge_units += (cta_of_h(U0 + u.n_tiles - 1) - cta_of_h(U0) >= kLastArriverMax);
                }
        }
    }
    long long mg = 0;
    if (merge_units > 0) {
        mg = merge_units * (kAttnMaxRows / 32) * (D / 16);
        const long long cap = static_cast<long long>(ctx->num_sms) * 4;
        mg = mg > cap ? cap : mg;
    }
    p.yield_flag = ctx->attn_yield_flag;
    p.progress = ctx->attn_progress;
    p.pass_state = ctx->attn_pass_state;
    p.slice = ctx->attn_slice;
    p.early_kv = (ctx->attn_kv_prefetch && !kFp8) ? 1 : 0;   // (the FP8 path reads the entry's codes back from the pages)
    p.resume = 0;
    // keep the launch: prepos_entry_attn_resume re-issues it with resume = 1 (same plan, same grid, same partial slots)
    static_assert(std::is_trivially_copyable<UmmaParams>::value, "UmmaParams is saved as bytes");
    ctx->pass_params.resize(sizeof(UmmaParams));
    memcpy(ctx->pass_params.data(), &p, sizeof(UmmaParams));
    ctx->pass_grid = static_cast<int>(grid);
    ctx->pass_merge_grid = static_cast<int>(mg);
    ctx->pass_smem = smem;
    ctx->pass_head_dim = D;
    ctx->pass_fp8 = kFp8;
    return issue<D, kFp8>(ctx, stream, 0);
}

// one launch of the saved pass (fresh or resumed) + the merge launch behind it
template <int D, bool kFp8>
int issue(prepos_ctx *ctx, cudaStream_t stream, int resume)
{
    UmmaParams p;
    memcpy(&p, ctx->pass_params.data(), sizeof(UmmaParams));
    p.resume = resume;
    p.launch_seq = ++ctx->attn_launch_seq;
    PREPOS_CUDA_TRY(cudaFuncSetAttribute(attn_umma_kernel<D, kFp8>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         static_cast<int>(ctx->pass_smem)));
    PREPOS_CUDA_TRY(prepos_launch_pdl(attn_umma_kernel<D, kFp8>, dim3(static_cast<unsigned>(ctx->pass_grid)), dim3(kThreads),
                                      ctx->pass_smem, stream, ctx->tm_k, ctx->tm_v, ctx->tm_kn, ctx->tm_vn, ctx->tm_q, p));
    ctx->launches += 1;
    if (ctx->pass_merge_grid > 0) {
        PREPOS_CUDA_TRY(prepos_launch_pdl(attn_merge_kernel<D>, dim3(static_cast<unsigned>(ctx->pass_merge_grid)), dim3(128),
                                          0, stream, p, ctx->pass_grid));
        ctx->launches += 1;
    }
    ctx->pass_open = true;
    ctx->pass_sliced = p.slice > 0;
    return PREPOS_OK;
}

}  // namespace

bool prepos_attn_umma_supported(const prepos_ctx *ctx)
{
    const prepos_model_shape &s = ctx->shape;
    const int G = s.n_q_heads / s.n_kv_heads;
    return (s.head_dim == 64 || s.head_dim == 128) && s.page_size >= 8 && s.page_size <= kTile &&
           (G & (G - 1)) == 0;  // the Q boxes take whole 8-row groups of (token, head) rows
}

int prepos_resume_attn_umma(prepos_ctx *ctx, cudaStream_t stream)
{
    if (ctx->pass_params.size() != sizeof(UmmaParams)) return PREPOS_E_INVALID_ARG;
    if (ctx->pass_fp8) return issue<128, true>(ctx, stream, 1);
    if (ctx->pass_head_dim == 128) return issue<128, false>(ctx, stream, 1);
    return issue<64, false>(ctx, stream, 1);
}

int prepos_launch_attn_umma(prepos_ctx *ctx, const AttnArgs &a, int tiles_per_lh, cudaStream_t stream)
{
    if (!prepos_attn_umma_supported(ctx)) return PREPOS_E_SHAPE;
    if (ctx->shape.head_dim == 128) return launch<128, false>(ctx, a, tiles_per_lh, stream);
    return launch<64, false>(ctx, a, tiles_per_lh, stream);
}

// the tcgen05 kernel over an e4m3 KV cache: d = 128, pages of 16..128 tokens (one scale per 16-column block or more)
bool prepos_attn_umma_fp8_supported(const prepos_ctx *ctx)
{
    const prepos_model_shape &s = ctx->shape;
    const int G = s.n_q_heads / s.n_kv_heads;
    return s.head_dim == 128 && s.page_size >= 16 && s.page_size <= kTile && (G & (G - 1)) == 0;
}

int prepos_launch_attn_umma_fp8(prepos_ctx *ctx, const AttnArgs &a, int tiles_per_lh, cudaStream_t stream)
{
    if (!prepos_attn_umma_fp8_supported(ctx)) return PREPOS_E_SHAPE;
    return launch<128, true>(ctx, a, tiles_per_lh, stream);
}
