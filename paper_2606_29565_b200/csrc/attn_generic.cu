// attn_generic.cu -- shape-generic CUDA-core kernel for a1 + a2 (Alg. 1 l.5-6):
// entry rows attend the session's paged KV cache and, causally, the entry tokens; entry K/V are
// appended to the session's pages.  It serves the shapes the tcgen05 kernel does not take (head_dim
// not in {64,128}, page size != 16, tiny launch-bound cases such as BASELINE config 1) and is the
// straightforward streaming formulation: one CTA per (unit, kv head, layer), 32-token tiles staged in
// shared memory, one warp per query row, online softmax in fp32.
#include <math_constants.h>

#include "common.cuh"

namespace {

constexpr int kThreads = 256;
constexpr int kWarps = kThreads / 32;
constexpr int kTile = 32;       // tokens per smem tile
constexpr int kRowsPerWarp = 8; // rows <= 64 per unit
constexpr int kKPad = 8;        // bf16 padding of K rows in smem

struct GenParams {
    AttnArgs a;
    const AttnUnit *units;
    int Hq, Hkv, d, page, page_shift;
    float scale_log2;
};

__device__ __forceinline__ const __nv_bfloat16 *kv_row_ptr(const GenParams &p, const AttnUnit &u, int layer, int kvh,
                                                           int j, bool is_v)
{
    // logical token j of the session: cached (through the page table) or entry token j - n_s
    if (j < u.n_s) {
        const int pg = p.a.page_table[static_cast<size_t>(u.session) * p.a.page_table_stride + (j >> p.page_shift)];
        const __nv_bfloat16 *pool = (is_v ? p.a.v_pool : p.a.k_pool) + static_cast<size_t>(layer) * p.a.pool_layer_stride;
        return pool + ((static_cast<size_t>(pg) * p.Hkv + kvh) * p.page + (j & (p.page - 1))) * p.d;
    }
    const __nv_bfloat16 *nw = (is_v ? p.a.v_new : p.a.k_new) + static_cast<size_t>(layer) * p.a.kv_new_layer_stride;
    return nw + (static_cast<size_t>(u.row0 + (j - u.n_s)) * p.Hkv + kvh) * p.d;
}

__global__ void __launch_bounds__(kThreads) attn_generic_kernel(const GenParams p)
{
    extern __shared__ __align__(16) uint8_t smem[];
    const AttnUnit u = p.units[blockIdx.x];
    const int kvh = blockIdx.y;
    const int layer = p.a.layer_begin + blockIdx.z;
    const int G = p.Hq / p.Hkv;
    const int d = p.d;
    const int rows = u.ntok * G;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int kstride = d + kKPad;

    float *q_s = reinterpret_cast<float *>(smem);                       // [rows][d], pre-scaled by scale*log2(e)
    float *o_s = q_s + static_cast<size_t>(rows) * d;                   // [rows][d]
    __nv_bfloat16 *k_s = reinterpret_cast<__nv_bfloat16 *>(o_s + static_cast<size_t>(rows) * d);  // [kTile][d+pad]
    __nv_bfloat16 *v_s = k_s + kTile * kstride;                         // [kTile][d]

    // ---- a1: Append(E).  The first row chunk of each (session, layer, kv head) writes all L entry tokens.
    if (u.tok0 == 0) {
        const int cpr = d / 8;  // 16-byte chunks per row
        for (int idx = threadIdx.x; idx < u.l_entry * cpr; idx += kThreads) {
            const int t = idx / cpr, c = idx - t * cpr;
            const int j = u.n_s + t;
            const int pg = p.a.page_table[static_cast<size_t>(u.session) * p.a.page_table_stride + (j >> p.page_shift)];
            const size_t dst = ((static_cast<size_t>(pg) * p.Hkv + kvh) * p.page + (j & (p.page - 1))) * d + c * 8;
            const size_t src = (static_cast<size_t>(u.row0 + t) * p.Hkv + kvh) * d + c * 8;
            const size_t lo = static_cast<size_t>(layer);
            *reinterpret_cast<uint4 *>(p.a.k_pool + lo * p.a.pool_layer_stride + dst) =
                *reinterpret_cast<const uint4 *>(p.a.k_new + lo * p.a.kv_new_layer_stride + src);
            *reinterpret_cast<uint4 *>(p.a.v_pool + lo * p.a.pool_layer_stride + dst) =
                *reinterpret_cast<const uint4 *>(p.a.v_new + lo * p.a.kv_new_layer_stride + src);
        }
    }

    // ---- Q rows -> smem (fp32, scaled), O accumulators = 0.  Row r = (entry token tok0 + r / G, head kvh*G + r % G)
    const __nv_bfloat16 *qb = p.a.q + static_cast<size_t>(layer) * p.a.q_layer_stride;
    for (int idx = threadIdx.x; idx < rows * d; idx += kThreads) {
        const int r = idx / d, c = idx - r * d;
        const int tok = u.tok0 + r / G, h = kvh * G + r % G;
        q_s[idx] = __bfloat162float(qb[(static_cast<size_t>(u.row0 + tok) * p.Hq + h) * d + c]) * p.scale_log2;
        o_s[idx] = 0.f;
    }
    float m_run[kRowsPerWarp], l_run[kRowsPerWarp];
#pragma unroll
    for (int i = 0; i < kRowsPerWarp; ++i) {
        m_run[i] = -CUDART_INF_F;
        l_run[i] = 0.f;
    }

    const int kv_len = u.n_s + u.tok0 + u.ntok;  // tokens visible to the last row of this chunk
    for (int t0 = 0; t0 < kv_len; t0 += kTile) {
        __syncthreads();  // previous tile consumed (and q_s/o_s initialised on the first pass)
        {
            const int cpr = d / 8;
            for (int idx = threadIdx.x; idx < kTile * cpr; idx += kThreads) {
                const int t = idx / cpr, c = idx - t * cpr;
                const int j = t0 + t;
                uint4 kk = make_uint4(0, 0, 0, 0), vv = make_uint4(0, 0, 0, 0);
                if (j < kv_len) {
                    kk = *reinterpret_cast<const uint4 *>(kv_row_ptr(p, u, layer, kvh, j, false) + c * 8);
                    vv = *reinterpret_cast<const uint4 *>(kv_row_ptr(p, u, layer, kvh, j, true) + c * 8);
                }
                *reinterpret_cast<uint4 *>(k_s + t * kstride + c * 8) = kk;
                *reinterpret_cast<uint4 *>(v_s + t * d + c * 8) = vv;
            }
        }
        __syncthreads();
#pragma unroll
        for (int i = 0; i < kRowsPerWarp; ++i) {
            const int r = warp + i * kWarps;
            if (r >= rows) break;
            const int j = t0 + lane;
            const int last_visible = u.n_s + u.tok0 + r / G;  // causal: entry row sees itself (reading Q5)
            float s = -CUDART_INF_F;
            if (j <= last_visible) {
                float acc = 0.f;
                const float *qr = q_s + r * d;
                const __nv_bfloat16 *kr = k_s + lane * kstride;
                for (int c = 0; c < d; c += 8) {
                    const uint4 kv = *reinterpret_cast<const uint4 *>(kr + c);
                    const float4 qa = *reinterpret_cast<const float4 *>(qr + c);
                    const float4 qc = *reinterpret_cast<const float4 *>(qr + c + 4);
                    acc = fmaf(qa.x, __uint_as_float(kv.x << 16), acc);
                    acc = fmaf(qa.y, __uint_as_float(kv.x & 0xffff0000u), acc);
                    acc = fmaf(qa.z, __uint_as_float(kv.y << 16), acc);
                    acc = fmaf(qa.w, __uint_as_float(kv.y & 0xffff0000u), acc);
                    acc = fmaf(qc.x, __uint_as_float(kv.z << 16), acc);
                    acc = fmaf(qc.y, __uint_as_float(kv.z & 0xffff0000u), acc);
                    acc = fmaf(qc.z, __uint_as_float(kv.w << 16), acc);
                    acc = fmaf(qc.w, __uint_as_float(kv.w & 0xffff0000u), acc);
                }
                s = acc;  // already in log2 units
            }
            float mt = s;
#pragma unroll
            for (int mask = 16; mask; mask >>= 1) mt = fmaxf(mt, __shfl_xor_sync(0xffffffffu, mt, mask));
            const float m_new = fmaxf(m_run[i], mt);
            // every tile holds at least one visible token for every row (t0 < kv_len and rows see >= n_s+tok0+1
            // tokens) only for the last rows; a row may see none of this tile: then m_new may stay -inf
            const float corr = (m_new == -CUDART_INF_F) ? 1.f : exp2f(m_run[i] - m_new);
            const float pj = (s == -CUDART_INF_F) ? 0.f : exp2f(s - m_new);
            float ps = pj;
#pragma unroll
            for (int mask = 16; mask; mask >>= 1) ps += __shfl_xor_sync(0xffffffffu, ps, mask);
            l_run[i] = l_run[i] * corr + ps;
            m_run[i] = m_new;
            float *orow = o_s + r * d;
            float oreg[8];  // d <= 256: this lane's columns lane, lane+32, ...
#pragma unroll
            for (int cc = 0; cc < 8; ++cc) oreg[cc] = (lane + cc * 32 < d) ? orow[lane + cc * 32] * corr : 0.f;
            for (int t = 0; t < kTile; ++t) {
                const float pt = __shfl_sync(0xffffffffu, pj, t);
#pragma unroll
                for (int cc = 0; cc < 8; ++cc)
                    if (lane + cc * 32 < d) oreg[cc] = fmaf(pt, __bfloat162float(v_s[t * d + lane + cc * 32]), oreg[cc]);
            }
#pragma unroll
            for (int cc = 0; cc < 8; ++cc)
                if (lane + cc * 32 < d) orow[lane + cc * 32] = oreg[cc];
        }
    }
    // ---- normalise and store
    __nv_bfloat16 *ob = p.a.out + static_cast<size_t>(layer) * p.a.out_layer_stride;
#pragma unroll
    for (int i = 0; i < kRowsPerWarp; ++i) {
        const int r = warp + i * kWarps;
        if (r >= rows) break;
        const int tok = u.tok0 + r / G, h = kvh * G + r % G;
        const float inv = 1.f / l_run[i];
        for (int c = lane; c < d; c += 32)
            ob[(static_cast<size_t>(u.row0 + tok) * p.Hq + h) * d + c] = __float2bfloat16(o_s[r * d + c] * inv);
    }
}

}  // namespace

int prepos_launch_attn_generic(prepos_ctx *ctx, const AttnArgs &a, cudaStream_t stream)
{
    GenParams p;
    p.a = a;
    p.units = ctx->attn_units;
    p.Hq = ctx->shape.n_q_heads;
    p.Hkv = ctx->shape.n_kv_heads;
    p.d = ctx->shape.head_dim;
    p.page = ctx->shape.page_size;
    p.page_shift = 0;
    while ((1 << p.page_shift) < p.page) ++p.page_shift;
    p.scale_log2 = a.scale * 1.4426950408889634f;
    const int G = p.Hq / p.Hkv;
    const int max_rows = (G > 16) ? G : (16 / G) * G;
    const size_t smem = static_cast<size_t>(max_rows) * p.d * 4 * 2 + static_cast<size_t>(kTile) * (p.d + kKPad) * 2 +
                        static_cast<size_t>(kTile) * p.d * 2;
    PREPOS_CUDA_TRY(cudaFuncSetAttribute(attn_generic_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         static_cast<int>(smem)));
    const dim3 grid(a.n_units, p.Hkv, a.layer_end - a.layer_begin);
    attn_generic_kernel<<<grid, kThreads, smem, stream>>>(p);
    PREPOS_CUDA_TRY(cudaGetLastError());
    ctx->launches += 1;
    return PREPOS_OK;
}
