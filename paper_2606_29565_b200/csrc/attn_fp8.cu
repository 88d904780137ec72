// attn_fp8.cu -- a1 + a2 over an FP8 (e4m3) KV cache (the paper's headline model "runs at
// 4-bit precision", without naming a storage format: DESIGN.md reading Q20).
//
//   K/V pages hold OCP e4m3 codes; one caller-owned fp32 scale per (layer, page, kv head) for K and one for V;
//   cached value = decode(code) * scale.  Alg. 1 order: Append(E) first -- code =
//   e4m3(fp32(x) / scale), division and conversion round-to-nearest-even, saturating at +-448 -- then Forward(E),
//   so entry row i sees the entry tokens j' <= i through their STORED codes.
//
// Two launches per call:
//   fp8_append_kernel   quantises K_new / V_new with the scale of the page each token lands in and writes the codes
//                       into the session's pages (a1)
//   attn_fp8_kernel     every row then reads ALL its keys -- the n_s cached tokens and the entry tokens up to its
//                       own -- from the pages: one load path, the causal limit is just a per-row key count (a2).
//                       d = 128 with pages of >= 16 tokens takes the tcgen05 kernel instead (attn_umma.cu, kFp8).
//                       Shape-generic CUDA-core formulation (one CTA per (row chunk, kv head, layer), 32-token tiles
//                       dequantised into shared memory as fp32, one warp per query row, fp32 online softmax).
#include <cuda_fp8.h>
#include <math_constants.h>

#include "common.cuh"
#include "ptx.cuh"

namespace {

constexpr int kThreads = 256;
constexpr int kWarps = kThreads / 32;
constexpr int kTile = 32;        // tokens per smem tile
constexpr int kRowsPerWarp = 8;  // rows <= 64 per unit
constexpr int kKPad = 4;         // fp32 padding of K rows in smem

struct Fp8Params {
    AttnArgs a;
    const AttnUnit *units;
    int Hq, Hkv, d, page, page_shift;
    float scale_log2;
};

// 16 bf16 values / scale -> 16 e4m3 codes (fp32 division and conversion both round to nearest even; saturating)
__device__ __forceinline__ uint4 quantise16(const uint4 lo, const uint4 hi, float scale)
{
    const uint32_t w[8] = {lo.x, lo.y, lo.z, lo.w, hi.x, hi.y, hi.z, hi.w};
    uint32_t out[4];
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        uint32_t r = 0;
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const uint32_t pair = w[2 * i + h];
            const float x0 = __uint_as_float(pair << 16), x1 = __uint_as_float(pair & 0xffff0000u);
            const __nv_fp8x2_storage_t c =
                __nv_cvt_float2_to_fp8x2(make_float2(__fdiv_rn(x0, scale), __fdiv_rn(x1, scale)), __NV_SATFINITE, __NV_E4M3);
            r |= static_cast<uint32_t>(c) << (16 * h);
        }
        out[i] = r;
    }
    return make_uint4(out[0], out[1], out[2], out[3]);
}

// a1: Append(E) for every (session, layer, kv head); the first row chunk of a session carries its whole entry
__global__ void __launch_bounds__(kThreads) fp8_append_kernel(const Fp8Params p)
{
    ptx::griddep_wait();
    ptx::griddep_launch();
    const AttnUnit u = p.units[blockIdx.x];
    if (u.tok0 != 0) return;
    const int kvh = blockIdx.y;
    const int layer = p.a.layer_begin + blockIdx.z;
    const int d = p.d;
    const int cpr = d / 16;  // 16-element chunks per row
    const size_t lo = static_cast<size_t>(layer);
    const int32_t *pt = p.a.page_table + static_cast<size_t>(u.session) * p.a.page_table_stride;
    for (int idx = threadIdx.x; idx < u.l_entry * cpr; idx += kThreads) {
        const int t = idx / cpr, c = idx - t * cpr;
        const int j = u.n_s + t;
        const int pg = pt[j >> p.page_shift];
        const size_t src = (static_cast<size_t>(u.row0 + t) * p.Hkv + kvh) * d + c * 16;
        const size_t dst = ((static_cast<size_t>(pg) * p.Hkv + kvh) * p.page + (j & (p.page - 1))) * d + c * 16;
        const size_t sidx = lo * p.a.scale_layer_stride + static_cast<size_t>(pg) * p.Hkv + kvh;
        const __nv_bfloat16 *ks = p.a.k_new + lo * p.a.kv_new_layer_stride + src;
        const __nv_bfloat16 *vs = p.a.v_new + lo * p.a.kv_new_layer_stride + src;
        const uint4 k0 = *reinterpret_cast<const uint4 *>(ks), k1 = *reinterpret_cast<const uint4 *>(ks + 8);
        const uint4 v0 = *reinterpret_cast<const uint4 *>(vs), v1 = *reinterpret_cast<const uint4 *>(vs + 8);
        *reinterpret_cast<uint4 *>(p.a.k_pool8 + lo * p.a.pool_layer_stride + dst) = quantise16(k0, k1, p.a.k_scale[sidx]);
        *reinterpret_cast<uint4 *>(p.a.v_pool8 + lo * p.a.pool_layer_stride + dst) = quantise16(v0, v1, p.a.v_scale[sidx]);
    }
}

// 16 e4m3 codes * scale -> 16 fp32 (decode is exact; the product rounds once, in fp32)
__device__ __forceinline__ void dequant16(const uint4 c, float scale, float *dst)
{
    const uint32_t w[4] = {c.x, c.y, c.z, c.w};
#pragma unroll
    for (int i = 0; i < 4; ++i) {
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const __half2_raw hr =
                __nv_cvt_fp8x2_to_halfraw2(static_cast<__nv_fp8x2_storage_t>((w[i] >> (16 * h)) & 0xffffu), __NV_E4M3);
            const float2 f = __half22float2(*reinterpret_cast<const __half2 *>(&hr));
            dst[4 * i + 2 * h] = f.x * scale;
            dst[4 * i + 2 * h + 1] = f.y * scale;
        }
    }
}

__global__ void __launch_bounds__(kThreads) attn_fp8_kernel(const Fp8Params p)
{
    extern __shared__ __align__(16) uint8_t smem[];
    ptx::griddep_wait();   // the codes of the entry tokens were written by fp8_append_kernel, the launch before
    ptx::griddep_launch();
    const AttnUnit u = p.units[blockIdx.x];
    const int kvh = blockIdx.y;
    const int layer = p.a.layer_begin + blockIdx.z;
    const int G = p.Hq / p.Hkv;
    const int d = p.d;
    const int rows = u.ntok * G;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int kstride = d + kKPad;

    float *q_s = reinterpret_cast<float *>(smem);      // [rows][d], pre-scaled by scale * log2(e)
    float *o_s = q_s + static_cast<size_t>(rows) * d;  // [rows][d]
    float *k_s = o_s + static_cast<size_t>(rows) * d;  // [kTile][d + pad]
    float *v_s = k_s + kTile * kstride;                // [kTile][d]

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

    const size_t lo = static_cast<size_t>(layer);
    const int32_t *pt = p.a.page_table + static_cast<size_t>(u.session) * p.a.page_table_stride;
    const uint8_t *kpool = p.a.k_pool8 + lo * p.a.pool_layer_stride;
    const uint8_t *vpool = p.a.v_pool8 + lo * p.a.pool_layer_stride;
    const float *ksc = p.a.k_scale + lo * p.a.scale_layer_stride;
    const float *vsc = p.a.v_scale + lo * p.a.scale_layer_stride;
    const int kv_len = u.n_load;  // = n_s + tok0 + ntok: keys visible to the last row of this chunk
    for (int t0 = 0; t0 < kv_len; t0 += kTile) {
        __syncthreads();
        {
            const int cpr = d / 16;
            for (int idx = threadIdx.x; idx < kTile * cpr; idx += kThreads) {
                const int t = idx / cpr, c = idx - t * cpr;
                const int j = t0 + t;
                float *kd = k_s + t * kstride + c * 16, *vd = v_s + t * d + c * 16;
                if (j < kv_len) {
                    const int pg = pt[j >> p.page_shift];
                    const size_t off = ((static_cast<size_t>(pg) * p.Hkv + kvh) * p.page + (j & (p.page - 1))) * d + c * 16;
                    const size_t sidx = static_cast<size_t>(pg) * p.Hkv + kvh;
                    dequant16(*reinterpret_cast<const uint4 *>(kpool + off), ksc[sidx], kd);
                    dequant16(*reinterpret_cast<const uint4 *>(vpool + off), vsc[sidx], vd);
                } else {
#pragma unroll
                    for (int e = 0; e < 16; ++e) kd[e] = vd[e] = 0.f;
                }
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
                const float *kr = k_s + lane * kstride;
                for (int c = 0; c < d; c += 4) {
                    const float4 kv = *reinterpret_cast<const float4 *>(kr + c);
                    const float4 qa = *reinterpret_cast<const float4 *>(qr + c);
                    acc = fmaf(qa.x, kv.x, acc);
                    acc = fmaf(qa.y, kv.y, acc);
                    acc = fmaf(qa.z, kv.z, acc);
                    acc = fmaf(qa.w, kv.w, acc);
                }
                s = acc;  // already in log2 units
            }
            float mt = s;
#pragma unroll
            for (int mask = 16; mask; mask >>= 1) mt = fmaxf(mt, __shfl_xor_sync(0xffffffffu, mt, mask));
            const float m_new = fmaxf(m_run[i], mt);
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
                const float pt_ = __shfl_sync(0xffffffffu, pj, t);
#pragma unroll
                for (int cc = 0; cc < 8; ++cc)
                    if (lane + cc * 32 < d) oreg[cc] = fmaf(pt_, v_s[t * d + lane + cc * 32], oreg[cc]);
            }
#pragma unroll
            for (int cc = 0; cc < 8; ++cc)
                if (lane + cc * 32 < d) orow[lane + cc * 32] = oreg[cc];
        }
    }
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

int prepos_launch_attn_fp8(prepos_ctx *ctx, const AttnArgs &a, bool use_umma, int total_tiles_per_lh, cudaStream_t stream)
{
    Fp8Params p;
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
    const size_t smem = static_cast<size_t>(max_rows) * p.d * 4 * 2 + static_cast<size_t>(kTile) * (p.d + kKPad) * 4 +
                        static_cast<size_t>(kTile) * p.d * 4;
    PREPOS_CUDA_TRY(cudaFuncSetAttribute(attn_fp8_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         static_cast<int>(smem)));
    const dim3 grid(a.n_units, p.Hkv, a.layer_end - a.layer_begin);
    PREPOS_CUDA_TRY(prepos_launch_pdl(fp8_append_kernel, grid, dim3(kThreads), 0, stream, p));
    ctx->launches += 1;
    // d = 128 with pages of >= 16 tokens: the tcgen05 kernel (attn_umma.cu, kFp8) reads the codes back from the pages
    if (use_umma) return prepos_launch_attn_umma_fp8(ctx, a, total_tiles_per_lh, stream);
    PREPOS_CUDA_TRY(prepos_launch_pdl(attn_fp8_kernel, grid, dim3(kThreads), smem, stream, p));
    ctx->launches += 1;
    return PREPOS_OK;
}
