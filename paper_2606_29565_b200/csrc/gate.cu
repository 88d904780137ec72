// gate.cu -- the serve-side kernels: batched confidence gate (Alg. 2; Eq. 12,
// PAPER.md:111) and invalidation (Sec. 3.6).  Both are a handful of bytes per
// request: launch-latency bound, one thread per request.
#include "common.cuh"
#include "ptx.cuh"

namespace {

__device__ __forceinline__ uint4 ld_relaxed_v4(const uint4 *p)
{
    uint4 v;
    asm volatile("ld.relaxed.gpu.global.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(p) : "memory");
    return v;
}

// Alg. 2 for one request.  The version compare is the authority for staleness (reading Q11), the VALID
// bit is redundant with it.
__global__ void __launch_bounds__(128) gate_serve_kernel(int n, const int32_t *__restrict__ session_ids,
                                                         const uint64_t *__restrict__ req_hash,
                                                         const prepos_record *records,
                                                         const uint64_t *session_version,
                                                         const uint32_t *__restrict__ bitmap, int vocab, float tau,
                                                         int strict_gt, int32_t *__restrict__ decision,
                                                         int32_t *__restrict__ token)
{
    ptx::griddep_wait();
    ptx::griddep_launch();
    const int r = blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= n) return;
    const int sid = session_ids[r];
    // Reader side of the publication protocol (include/prepos.h "Record publication"): the record may be re-published
    // or invalidated on another stream while this serve runs.  Word 1 (gap, flags + sequence, version) is read before
    // and after the payload words; if the two reads differ a publication was in progress and the request falls
    // through.  The live version is read last: a record is served only if it was computed at the version that is
    // live after its fields were read (Sec. 3.6).
    const uint4 *p = reinterpret_cast<const uint4 *>(records + sid);
    const uint4 w1a = ld_relaxed_v4(p + 1);  // gap, flags, version
    ptx::fence_acq_rel_gpu();
    const uint4 w0 = ld_relaxed_v4(p);       // max_logit, lse, top1, top2
    const uint4 w2 = ld_relaxed_v4(p + 2);   // entry_hash, position
    ptx::fence_acq_rel_gpu();
    const uint4 w1 = ld_relaxed_v4(p + 1);
    const bool torn = (w1a.x != w1.x) | (w1a.y != w1.y) | (w1a.z != w1.z) | (w1a.w != w1.w);
    const int32_t top1 = static_cast<int32_t>(w0.z);
    const float gap = __uint_as_float(w1.x);
    const uint32_t flags = w1.y;
    const uint64_t rec_version = (static_cast<uint64_t>(w1.w) << 32) | w1.z;
    const uint64_t rec_hash = (static_cast<uint64_t>(w2.y) << 32) | w2.x;
    const uint64_t live = *reinterpret_cast<const volatile uint64_t *>(session_version + sid);
    const uint64_t rh = req_hash ? req_hash[r] : 0ull;

    int dec;
    if (torn || !(flags & PREPOS_FLAG_VALID) || (flags & PREPOS_FLAG_NONFINITE) || rec_version != live) {
        dec = PREPOS_STALE_OR_INVALID;  // Alg. 2 l.1-2
    } else if (rec_hash != 0ull && rh != 0ull && rec_hash != rh) {
        dec = PREPOS_INELIGIBLE;  // Alg. 2 l.1-2, realised entry != pre-positioned entry
    } else if (top1 < 0 || top1 >= vocab || !((bitmap[top1 >> 5] >> (top1 & 31)) & 1u)) {
        dec = PREPOS_NOT_IN_FAST_SET;  // Eq. 12, argmax not in A
    } else if (strict_gt ? !(gap > tau) : !(gap >= tau)) {
        dec = PREPOS_GAP_BELOW_TAU;  // Eq. 12, gamma vs tau
    } else {
        dec = PREPOS_SERVED;  // Alg. 2 l.6
    }
    decision[r] = dec;
    token[r] = (dec == PREPOS_SERVED) ? top1 : -1;
}

// Sec. 3.6: version bump + valid clear.  Atomics so that repeated ids each count as one mutation.
__global__ void __launch_bounds__(128) invalidate_kernel(int n, const int32_t *__restrict__ session_ids,
                                                         unsigned long long *__restrict__ session_version,
                                                         prepos_record *__restrict__ records)
{
    ptx::griddep_wait();
    ptx::griddep_launch();
    const int r = blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= n) return;
    const int sid = session_ids[r];
    atomicAnd(&records[sid].flags, ~PREPOS_FLAG_VALID);
    __threadfence();
    atomicAdd(&session_version[sid], 1ull);
}

// Wilson score interval of k successes in n trials, fp64 (z = the two-sided 95% normal quantile)
__device__ __forceinline__ void wilson95(int k, int n, double &lo, double &hi)
{
    if (n <= 0) {
        lo = 0.0;
        hi = 1.0;
        return;
    }
    const double z = 1.959963984540054;
    const double p = static_cast<double>(k) / n;
    const double den = 1.0 + z * z / n;
    const double centre = (p + z * z / (2.0 * n)) / den;
    const double half = z * sqrt(p * (1.0 - p) / n + z * z / (4.0 * static_cast<double>(n) * n)) / den;
    lo = centre - half;
    hi = centre + half;
}

// Eq. 13-14 for one threshold per CTA: two integer counts over the n records, then the rates and intervals.
__global__ void __launch_bounds__(256) gate_sweep_kernel(int n, const prepos_record *__restrict__ records,
                                                         const uint64_t *__restrict__ session_version,
                                                         const uint32_t *__restrict__ bitmap, int vocab,
                                                         const int32_t *__restrict__ full_path_token,
                                                         const float *__restrict__ taus, int strict_gt,
                                                         prepos_sweep_point *__restrict__ out)
{
    ptx::griddep_wait();
    ptx::griddep_launch();
    const float tau = taus[blockIdx.x];
    int acc = 0, bad = 0;
    for (int i = threadIdx.x; i < n; i += blockDim.x) {
        const uint4 *p = reinterpret_cast<const uint4 *>(records + i);
        const uint4 w0 = p[0];  // max_logit, lse, top1, top2
        const uint4 w1 = p[1];  // gap, flags, version
        const int32_t top1 = static_cast<int32_t>(w0.z);
        const float gap = __uint_as_float(w1.x);
        const uint32_t flags = w1.y;
        const uint64_t rec_version = (static_cast<uint64_t>(w1.w) << 32) | w1.z;
        const bool servable = (flags & PREPOS_FLAG_VALID) && !(flags & PREPOS_FLAG_NONFINITE) &&
                              rec_version == session_version[i] && top1 >= 0 && top1 < vocab &&
                              ((bitmap[top1 >> 5] >> (top1 & 31)) & 1u);
        const bool a = servable && (strict_gt ? (gap > tau) : (gap >= tau)) && (fabsf(gap) <= 3.0e38f);
        acc += a;
        bad += a && (top1 != full_path_token[i]);
    }
    __shared__ int s_acc[8], s_bad[8];
#pragma unroll
    for (int m = 16; m > 0; m >>= 1) {
        acc += __shfl_xor_sync(0xffffffffu, acc, m);
        bad += __shfl_xor_sync(0xffffffffu, bad, m);
    }
    if ((threadIdx.x & 31) == 0) {
        s_acc[threadIdx.x >> 5] = acc;
        s_bad[threadIdx.x >> 5] = bad;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        int a = 0, f = 0;
        for (int w = 0; w < static_cast<int>(blockDim.x >> 5); ++w) {
            a += s_acc[w];
            f += s_bad[w];
        }
        prepos_sweep_point r;
        r.tau = tau;
        r.n = n;
        r.accepted = a;
        r.false_accepts = f;
        r.coverage = n > 0 ? static_cast<double>(a) / n : 0.0;
        r.far = a > 0 ? static_cast<double>(f) / a : 0.0;
        wilson95(a, n, r.cov_lo, r.cov_hi);
        wilson95(f, a, r.far_lo, r.far_hi);
        out[blockIdx.x] = r;
    }
}

}  // namespace

int prepos_launch_gate_sweep(prepos_ctx *ctx, int n, const prepos_record *records, const uint64_t *session_version,
                             const uint32_t *bitmap, const int32_t *full_path_token, int n_tau, const float *taus,
                             int strict_gt, prepos_sweep_point *out, cudaStream_t stream)
{
    if (n_tau == 0) return PREPOS_OK;
    PREPOS_CUDA_TRY(prepos_launch_pdl(gate_sweep_kernel, dim3(n_tau), dim3(256), 0, stream, n, records, session_version,
                                      bitmap, ctx->shape.vocab, full_path_token, taus, strict_gt, out));
    ctx->launches += 1;
    return PREPOS_OK;
}

int prepos_launch_gate_serve(prepos_ctx *ctx, int n, const int32_t *session_ids, const uint64_t *req_hash,
                             const prepos_record *records, const uint64_t *session_version,
                             const uint32_t *bitmap, float tau, int strict_gt, int32_t *decision, int32_t *token,
                             cudaStream_t stream)
{
    if (n == 0) return PREPOS_OK;
    const int threads = 128;
    PREPOS_CUDA_TRY(prepos_launch_pdl(gate_serve_kernel, dim3((n + threads - 1) / threads), dim3(threads), 0, stream, n,
                                      session_ids, req_hash, records, session_version, bitmap, ctx->shape.vocab, tau,
                                      strict_gt, decision, token));
    ctx->launches += 1;
    return PREPOS_OK;
}

int prepos_launch_invalidate(prepos_ctx *ctx, int n, const int32_t *session_ids, uint64_t *session_version,
                             prepos_record *records, cudaStream_t stream)
{
    if (n == 0) return PREPOS_OK;
    const int threads = 128;
    PREPOS_CUDA_TRY(prepos_launch_pdl(invalidate_kernel, dim3((n + threads - 1) / threads), dim3(threads), 0, stream, n,
                                      session_ids, reinterpret_cast<unsigned long long *>(session_version), records));
    ctx->launches += 1;
    return PREPOS_OK;
}
