/*
 * prepos_oracle.c -- the CPU ORACLE for the speculative pre-positioning hot path.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may build, load or call it.
 * It shares no code, header, table or helper with the CUDA path
 * (paper_2606_29565_b200/csrc) and neither side includes the other.
 *
 * Every function is the plain definition of what the paper's step computes, written
 * out in fp64 (inputs are the exact bf16 bit patterns widened to double), with no
 * blocking, fusion or reordering beyond the definition, so it can be checked
 * against /root/reference/PAPER.md by eye.  Citations are PAPER.md:<line>.
 *
 *   O1 oracle_entry_attn   Alg. 1 l.2-6, Eq. 1
 *   O2 oracle_logits       "logits at the final entry position"
 *   O3 oracle_record       Eq. 11, Alg. 2 l.3-4
 *   O4 oracle_gate         Eq. 12, Alg. 2
 *   O5 oracle_invalidate / oracle_stamp   Sec. 3.6, Fig. 3
 *   O7 oracle_entry_attn_fp8  O1 over an FP8 (e4m3) KV cache   } the quantised variants of SURVEY.md 8(f) NEXT-4
 *   O8 oracle_logits_w4       O2 over a 4-bit W_vocab          } (the paper's headline model "runs at 4-bit
 *                             precision").  The paper gives no storage format: the rules are
 *                             this build's reading, Q20 / Q21; each dequantises exactly and then IS O1 / O2.
 *
 * Pins (tests/test_oracle_*.py, all `-m "not gpu"`): every function here is pinned by
 * closed forms, invariants, library cross-checks and brute force; none is "parity unpinned".
 * O7 / O8: the e4m3 codec against a library's e4m3 on all 256 codes and a dense grid of values, and
 * equality with O1 / O2 wherever code * scale is exactly representable (tests/test_oracle_quant.py).
 *
 * OpenMP is used only over independent outputs (query rows, vocabulary rows); each
 * output is still computed by the serial definition.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* exact widening of a bf16 bit pattern: bf16 is the top 16 bits of an IEEE fp32 */
static double bf16_to_double(uint16_t b)
{
    uint32_t u = ((uint32_t)b) << 16;
    float f;
    memcpy(&f, &u, sizeof f);
    return (double)f;
}

/* physical element offset of logical cache token j for kv head g.
 * Pool layout [n_pages][Hkv][page][d] (reading Q6): page = table[j / page]. */
static size_t pool_offset(const int32_t *page_table, int j, int g, int Hkv, int page, int d)
{
    size_t pg = (size_t)page_table[j / page];
    return ((pg * (size_t)Hkv + (size_t)g) * (size_t)page + (size_t)(j % page)) * (size_t)d;
}

/*
 * O1.  Pre-position entry attention for ONE session and ONE layer.
 *
 * Alg. 1:
 *   l.2-3  if L_entry > B (headroom = capacity_tokens - n_s): skip, no side effect  -> returns 1
 *   l.5    Append(E) at end position n_s: K_new/V_new written to cache positions n_s..n_s+L-1
 *   l.6    Forward(E): here, its attention part.  Entry row i (position n_s+i) attends the
 *          resident state j < n_s and the entry tokens j' <= i ("causal among themselves",
 *          BASELINE.json north_star; reading Q5), i.e. cache positions 0..n_s+i:
 *              s_j = (q_i . k_j) * scale ;  p_j = exp(s_j - m) / sum_j exp(s_j - m) ;  o_i = sum_j p_j v_j
 *          GQA: query head h reads kv head g = h / (Hq/Hkv)  (reading Q4).
 *   l.7    p = n_s + L  (Eq. 1) -> *position_out
 *
 * q      [L][Hq][d]   bf16 bits          k_new,v_new [L][Hkv][d] bf16 bits
 * k_pool,v_pool [n_pages][Hkv][page][d] bf16 bits, modified in place by the append
 * page_table    [>= ceil((n_s+L)/page)] physical page ids of this session
 * out    [L][Hq][d]   fp64   (untouched when skipped)
 * rowsum [L][Hq]      fp64   sum_j p_j of every row (for the "softmax sums to 1" pin); may be NULL
 * returns 0 = done, 1 = skipped on budget, -1 = bad argument
 */
/* The same pass, producing only the outputs (h, i) with h_lo <= h < h_hi, i_lo <= i < i_hi (the other rows of `out`
 * and `rowsum` are left untouched; the append is always done in full).  oracle_entry_attn below IS this function
 * over the full ranges, so every pin of O1 exercises this code; the sampled full-size parity tests use the ranges. */
int oracle_entry_attn_ranged(const uint16_t *q, const uint16_t *k_new, const uint16_t *v_new,
                             uint16_t *k_pool, uint16_t *v_pool, const int32_t *page_table,
                             int n_s, int L, int capacity_tokens,
                             int Hq, int Hkv, int d, int page, double scale,
                             int h_lo, int h_hi, int i_lo, int i_hi,
                             double *out, double *rowsum, int64_t *position_out)
{
    if (n_s < 0 || L < 0 || Hq <= 0 || Hkv <= 0 || d <= 0 || page <= 0 || Hq % Hkv != 0)
        return -1;
    if (h_lo < 0 || h_hi > Hq || i_lo < 0 || i_hi > L)
        return -1;
    /* Alg. 1 l.2-3: cell-budget headroom B = capacity - n_s */
    if (L > capacity_tokens - n_s)
        return 1;
    const int G = Hq / Hkv;

    /* Alg. 1 l.5: Append(E) at end position n_s */
    for (int jp = 0; jp < L; ++jp)
        for (int g = 0; g < Hkv; ++g) {
            size_t dst = pool_offset(page_table, n_s + jp, g, Hkv, page, d);
            size_t src = ((size_t)jp * (size_t)Hkv + (size_t)g) * (size_t)d;
            memcpy(k_pool + dst, k_new + src, (size_t)d * sizeof(uint16_t));
            memcpy(v_pool + dst, v_new + src, (size_t)d * sizeof(uint16_t));
        }

    /* Alg. 1 l.6: attention of each entry row over cache positions 0..n_s+i */
    int bad = 0;
#pragma omp parallel for collapse(2) schedule(dynamic, 1)
    for (int h = h_lo; h < h_hi; ++h)
        for (int i = i_lo; i < i_hi; ++i) {
            const int g = h / G;
            const int n_keys = n_s + i + 1;
            double *s = (double *)malloc((size_t)n_keys * sizeof(double));
            if (!s) {
                bad = 1;
                continue;
            }
            const uint16_t *qi = q + ((size_t)i * (size_t)Hq + (size_t)h) * (size_t)d;
            double m = -INFINITY;
            for (int j = 0; j < n_keys; ++j) {
                const uint16_t *kj = k_pool + pool_offset(page_table, j, g, Hkv, page, d);
                double acc = 0.0;
                for (int c = 0; c < d; ++c)
                    acc += bf16_to_double(qi[c]) * bf16_to_double(kj[c]);
                s[j] = acc * scale;
                if (s[j] > m)
                    m = s[j];
            }
            double denom = 0.0;
            for (int j = 0; j < n_keys; ++j) {
                s[j] = exp(s[j] - m);
                denom += s[j];
            }
            double *oi = out + ((size_t)i * (size_t)Hq + (size_t)h) * (size_t)d;
            for (int c = 0; c < d; ++c)
                oi[c] = 0.0;
            double psum = 0.0;
            for (int j = 0; j < n_keys; ++j) {
                const double p = s[j] / denom;
                psum += p;
                const uint16_t *vj = v_pool + pool_offset(page_table, j, g, Hkv, page, d);
                for (int c = 0; c < d; ++c)
                    oi[c] += p * bf16_to_double(vj[c]);
            }
            if (rowsum)
                rowsum[(size_t)i * (size_t)Hq + (size_t)h] = psum;
            free(s);
        }
    if (bad)
        return -1;
    if (position_out)
        *position_out = (int64_t)n_s + (int64_t)L; /* Eq. 1 */
    return 0;
}

int oracle_entry_attn(const uint16_t *q, const uint16_t *k_new, const uint16_t *v_new,
                      uint16_t *k_pool, uint16_t *v_pool, const int32_t *page_table,
                      int n_s, int L, int capacity_tokens,
                      int Hq, int Hkv, int d, int page, double scale,
                      double *out, double *rowsum, int64_t *position_out)
{
    return oracle_entry_attn_ranged(q, k_new, v_new, k_pool, v_pool, page_table, n_s, L, capacity_tokens, Hq, Hkv, d,
                                    page, scale, 0, Hq, 0, L < 0 ? 0 : L, out, rowsum, position_out);
}

/*
 * O2.  Ready-distribution logits: l_v = sum_k W[v][k] * x[k].
 * w [V][H] bf16 bits row-major, x [H] bf16 bits (reading Q7: the caller's final hidden
 * state of the last entry position), logits [V] fp64.
 */
void oracle_logits(const uint16_t *w, const uint16_t *x, int V, int H, double *logits)
{
#pragma omp parallel for schedule(static)
    for (int v = 0; v < V; ++v) {
        const uint16_t *wv = w + (size_t)v * (size_t)H;
        double acc = 0.0;
        for (int k = 0; k < H; ++k)
            acc += bf16_to_double(wv[k]) * bf16_to_double(x[k]);
        logits[v] = acc;
    }
}

/* ------------------------------------------------------------------------------------------------------------------
 * Quantised variants ("4-bit precision").  The paper states no format, so
 * these follow DESIGN.md readings Q20 (FP8 KV) and Q21 (4-bit W_vocab).  Both dequantise EXACTLY (every code times
 * its scale is formed in fp64) and then apply the fp64 definitions O1 / O2 unchanged.
 * ---------------------------------------------------------------------------------------------------------------- */

/* OCP FP8 E4M3 ("e4m3fn"): 1 sign, 4 exponent (bias 7), 3 mantissa bits; no infinities; S.1111.111 is NaN;
 * exponent field 0 is subnormal: (m/8) * 2^-6.  Largest finite value 448 = 1.75 * 2^8. */
double oracle_e4m3_decode(uint8_t b)
{
    const int sign = b >> 7, e = (b >> 3) & 15, m = b & 7;
    double v;
    if (e == 15 && m == 7)
        return NAN;
    if (e == 0)
        v = ldexp((double)m / 8.0, -6);
    else
        v = ldexp(1.0 + (double)m / 8.0, e - 7);
    return sign ? -v : v;
}

/* fp32 -> e4m3, round to nearest, ties to the even code, saturating to +-448 (NaN -> 0x7f).  Written as a search
 * over the 127 finite magnitudes (codes 0x00..0x7e are monotone in value), not as bit manipulation. */
uint8_t oracle_e4m3_encode(float y)
{
    if (isnan(y))
        return 0x7f;
    const uint8_t sign = signbit(y) ? 0x80 : 0x00;
    const double a = fabs((double)y);
    if (a >= 448.0)
        return (uint8_t)(sign | 0x7e);
    int lo = 0; /* largest code with value <= a */
    for (int c = 0; c <= 0x7e; ++c)
        if (oracle_e4m3_decode((uint8_t)c) <= a)
            lo = c;
    if (lo == 0x7e)
        return (uint8_t)(sign | 0x7e);
    const double vlo = oracle_e4m3_decode((uint8_t)lo), vhi = oracle_e4m3_decode((uint8_t)(lo + 1));
    int pick;
    if (a - vlo < vhi - a)
        pick = lo;
    else if (a - vlo > vhi - a)
        pick = lo + 1;
    else
        pick = (lo & 1) ? lo + 1 : lo; /* tie: even mantissa */
    return (uint8_t)(sign | pick);
}

/* scale of logical cache token j, kv head g: scales are [n_pages][Hkv] fp32, one per (page, kv head) (Q20) */
static double page_scale(const float *scale, const int32_t *page_table, int j, int g, int Hkv, int page)
{
    return (double)scale[(size_t)page_table[j / page] * (size_t)Hkv + (size_t)g];
}

/*
 * O7.  O1 over an FP8 KV cache (reading Q20).  k_pool8 / v_pool8 [n_pages][Hkv][page][d] are e4m3 codes;
 * k_scale / v_scale [n_pages][Hkv] fp32 are caller-owned, one per (page, kv head), for every page of the session
 * including the ones the entry is appended to.  Cached value = decode(code) * scale.
 *   l.5  Append(E): code = e4m3(fp32(x) / scale) with the fp32 division and the conversion rounded to nearest even,
 *        saturating (both sides take this decision in fp32, the kernel's precision)
 *   l.6  Forward(E) runs after the append (Alg. 1 order), so entry row i sees the entry tokens j' <= i through
 *        their STORED codes -- which makes a pre-position of L1 then L2 tokens identical to one of L1 + L2.
 * Everything else (budget skip, scale, GQA map, two-pass softmax in fp64) is O1 word for word.
 */
int oracle_entry_attn_fp8(const uint16_t *q, const uint16_t *k_new, const uint16_t *v_new,
                          uint8_t *k_pool8, uint8_t *v_pool8, const float *k_scale, const float *v_scale,
                          const int32_t *page_table, int n_s, int L, int capacity_tokens,
                          int Hq, int Hkv, int d, int page, double scale,
                          int h_lo, int h_hi, int i_lo, int i_hi,
                          double *out, int64_t *position_out)
{
    if (n_s < 0 || L < 0 || Hq <= 0 || Hkv <= 0 || d <= 0 || page <= 0 || Hq % Hkv != 0)
        return -1;
    if (h_lo < 0 || h_hi > Hq || i_lo < 0 || i_hi > L)
        return -1;
    if (L > capacity_tokens - n_s)
        return 1;
    const int G = Hq / Hkv;

    for (int jp = 0; jp < L; ++jp)
        for (int g = 0; g < Hkv; ++g) {
            const size_t dst = pool_offset(page_table, n_s + jp, g, Hkv, page, d);
            const size_t src = ((size_t)jp * (size_t)Hkv + (size_t)g) * (size_t)d;
            const float ks = k_scale[(size_t)page_table[(n_s + jp) / page] * (size_t)Hkv + (size_t)g];
            const float vs = v_scale[(size_t)page_table[(n_s + jp) / page] * (size_t)Hkv + (size_t)g];
            for (int c = 0; c < d; ++c) {
                k_pool8[dst + c] = oracle_e4m3_encode((float)bf16_to_double(k_new[src + c]) / ks);
                v_pool8[dst + c] = oracle_e4m3_encode((float)bf16_to_double(v_new[src + c]) / vs);
            }
        }

    int bad = 0;
#pragma omp parallel for collapse(2) schedule(dynamic, 1)
    for (int h = h_lo; h < h_hi; ++h)
        for (int i = i_lo; i < i_hi; ++i) {
            const int g = h / G;
            const int n_keys = n_s + i + 1;
            double *s = (double *)malloc((size_t)n_keys * sizeof(double));
            if (!s) {
                bad = 1;
                continue;
            }
            const uint16_t *qi = q + ((size_t)i * (size_t)Hq + (size_t)h) * (size_t)d;
            double m = -INFINITY;
            for (int j = 0; j < n_keys; ++j) {
                const uint8_t *kj = k_pool8 + pool_offset(page_table, j, g, Hkv, page, d);
                const double ks = page_scale(k_scale, page_table, j, g, Hkv, page);
                double acc = 0.0;
                for (int c = 0; c < d; ++c)
                    acc += bf16_to_double(qi[c]) * (oracle_e4m3_decode(kj[c]) * ks);
                s[j] = acc * scale;
                if (s[j] > m)
                    m = s[j];
            }
            double denom = 0.0;
            for (int j = 0; j < n_keys; ++j) {
                s[j] = exp(s[j] - m);
                denom += s[j];
            }
            double *oi = out + ((size_t)i * (size_t)Hq + (size_t)h) * (size_t)d;
            for (int c = 0; c < d; ++c)
                oi[c] = 0.0;
            for (int j = 0; j < n_keys; ++j) {
                const double p = s[j] / denom;
                const uint8_t *vj = v_pool8 + pool_offset(page_table, j, g, Hkv, page, d);
                const double vs = page_scale(v_scale, page_table, j, g, Hkv, page);
                for (int c = 0; c < d; ++c)
                    oi[c] += p * (oracle_e4m3_decode(vj[c]) * vs);
            }
            free(s);
        }
    if (bad)
        return -1;
    if (position_out)
        *position_out = (int64_t)n_s + (int64_t)L;
    return 0;
}

/*
 * O8.  O2 over a 4-bit W_vocab (reading Q21).  w4 [V][H/2]: two codes per byte, the element with even k in the low
 * nibble; a code is a two's-complement int4 in -8..7.  w_scale [V][H/group] bf16 bits, one per (row, group of `group`
 * consecutive k).  W[v][k] = code * scale[v][k / group]; then l_v = sum_k W[v][k] x[k] exactly as O2.
 */
void oracle_logits_w4(const uint8_t *w4, const uint16_t *w_scale, const uint16_t *x, int V, int H, int group,
                      double *logits)
{
#pragma omp parallel for schedule(static)
    for (int v = 0; v < V; ++v) {
        const uint8_t *wv = w4 + (size_t)v * (size_t)(H / 2);
        const uint16_t *sv = w_scale + (size_t)v * (size_t)(H / group);
        double acc = 0.0;
        for (int k = 0; k < H; ++k) {
            const int nib = (k & 1) ? (wv[k >> 1] >> 4) : (wv[k >> 1] & 15);
            const int code = nib >= 8 ? nib - 16 : nib;
            acc += ((double)code * bf16_to_double(sv[k / group])) * bf16_to_double(x[k]);
        }
        logits[v] = acc;
    }
}

/* the ready-distribution record of BASELINE.json north_star: max, logsumexp, top-1, top-2, gap */
typedef struct {
    double max_logit; /* l^(1) */
    double lse;       /* log sum_v exp(l_v), natural log (reading Q10) */
    double gap;       /* gamma = l^(1) - l^(2), Eq. 11 */
    int32_t top1;     /* argmax, Alg. 2 l.4 */
    int32_t top2;     /* index of l^(2) */
    int32_t nonfinite;/* 1 if any logit is NaN/Inf (reading Q18): such a record never serves */
    int32_t pad_;
} oracle_record_t;

/*
 * O3.  Top2 / gap / argmax (Eq. 11; Alg. 2 l.3-4) plus
 * max and logsumexp.  Tokens are ordered by (logit descending, id ascending) (reading Q8):
 * top1, top2 are the first two in that order.  V == 1: top2 = -1, gap = +inf.
 */
void oracle_record(const double *logits, int V, oracle_record_t *rec)
{
    int t1 = -1, t2 = -1;
    int nonfinite = 0;
    for (int v = 0; v < V; ++v) {
        const double l = logits[v];
        if (!isfinite(l))
            nonfinite = 1;
        /* strict '>' keeps the lowest id among equal logits ahead */
        if (t1 < 0 || l > logits[t1]) {
            t2 = t1;
            t1 = v;
        } else if (t2 < 0 || l > logits[t2]) {
            t2 = v;
        }
    }
    rec->top1 = t1;
    rec->top2 = t2;
    rec->nonfinite = nonfinite;
    rec->pad_ = 0;
    rec->max_logit = (t1 >= 0) ? logits[t1] : -INFINITY;
    rec->gap = (t2 >= 0) ? logits[t1] - logits[t2] : INFINITY;
    double sum = 0.0;
    for (int v = 0; v < V; ++v)
        sum += exp(logits[v] - rec->max_logit);
    rec->lse = rec->max_logit + log(sum);
}

/* decision codes of the serve (shared vocabulary with include/prepos.h by value only) */
enum {
    ORACLE_SERVED = 0,
    ORACLE_GAP_BELOW_TAU = 1,
    ORACLE_NOT_IN_FAST_SET = 2,
    ORACLE_STALE_OR_INVALID = 3,
    ORACLE_INELIGIBLE = 4
};

/*
 * O4.  Confidence-gated serve for one request (Alg. 2; Eq. 12).
 *   l.1  not valid (flag clear, version stamp != live session version, non-finite) -> fall through
 *        ineligible (realised entry hash != pre-positioned entry hash; hash 0 on either
 *        side = the relaxed streaming match of PAPER.md:172)                       -> fall through
 *   l.5  serve top1 iff gamma >= tau (strict_gt: gamma > tau, the paper's form; reading Q1)
 *        and top1 in A (bitmap over the vocabulary)
 * First failing reason is reported in the order stale/invalid, ineligible, not-in-set, gap.
 * Returns the decision code; *token = top1 when SERVED else -1.
 */
int oracle_gate(double gap, int32_t top1, int valid, int nonfinite,
                uint64_t record_version, uint64_t session_version,
                uint64_t record_hash, uint64_t request_hash,
                const uint32_t *fast_set_bitmap, int V, double tau, int strict_gt,
                int32_t *token)
{
    *token = -1;
    if (!valid || nonfinite || record_version != session_version)
        return ORACLE_STALE_OR_INVALID;
    if (record_hash != 0 && request_hash != 0 && record_hash != request_hash)
        return ORACLE_INELIGIBLE;
    if (top1 < 0 || top1 >= V || !((fast_set_bitmap[top1 >> 5] >> (top1 & 31)) & 1u))
        return ORACLE_NOT_IN_FAST_SET;
    if (strict_gt ? !(gap > tau) : !(gap >= tau))
        return ORACLE_GAP_BELOW_TAU;
    *token = top1;
    return ORACLE_SERVED;
}

/*
 * O5.  Invalidation (Fig. 3): every mutation of the
 * persistent state bumps the session's version and clears the validity flag of its record
 * in the same step.  ids may repeat; each occurrence is one mutation.
 */
void oracle_invalidate(const int32_t *session_ids, int n, uint64_t *session_version, int32_t *record_valid)
{
    for (int r = 0; r < n; ++r) {
        session_version[session_ids[r]] += 1;
        record_valid[session_ids[r]] = 0;
    }
}

/* Alg. 1 l.10-12: the record is stamped with the version current at pre-position time. */
void oracle_stamp(int32_t session_id, const uint64_t *session_version,
                  uint64_t *record_version, int32_t *record_valid)
{
    record_version[session_id] = session_version[session_id];
    record_valid[session_id] = 1;
}

/* host helper mirrored by tests: A as a bitmap over the vocabulary */
void oracle_fastset_bitmap(const int32_t *ids, int n, int V, uint32_t *bitmap)
{
    const int words = (V + 31) / 32;
    for (int w = 0; w < words; ++w)
        bitmap[w] = 0u;
    for (int r = 0; r < n; ++r)
        if (ids[r] >= 0 && ids[r] < V)
            bitmap[ids[r] >> 5] |= 1u << (ids[r] & 31);
}

/* test-infrastructure plumbing: the 1-thread figure of bench.py's cpu_baseline */
void oracle_set_num_threads(int n)
{
#ifdef _OPENMP
    omp_set_num_threads(n > 0 ? n : 1);
#else
    (void)n;
#endif
}

int oracle_num_threads(void)
{
    int n = 1;
#ifdef _OPENMP
#pragma omp parallel
    {
#pragma omp single
        n = omp_get_num_threads();
    }
#endif
    return n;
}
