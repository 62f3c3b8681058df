/*
 * oracle/attention.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, obviously-correct CPU oracle (fp64) for the hot path of KernelFlume
 * (arxiv/paper_2606_29207): decode core-attention of one new-token query over a request's KV
 * cache, the same restricted to one token range (the "partial" an attention node returns), and
 * the log-sum-exp merge of partials.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may build, link, import or call this file.  It shares no
 * code, header, table or helper with the CUDA path and includes nothing from include/ or
 * paper_2606_29207_b200/.
 *
 * What it follows:
 *  - PAPER.md:81  (sec 2.2): decode attention of the new token over the whole accumulated KV cache.
 *  - PAPER.md:145-147 (sec 3.2 steps 3-4): each attention node computes local attention over its
 *    token-range partition and returns partials (o_i, m_i, l_i), combined "with the standard
 *    online-softmax (log-sum-exp) reduction".
 *  - PAPER.md:254 (sec 5.1): "This merge produces the same result as computing attention over the
 *    full KV range" -- so the oracle for the merged result is the plain softmax definition.
 *  The paper prints no attention formula; the textbook definition is used (readings 1-6):
 *      s_t  = scale * sum_i q[h][i] * K[g][t][i],   g = h / G  (G = H_q / H_kv, integer division)
 *      m    = max_t s_t ;  l = sum_t exp(s_t - m) ;  lse = m + ln(l)
 *      o[j] = ( sum_t exp(s_t - m) * V[g][t][j] ) / l
 *  Partials are returned as (o_i normalised, lse_i = m_i + ln l_i)  (reading 3).
 *  merge:  M = max_j lse_j ; lse = M + ln sum_j exp(lse_j - M) ; o = sum_j exp(lse_j - lse) * o_j
 *
 * No blocking, tiling, fusion or reordering beyond the definition: two plain passes over t.
 * fp16 inputs are converted to double exactly, all arithmetic is IEEE double.
 * OpenMP is used only ACROSS independent (request, head) problems in the batch entry point.
 *
 * Pins (tests/test_oracle_*.py): 1-token context, identical keys, q = 0, two-token sigmoid, the
 * d=1 hand example (lse = ln 6, o = 14), constant V, convexity bounds, permutation and shift
 * invariance, scipy/numpy fp64, 40-digit mpmath brute force, golden values of SURVEY.md App. B,
 * split/merge invariance, GQA head-mapping.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* POW2_M25[e] = 2^(e-25) for the biased binary16 exponent e = 1..30 (entries 0 and 31 unused). */
static const double POW2_M25[32] = {
    0.0,     0x1p-24, 0x1p-23, 0x1p-22, 0x1p-21, 0x1p-20, 0x1p-19, 0x1p-18, 0x1p-17, 0x1p-16, 0x1p-15,
    0x1p-14, 0x1p-13, 0x1p-12, 0x1p-11, 0x1p-10, 0x1p-9,  0x1p-8,  0x1p-7,  0x1p-6,  0x1p-5,  0x1p-4,
    0x1p-3,  0x1p-2,  0x1p-1,  0x1p0,   0x1p1,   0x1p2,   0x1p3,   0x1p4,   0x1p5,   0.0};

/* IEEE binary16 -> double, exact (handles zero, subnormal, inf, nan). */
static double half_to_double(uint16_t h)
{
    int sign = (h >> 15) & 1;
    int expo = (h >> 10) & 0x1f;
    int mant = h & 0x3ff;
    double v;
    if (expo == 0) {
        v = (double)mant * 0x1p-24;                   /* subnormal: mant * 2^-24 (exact) */
    } else if (expo == 31) {
        v = mant ? NAN : INFINITY;
    } else {
        v = (double)(mant | 0x400) * POW2_M25[expo];  /* (1024+mant) * 2^(expo-25), exact */
    }
    return sign ? -v : v;
}

/*
 * Attention of ONE query head over tokens [t_begin, t_end) of ONE kv head.
 *   q      : [d] fp16 bits
 *   K, V   : [n_tokens_total][d] fp16 bits (row t = token t)
 *   o      : [d] double out;  lse : double out
 * Returns 0, or -1 if the token range is empty (o, lse untouched) or allocation fails.
 */
int kfo_attend_head(const uint16_t *q, const uint16_t *K, const uint16_t *V, int64_t t_begin,
                    int64_t t_end, int d, double scale, double *o, double *lse)
{
    int64_t n = t_end - t_begin;
    if (n <= 0) return -1;
    double *s = (double *)malloc((size_t)n * sizeof(double));
    double *qd = (double *)malloc((size_t)d * sizeof(double));
    if (!s || !qd) { free(s); free(qd); return -1; }
    for (int i = 0; i < d; ++i) qd[i] = half_to_double(q[i]);
    double m = -INFINITY;
    for (int64_t t = 0; t < n; ++t) {
        const uint16_t *k = K + (size_t)(t_begin + t) * d;
        double acc = 0.0;
        for (int i = 0; i < d; ++i) acc += qd[i] * half_to_double(k[i]);
        s[t] = scale * acc;
        if (s[t] > m) m = s[t];
    }
    double l = 0.0;
    for (int j = 0; j < d; ++j) o[j] = 0.0;
    for (int64_t t = 0; t < n; ++t) {
        double p = exp(s[t] - m);
        const uint16_t *v = V + (size_t)(t_begin + t) * d;
        l += p;
        for (int j = 0; j < d; ++j) o[j] += p * half_to_double(v[j]);
    }
    for (int j = 0; j < d; ++j) o[j] /= l;
    *lse = m + log(l);
    free(s);
    free(qd);
    return 0;
}

/*
 * One request, all query heads, tokens [t_begin, t_end).
 *   q : [H_q][d];  K, V : [H_kv][n_tokens_total][d];  o : [H_q][d];  lse : [H_q]
 * GQA mapping: query head h uses kv head h / (H_q / H_kv)   (reading 2).
 */
int kfo_attend_request(const uint16_t *q, const uint16_t *K, const uint16_t *V, int n_q_heads,
                       int n_kv_heads, int64_t n_tokens_total, int64_t t_begin, int64_t t_end, int d,
                       double scale, double *o, double *lse, int n_threads)
{
    if (n_q_heads % n_kv_heads) return -2;
    int G = n_q_heads / n_kv_heads;
    int rc = 0;
#ifdef _OPENMP
    if (n_threads <= 0) n_threads = omp_get_max_threads();
#pragma omp parallel for schedule(dynamic, 1) num_threads(n_threads)
#endif
    for (int h = 0; h < n_q_heads; ++h) {
        int g = h / G;
        int r = kfo_attend_head(q + (size_t)h * d, K + (size_t)g * n_tokens_total * d,
                                V + (size_t)g * n_tokens_total * d, t_begin, t_end, d, scale,
                                o + (size_t)h * d, lse + h);
        if (r) {
#ifdef _OPENMP
#pragma omp critical
#endif
            rc = r;
        }
    }
    return rc;
}

/*
 * Merge J partials of one head:  lse_j [J], o_j [J][d]  ->  o [d], lse.
 * A partial with lse_j = -inf has weight 0 (reading 13).  If every lse_j = -inf the
 * result is lse = -inf, o = 0.
 */
int kfo_merge_head(const double *lse_j, const double *o_j, int J, int d, double *o, double *lse)
{
    double M = -INFINITY;
    for (int j = 0; j < J; ++j)
        if (lse_j[j] > M) M = lse_j[j];
    for (int i = 0; i < d; ++i) o[i] = 0.0;
    if (M == -INFINITY) { *lse = -INFINITY; return 0; }
    double sum = 0.0;
    for (int j = 0; j < J; ++j) sum += exp(lse_j[j] - M);
    *lse = M + log(sum);
    for (int j = 0; j < J; ++j) {
        double w = exp(lse_j[j] - *lse);
        if (w == 0.0) continue;  /* also skips 0 * (garbage o_j) for lse_j = -inf */
        for (int i = 0; i < d; ++i) o[i] += w * o_j[(size_t)j * d + i];
    }
    return 0;
}

int kfo_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
