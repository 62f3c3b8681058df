/*
 * oracle/wside.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain fp64 oracle of the W-node stages that surround core attention in a decode layer of KernelFlume
 * (arxiv/paper_2606_29207): the QKV projection in front of it (PAPER.md:143 step 1, :137 "W nodes keep weights"),
 * and W_O and the feed-forward network behind it (PAPER.md:147 step 5, :254 "merge ... before applying W_O and FFN",
 * :266-268 T_p and T_f of the inter-layer pipeline).  Each of these is a dense contraction with a plain definition,
 *
 *      y[b][n] = sum_k x[b][k] * W[n][k]            (W stored [out_features][in_features], the nn.Linear convention)
 *
 * written out as the triple loop, k ascending, in IEEE double; and the FFN's gated activation of the Llama models
 * the paper serves, SwiGLU:  h = silu(g) * u,  silu(z) = z / (1 + exp(-z)).
 * No blocking, no reordering, no library call.  OpenMP only across independent output elements.
 * It shares nothing with the CUDA path and includes nothing from include/ or paper_2606_29207_b200/.
 *
 * Pins (tests/test_oracle_wside.py): identity weights, one-hot rows, a 2x3 hand example, linearity, numpy's fp64
 * matmul, silu at 0 / ln 3 / -ln 3, silu(z) - silu(-z) = z.
 */
#include <math.h>
#include <stdint.h>
#ifdef _OPENMP
#include <omp.h>
#endif

int kfo_linear(const double *x, const double *w, int64_t B, int64_t N, int64_t K, double *y)
{
    if (!x || !w || !y || B < 0 || N < 0 || K < 0) return -1;
    int64_t bn;
#pragma omp parallel for schedule(static)
    for (bn = 0; bn < B * N; ++bn) {
        const int64_t b = bn / N, n = bn % N;
        double acc = 0.0;
        for (int64_t k = 0; k < K; ++k) acc += x[b * K + k] * w[n * K + k];
        y[bn] = acc;
    }
    return 0;
}

int kfo_swiglu(const double *g, const double *u, int64_t n, double *h)
{
    if (!g || !u || !h || n < 0) return -1;
    for (int64_t i = 0; i < n; ++i) h[i] = g[i] / (1.0 + exp(-g[i])) * u[i];
    return 0;
}
