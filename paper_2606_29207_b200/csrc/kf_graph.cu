// kf_graph.cu -- one decode step as a static CUDA graph (kf_step_graph_*, include/kflume.h).
//
// The paper keeps the W-node computation in ONE static CUDA Graph and moves every elasticity decision into a
// routing table that the graph never sees (PAPER.md:127 requirement R1, :165-179).  Here the same property
// holds on the device: all hot kernels launch fixed grids and read lengths, routes and the work plan from device
// memory, so a graph captured once stays valid across route updates, range fills and open / close of requests.
// A replay removes the per-launch submission latency between the small kernels of a step (route update, append,
// commit) and the attend kernel.  Input / output pointers may be re-bound at every launch
// (cudaGraphExecKernelNodeSetParams: host-side only, the graph is not re-instantiated).
#include <stdio.h>

#include <new>
#include <vector>

#include "kf_ctx.h"

using namespace kf;

struct kf_graph {
    kf_ctx *ctx;
    cudaGraph_t graph;
    cudaGraphExec_t exec;
    int n;                                  // layer-steps per launch
    int host_io;                            // 1: q/k/v/o/lse are pinned host buffers
    bool zero_copy;                         // host_io graph made of kernels only (no copy nodes): re-bindable
    int kernels_per_launch;
    std::vector<int32_t> layers;
    std::vector<cudaGraphNode_t> append_nodes, attend_nodes;   // [n] (device-pointer graphs only)
    std::vector<cudaKernelNodeParams> append_params, attend_params;
    std::vector<const void *> q, k, v;      // currently bound pointers
    std::vector<float *> o, lse;
};

namespace {

// kernel nodes of a linear (single-stream capture) graph, in execution order
int kernel_chain(cudaGraph_t g, std::vector<cudaGraphNode_t> &out) {
    size_t n = 0;
    if (cudaGraphGetNodes(g, nullptr, &n) != cudaSuccess) return -1;
    std::vector<cudaGraphNode_t> roots(n);
    size_t nr = n;
    if (cudaGraphGetRootNodes(g, roots.data(), &nr) != cudaSuccess || nr != 1) return -1;
    cudaGraphNode_t cur = roots[0];
    for (size_t i = 0; i < n; ++i) {
        cudaGraphNodeType t;
        if (cudaGraphNodeGetType(cur, &t) != cudaSuccess) return -1;
        if (t == cudaGraphNodeTypeKernel) out.push_back(cur);
        size_t nd = 0;
        if (cudaGraphNodeGetDependentNodes(cur, nullptr, &nd) != cudaSuccess) return -1;
        if (nd == 0) break;
        if (nd != 1) return -1;
        cudaGraphNode_t next;
        if (cudaGraphNodeGetDependentNodes(cur, &next, &nd) != cudaSuccess) return -1;
        cur = next;
    }
    return 0;
}

}  // namespace

extern "C" {

int kf_step_graph_create(kf_ctx *ctx, int32_t n_layer_steps, const int32_t *layers, int32_t host_io,
                         const void *const *q, const void *const *k_new, const void *const *v_new, float *const *o,
                         float *const *lse, kf_stream stream, kf_graph **out) {
    if (!out) return KF_EINVAL;
    *out = nullptr;
    if (!ctx || n_layer_steps < 1 || n_layer_steps > 4096 || !layers || !q || !k_new || !v_new || !o || !lse || !stream)
        return KF_EINVAL;
    for (int i = 0; i < n_layer_steps; ++i)
        if (layers[i] < 0 || layers[i] >= ctx->cfg.n_layers || !q[i] || !k_new[i] || !v_new[i] || !o[i] || !lse[i])
            return KF_EINVAL;
    cudaStream_t s = (cudaStream_t)stream;
    kf_graph *g = new (std::nothrow) kf_graph();
    if (!g) return KF_EINVAL;
    g->ctx = ctx;
    g->graph = nullptr;
    g->exec = nullptr;
    g->n = n_layer_steps;
    g->host_io = host_io ? 1 : 0;
    g->zero_copy = false;
    g->layers.assign(layers, layers + n_layer_steps);
    g->q.assign(q, q + n_layer_steps);
    g->k.assign(k_new, k_new + n_layer_steps);
    g->v.assign(v_new, v_new + n_layer_steps);
    g->o.assign(o, o + n_layer_steps);
    g->lse.assign(lse, lse + n_layer_steps);

    const int64_t launches0 = ctx->launches;
    cudaError_t e = cudaStreamBeginCapture(s, cudaStreamCaptureModeThreadLocal);
    if (e != cudaSuccess) {
        delete g;
        return cuda_fail(ctx, e);
    }
    // One fusion that only exists inside the captured step: the step commit is done by the last worker of the last
    // attend launch (2n + 1 kernels per step instead of 2n + 2); the observable state after a launch is that of
    // the public call sequence.  (Folding the first append into the single-CTA plan kernel was measured and
    // dropped: one CTA needs 13 us to copy B = 64 rows that B CTAs copy in 4.)
    int rc = kf_token_boundary(ctx, stream);
    for (int i = 0; i < n_layer_steps && rc == KF_OK; ++i) {
        const int commit = i == n_layer_steps - 1;
        if (g->host_io) {
            rc = kf_layer_step_host_impl(ctx, layers[i], q[i], k_new[i], v_new[i], o[i], lse[i], commit, stream);
        } else {
            rc = kf_kv_append(ctx, layers[i], k_new[i], v_new[i], stream);
            if (rc == KF_OK) rc = kf_attend_impl(ctx, layers[i], q[i], o[i], lse[i], nullptr, nullptr, commit, stream);
        }
    }
    e = cudaStreamEndCapture(s, &g->graph);
    g->kernels_per_launch = (int)(ctx->launches - launches0);
    ctx->launches = launches0;  // nothing ran yet
    if (rc == KF_OK && e != cudaSuccess) rc = cuda_fail(ctx, e);
    if (rc == KF_OK) {
        e = cudaGraphInstantiate(&g->exec, g->graph, 0);
        if (e != cudaSuccess) rc = cuda_fail(ctx, e);
    }
    size_t n_nodes = 0;
    if (rc == KF_OK && cudaGraphGetNodes(g->graph, nullptr, &n_nodes) != cudaSuccess) n_nodes = 0;
    // a host-io graph whose layer-steps all took the zero-copy path consists of kernels only: same shape as a
    // device graph (the staging kernel in place of the append kernel), so it can be re-bound the same way
    g->zero_copy = g->host_io && n_nodes == (size_t)(2 * n_layer_steps + 1);
    if (rc == KF_OK && (!g->host_io || g->zero_copy)) {
        // kernel order of the capture: plan, n x (append or stage, attend)
        std::vector<cudaGraphNode_t> chain;
        if (kernel_chain(g->graph, chain) != 0 || (int)chain.size() != 2 * n_layer_steps + 1) {
            snprintf(ctx->cuda_err, sizeof(ctx->cuda_err), "unexpected step-graph topology");
            rc = KF_ECUDA;
        } else {
            for (int i = 0; i < n_layer_steps && rc == KF_OK; ++i) {
                g->append_nodes.push_back(chain[1 + 2 * i]);
                g->attend_nodes.push_back(chain[2 + 2 * i]);
                cudaKernelNodeParams pa, pt;
                e = cudaGraphKernelNodeGetParams(chain[1 + 2 * i], &pa);
                if (e == cudaSuccess) e = cudaGraphKernelNodeGetParams(chain[2 + 2 * i], &pt);
                if (e != cudaSuccess) rc = cuda_fail(ctx, e);
                g->append_params.push_back(pa);
                g->attend_params.push_back(pt);
            }
        }
    }
    if (rc != KF_OK) {
        cudaGetLastError();
        if (g->exec) cudaGraphExecDestroy(g->exec);
        if (g->graph) cudaGraphDestroy(g->graph);
        delete g;
        return rc;
    }
    *out = g;
    return KF_OK;
}

int kf_step_graph_launch(kf_graph *g, const void *const *q, const void *const *k_new, const void *const *v_new,
                         float *const *o, float *const *lse, kf_stream stream) {
    if (!g || !stream) return KF_EINVAL;
    kf_ctx *ctx = g->ctx;
    const bool rebind = q || k_new || v_new || o || lse;
    if (rebind && ((g->host_io && !g->zero_copy) || !q || !k_new || !v_new || !o || !lse)) return KF_EINVAL;
    if (rebind) {
        for (int i = 0; i < g->n; ++i) {
            if (!q[i] || !k_new[i] || !v_new[i] || !o[i] || !lse[i] || ((uintptr_t)q[i] & 15) || ((uintptr_t)k_new[i] & 15) ||
                ((uintptr_t)v_new[i] & 15) || ((uintptr_t)o[i] & 15))
                return KF_EINVAL;
            if (g->host_io) {
                // kv_append_stage_kernel(Dev d, int layer, k_new, v_new, q_src, q_dst); the attend node reads stage_q
                const bool in_changed = q[i] != g->q[i] || k_new[i] != g->k[i] || v_new[i] != g->v[i];
                const bool out_changed = o[i] != g->o[i] || lse[i] != g->lse[i];
                if ((in_changed && !(device_can_read(q[i]) && device_can_read(k_new[i]) && device_can_read(v_new[i]))) ||
                    (out_changed && !(device_can_read(o[i]) && device_can_read(lse[i]))))
                    return KF_EINVAL;
                if (in_changed) {
                    int layer = g->layers[i];
                    const void *kk = k_new[i], *vv = v_new[i], *qq = q[i];
                    void *qd = ctx->dev.stage_q;
                    void *args[6] = {&ctx->dev, &layer, &kk, &vv, &qq, &qd};
                    cudaKernelNodeParams p = g->append_params[i];
                    p.kernelParams = args;
                    p.extra = nullptr;
                    const cudaError_t e = cudaGraphExecKernelNodeSetParams(g->exec, g->append_nodes[i], &p);
                    if (e != cudaSuccess) return cuda_fail(ctx, e);
                    g->k[i] = k_new[i];
                    g->v[i] = v_new[i];
                }
            } else if (k_new[i] != g->k[i] || v_new[i] != g->v[i]) {
                // kv_append_kernel(Dev d, int layer, const __half *k_new, const __half *v_new)
                int layer = g->layers[i];
                const void *kk = k_new[i], *vv = v_new[i];
                void *args[4] = {&ctx->dev, &layer, &kk, &vv};
                cudaKernelNodeParams p = g->append_params[i];
                p.kernelParams = args;
                p.extra = nullptr;
                const cudaError_t e = cudaGraphExecKernelNodeSetParams(g->exec, g->append_nodes[i], &p);
                if (e != cudaSuccess) return cuda_fail(ctx, e);
                g->k[i] = k_new[i];
                g->v[i] = v_new[i];
            }
            if ((!g->host_io && q[i] != g->q[i]) || o[i] != g->o[i] || lse[i] != g->lse[i]) {
                // attend_*_kernel(AttendParams p): same struct as kf_attend builds, new q / o / lse
                AttendParams ap;
                ap.d = ctx->dev;
                ap.layer = g->layers[i];
                ap.q = g->host_io ? ctx->dev.stage_q : (const __half *)q[i];
                ap.o_part = ctx->dev.range_o;
                ap.lse_part = ctx->dev.range_lse;
                ap.o = o[i];
                ap.lse = lse[i];
                ap.fused = 1;
                ap.commit = i == g->n - 1;
                ap.part_mask = ~0ull;
                void *args[1] = {&ap};
                cudaKernelNodeParams p = g->attend_params[i];
                p.kernelParams = args;
                p.extra = nullptr;
                const cudaError_t e = cudaGraphExecKernelNodeSetParams(g->exec, g->attend_nodes[i], &p);
                if (e != cudaSuccess) return cuda_fail(ctx, e);
                g->o[i] = o[i];
                g->lse[i] = lse[i];
            }
            g->q[i] = q[i];
        }
    }
    const cudaError_t e = cudaGraphLaunch(g->exec, (cudaStream_t)stream);
    if (e != cudaSuccess) return cuda_fail(ctx, e);
    ctx->launches += g->kernels_per_launch;
    ctx->plan_dirty = true;  // the graph ends with the step commit
    return KF_OK;
}

int kf_step_graph_destroy(kf_graph *g) {
    if (!g) return KF_EINVAL;
    if (g->exec) cudaGraphExecDestroy(g->exec);
    if (g->graph) cudaGraphDestroy(g->graph);
    delete g;
    return KF_OK;
}

}  // extern "C"
