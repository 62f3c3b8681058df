// kf_graph.cu -- one decode step as a static CUDA graph (kf_step_graph_*, include/kflume.h).
//
// The paper keeps the W-node computation in ONE static CUDA Graph and moves every elasticity decision into a
// routing table that the graph never sees (PAPER.md:127 requirement R1, :165-179).  Here the same property
// holds on the device: all hot kernels launch fixed grids and read lengths, routes and the work plan from device
// memory, so a graph captured once stays valid across route updates, range fills and open / close of requests.
// A replay removes the per-launch submission latency between the small kernels of a step (route update, append,
// commit) and the attend kernel.  Input / output pointers may be re-bound at every launch
// (cudaGraphExecKernelNodeSetParams: host-side only, the graph is not re-instantiated).
#include <cuda.h>
#include <stdio.h>
#include <time.h>

#include <algorithm>
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
    bool fused_append;                      // device graph with the TMA kernel: the append rides in the attend launch
    int kernels_per_launch;
    std::vector<int32_t> layers;
    std::vector<cudaGraphNode_t> append_nodes, attend_nodes;   // [n] (device-pointer graphs only)
    std::vector<cudaKernelNodeParams> append_params, attend_params;
    std::vector<const void *> q, k, v;      // currently bound pointers
    std::vector<float *> o, lse;
    // graph progress signalling (kf_step_graph_flags)
    uint32_t *ready;                        // [n] pinned host words written after each layer-step, or nullptr
    bool gates;                             // a wait on gate word i (device memory) precedes layer-step i
    std::vector<cudaGraphNode_t> wait_nodes, write_nodes;   // batch mem-op nodes, [n] each (or empty)
    uint64_t n_launches;                    // launches so far: launch L (1-based) uses seq(L, i) = (L-1)*n + i + 1
    cudaStream_t last_stream;               // stream of the last launch: a gate must not be released on it
};

namespace {

// Driver entry points of the stream memory operations ("WriteValue32-style" signal writes and "ReadValue32-style"
// waits of PAPER.md:167, :175) and of their graph nodes, resolved through the runtime (the library does not link
// libcuda directly).
struct MemOps {
    CUresult (*write32)(CUstream, CUdeviceptr, cuuint32_t, unsigned int);
    CUresult (*wait32)(CUstream, CUdeviceptr, cuuint32_t, unsigned int);
    CUresult (*node_get)(CUgraphNode, CUDA_BATCH_MEM_OP_NODE_PARAMS *);
    CUresult (*exec_set)(CUgraphExec, CUgraphNode, const CUDA_BATCH_MEM_OP_NODE_PARAMS *);
    CUresult (*node_type)(CUgraphNode, CUgraphNodeType *);
    bool ok;
};
const MemOps &memops() {
    static MemOps m = [] {
        MemOps x = {};
        auto get = [](const char *name) -> void * {
            void *fn = nullptr;
            cudaDriverEntryPointQueryResult q;
            if (cudaGetDriverEntryPoint(name, &fn, cudaEnableDefault, &q) != cudaSuccess || q != cudaDriverEntryPointSuccess) {
                cudaGetLastError();
                return nullptr;
            }
            return fn;
        };
        x.write32 = (decltype(x.write32))get("cuStreamWriteValue32");
        x.wait32 = (decltype(x.wait32))get("cuStreamWaitValue32");
        x.node_get = (decltype(x.node_get))get("cuGraphBatchMemOpNodeGetParams");
        x.exec_set = (decltype(x.exec_set))get("cuGraphExecBatchMemOpNodeSetParams");
        x.node_type = (decltype(x.node_type))get("cuGraphNodeGetType");
        x.ok = x.write32 && x.wait32 && x.node_get && x.exec_set && x.node_type;
        return x;
    }();
    return m;
}

int drv_fail(kf_ctx *ctx, const char *what, CUresult r) {
    snprintf(ctx->cuda_err, sizeof(ctx->cuda_err), "%s failed: CUresult %d", what, (int)r);
    return KF_ECUDA;
}

// set the value of a one-operation batch mem-op node (wait or write) in the executable graph
int set_memop_value(kf_graph *g, cudaGraphNode_t node, uint32_t value) {
    CUstreamBatchMemOpParams op;
    CUDA_BATCH_MEM_OP_NODE_PARAMS np;
    CUresult r = memops().node_get((CUgraphNode)node, &np);
    if (r != CUDA_SUCCESS || np.count != 1) return drv_fail(g->ctx, "cuGraphBatchMemOpNodeGetParams", r);
    op = np.paramArray[0];
    if (op.operation == CU_STREAM_MEM_OP_WAIT_VALUE_32)
        op.waitValue.value = value;
    else
        op.writeValue.value = value;
    np.paramArray = &op;
    r = memops().exec_set((CUgraphExec)g->exec, (CUgraphNode)node, &np);
    if (r != CUDA_SUCCESS) return drv_fail(g->ctx, "cuGraphExecBatchMemOpNodeSetParams", r);
    return KF_OK;
}

// kernel nodes (and, separately, batch mem-op nodes) of a linear (single-stream capture) graph, in execution order
int kernel_chain(cudaGraph_t g, std::vector<cudaGraphNode_t> &out, std::vector<cudaGraphNode_t> *memop = nullptr) {
    size_t n = 0;
    if (cudaGraphGetNodes(g, nullptr, &n) != cudaSuccess) return -1;
    std::vector<cudaGraphNode_t> roots(n);
    size_t nr = n;
    if (cudaGraphGetRootNodes(g, roots.data(), &nr) != cudaSuccess || nr != 1) return -3;
    cudaGraphNode_t cur = roots[0];
    for (size_t i = 0; i < n; ++i) {
        // the runtime's node-type enum has no name for batch mem-op nodes: ask the driver when it is there
        if (memops().node_type) {
            CUgraphNodeType t;
            if (memops().node_type((CUgraphNode)cur, &t) != CUDA_SUCCESS) return -2;
            if (t == CU_GRAPH_NODE_TYPE_KERNEL) out.push_back(cur);
            if (t == CU_GRAPH_NODE_TYPE_BATCH_MEM_OP && memop) memop->push_back(cur);
        } else {
            cudaGraphNodeType t;
            if (cudaGraphNodeGetType(cur, &t) != cudaSuccess) return -2;
            if (t == cudaGraphNodeTypeKernel) out.push_back(cur);
        }
        // the _v2 query also reports programmatic (PDL) edges, which the plain one refuses
        size_t nd = 0;
        if (cudaGraphNodeGetDependentNodes_v2(cur, nullptr, nullptr, &nd) != cudaSuccess) return -1;
        if (nd == 0) break;
        if (nd != 1) return -4;
        cudaGraphNode_t next;
        cudaGraphEdgeData edge;
        if (cudaGraphNodeGetDependentNodes_v2(cur, &next, &edge, &nd) != cudaSuccess) return -1;
        cur = next;
    }
    return 0;
}

}  // namespace

namespace {

// Capture the step on `s`, instantiate, and locate the nodes that are re-bound / re-valued per launch.  Replaces
// whatever graph `g` held.  With g->gates a ReadValue32-style wait on gate word i precedes layer-step i; with
// g->ready a WriteValue32-style write of the sequence number to ready[i] follows it.
int build_graph(kf_graph *g, cudaStream_t s) {
    kf_ctx *ctx = g->ctx;
    const int n = g->n;
    kf_stream stream = (kf_stream)s;
    if ((g->gates || g->ready) && !memops().ok) {
        snprintf(ctx->cuda_err, sizeof(ctx->cuda_err), "stream memory operations unavailable in this driver");
        return KF_ECUDA;
    }
    if (g->exec) cudaGraphExecDestroy(g->exec);
    if (g->graph) cudaGraphDestroy(g->graph);
    g->exec = nullptr;
    g->graph = nullptr;
    g->append_nodes.clear();
    g->attend_nodes.clear();
    g->append_params.clear();
    g->attend_params.clear();
    g->wait_nodes.clear();
    g->write_nodes.clear();

    const int64_t launches0 = ctx->launches;
    cudaError_t e = cudaStreamBeginCapture(s, cudaStreamCaptureModeThreadLocal);
    if (e != cudaSuccess) return cuda_fail(ctx, e);
    // One fusion that only exists inside the captured step: the step commit is done by the last worker of the last
    // attend launch (2n + 1 kernels per step instead of 2n + 2); the observable state after a launch is that of
    // the public call sequence.  (Folding the first append into the single-CTA plan kernel was measured and
    // dropped: one CTA needs 13 us to copy B = 64 rows that B CTAs copy in 4.)
    int rc = kf_token_boundary(ctx, stream);
    CUresult dr = CUDA_SUCCESS;
    for (int i = 0; i < n && rc == KF_OK; ++i) {
        const int commit = i == n - 1;
        if (g->gates) {  // the inputs of layer-step i are "received" when gate i reaches this launch's sequence number
            dr = memops().wait32((CUstream)s, (CUdeviceptr)(uintptr_t)(ctx->dev.gates + i), 0, CU_STREAM_WAIT_VALUE_GEQ);
            if (dr != CUDA_SUCCESS) rc = drv_fail(ctx, "cuStreamWaitValue32 (capture)", dr);
        }
        if (rc != KF_OK) break;
        if (g->host_io) {
            rc = kf_layer_step_host_impl(ctx, g->layers[i], g->q[i], g->k[i], g->v[i], g->o[i], g->lse[i], commit, stream);
        } else {
            // with the TMA kernel the append rides in the attend launch (n + 1 kernels per step instead of 2n + 1)
            if (!g->fused_append) rc = kf_kv_append(ctx, g->layers[i], g->k[i], g->v[i], stream);
            if (rc == KF_OK)
                rc = kf_attend_impl(ctx, g->layers[i], g->q[i], g->o[i], g->lse[i], nullptr, nullptr, commit,
                                    g->fused_append ? g->k[i] : nullptr, g->fused_append ? g->v[i] : nullptr, stream);
        }
        if (rc == KF_OK && g->ready) {  // o[i] / lse[i] are complete: signal the host (default flags: the write is
                                        // ordered after all prior writes of the stream, system-wide)
            dr = memops().write32((CUstream)s, (CUdeviceptr)(uintptr_t)(g->ready + i), 0, CU_STREAM_WRITE_VALUE_DEFAULT);
            if (dr != CUDA_SUCCESS) rc = drv_fail(ctx, "cuStreamWriteValue32 (capture)", dr);
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
    std::vector<cudaGraphNode_t> chain, mem;
    const size_t n_mem = (size_t)n * ((g->gates ? 1 : 0) + (g->ready ? 1 : 0));
    int kc = 0;
    if (rc == KF_OK && (kc = kernel_chain(g->graph, chain, &mem)) != 0) {
        snprintf(ctx->cuda_err, sizeof(ctx->cuda_err), "unexpected step-graph topology (%d, %zu nodes)", kc, n_nodes);
        rc = KF_ECUDA;
    }
    // a host-io graph whose layer-steps all took the zero-copy path consists of kernels (and mem-ops) only: same
    // shape as a device graph (the staging kernel in place of the append kernel), so it can be re-bound the same way
    g->zero_copy = g->host_io && rc == KF_OK && n_nodes == (size_t)(2 * n + 1) + n_mem && (int)chain.size() == 2 * n + 1;
    const int per = g->fused_append ? 1 : 2;  // kernels per layer-step
    if (rc == KF_OK && mem.size() != n_mem) {
        snprintf(ctx->cuda_err, sizeof(ctx->cuda_err), "step graph: %zu mem-op nodes captured, %zu expected", mem.size(), n_mem);
        rc = KF_ECUDA;
    }
    if (rc == KF_OK && (!g->host_io || g->zero_copy)) {
        // kernel order of the capture: plan, n x ([append or stage,] attend)
        if ((int)chain.size() != per * n + 1) {
            snprintf(ctx->cuda_err, sizeof(ctx->cuda_err), "unexpected step-graph topology");
            rc = KF_ECUDA;
        } else {
            for (int i = 0; i < n && rc == KF_OK; ++i) {
                g->append_nodes.push_back(chain[1 + per * i]);  // (the attend node itself when the append is fused)
                g->attend_nodes.push_back(chain[per + per * i]);
                cudaKernelNodeParams pa, pt;
                e = cudaGraphKernelNodeGetParams(chain[1 + per * i], &pa);
                if (e == cudaSuccess) e = cudaGraphKernelNodeGetParams(chain[per + per * i], &pt);
                if (e != cudaSuccess) rc = cuda_fail(ctx, e);
                g->append_params.push_back(pa);
                g->attend_params.push_back(pt);
            }
        }
    }
    if (rc == KF_OK) {  // mem-op order of the capture: per layer-step [wait], ..., [write]
        size_t m = 0;
        for (int i = 0; i < n; ++i) {
            if (g->gates) g->wait_nodes.push_back(mem[m++]);
            if (g->ready) g->write_nodes.push_back(mem[m++]);
        }
    }
    if (rc != KF_OK) {
        cudaGetLastError();
        if (g->exec) cudaGraphExecDestroy(g->exec);
        if (g->graph) cudaGraphDestroy(g->graph);
        g->exec = nullptr;
        g->graph = nullptr;
    }
    return rc;
}

}  // namespace

extern "C" {

int kf_step_graph_create(kf_ctx *ctx, int32_t n_layer_steps, const int32_t *layers, int32_t host_io,
                         const void *const *q, const void *const *k_new, const void *const *v_new, float *const *o,
                         float *const *lse, kf_stream stream, kf_graph **out) {
    if (!out) return KF_EINVAL;
    *out = nullptr;
    if (!ctx || n_layer_steps < 1 || n_layer_steps > kMaxGraphLayerSteps || !layers || !q || !k_new || !v_new || !o || !lse || !stream)
        return KF_EINVAL;
    for (int i = 0; i < n_layer_steps; ++i)
        if (layers[i] < 0 || layers[i] >= ctx->cfg.n_layers || !q[i] || !k_new[i] || !v_new[i] || !o[i] || !lse[i])
            return KF_EINVAL;
    kf_graph *g = new (std::nothrow) kf_graph();
    if (!g) return KF_EINVAL;
    g->ctx = ctx;
    g->graph = nullptr;
    g->exec = nullptr;
    g->n = n_layer_steps;
    g->host_io = host_io ? 1 : 0;
    g->zero_copy = false;
    g->fused_append = !g->host_io && ctx->impl == KF_IMPL_TMA;
    g->ready = nullptr;
    g->gates = false;
    g->n_launches = 0;
    g->last_stream = nullptr;
    g->layers.assign(layers, layers + n_layer_steps);
    g->q.assign(q, q + n_layer_steps);
    g->k.assign(k_new, k_new + n_layer_steps);
    g->v.assign(v_new, v_new + n_layer_steps);
    g->o.assign(o, o + n_layer_steps);
    g->lse.assign(lse, lse + n_layer_steps);
    const int rc = build_graph(g, (cudaStream_t)stream);
    if (rc != KF_OK) {
        delete g;
        return rc;
    }
    *out = g;
    return KF_OK;
}

int kf_step_graph_flags(kf_graph *g, uint32_t *ready_host, int32_t gates, kf_stream stream) {
    if (!g || !stream) return KF_EINVAL;
    if (g->n_launches != 0) return KF_ESTATE;  // the sequence numbers of a graph start at its first launch
    if (ready_host && (((uintptr_t)ready_host & 3) || !device_can_read(ready_host))) return KF_EINVAL;
    g->ready = ready_host;
    g->gates = gates != 0;
    if (g->gates) {  // gate words start below every sequence number
        // ... and they do so BEFORE this call returns: a gate "may be released before the launch that waits on it", on
        // another stream, so a memset still queued behind earlier work of `stream` could land after such a release, erase
        // it and leave the graph waiting for ever.  The call is off the hot path; it waits for the memset.
        cudaError_t e = cudaMemsetAsync(g->ctx->dev.gates, 0, (size_t)g->n * 4, (cudaStream_t)stream);
        if (e == cudaSuccess) e = cudaStreamSynchronize((cudaStream_t)stream);
        if (e != cudaSuccess) return cuda_fail(g->ctx, e);
    }
    if (ready_host)
        for (int i = 0; i < g->n; ++i) ready_host[i] = 0;
    return build_graph(g, (cudaStream_t)stream);
}

uint32_t kf_step_graph_seq(const kf_graph *g, int32_t layer_step) {
    if (!g || layer_step < 0 || layer_step >= g->n) return 0;
    return (uint32_t)(g->n_launches * (uint64_t)g->n + (uint64_t)layer_step + 1);
}

int kf_step_graph_release(kf_graph *g, int32_t layer_step, uint32_t seq, kf_stream signal_stream) {
    if (!g || layer_step < 0 || layer_step >= g->n) return KF_EINVAL;
    if (!g->gates) return KF_ESTATE;
    // "the execution stream is already blocked on that wait, so enqueuing the flag write on the same
    // stream would place it behind the wait and deadlock" -- refused instead of deadlocking
    if ((cudaStream_t)signal_stream == g->last_stream) return KF_ESTATE;
    const CUresult r = memops().write32((CUstream)signal_stream, (CUdeviceptr)(uintptr_t)(g->ctx->dev.gates + layer_step),
                                        seq, CU_STREAM_WRITE_VALUE_DEFAULT);
    if (r != CUDA_SUCCESS) return drv_fail(g->ctx, "cuStreamWriteValue32", r);
    return KF_OK;
}

int kf_step_graph_launch(kf_graph *g, const void *const *q, const void *const *k_new, const void *const *v_new,
                         float *const *o, float *const *lse, kf_stream stream) {
    if (!g || !stream || !g->exec) return KF_EINVAL;
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
                if ((in_changed && !(host_ptr_ok(ctx, q[i]) && host_ptr_ok(ctx, k_new[i]) && host_ptr_ok(ctx, v_new[i]))) ||
                    (out_changed && !(host_ptr_ok(ctx, o[i]) && host_ptr_ok(ctx, lse[i]))))
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
            } else if (!g->fused_append && (k_new[i] != g->k[i] || v_new[i] != g->v[i])) {
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
            if ((!g->host_io && q[i] != g->q[i]) || o[i] != g->o[i] || lse[i] != g->lse[i] ||
                (g->fused_append && (k_new[i] != g->k[i] || v_new[i] != g->v[i]))) {
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
                ap.k_new = g->fused_append ? (const __half *)k_new[i] : nullptr;
                ap.v_new = g->fused_append ? (const __half *)v_new[i] : nullptr;
                void *args[1] = {&ap};
                cudaKernelNodeParams p = g->attend_params[i];
                p.kernelParams = args;
                p.extra = nullptr;
                const cudaError_t e = cudaGraphExecKernelNodeSetParams(g->exec, g->attend_nodes[i], &p);
                if (e != cudaSuccess) return cuda_fail(ctx, e);
                g->o[i] = o[i];
                g->lse[i] = lse[i];
                if (g->fused_append) {
                    g->k[i] = k_new[i];
                    g->v[i] = v_new[i];
                }
            }
            g->q[i] = q[i];
        }
    }
    // this launch's sequence numbers: seq(L, i) = (L - 1) * n + i + 1 (host-side node update, like the pointers)
    for (int i = 0; i < g->n; ++i) {
        const uint32_t seq = kf_step_graph_seq(g, i);
        int rc = KF_OK;
        if (g->gates) rc = set_memop_value(g, g->wait_nodes[i], seq);
        if (rc == KF_OK && g->ready) rc = set_memop_value(g, g->write_nodes[i], seq);
        if (rc != KF_OK) return rc;
    }
    const cudaError_t e = cudaGraphLaunch(g->exec, (cudaStream_t)stream);
    if (e != cudaSuccess) return cuda_fail(ctx, e);
    g->n_launches += 1;
    g->last_stream = (cudaStream_t)stream;
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


// Diagnostics: round trip of one gate release and one readiness signal through a two-node graph
// [wait gate >= seq] -> [write seq to a pinned host word]: the host releases the gate with a WriteValue32 on the
// signalling stream and spins on the host word.  t = host enqueue + GPU sees the gate + GPU write becomes visible to
// the host: an upper bound on the "GPU store -> host sees it" latency of a readiness flag.
int kf_signal_roundtrip(kf_ctx *ctx, int32_t iters, kf_stream exec_stream, kf_stream signal_stream, double *median_us,
                        double *min_us) {
    if (!ctx || iters < 1 || iters > 100000 || !exec_stream || !signal_stream || exec_stream == signal_stream || !median_us ||
        !min_us)
        return KF_EINVAL;
    if (!memops().ok) return KF_ECUDA;
    cudaStream_t es = (cudaStream_t)exec_stream, ss = (cudaStream_t)signal_stream;
    uint32_t *gate = ctx->dev.gates + kMaxGraphLayerSteps;  // a word of its own, behind the gates a step graph can use
    volatile uint32_t *ready = nullptr;
    cudaError_t e = cudaHostAlloc((void **)&ready, 64, cudaHostAllocMapped);
    if (e != cudaSuccess) return cuda_fail(ctx, e);
    *ready = 0;
    cudaGraph_t graph = nullptr;
    cudaGraphExec_t exec = nullptr;
    int rc = KF_OK;
    e = cudaMemsetAsync(gate, 0, 4, es);
    if (e == cudaSuccess) e = cudaStreamSynchronize(es);
    if (e == cudaSuccess) e = cudaStreamBeginCapture(es, cudaStreamCaptureModeThreadLocal);
    if (e != cudaSuccess) rc = cuda_fail(ctx, e);
    if (rc == KF_OK) {
        CUresult r = memops().wait32((CUstream)es, (CUdeviceptr)(uintptr_t)gate, 0, CU_STREAM_WAIT_VALUE_GEQ);
        if (r == CUDA_SUCCESS) r = memops().write32((CUstream)es, (CUdeviceptr)(uintptr_t)ready, 0, CU_STREAM_WRITE_VALUE_DEFAULT);
        e = cudaStreamEndCapture(es, &graph);
        if (r != CUDA_SUCCESS) rc = drv_fail(ctx, "stream mem-op capture", r);
        else if (e != cudaSuccess) rc = cuda_fail(ctx, e);
    }
    if (rc == KF_OK && (e = cudaGraphInstantiate(&exec, graph, 0)) != cudaSuccess) rc = cuda_fail(ctx, e);
    std::vector<cudaGraphNode_t> kern, mem;
    if (rc == KF_OK && (kernel_chain(graph, kern, &mem) != 0 || mem.size() != 2)) {
        snprintf(ctx->cuda_err, sizeof(ctx->cuda_err), "roundtrip graph: unexpected topology");
        rc = KF_ECUDA;
    }
    std::vector<double> t;
    kf_graph tmp;  // set_memop_value only needs ctx and exec
    tmp.ctx = ctx;
    tmp.exec = exec;
    auto now_us = [] {
        timespec ts;
        clock_gettime(CLOCK_MONOTONIC, &ts);
        return ts.tv_sec * 1e6 + ts.tv_nsec * 1e-3;
    };
    for (int it = 0; it < iters + 10 && rc == KF_OK; ++it) {
        const uint32_t seq = (uint32_t)it + 1;
        rc = set_memop_value(&tmp, mem[0], seq);
        if (rc == KF_OK) rc = set_memop_value(&tmp, mem[1], seq);
        if (rc != KF_OK) break;
        if ((e = cudaGraphLaunch(exec, es)) != cudaSuccess) {
            rc = cuda_fail(ctx, e);
            break;
        }
        const double t_arm = now_us();
        while (now_us() - t_arm < 30.0) {}  // let the graph reach its wait
        const double t0 = now_us();
        const CUresult r = memops().write32((CUstream)ss, (CUdeviceptr)(uintptr_t)gate, seq, CU_STREAM_WRITE_VALUE_DEFAULT);
        if (r != CUDA_SUCCESS) {
            rc = drv_fail(ctx, "cuStreamWriteValue32", r);
            // unblock the graph through a plain copy so that nothing is left waiting
            cudaMemcpyAsync(gate, &seq, 4, cudaMemcpyHostToDevice, ss);
            break;
        }
        while (*ready != seq && now_us() - t0 < 2e6) {}
        const double t1 = now_us();
        if (*ready != seq) {
            snprintf(ctx->cuda_err, sizeof(ctx->cuda_err), "roundtrip: readiness flag not seen within 2 s");
            rc = KF_ECUDA;
            break;
        }
        if (it >= 10) t.push_back(t1 - t0);
    }
    if (rc != KF_OK) {
        // something went wrong with a graph possibly still waiting at the gate: open it for good with a plain copy (a
        // value every wait of this call accepts) BEFORE synchronising the execution stream, or that would block for ever
        static const uint32_t open_value = 0x7fffffffu;
        cudaMemcpyAsync(gate, &open_value, 4, cudaMemcpyHostToDevice, ss);
    }
    cudaStreamSynchronize(ss);
    cudaStreamSynchronize(es);
    if (exec) cudaGraphExecDestroy(exec);
    if (graph) cudaGraphDestroy(graph);
    cudaFreeHost((void *)ready);
    if (rc == KF_OK) {
        std::sort(t.begin(), t.end());
        *median_us = t[t.size() / 2];
        *min_us = t[0];
    }
    return rc;
}

}  // extern "C"
