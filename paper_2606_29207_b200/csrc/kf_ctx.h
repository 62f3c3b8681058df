// kf_ctx.h -- the host-side context of libkflume (private to the library).
#pragma once
#include "kf_common.cuh"

struct kf_ctx {
    kf_config cfg;
    kf::Dev dev;
    int sm_count;
    int n_ctas;
    int impl;
    bool plan_dirty;  // lengths moved (step commit) or routes were edited since the plan kernel last ran
    int64_t launches;
    char cuda_err[256];
    static constexpr int kPinnedCache = 1024;
    const void *pinned[kPinnedCache];  // host pointers already verified as device-readable (kf_layer_step_host,
                                       // kf_step_graph_launch): direct-mapped by address
};

// library-internal entry points of the static step graph (kf_graph.cu); not exported through include/kflume.h:
// the same calls as their public namesakes plus a fusion that only makes sense inside one captured step
#define KF_INTERNAL __attribute__((visibility("hidden")))
extern "C" {
KF_INTERNAL int kf_attend_impl(kf_ctx *ctx, int32_t layer, const void *q, float *o, float *lse, float *o_part, float *lse_part,
                   int commit, const void *k_new, const void *v_new,   // commit != 0: + kf_step_commit in the same launch
                   kf_stream stream);                                  // k_new / v_new != NULL: + kf_kv_append, ditto
KF_INTERNAL int kf_layer_step_host_impl(kf_ctx *ctx, int32_t layer, const void *q_host, const void *k_new_host,
                                        const void *v_new_host, float *o_host, float *lse_host, int commit,
                                        kf_stream stream);
}

namespace kf {
int cuda_fail(kf_ctx *ctx, cudaError_t e);  // records the error text in the ctx, returns KF_ECUDA
bool device_can_read(const void *host_ptr);  // pinned host memory the GPU can dereference as it is
bool host_ptr_ok(kf_ctx *ctx, const void *p);  // the same through the ctx's cache of verified pointers
}
