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
};

namespace kf {
int cuda_fail(kf_ctx *ctx, cudaError_t e);  // records the error text in the ctx, returns KF_ECUDA
}
