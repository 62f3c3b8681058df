// kf_static.cu -- kf_attend_static (include/kflume.h): kf_attend for callers that have no device memory to spare for the
// range partials and no way to get any.  The partials live in ONE array that is part of the library image.
//
// Why it exists.  kf_attend needs room for every range's partial (o_j, lse_j) between the attention phase and the merge
// (PAPER.md:147, :254).  Normally that room is the caller's: an o_part / lse_part pair, or a slice of the workspace handed
// to kf_create.  Some callers cannot provide either at the moment they need it:
//   - an attention node that has already given all of its HBM to KV pools (the paper's A nodes are "weightless": their
//     memory IS the KV capacity) and joins a running decode loop -- cudaMalloc at that point may fail, and
//     when it succeeds it synchronises the whole device, stalling the step graphs of every other stream;
//   - code that runs inside a region where the CUDA allocator must not be entered at all: between the begin and end of a
//     stream capture on another thread's behalf, inside a framework whose caching allocator owns all device memory, or
//     in a latency-critical loop that has promised never to take the driver's allocation lock.
// For them the scratch is a fixed-size, file-scope __device__ array: it is reserved when the library is loaded onto a
// GPU and released when the process exits, so the call itself never allocates or frees anything.
//
// What that costs.  KF_STATIC_SCRATCH_BYTES of device memory on EVERY GPU the process uses with this library, until
// exit, whether or not the entry point is ever called.  There is one array per GPU, not per ctx: all callers share it.
#include <mutex>

#include <stdio.h>

#include "kf_ctx.h"

namespace {

// The scratch itself.  In HOST code the name below is only a handle for the runtime (a host-side shadow variable):
// taking its address on the host and giving that to a kernel would make the kernel read host memory or fault.  Host
// code gets the real device address from cudaGetSymbolAddress, once per device (scratch_address below).
static __device__ __align__(256) unsigned char g_static_scratch[KF_STATIC_SCRATCH_BYTES];

constexpr int kMaxDevices = 64;
std::mutex g_mutex;
unsigned char *g_device_address[kMaxDevices];  // [dev] device address of g_static_scratch on that GPU, nullptr = not asked yet

// Device address of the array on the CURRENT device.  The first call per device asks the runtime (this is the set-up
// step: it can make the runtime load this module onto the device, so it belongs before any stream capture); later calls
// read the cached pointer.  Returns KF_OK or an error with the text left in the ctx.
int scratch_address(kf_ctx *ctx, unsigned char **out) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return kf::cuda_fail(ctx, e);
    if (dev < 0 || dev >= kMaxDevices) {
        snprintf(ctx->cuda_err, sizeof(ctx->cuda_err), "kf_attend_static: device ordinal %d is beyond the %d this entry point tracks",
                 dev, kMaxDevices);
        return KF_EINVAL;
    }
    std::lock_guard<std::mutex> lock(g_mutex);
    if (!g_device_address[dev]) {
        void *p = nullptr;
        e = cudaGetSymbolAddress(&p, g_static_scratch);
        if (e != cudaSuccess) return kf::cuda_fail(ctx, e);
        if (!p || ((uintptr_t)p & 255)) {
            snprintf(ctx->cuda_err, sizeof(ctx->cuda_err), "kf_attend_static: cudaGetSymbolAddress returned an unusable address");
            return KF_ECUDA;
        }
        g_device_address[dev] = (unsigned char *)p;
    }
    *out = g_device_address[dev];
    return KF_OK;
}

inline size_t align256(size_t x) { return (x + 255) & ~(size_t)255; }

}  // namespace

extern "C" int kf_attend_static(kf_ctx *ctx, int32_t layer, const void *q, float *o, float *lse, kf_stream stream) {
    if (!ctx) return KF_EINVAL;
    // layout inside the array: o_part [B][Jmax][H_q][128] fp32, then (256-byte aligned) lse_part [B][Jmax][H_q] fp32
    const size_t rows = (size_t)ctx->cfg.max_requests * ctx->cfg.max_ranges_per_request * ctx->cfg.n_q_heads;
    const size_t o_bytes = align256(rows * kf::kHeadDim * sizeof(float));
    const size_t need = o_bytes + rows * sizeof(float);
    if (need > (size_t)KF_STATIC_SCRATCH_BYTES) {
        snprintf(ctx->cuda_err, sizeof(ctx->cuda_err),
                 "kf_attend_static: max_requests * max_ranges_per_request * n_q_heads = %zu partial rows need %zu bytes, the "
                 "static scratch holds %zu (KF_STATIC_SCRATCH_BYTES); use kf_attend with caller memory",
                 rows, need, (size_t)KF_STATIC_SCRATCH_BYTES);
        return KF_EINVAL;
    }
    unsigned char *base = nullptr;
    const int rc = scratch_address(ctx, &base);
    if (rc != KF_OK) return rc;
    // From here on this IS kf_attend: same plan, same kernel, same fixed merge order -- only the partials' address differs.
    // Nothing in the array has to be cleared: the merge reads only range partials that an earlier phase of the SAME launch
    // wrote (completion counters in the ctx workspace order the two), so whatever an earlier call left behind is never read.
    return kf_attend_impl(ctx, layer, q, o, lse, (float *)base, (float *)(base + o_bytes), 0, nullptr, nullptr, stream);
}
