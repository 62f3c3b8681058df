// kf_probe.cu -- read-only HBM bandwidth probe (measurement aid, not on the hot path).
//
// MEASURED_PEAKS.json's HBM figure is a COPY (read + write) bandwidth; the attend kernel only reads.  This probe
// streams every KV pool of the ctx once, in ONE launch, with plain 128-bit loads (16 independent loads in flight per thread, persistent grid) and
// folds the data into one word so nothing is optimised away.  bench.py runs it on the KV pools right after the
// timed region and reports the attend kernel's bandwidth as a fraction of it (third denominator).
#include <time.h>

#include <algorithm>
#include <vector>

#include "kf_ctx.h"

namespace kf {

constexpr int kProbeThreads = 512;
constexpr int kProbeUnroll = 16;

__global__ void __launch_bounds__(kProbeThreads) probe_read_kernel(Dev d, size_t n_vec, uint32_t *sink) {
    const size_t stride = (size_t)gridDim.x * kProbeThreads;
    uint32_t acc = 0;
    for (int p = 0; p < d.P; ++p) {  // one launch covers every partition pool (K and V halves)
        const int4 *buf = reinterpret_cast<const int4 *>(d.pool[p]);
        size_t i = (size_t)blockIdx.x * kProbeThreads + threadIdx.x;
        for (; i + (kProbeUnroll - 1) * stride < n_vec; i += kProbeUnroll * stride) {
            int4 v[kProbeUnroll];
#pragma unroll
            for (int k = 0; k < kProbeUnroll; ++k) v[k] = __ldcs(buf + i + k * stride);  // streaming: evict first
#pragma unroll
            for (int k = 0; k < kProbeUnroll; ++k) acc ^= (uint32_t)(v[k].x ^ v[k].y ^ v[k].z ^ v[k].w);
        }
        for (; i < n_vec; i += stride) {
            const int4 v = __ldcs(buf + i);
            acc ^= (uint32_t)(v.x ^ v.y ^ v.z ^ v.w);
        }
    }
    if (acc == 0x9E3779B9u) atomicAdd(sink, 1u);  // practically never: keeps the loads alive
}

}  // namespace kf

extern "C" int kf_probe_read(kf_ctx *ctx, void *sink, size_t *bytes_read, kf_stream stream) {
    if (!ctx || !sink) return KF_EINVAL;
    const size_t pool_bytes = 2 * ctx->dev.v_off;
    const int ctas = ctx->sm_count * 4;
    kf::probe_read_kernel<<<ctas, kf::kProbeThreads, 0, (cudaStream_t)stream>>>(ctx->dev, pool_bytes / 16, (uint32_t *)sink);
    const cudaError_t e = cudaPeekAtLastError();
    if (e != cudaSuccess) {
        cudaGetLastError();
        return kf::cuda_fail(ctx, e);
    }
    if (bytes_read) *bytes_read = pool_bytes * (size_t)ctx->dev.P;
    return KF_OK;
}

// Diagnostics: what a route install (kf_set_active_partitions: PAPER.md:216-219, :308) costs when it is issued from C,
// without a language binding in the way.  Per iteration the published active set is replaced by a neighbouring one
// (one partition toggled, never empty) with the same tiny kernel the public call launches.
//   enqueue: host time of the launch call alone -- what the caller's routing loop spends before it can go on;
//   complete: launch call + cudaStreamSynchronize -- the new set is in device memory and every later kernel sees it.
// The set found at entry is re-published before the call returns.
extern "C" int kf_route_install_latency(kf_ctx *ctx, int32_t iters, kf_stream stream, double *enqueue_us_median,
                                        double *complete_us_median) {
    if (!ctx || iters < 1 || iters > 100000 || !enqueue_us_median || !complete_us_median) return KF_EINVAL;
    cudaStream_t s = (cudaStream_t)stream;
    const int P = ctx->dev.P;
    int32_t act[kf::kMaxPartitions];
    cudaError_t e = cudaMemcpyAsync(act, ctx->dev.active, (size_t)P * 4, cudaMemcpyDeviceToHost, s);
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);
    if (e != cudaSuccess) return kf::cuda_fail(ctx, e);
    unsigned long long orig = 0;
    for (int p = 0; p < P; ++p)
        if (act[p]) orig |= 1ull << p;
    if (!orig) return KF_ESTATE;
    auto now_us = [] {
        timespec ts;
        clock_gettime(CLOCK_MONOTONIC, &ts);
        return ts.tv_sec * 1e6 + ts.tv_nsec * 1e-3;
    };
    std::vector<double> tq, tc;
    const int warm = 10;
    for (int it = 0; it < iters + warm && e == cudaSuccess; ++it) {
        unsigned long long m = orig ^ (1ull << (it % P));
        if (!m) m = orig;
        const double t0 = now_us();
        const int n = kf::launch_set_active(ctx->dev, m, s);
        const double t1 = now_us();
        e = cudaStreamSynchronize(s);
        const double t2 = now_us();
        if (n > 0) ctx->launches += n;
        if (it >= warm) {
            tq.push_back(t1 - t0);
            tc.push_back(t2 - t0);
        }
    }
    const int n = kf::launch_set_active(ctx->dev, orig, s);  // leave the routing state as it was found
    if (n > 0) ctx->launches += n;
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);
    if (e == cudaSuccess) e = cudaPeekAtLastError();
    if (e != cudaSuccess) {
        cudaGetLastError();
        return kf::cuda_fail(ctx, e);
    }
    std::sort(tq.begin(), tq.end());
    std::sort(tc.begin(), tc.end());
    *enqueue_us_median = tq[tq.size() / 2];
    *complete_us_median = tc[tc.size() / 2];
    return KF_OK;
}
