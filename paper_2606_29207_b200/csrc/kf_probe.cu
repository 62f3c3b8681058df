// kf_probe.cu -- read-only HBM bandwidth probe (measurement aid, not on the hot path).
//
// MEASURED_PEAKS.json's HBM figure is a COPY (read + write) bandwidth; the attend kernel only reads.  This probe
// streams every KV pool of the ctx once, in ONE launch, with plain 128-bit loads (16 independent loads in flight per thread, persistent grid) and
// folds the data into one word so nothing is optimised away.  bench.py runs it on the KV pools right after the
// timed region and reports the attend kernel's bandwidth as a fraction of it (third denominator).
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
