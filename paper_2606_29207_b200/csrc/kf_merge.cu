// kf_merge.cu -- stand-alone merge kernels of the unfused path: pieces -> range partials (tail of
// kf_partial_attend) and range partials -> final output (kf_merge_partials).
#include "kf_merge.cuh"

namespace kf {

// warp per (unit, head of its group), grid-stride: units cut into several pieces are reduced into their range partial
__global__ void __launch_bounds__(256) merge_units_kernel(AttendParams p) {
    const Dev &d = p.d;
    const int lane = threadIdx.x & 31;
    const int warps = gridDim.x * (blockDim.x >> 5);
    const int n = d.plan->n_units * d.G;
    for (int t = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5); t < n; t += warps) {
        const int u = t / d.G, i = t - u * d.G;
        const Unit un = d.units[u];
        if (un.n_pieces <= 1) continue;
        if (!((p.part_mask >> un.part) & 1ull)) continue;
        merge_unit_head(p, un, u % d.Hkv, i, false, lane);
    }
}

// warp per (request, query head), grid-stride
__global__ void __launch_bounds__(256) merge_ranges_kernel(Dev d, const float *o_part, const float *lse_part,
                                                           float *o, float *lse) {
    const int lane = threadIdx.x & 31;
    const int warps = gridDim.x * (blockDim.x >> 5);
    const int n = d.B * d.Hq;
    for (int i = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5); i < n; i += warps) {
        const int req = i / d.Hq, h = i - req * d.Hq;
        const int J = d.scratch[req];  // J_r of the current plan; 0 for closed requests
        if (J <= 0) continue;
        merge_request_head(d, o_part, lse_part, o, lse, req, h, J, lane);
    }
}

int launch_merge_units(const AttendParams &p, int n_ctas, cudaStream_t s) {
    merge_units_kernel<<<n_ctas, 256, 0, s>>>(p);
    return 1;
}

int launch_merge_ranges(const Dev &d, const float *o_part, const float *lse_part, float *o, float *lse,
                        cudaStream_t s) {
    const int n = d.B * d.Hq;
    int ctas = (n + 7) / 8;
    if (ctas > 592) ctas = 592;
    merge_ranges_kernel<<<ctas, 256, 0, s>>>(d, o_part, lse_part, o, lse);
    return 1;
}

}  // namespace kf
