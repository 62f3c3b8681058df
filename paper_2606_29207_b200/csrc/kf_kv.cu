// kf_kv.cu -- KV placement into the token-range pools: bulk context load (post-prefill initialisation,
// PAPER.md:234) and the per-step append of (K_new, V_new) on the tail range.
#include "kf_common.cuh"

namespace kf {

// One thread moves one 16-byte chunk (8 halfs) of one token row.  grid = (chunks, H_kv, 2 {K,V}).
__global__ void __launch_bounds__(256) load_context_kernel(Dev d, int layer, int req, int tok_begin, int n_tokens,
                                                           const __half *__restrict__ k,
                                                           const __half *__restrict__ v) {
    const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int t = (int)(idx >> 4), c = (int)(idx & 15);
    if (t >= n_tokens) return;
    const int g = blockIdx.y, is_v = blockIdx.z;
    const int pos = tok_begin + t;
    // range that holds position pos: begin_j <= pos < begin_j+1 (j * R unless a tail was redirected, reading 28)
    const int nr = d.len[req] < 0 ? 0 : d.n_ranges[req];
    const int *bg = d.range_begin + (size_t)req * d.Jmax;
    int j = min(pos / d.R, nr - 1);
    while (j + 1 < nr && bg[j + 1] <= pos) ++j;
    const int off = nr > 0 ? pos - bg[j] : 0;
    if (nr == 0 || off >= d.R) {
        if (c == 0 && g == 0 && is_v == 0) set_error(d, KF_ESTATE);
        return;
    }
    const int p = d.route_part[(size_t)req * d.Jmax + j];
    const int slot = d.route_slot[(size_t)req * d.Jmax + j];
    const __half *src = (is_v ? v : k) + ((size_t)g * n_tokens + t) * kHeadDim + c * 8;
    unsigned char *dst = d.pool[p] + (is_v ? d.v_off : 0) + row_offset(d, layer, slot, g, off) + c * 16;
    *reinterpret_cast<int4 *>(dst) = __ldg(reinterpret_cast<const int4 *>(src));
}

// (a2) grid = B; each block copies the 2 * H_kv rows of one request to position len_r of its tail range.
__global__ void __launch_bounds__(256) kv_append_kernel(Dev d, int layer, const __half *__restrict__ k_new,
                                                        const __half *__restrict__ v_new) {
    const int r = blockIdx.x;
    const int len = d.len[r];
    if (len < 0 || !d.req_active[r]) return;
    const int j = d.n_ranges[r] - 1;  // the tail range
    const int off = j >= 0 ? len - d.range_begin[(size_t)r * d.Jmax + j] : d.R;
    if (off >= d.R) {  // no route for position len
        if (threadIdx.x == 0) set_error(d, KF_ESTATE);
        return;
    }
    const int p = d.route_part[(size_t)r * d.Jmax + j];
    const int slot = d.route_slot[(size_t)r * d.Jmax + j];
    const int chunks = 2 * d.Hkv * 16;
    for (int i = threadIdx.x; i < chunks; i += blockDim.x) {
        const int c = i & 15, g = (i >> 4) % d.Hkv, is_v = (i >> 4) / d.Hkv;
        const __half *src = (is_v ? v_new : k_new) + ((size_t)r * d.Hkv + g) * kHeadDim + c * 8;
        unsigned char *dst = d.pool[p] + (is_v ? d.v_off : 0) + row_offset(d, layer, slot, g, off) + c * 16;
        *reinterpret_cast<int4 *>(dst) = __ldg(reinterpret_cast<const int4 *>(src));
    }
}

// (a2) for the end-to-end path: k_new / v_new / q_src are PINNED HOST buffers read straight over the bus (zero-copy,
// uncached loads: the host rewrites them between launches); the q rows are staged into device memory for the attend
// kernel in the same launch.  Replaces three host->device copies by one kernel.
__global__ void __launch_bounds__(256) kv_append_stage_kernel(Dev d, int layer, const __half *k_new,
                                                              const __half *v_new, const __half *q_src,
                                                              __half *q_dst) {
    // grid (B, kStageSplit): bus reads are latency-bound (~2 us each), so a request's q rows are spread over several
    // CTAs; slice 0 also appends the K/V rows
    const int r = blockIdx.x;
    const int q_chunks = d.Hq * 16;  // 16-byte chunks of this request's q rows
    for (int i = blockIdx.y * blockDim.x + threadIdx.x; i < q_chunks; i += gridDim.y * blockDim.x) {
        const size_t off = (size_t)r * q_chunks + i;
        reinterpret_cast<int4 *>(q_dst)[off] = __ldcv(reinterpret_cast<const int4 *>(q_src) + off);
    }
    if (blockIdx.y != 0) return;
    const int len = d.len[r];
    if (len < 0 || !d.req_active[r]) return;
    const int j = d.n_ranges[r] - 1;  // the tail range
    const int off = j >= 0 ? len - d.range_begin[(size_t)r * d.Jmax + j] : d.R;
    if (off >= d.R) {  // no route for position len
        if (threadIdx.x == 0) set_error(d, KF_ESTATE);
        return;
    }
    const int p = d.route_part[(size_t)r * d.Jmax + j];
    const int slot = d.route_slot[(size_t)r * d.Jmax + j];
    const int chunks = 2 * d.Hkv * 16;
    for (int i = threadIdx.x; i < chunks; i += blockDim.x) {
        const int c = i & 15, g = (i >> 4) % d.Hkv, is_v = (i >> 4) / d.Hkv;
        const __half *src = (is_v ? v_new : k_new) + ((size_t)r * d.Hkv + g) * kHeadDim + c * 8;
        unsigned char *dst = d.pool[p] + (is_v ? d.v_off : 0) + row_offset(d, layer, slot, g, off) + c * 16;
        *reinterpret_cast<int4 *>(dst) = __ldcv(reinterpret_cast<const int4 *>(src));
    }
}

int launch_load_context(const Dev &d, int layer, int req, int tok_begin, int n_tokens, const __half *k,
                        const __half *v, cudaStream_t s) {
    if (n_tokens <= 0) return 0;
    const int64_t chunks = (int64_t)n_tokens * 16;
    dim3 grid((unsigned)((chunks + 255) / 256), d.Hkv, 2);
    load_context_kernel<<<grid, 256, 0, s>>>(d, layer, req, tok_begin, n_tokens, k, v);
    return 1;
}

int launch_kv_append(const Dev &d, int layer, const __half *k_new, const __half *v_new, cudaStream_t s) {
    kv_append_kernel<<<d.B, 256, 0, s>>>(d, layer, k_new, v_new);
    return 1;
}

int launch_kv_append_stage(const Dev &d, int layer, const __half *k_new, const __half *v_new, const __half *q_src,
                           __half *q_dst, cudaStream_t s) {
    const int split = d.Hq * 16 > 256 ? (d.Hq * 16 + 255) / 256 : 1;  // one q chunk per thread
    kv_append_stage_kernel<<<dim3(d.B, split), 256, 0, s>>>(d, layer, k_new, v_new, q_src, q_dst);
    return 1;
}

}  // namespace kf
