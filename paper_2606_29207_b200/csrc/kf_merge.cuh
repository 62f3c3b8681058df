// kf_merge.cuh -- log-sum-exp merge of attention partials, shared by the fused
// tail of the attend kernels (last-arriver pattern) and the stand-alone merge kernels.
//
//   lse = M + ln sum_j exp(lse_j - M),  M = max_j lse_j ;   o = sum_j exp(lse_j - lse) * o_j
//
// The reduction always runs over j in ascending index order, whichever work item arrives last, so results
// are run-to-run identical and the fused and unfused paths agree bit for bit.
#pragma once
#include "kf_common.cuh"

namespace kf {

__device__ __forceinline__ float warp_max(float v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}
__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// Where a worker writes the partial of one piece.  o rows are [G][128] fp32 (row stride 128), lse is [G].
// o2/lse2 (optional) receive a second copy: the final output when the piece is the whole request-head.
struct PieceDest {
    float *o, *lse, *o2, *lse2;
};

__device__ __forceinline__ size_t range_row(const Dev &d, int req, int range, int head) {
    return ((size_t)req * d.Jmax + range) * d.Hq + head;
}

// Pieces of a unit cut by c >= 1 span boundaries use piece-buffer slots 2*cb .. 2*cb + c, where cb = cuts before
// the unit = piece_begin - u: slots of different units never overlap and at most 2*workers + 1 slots are used.
__device__ __forceinline__ int piece_slot(const Unit &un, int u, int piece) {
    return 2 * (un.piece_begin - u) + (piece - un.piece_begin);
}

__device__ __forceinline__ PieceDest piece_dest(const AttendParams &p, const Unit &un, int u, int g, int piece) {
    const Dev &d = p.d;
    PieceDest pd;
    pd.o2 = nullptr;
    pd.lse2 = nullptr;
    if (un.n_pieces == 1) {
        const size_t row = range_row(d, un.req, un.range, g * d.G);
        pd.o = p.o_part + row * kHeadDim;
        pd.lse = p.lse_part + row;
        if (p.fused && d.scratch[un.req] == 1) {  // J_r == 1: this piece is the final result
            const size_t frow = (size_t)un.req * d.Hq + g * d.G;
            pd.o2 = p.o + frow * kHeadDim;
            pd.lse2 = p.lse + frow;
        }
    } else {
        const int ps = piece_slot(un, u, piece);
        pd.o = d.piece_o + (size_t)ps * d.G * kHeadDim;
        pd.lse = d.piece_lse + (size_t)ps * d.G;
    }
    return pd;
}

// One warp merges n partials of a head group: source partial j has o rows at src_o + j*o_stride + i*128 and
// lse at src_lse[j*lse_stride + i], i < G.  Lane l owns columns [4l, 4l+4).  Loads bypass L1 (__ldcg): the
// partials were written by other SMs in this same launch.  Four heads are reduced together and the inner loop
// is unrolled so that ~16 independent 16-byte loads are in flight per lane (the merge is L2-latency bound).
// The accumulation order is j ascending for every head, whoever calls this.
__device__ __forceinline__ void warp_merge(const float *src_o, size_t o_stride, const float *src_lse,
                                           size_t lse_stride, int n, int G, float *dst_o, float *dst_lse,
                                           float *dst2_o, float *dst2_lse, int lane) {
    for (int i0 = 0; i0 < G; i0 += 4) {
        const int nh = min(4, G - i0);
        float4 acc[4];
        float lse_h[4];
#pragma unroll
        for (int hh = 0; hh < 4; ++hh) {
            acc[hh] = make_float4(0.f, 0.f, 0.f, 0.f);
            lse_h[hh] = -INFINITY;
        }
        if (n == 1) {  // exact copy
#pragma unroll
            for (int hh = 0; hh < 4; ++hh) {
                if (hh < nh) {
                    lse_h[hh] = __ldcg(src_lse + i0 + hh);
                    acc[hh] = __ldcg(reinterpret_cast<const float4 *>(src_o + (size_t)(i0 + hh) * kHeadDim) + lane);
                }
            }
        } else {
#pragma unroll
            for (int hh = 0; hh < 4; ++hh) {
                if (hh < nh) {
                    const float *lp = src_lse + i0 + hh;
                    float M = -INFINITY;
                    for (int j = lane; j < n; j += 32) M = fmaxf(M, __ldcg(lp + (size_t)j * lse_stride));
                    M = warp_max(M);
                    if (M != -INFINITY) {
                        float sum = 0.f;
                        for (int j = lane; j < n; j += 32) sum += expf(__ldcg(lp + (size_t)j * lse_stride) - M);
                        sum = warp_sum(sum);
                        lse_h[hh] = M + logf(sum);
                    }
                }
            }
            for (int jb = 0; jb < n; jb += 32) {
                float wl[4];  // this lane's weights of partial jb + lane
#pragma unroll
                for (int hh = 0; hh < 4; ++hh) {
                    wl[hh] = 0.f;
                    if (hh < nh && jb + lane < n && lse_h[hh] != -INFINITY)
                        wl[hh] = expf(__ldcg(src_lse + (size_t)(jb + lane) * lse_stride + i0 + hh) - lse_h[hh]);
                }
                const int cnt = min(32, n - jb);
#pragma unroll 4
                for (int jj = 0; jj < cnt; ++jj) {
                    const float *row = src_o + (size_t)(jb + jj) * o_stride + (size_t)i0 * kHeadDim;
#pragma unroll
                    for (int hh = 0; hh < 4; ++hh) {
                        const float w = __shfl_sync(0xffffffffu, wl[hh], jj);
                        if (hh < nh) {
                            float4 v = __ldcg(reinterpret_cast<const float4 *>(row + (size_t)hh * kHeadDim) + lane);
                            if (w == 0.f) v = make_float4(0.f, 0.f, 0.f, 0.f);  // lse_j = -inf: ignore its o_j
                            acc[hh].x = fmaf(w, v.x, acc[hh].x);
                            acc[hh].y = fmaf(w, v.y, acc[hh].y);
                            acc[hh].z = fmaf(w, v.z, acc[hh].z);
                            acc[hh].w = fmaf(w, v.w, acc[hh].w);
                        }
                    }
                }
            }
        }
#pragma unroll
        for (int hh = 0; hh < 4; ++hh) {
            if (hh < nh) {
                reinterpret_cast<float4 *>(dst_o + (size_t)(i0 + hh) * kHeadDim)[lane] = acc[hh];
                if (lane == 0) dst_lse[i0 + hh] = lse_h[hh];
                if (dst2_o) {
                    reinterpret_cast<float4 *>(dst2_o + (size_t)(i0 + hh) * kHeadDim)[lane] = acc[hh];
                    if (lane == 0) dst2_lse[i0 + hh] = lse_h[hh];
                }
            }
        }
    }
}

// merge the pieces of unit u into its range partial (and into the final output if J_r == 1 and fused)
__device__ __forceinline__ void merge_unit_pieces(const AttendParams &p, const Unit &un, int u, int g, int lane) {
    const Dev &d = p.d;
    const size_t row = range_row(d, un.req, un.range, g * d.G);
    float *o2 = nullptr, *l2 = nullptr;
    if (p.fused && d.scratch[un.req] == 1) {
        const size_t frow = (size_t)un.req * d.Hq + g * d.G;
        o2 = p.o + frow * kHeadDim;
        l2 = p.lse + frow;
    }
    const int ps = piece_slot(un, u, un.piece_begin);
    warp_merge(d.piece_o + (size_t)ps * d.G * kHeadDim, (size_t)d.G * kHeadDim,
               d.piece_lse + (size_t)ps * d.G, d.G, un.n_pieces, d.G, p.o_part + row * kHeadDim,
               p.lse_part + row, o2, l2, lane);
}

// merge the J range partials of (req, kv head g) into the final output
__device__ __forceinline__ void merge_request_ranges(const Dev &d, const float *o_part, const float *lse_part,
                                                     float *o, float *lse, int req, int g, int J, int lane) {
    const size_t row = range_row(d, req, 0, g * d.G);
    const size_t frow = (size_t)req * d.Hq + g * d.G;
    warp_merge(o_part + row * kHeadDim, (size_t)d.Hq * kHeadDim, lse_part + row, d.Hq, J, d.G,
               o + frow * kHeadDim, lse + frow, nullptr, nullptr, lane);
}

// Fused tail: called by the whole warp after it has written the partial of one piece of unit u.
// The last piece of a unit merges the unit; the last unit of a (request, kv head) merges the request.
__device__ __forceinline__ void finish_piece(const AttendParams &p, int u, const Unit &un, int g, int lane) {
    const Dev &d = p.d;
    if (un.n_pieces > 1) {
        __threadfence();
        __syncwarp();
        int old = 0;
        if (lane == 0) old = atomicAdd(&d.unit_counter[u], 1);
        old = __shfl_sync(0xffffffffu, old, 0);
        if (old != un.n_pieces - 1) return;
        __threadfence();
        merge_unit_pieces(p, un, u, g, lane);
        if (lane == 0) d.unit_counter[u] = 0;
    }
    const int J = d.scratch[un.req];
    if (J <= 1) return;  // piece_dest / merge_unit_pieces already wrote the final rows
    __threadfence();
    __syncwarp();
    int old = 0;
    if (lane == 0) old = atomicAdd(&d.group_counter[un.req * d.Hkv + g], 1);
    old = __shfl_sync(0xffffffffu, old, 0);
    if (old != J - 1) return;
    __threadfence();
    merge_request_ranges(d, p.o_part, p.lse_part, p.o, p.lse, un.req, g, J, lane);
    if (lane == 0) d.group_counter[un.req * d.Hkv + g] = 0;
}

}  // namespace kf
