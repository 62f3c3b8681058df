// kf_attend_simple.cu -- KF_IMPL_SIMPLE: CUDA-core split-KV decode attention over token-range partitions
// (PAPER.md:137, :145).  One warp = one worker taking chunks of the work plan round-robin; 128-bit coalesced loads of
// K rows, 64-bit coalesced loads of V rows, fp32 online softmax (base-2), warp-shuffle reductions.  It is the
// plain reference GPU kernel: the TMA / tensor-core kernel (kf_attend_tma.cu) must agree with it.
#include "kf_merge.cuh"

namespace kf {

__global__ void __launch_bounds__(kWarpsPerCta * 32) attend_simple_kernel(AttendParams p) {
    __shared__ float q_s[kWarpsPerCta][kMaxGroup * kHeadDim];
    const Dev &d = p.d;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int W = gridDim.x * kWarpsPerCta;
    const int n_chunks = d.plan->n_pieces;
    const int w = warp * gridDim.x + blockIdx.x;  // warp-major: small launches spread over all SMs
    const Counters ctr = launch_prologue(d, w, W, lane);
    const int G = d.G;
    float *qs = q_s[warp];

    // static round-robin over the chunk list (one chunk = one piece of one unit)
    for (int c = w; c < n_chunks; c += W) {
        const Chunk ch = d.chunks[c];
        const int u = ch.unit, piece = ch.piece;
        const Unit un = d.units[u];
        const int g = u % d.Hkv;
        const int cnt = live_cnt(d, un);  // the plan may be older than this step (kf_common.cuh)
        const int t0 = ch.tile_begin, t1 = ch.tile_begin + live_tiles(un, cnt, ch.tile_begin, ch.n_tiles);
        if ((p.part_mask >> un.part) & 1ull) {
            const __half *qg = p.q + ((size_t)un.req * d.Hq + (size_t)g * G) * kHeadDim;
            __syncwarp();
            for (int i = lane; i < G * kHeadDim; i += 32) qs[i] = __half2float(qg[i]) * d.scale_log2;
            __syncwarp();

            float m[kMaxGroup], l[kMaxGroup], acc[kMaxGroup][4];
#pragma unroll
            for (int i = 0; i < kMaxGroup; ++i) {
                m[i] = -INFINITY;
                l[i] = 0.f;
                acc[i][0] = acc[i][1] = acc[i][2] = acc[i][3] = 0.f;
            }
            const unsigned char *Kb = d.pool[un.part] + row_offset(d, p.layer, un.slot, g, 0);
            const unsigned char *Vb = Kb + d.v_off;
            const int half = lane >> 4;

            for (int tile = t0; tile < t1; ++tile) {
                const int tok = tile * kTileTokens + (lane & 15);
                const bool valid = tok < cnt;
                float s[kMaxGroup];
#pragma unroll
                for (int i = 0; i < kMaxGroup; ++i) s[i] = 0.f;
                if (valid) {
                    const int4 *kp = reinterpret_cast<const int4 *>(Kb + (size_t)tok * 256 + half * 128);
#pragma unroll
                    for (int c = 0; c < 8; ++c) {
                        const int4 kk = __ldg(kp + c);
                        const __half2 *h2 = reinterpret_cast<const __half2 *>(&kk);
                        float kf[8];
#pragma unroll
                        for (int e = 0; e < 4; ++e) {
                            const float2 f = __half22float2(h2[e]);
                            kf[2 * e] = f.x;
                            kf[2 * e + 1] = f.y;
                        }
#pragma unroll
                        for (int i = 0; i < kMaxGroup; ++i) {
                            if (i < G) {
                                const float *qq = qs + i * kHeadDim + half * 64 + c * 8;
#pragma unroll
                                for (int e = 0; e < 8; ++e) s[i] = fmaf(kf[e], qq[e], s[i]);
                            }
                        }
                    }
                }
                float pr[kMaxGroup];
#pragma unroll
                for (int i = 0; i < kMaxGroup; ++i) {
                    pr[i] = 0.f;
                    if (i < G) {
                        float si = s[i] + __shfl_xor_sync(0xffffffffu, s[i], 16);
                        if (!valid) si = -INFINITY;
                        float mx = si;
#pragma unroll
                        for (int o = 8; o > 0; o >>= 1) mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, o));
                        const float m_new = fmaxf(m[i], mx);  // finite: every tile has >= 1 valid token
                        const float alpha = exp2f(m[i] - m_new);
                        pr[i] = valid ? exp2f(si - m_new) : 0.f;
                        l[i] = l[i] * alpha + (half == 0 ? pr[i] : 0.f);
                        acc[i][0] *= alpha;
                        acc[i][1] *= alpha;
                        acc[i][2] *= alpha;
                        acc[i][3] *= alpha;
                        m[i] = m_new;
                    }
                }
                const int nvalid = min(kTileTokens, cnt - tile * kTileTokens);
                for (int tt = 0; tt < nvalid; ++tt) {
                    const uint2 vv = __ldg(reinterpret_cast<const uint2 *>(
                        Vb + (size_t)(tile * kTileTokens + tt) * 256 + lane * 8));
                    const float2 v01 = __half22float2(*reinterpret_cast<const __half2 *>(&vv.x));
                    const float2 v23 = __half22float2(*reinterpret_cast<const __half2 *>(&vv.y));
#pragma unroll
                    for (int i = 0; i < kMaxGroup; ++i) {
                        if (i < G) {
                            const float pt = __shfl_sync(0xffffffffu, pr[i], tt);
                            acc[i][0] = fmaf(pt, v01.x, acc[i][0]);
                            acc[i][1] = fmaf(pt, v01.y, acc[i][1]);
                            acc[i][2] = fmaf(pt, v23.x, acc[i][2]);
                            acc[i][3] = fmaf(pt, v23.y, acc[i][3]);
                        }
                    }
                }
            }

            const PieceDest pd = piece_dest(p, un, u, g, piece);
#pragma unroll
            for (int i = 0; i < kMaxGroup; ++i) {
                if (i < G) {
                    const float lt = warp_sum(l[i]);
                    const float inv = 1.f / lt;
                    const float lse = (m[i] + log2f(lt)) * 0.6931471805599453f;
                    const float4 o4 = make_float4(acc[i][0] * inv, acc[i][1] * inv, acc[i][2] * inv, acc[i][3] * inv);
                    reinterpret_cast<float4 *>(pd.o + (size_t)i * kHeadDim)[lane] = o4;
                    if (lane == 0) pd.lse[i] = lse;
                    if (pd.o2) {
                        reinterpret_cast<float4 *>(pd.o2 + (size_t)i * kHeadDim)[lane] = o4;
                        if (lane == 0) pd.lse2[i] = lse;
                    }
                }
            }
            if (p.fused) piece_done(p, ctr, u, un, g, lane);
        }
    }
    if (p.fused) merge_phase(p, ctr, W, lane);
    launch_epilogue(d, W, lane, p.commit);
}

int launch_attend_simple(const AttendParams &p, int n_ctas, cudaStream_t s) {
    cudaLaunchConfig_t cfg = {};  // cooperative: see launch_one() in kf_attend_tma.cu
    cfg.gridDim = dim3(n_ctas);
    cfg.blockDim = dim3(kWarpsPerCta * 32);
    cfg.dynamicSmemBytes = 0;
    cfg.stream = s;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeCooperative;
    attr[0].val.cooperative = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    cudaLaunchKernelEx(&cfg, attend_simple_kernel, p);
    return 1;
}

}  // namespace kf
