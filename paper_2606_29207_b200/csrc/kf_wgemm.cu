// kf_wgemm.cu -- the dense contractions of the W-node stages (PAPER.md:143 step 1: QKV projection; :147 step 5 and
// :254: W_O and FFN), as ONE weight-streaming GEMM kernel for decode-sized batches (B <= 128):
//
//      out[b][n] = sum_k x[b][k] * W[n][k]          x [B][K] fp16,  W [N][K] fp16 ([out][in]),  fp32 accumulate
//
// At B <= 128 these GEMMs are bound by reading W once from HBM (2*N*K bytes for 2*B*N*K flop: <= 128 flop/B), so the
// kernel is built around the memory pipeline, and the tensor cores are simply the cheapest way to keep the math off
// the critical path -- on sm_100a that means tcgen05:
//   * the WEIGHT tile is the M side of the MMA (128 output features = 128 TMEM lanes), the batch is the N side
//     (NB = 16..128 columns), so a small batch costs no padding traffic and no wasted accumulator rows;
//   * warp 0 (one lane) streams 128 x 64 weight tiles and the matching NB x 64 activation tile with TMA
//     (cp.async.bulk.tensor.2d, 128-byte swizzle) through a 4..6 stage mbarrier ring;
//   * warp 1 (one lane) issues tcgen05.mma.cta_group::1.kind::f16 (M = 128, N = NB, K = 16, both operands K-major
//     shared-memory descriptors), accumulators in TMEM; tcgen05.commit releases the ring stages;
//   * warps 2..5 read the accumulators back with tcgen05.ld (32x32b: one output feature per thread, the batch along
//     the registers) and store fp16;
//   * N / 128 tiles rarely fill 148 SMs (Q projection of Llama-3.1-8B: 32 tiles), so K is split across CTAs; partial
//     sums go through L2 as fp32 and the LAST CTA of a tile adds them in split order (deterministic) and writes fp16;
//   * the gate and up projections of the FFN run as two accumulators of the same CTA (two weight tiles per stage,
//     one shared activation tile), so SwiGLU is applied in the epilogue and g, u never exist in memory.
#include <cuda.h>

#include "kf_wside.cuh"

namespace kf {

namespace {

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred P1;\n"
        "WG_WAIT:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n"
        "@P1 bra WG_DONE;\n"
        "bra WG_WAIT;\n"
        "WG_DONE:\n"
        "}\n" ::"r"(bar),
        "r"(parity)
        : "memory");
}
__device__ __forceinline__ void tma_load_2d_hint(uint32_t dst, const CUtensorMap *tmap, int x, int y, uint32_t bar,
                                                 uint64_t policy) {
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1, {%3, %4}], "
        "[%2], %5;" ::"r"(dst),
        "l"(tmap), "r"(bar), "r"(x), "r"(y), "l"(policy)
        : "memory");
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }

// K-major operand tile in shared memory, rows of 128 bytes (64 halfs), 128-byte swizzle, 8-row atoms 1024 bytes apart
__device__ __forceinline__ uint64_t umma_desc(uint32_t smem_addr) {
    uint64_t d = 0;
    d |= (uint64_t)((smem_addr & 0x3FFFFu) >> 4);  // start address, 16-byte units
    d |= (uint64_t)1 << 16;                        // leading byte offset: unused for swizzled K-major operands
    d |= (uint64_t)(1024 >> 4) << 32;              // stride byte offset: next 8-row group
    d |= (uint64_t)1 << 46;                        // descriptor version (Blackwell)
    d |= (uint64_t)2 << 61;                        // SWIZZLE_128B
    return d;
}
// D[tmem] (+)= A[smem] * B[smem]^T : M = 128 rows of A, N rows of B, K = 16
__device__ __forceinline__ void umma_f16(uint32_t tmem_d, uint64_t desc_a, uint64_t desc_b, uint32_t idesc, uint32_t accumulate) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "setp.ne.b32 p, %4, 0;\n"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n"
        "}\n" ::"r"(tmem_d),
        "l"(desc_a), "l"(desc_b), "r"(idesc), "r"(accumulate)
        : "memory");
}
__device__ __forceinline__ void umma_commit(uint32_t bar) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void tmem_ld16(uint32_t taddr, float (&v)[16]) {
    uint32_t r[16];
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
        : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
          "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
        : "r"(taddr));
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
    for (int i = 0; i < 16; ++i) v[i] = __uint_as_float(r[i]);
}

__device__ __forceinline__ float silu_mul(float g, float u) { return g / (1.f + __expf(-g)) * u; }

__host__ __device__ constexpr int tmem_cols(int n) { return n <= 32 ? 32 : n <= 64 ? 64 : n <= 128 ? 128 : n <= 256 ? 256 : 512; }

}  // namespace

template <int NB, bool DUAL>
__global__ void __launch_bounds__(kWgThreads, 1)
    wgemm_kernel(const __grid_constant__ CUtensorMap tmW, const __grid_constant__ CUtensorMap tmX, const WGemmArgs a) {
    constexpr int kWBytes = kWgTileN * kWgBK * 2;  // 16 KB: 128 weight rows x 64 halfs
    constexpr int kXBytes = NB * kWgBK * 2;
    constexpr int kNW = DUAL ? 2 : 1;
    constexpr int kStageBytes = kWBytes * kNW + kXBytes;
    constexpr int kStages = wgemm_stages(NB, DUAL);
    constexpr int kCols = tmem_cols(NB * kNW);
    extern __shared__ unsigned char smem_raw[];
    __shared__ __align__(8) uint64_t full_bar[kStages], empty_bar[kStages], acc_bar;
    __shared__ uint32_t tmem_base_s;
    __shared__ int last_s;
    const uint32_t base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int tile = blockIdx.x / a.splits, split = blockIdx.x - tile * a.splits;
    const int nkb = a.kb_per_split, kb0 = split * nkb;

    if (warp == 0 && lane == 0) {
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tmW) : "memory");
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tmX) : "memory");
#pragma unroll
        for (int s = 0; s < kStages; ++s) {
            mbar_init(smem_u32(&full_bar[s]), 1);
            mbar_init(smem_u32(&empty_bar[s]), 1);
        }
        mbar_init(smem_u32(&acc_bar), 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    if (warp == 1) {  // the whole warp allocates (and later frees) the accumulator columns
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&tmem_base_s)),
                     "n"(kCols)
                     : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = tmem_base_s;

    if (warp == 0) {
        if (lane == 0) {
            // ---- TMA producer: weights are read once -> evict-first; the activation tile is re-read by every CTA ----
            uint64_t pol_w = 0, pol_x = 0;
            asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol_w));
            asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(pol_x));
            for (int i = 0; i < nkb; ++i) {
                const int s = i % kStages;
                mbar_wait(smem_u32(&empty_bar[s]), ((i / kStages) & 1) ^ 1);
                const uint32_t sb = base + s * kStageBytes, bar = smem_u32(&full_bar[s]);
                const int kx = (kb0 + i) * kWgBK;
                mbar_expect_tx(bar, kStageBytes);
                tma_load_2d_hint(sb, &tmW, kx, tile * kWgTileN, bar, pol_w);
                if (DUAL) tma_load_2d_hint(sb + kWBytes, &tmW, kx, a.up_row_offset + tile * kWgTileN, bar, pol_w);
                tma_load_2d_hint(sb + kWBytes * kNW, &tmX, kx, 0, bar, pol_x);
            }
        }
        __syncwarp();
    } else if (warp == 1) {
        if (lane == 0) {
            // ---- MMA issuer: instruction descriptor: D fp32, A/B fp16 K-major, N = NB, M = 128 ----
            constexpr uint32_t idesc = (1u << 4) | ((uint32_t)(NB >> 3) << 17) | ((uint32_t)(kWgTileN >> 4) << 24);
            for (int i = 0; i < nkb; ++i) {
                const int s = i % kStages;
                mbar_wait(smem_u32(&full_bar[s]), (i / kStages) & 1);
                tc_fence_after();
                const uint32_t sa = base + s * kStageBytes, sx = sa + kWBytes * kNW;
#pragma unroll
                for (int k = 0; k < kWgBK / 16; ++k) {
                    const uint64_t db = umma_desc(sx + k * 32);
                    umma_f16(tmem, umma_desc(sa + k * 32), db, idesc, (uint32_t)((i | k) != 0));
                    if (DUAL) umma_f16(tmem + NB, umma_desc(sa + kWBytes + k * 32), db, idesc, (uint32_t)((i | k) != 0));
                }
                umma_commit(smem_u32(&empty_bar[s]));  // the stage is free once these MMAs have read it
            }
            umma_commit(smem_u32(&acc_bar));  // accumulators complete
        }
        __syncwarp();
    } else {
        // ---- epilogue: thread = one output feature (TMEM lane), registers run along the batch ----
        const int slice = warp & 3;  // a warp may only touch TMEM lanes 32 * (warp % 4) ..
        const int row = slice * 32 + lane;
        const int n = tile * kWgTileN + row;
        const uint32_t taddr = tmem + ((uint32_t)(slice * 32) << 16);
        const int seg = (tile * kWgTileN >= a.seg_end[0]) + (tile * kWgTileN >= a.seg_end[1]);
        const int nn = n - (seg == 0 ? 0 : a.seg_end[seg - 1]);
        __half *out = a.out[seg] + nn;
        const int ld = a.ld[seg];
        mbar_wait(smem_u32(&acc_bar), 0);
        tc_fence_after();
        if (a.splits == 1) {
#pragma unroll 1
            for (int c0 = 0; c0 < NB; c0 += 16) {
                float g[16], u[16];
                tmem_ld16(taddr + c0, g);
                if (DUAL) tmem_ld16(taddr + NB + c0, u);
#pragma unroll
                for (int j = 0; j < 16; ++j)
                    if (c0 + j < a.B) out[(size_t)(c0 + j) * ld] = __float2half_rn(DUAL ? silu_mul(g[j], u[j]) : g[j]);
            }
        } else {
            float *part = a.partial + ((size_t)split * NB) * a.N + n;
            const size_t dual_off = (size_t)a.splits * NB * a.N;
#pragma unroll 1
            for (int c0 = 0; c0 < NB; c0 += 16) {
                float g[16];
                tmem_ld16(taddr + c0, g);
#pragma unroll
                for (int j = 0; j < 16; ++j)
                    if (c0 + j < a.B) __stcg(part + (size_t)(c0 + j) * a.N, g[j]);
                if (DUAL) {
                    tmem_ld16(taddr + NB + c0, g);
#pragma unroll
                    for (int j = 0; j < 16; ++j)
                        if (c0 + j < a.B) __stcg(part + dual_off + (size_t)(c0 + j) * a.N, g[j]);
                }
            }
            asm volatile("bar.sync 1, 128;" ::: "memory");  // the 128 epilogue threads
            if (threadIdx.x == 64) {
                asm volatile("fence.acq_rel.gpu;" ::: "memory");
                const int old = atomicAdd(a.counters + tile, 1);
                const int last = old == a.splits - 1;
                if (last) a.counters[tile] = 0;  // ready for the next launch
                asm volatile("fence.acq_rel.gpu;" ::: "memory");
                last_s = last;
            }
            asm volatile("bar.sync 1, 128;" ::: "memory");
            if (last_s) {
                // the last CTA of this tile adds the partial sums in split order and applies the epilogue
                const float *p0 = a.partial + n;
                for (int b = 0; b < a.B; ++b) {
                    float g = 0.f, u = 0.f;
                    for (int s = 0; s < a.splits; ++s) {
                        g += __ldcg(p0 + ((size_t)s * NB + b) * a.N);
                        if (DUAL) u += __ldcg(p0 + dual_off + ((size_t)s * NB + b) * a.N);
                    }
                    out[(size_t)b * ld] = __float2half_rn(DUAL ? silu_mul(g, u) : g);
                }
            }
        }
        tc_fence_before();
    }
    __syncthreads();
    if (warp == 1) {
        tc_fence_after();
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "n"(kCols) : "memory");
    }
}

// o [rows][cols] fp32 -> fp16 (the attention output that feeds W_O)
__global__ void cast_o_kernel(const float *__restrict__ o, __half *__restrict__ o16, size_t n4) {
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n4; i += (size_t)gridDim.x * blockDim.x) {
        const float4 v = __ldg(reinterpret_cast<const float4 *>(o) + i);
        __half2 a = __floats2half2_rn(v.x, v.y), b = __floats2half2_rn(v.z, v.w);
        uint2 w;
        w.x = *reinterpret_cast<uint32_t *>(&a);
        w.y = *reinterpret_cast<uint32_t *>(&b);
        reinterpret_cast<uint2 *>(o16)[i] = w;
    }
}

template <int NB, bool DUAL>
static int launch_one(const CUtensorMap &tmW, const CUtensorMap &tmX, const WGemmArgs &a, cudaStream_t s) {
    const int smem = wgemm_smem_bytes(NB, DUAL);
    static bool configured = false;  // per instantiation
    if (!configured) {
        if (cudaFuncSetAttribute(wgemm_kernel<NB, DUAL>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem) != cudaSuccess)
            return KF_ECUDA;
        configured = true;
    }
    wgemm_kernel<NB, DUAL><<<(a.N / kWgTileN) * a.splits, kWgThreads, smem, s>>>(tmW, tmX, a);
    return 1;
}

int launch_wgemm(const CUtensorMap &tmW, const CUtensorMap &tmX, const WGemmArgs &a, int nb, bool dual, cudaStream_t s) {
#define KF_WG(NBv)                                                          \
    if (nb == NBv) return dual ? launch_one<NBv, true>(tmW, tmX, a, s) : launch_one<NBv, false>(tmW, tmX, a, s);
    KF_WG(16) KF_WG(32) KF_WG(64) KF_WG(128)
#undef KF_WG
    return KF_EINVAL;
}

int launch_cast_o(const float *o, __half *o16, size_t n, cudaStream_t s) {
    const size_t n4 = n / 4;
    const int blocks = (int)((n4 + 255) / 256 < 592 ? (n4 + 255) / 256 : 592);
    cast_o_kernel<<<blocks > 0 ? blocks : 1, 256, 0, s>>>(o, o16, n4);
    return 1;
}

}  // namespace kf
