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
//   * persistent, stream-K: N / 128 tiles rarely fill 148 SMs (Q projection of Llama-3.1-8B: 32 tiles), so the flat
//     sequence of (tile, k-block) pairs is cut into one contiguous span per CTA; the TMA ring runs through a span
//     without draining at tile boundaries, two TMEM accumulator buffers let the epilogue of one tile overlap the MMAs
//     of the next; a tile that several spans share goes through L2 as fp32 pieces which a small fix-up kernel adds
//     in k order (deterministic; no CTA ever waits for another one, so any SM budget is safe) and writes as fp16;
//   * programmatic dependent launch along the kernel chain of a W-side call: the set-up of a kernel (barriers, TMEM,
//     descriptors) overlaps the tail of its predecessor;
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

// One span of the stream-K decomposition: CTA c owns the k-blocks [c * per, (c + 1) * per) of the flat sequence
// (tile 0: k-blocks 0 .. nkb-1, tile 1: ...).  A maximal run of k-blocks inside one tile is a SEGMENT: one accumulator.
struct Span {
    int k0, k1;
};
__device__ __forceinline__ Span span_of(const WGemmArgs &a, int cta, int n_ctas) {
    const int total = (a.N / kWgTileN) * a.nkb;
    const int per = (total + n_ctas - 1) / n_ctas;
    Span sp;
    sp.k0 = min(total, cta * per);
    sp.k1 = min(total, sp.k0 + per);
    return sp;
}

template <int NB, bool DUAL>
__global__ void __launch_bounds__(kWgThreads, 1)
    wgemm_kernel(const __grid_constant__ CUtensorMap tmW, const __grid_constant__ CUtensorMap tmX, const WGemmArgs a) {
    constexpr int kWBytes = kWgTileN * kWgBK * 2;  // 16 KB: 128 weight rows x 64 halfs
    constexpr int kXBytes = NB * kWgBK * 2;
    constexpr int kNW = DUAL ? 2 : 1;
    constexpr int kStageBytes = kWBytes * kNW + kXBytes;
    constexpr int kStages = wgemm_stages(NB, DUAL);
    constexpr int kAccCols = NB * kNW;               // TMEM columns of one accumulator buffer
    constexpr int kCols = tmem_cols(2 * kAccCols);   // two buffers: the epilogue of a segment overlaps the next one's MMAs
    extern __shared__ unsigned char smem_raw[];
    __shared__ __align__(8) uint64_t full_bar[kStages], empty_bar[kStages], acc_full[2], acc_empty[2];
    __shared__ uint32_t tmem_base_s;
    const uint32_t base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int nkb = a.nkb;
    const Span sp = span_of(a, blockIdx.x, gridDim.x);

    if (warp == 0 && lane == 0) {
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tmW) : "memory");
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tmX) : "memory");
#pragma unroll
        for (int s = 0; s < kStages; ++s) {
            mbar_init(smem_u32(&full_bar[s]), 1);
            mbar_init(smem_u32(&empty_bar[s]), 1);
        }
#pragma unroll
        for (int s = 0; s < 2; ++s) {
            mbar_init(smem_u32(&acc_full[s]), 1);
            mbar_init(smem_u32(&acc_empty[s]), 4);  // one arrival per epilogue warp
        }
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
    // Programmatic dependent launch along the chain of a W-side call: everything above (barriers, TMEM, descriptor
    // prefetch) touches no global memory and overlaps the tail of the preceding kernel; nothing below runs before that
    // kernel has completed.  The successor may set itself up from here on.
    asm volatile("griddepcontrol.wait;" ::: "memory");
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");

    if (warp == 0) {
        if (lane == 0) {
            // ---- TMA producer: runs through the whole span, across tile boundaries; weights are read once ->
            //      evict-first; the activation tile is re-read by every CTA -> evict-last ----
            uint64_t pol_w = 0, pol_x = 0;
            asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol_w));
            asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(pol_x));
            int tile = sp.k0 / nkb, kb = sp.k0 - tile * nkb;
            for (int i = 0; i < sp.k1 - sp.k0; ++i) {
                const int s = i % kStages;
                mbar_wait(smem_u32(&empty_bar[s]), ((i / kStages) & 1) ^ 1);
                const uint32_t sb = base + s * kStageBytes, bar = smem_u32(&full_bar[s]);
                const int kx = kb * kWgBK;
                mbar_expect_tx(bar, kStageBytes);
                tma_load_2d_hint(sb, &tmW, kx, tile * kWgTileN, bar, pol_w);
                if (DUAL) tma_load_2d_hint(sb + kWBytes, &tmW, kx, a.up_row_offset + tile * kWgTileN, bar, pol_w);
                tma_load_2d_hint(sb + kWBytes * kNW, &tmX, kx, 0, bar, pol_x);
                if (++kb == nkb) {
                    kb = 0;
                    ++tile;
                }
            }
        }
        __syncwarp();
    } else if (warp == 1) {
        if (lane == 0) {
            // ---- MMA issuer: instruction descriptor: D fp32, A/B fp16 K-major, N = NB, M = 128 ----
            constexpr uint32_t idesc = (1u << 4) | ((uint32_t)(NB >> 3) << 17) | ((uint32_t)(kWgTileN >> 4) << 24);
            int i = 0, seg = 0;
            for (int pos = sp.k0; pos < sp.k1; ++seg) {
                const int kb = pos % nkb;
                const int len = min(nkb - kb, sp.k1 - pos);
                const int buf = seg & 1;
                mbar_wait(smem_u32(&acc_empty[buf]), ((seg >> 1) & 1) ^ 1);  // the epilogue has drained this buffer
                tc_fence_after();
                const uint32_t acc = tmem + buf * kAccCols;
                for (int j = 0; j < len; ++j, ++i) {
                    const int s = i % kStages;
                    mbar_wait(smem_u32(&full_bar[s]), (i / kStages) & 1);
                    tc_fence_after();
                    const uint32_t sa = base + s * kStageBytes, sx = sa + kWBytes * kNW;
#pragma unroll
                    for (int k = 0; k < kWgBK / 16; ++k) {
                        const uint64_t db = umma_desc(sx + k * 32);
                        umma_f16(acc, umma_desc(sa + k * 32), db, idesc, (uint32_t)((j | k) != 0));
                        if (DUAL) umma_f16(acc + NB, umma_desc(sa + kWBytes + k * 32), db, idesc, (uint32_t)((j | k) != 0));
                    }
                    umma_commit(smem_u32(&empty_bar[s]));  // the stage is free once these MMAs have read it
                }
                umma_commit(smem_u32(&acc_full[buf]));  // this segment's accumulator is complete
                pos += len;
            }
        }
        __syncwarp();
    } else {
        // ---- epilogue: thread = one output feature (TMEM lane), registers run along the batch ----
        const int slice = warp & 3;  // a warp may only touch TMEM lanes 32 * (warp % 4) ..
        const int row = slice * 32 + lane;
        const size_t slot_floats = (size_t)NB * kWgTileN * kNW;  // one partial: [kNW][NB][128] fp32
        int seg = 0;
        for (int pos = sp.k0; pos < sp.k1; ++seg) {
            const int tile = pos / nkb, kb = pos - tile * nkb;
            const int len = min(nkb - kb, sp.k1 - pos);
            const int buf = seg & 1;
            const int n = tile * kWgTileN + row;
            // output segment of the tile (no dynamic indexing of the parameter struct: that would copy it to local memory)
            const bool s1 = tile * kWgTileN >= a.seg_end[0], s2 = tile * kWgTileN >= a.seg_end[1];
            __half *out = (s2 ? a.out[2] : s1 ? a.out[1] : a.out[0]) + (n - (s2 ? a.seg_end[1] : s1 ? a.seg_end[0] : 0));
            const int ld = s2 ? a.ld[2] : s1 ? a.ld[1] : a.ld[0];
            const uint32_t taddr = tmem + ((uint32_t)(slice * 32) << 16) + buf * kAccCols;
            mbar_wait(smem_u32(&acc_full[buf]), (seg >> 1) & 1);
            tc_fence_after();
            const bool whole = len == nkb;
            if (whole) {
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
                // a piece of a tile: fp32 partial into this CTA's slot (0: the span's first segment, 1: any later one)
                float *part = a.partial + ((size_t)blockIdx.x * 2 + (seg == 0 ? 0 : 1)) * slot_floats + row;
#pragma unroll 1
                for (int c0 = 0; c0 < NB; c0 += 16) {
                    float g[16];
                    tmem_ld16(taddr + c0, g);
#pragma unroll
                    for (int j = 0; j < 16; ++j)
                        if (c0 + j < a.B) __stcg(part + (size_t)(c0 + j) * kWgTileN, g[j]);
                    if (DUAL) {
                        tmem_ld16(taddr + NB + c0, g);
#pragma unroll
                        for (int j = 0; j < 16; ++j)
                            if (c0 + j < a.B) __stcg(part + (size_t)(NB + c0 + j) * kWgTileN, g[j]);
                    }
                }
            }
            // the accumulator buffer is free again
            tc_fence_before();
            __syncwarp();
            if (lane == 0) asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(&acc_empty[buf])) : "memory");
            pos += len;
        }
        tc_fence_before();
    }
    __syncthreads();
    if (warp == 1) {
        tc_fence_after();
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "n"(kCols) : "memory");
    }
}

// Fix-up of the tiles that several spans share: out[b][n] = epilogue(sum over the pieces, in k order = ascending CTA).
// One thread per (4 consecutive features, batch row): every piece is read once with 128-bit loads, coalesced along the
// features, all pieces of the thread in flight at once; 8-byte stores.  grid (tiles, ceil(B / 8)), block (32, 8).
template <bool DUAL>
__global__ void __launch_bounds__(256) wgemm_fixup_kernel(const WGemmArgs a, int nb) {
    asm volatile("griddepcontrol.wait;" ::: "memory");  // launched while the GEMM is still running (PDL)
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    const int tile = blockIdx.x, row = threadIdx.x * 4, b = blockIdx.y * 8 + threadIdx.y;
    const int nkb = a.nkb;
    const int total = (a.N / kWgTileN) * nkb;
    const int per = (total + a.n_ctas - 1) / a.n_ctas;
    const int k_lo = tile * nkb, k_hi = k_lo + nkb;  // the tile's k-blocks in the flat (tile, k-block) sequence
    const int c_first = k_lo / per, c_last = (k_hi - 1) / per;
    if (c_first == c_last || b >= a.B) return;  // the tile was whole: its CTA stored the result itself
    const size_t slot_floats = (size_t)nb * kWgTileN * (DUAL ? 2 : 1);
    float4 g = make_float4(0.f, 0.f, 0.f, 0.f), u = g;
    for (int c0 = c_first; c0 <= c_last; c0 += 8) {
        float4 t[8], tu[8];
#pragma unroll
        for (int e = 0; e < 8; ++e) {
            const int c = c0 + e;
            const int start = c * per;  // slot 0 holds the span's first segment: the span starts inside this tile
            const int slot = (start >= k_lo && start < k_hi) ? 0 : 1;
            const float *pp = a.partial + ((size_t)c * 2 + slot) * slot_floats + row;
            t[e] = c <= c_last ? __ldcg(reinterpret_cast<const float4 *>(pp + (size_t)b * kWgTileN)) : make_float4(0.f, 0.f, 0.f, 0.f);
            if (DUAL)
                tu[e] = c <= c_last ? __ldcg(reinterpret_cast<const float4 *>(pp + (size_t)(nb + b) * kWgTileN))
                                    : make_float4(0.f, 0.f, 0.f, 0.f);
        }
#pragma unroll
        for (int e = 0; e < 8; ++e) {
            g.x += t[e].x;
            g.y += t[e].y;
            g.z += t[e].z;
            g.w += t[e].w;
            if (DUAL) {
                u.x += tu[e].x;
                u.y += tu[e].y;
                u.z += tu[e].z;
                u.w += tu[e].w;
            }
        }
    }
    const int n = tile * kWgTileN + row;
    // output segment of the tile (no dynamic indexing of the parameter struct: that would copy it to local memory)
    const bool s1 = tile * kWgTileN >= a.seg_end[0], s2 = tile * kWgTileN >= a.seg_end[1];
    __half *base_out = s2 ? a.out[2] : s1 ? a.out[1] : a.out[0];
    const int ldo = s2 ? a.ld[2] : s1 ? a.ld[1] : a.ld[0];
    const int n0 = s2 ? a.seg_end[1] : s1 ? a.seg_end[0] : 0;
    __half *out = base_out + (n - n0) + (size_t)b * ldo;
    const __half2 lo = __floats2half2_rn(DUAL ? silu_mul(g.x, u.x) : g.x, DUAL ? silu_mul(g.y, u.y) : g.y);
    const __half2 hi = __floats2half2_rn(DUAL ? silu_mul(g.z, u.z) : g.z, DUAL ? silu_mul(g.w, u.w) : g.w);
    uint2 w;
    w.x = *reinterpret_cast<const uint32_t *>(&lo);
    w.y = *reinterpret_cast<const uint32_t *>(&hi);
    *reinterpret_cast<uint2 *>(out) = w;
}

// o [rows][cols] fp32 -> fp16 (the attention output that feeds W_O)
__global__ void cast_o_kernel(const float *__restrict__ o, __half *__restrict__ o16, size_t n4) {
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");  // the W_O GEMM may set itself up meanwhile
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
static int launch_one(const CUtensorMap &tmW, const CUtensorMap &tmX, const WGemmArgs &a, bool pdl, cudaStream_t s) {
    const int smem = wgemm_smem_bytes(NB, DUAL);
    // the opt-in to > 48 KB of dynamic shared memory is a per-DEVICE property of the function: once per instantiation
    // and device (a second GPU in the same process would otherwise launch without it and fail)
    constexpr int kDevs = 64;
    static bool configured[kDevs] = {};
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return KF_ECUDA;
    if (dev < 0 || dev >= kDevs || !configured[dev]) {
        if (cudaFuncSetAttribute(wgemm_kernel<NB, DUAL>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem) != cudaSuccess)
            return KF_ECUDA;
        if (dev >= 0 && dev < kDevs) configured[dev] = true;
    }
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(a.n_ctas);
    cfg.blockDim = dim3(kWgThreads);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = s;
    cfg.attrs = attr;
    cfg.numAttrs = pdl ? 1 : 0;  // safe behind any kernel: nothing before the kernel's griddepcontrol.wait touches global memory
    if (cudaLaunchKernelEx(&cfg, wgemm_kernel<NB, DUAL>, tmW, tmX, a) != cudaSuccess) return KF_ECUDA;
    // tiles shared between spans exist unless every span boundary is a tile boundary
    const int tiles = a.N / kWgTileN, total = tiles * a.nkb, per = (total + a.n_ctas - 1) / a.n_ctas;
    if (per % a.nkb == 0) return 1;
    cfg.gridDim = dim3(tiles, (a.B + 7) / 8);
    cfg.blockDim = dim3(kWgTileN / 4, 8);
    cfg.dynamicSmemBytes = 0;
    cfg.numAttrs = 1;            // the fix-up always follows its GEMM
    if (cudaLaunchKernelEx(&cfg, wgemm_fixup_kernel<DUAL>, a, (int)NB) != cudaSuccess) return KF_ECUDA;
    return 2;
}

int launch_wgemm(const CUtensorMap &tmW, const CUtensorMap &tmX, const WGemmArgs &a, int nb, bool dual, bool pdl,
                 cudaStream_t s) {
#define KF_WG(NBv)                                                          \
    if (nb == NBv) return dual ? launch_one<NBv, true>(tmW, tmX, a, pdl, s) : launch_one<NBv, false>(tmW, tmX, a, pdl, s);
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
