// kf_attend_tma.cu -- KF_IMPL_TMA: the roofline kernel for split-KV decode attention over token-range
// partitions (PAPER.md:137, :145; "decode attention is bandwidth-bound", :225).
//
// Design (B200 / sm_100a):
//  * Persistent grid, one CTA of 8 warps per SM.  Every WARP is an independent worker that owns an equal,
//    contiguous span of the step's 16-token tiles (stream-K split built on the device by plan_kernel), its
//    own 3-stage shared-memory ring and its own mbarriers: there is no CTA-wide synchronisation at all.
//  * K/V tiles are fetched by TMA (cp.async.bulk.tensor.2d, one elected lane) straight from the routed pool
//    slot into 128B-swizzled shared memory; each of the 1184 workers keeps up to 24 KB in flight
//    (~190 KB per SM) -- Little's law at ~6.5 TB/s x ~1 us needs ~50 KB per SM.
//  * The G query heads of a GQA group are packed into the M dimension of mma.sync.m16n8k16 (fp16 in, fp32
//    accumulate): S = Q K^T and O += P V run on the tensor cores so the ALUs only do the online softmax.
//    K fragments come from ldmatrix, V fragments from ldmatrix.trans; the hardware swizzle makes both
//    bank-conflict free.
//  * Online softmax in fp32, base 2, quad shuffles; the accumulator rescale is skipped when no running
//    maximum moved.
//  * The partial (o, lse) of each piece goes to the range-partial rows or to a piece buffer; in fused mode
//    the last-arriving worker merges pieces -> range -> request (kf_merge.cuh).
#include <cuda.h>

#include "kf_merge.cuh"

namespace kf {

constexpr int kSubTile = kTileTokens * 128;     // 16 rows x 128 B (64 halfs): one TMA box
constexpr int kStageBytes = 4 * kSubTile;       // K lo | K hi | V lo | V hi = 8 KB
constexpr int kRing = 8;                        // chunk descriptors in flight between the load and compute cursors
// P is rounded to fp16 for the P.V MMA.  With p = exp2(s - m) in (0, 1] every weight below 2^-25 would flush to zero
// there while the fp32 row sum l keeps it: on a long, peaked context (1M tokens, each 2^-25 below the maximum) that
// is up to 3% of the mass missing from o but present in l.  So P (and l with it) is carried scaled up:
// p' = exp2(s - m_ref + kPShift), where m_ref trails the true maximum by at most kLazy, so p' <= 2^14;
// o'/l' = o/l, lse = m_ref + log2(l') - kPShift.
constexpr float kLazy = 8.f;     // the reference maximum of a head moves only when a score exceeds it by 2^8
constexpr float kPShift = 6.f;   // p = exp2(s - m_ref + 6) <= 2^14: fits fp16; flush threshold 2^-31 .. 2^-39 below the maximum

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
        "KF_WAIT:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n"
        "@P1 bra KF_DONE;\n"
        "bra KF_WAIT;\n"
        "KF_DONE:\n"
        "}\n" ::"r"(bar),
        "r"(parity)
        : "memory");
}
__device__ __forceinline__ void tma_load_2d(uint32_t dst, const void *tmap, int x, int y, uint32_t bar) {
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4}], [%2];" ::"r"(dst),
        "l"(tmap), "r"(bar), "r"(x), "r"(y)
        : "memory");
}
__device__ __forceinline__ void tma_load_2d_hint(uint32_t dst, const void *tmap, int x, int y, uint32_t bar,
                                                 uint64_t policy) {
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1, {%3, %4}], "
        "[%2], %5;" ::"r"(dst),
        "l"(tmap), "r"(bar), "r"(x), "r"(y), "l"(policy)
        : "memory");
}
__device__ __forceinline__ void ldsm_x4(uint32_t addr, uint32_t &r0, uint32_t &r1, uint32_t &r2, uint32_t &r3) {
    asm volatile("ldmatrix.sync.aligned.m8n8.x4.shared.b16 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r0), "=r"(r1), "=r"(r2), "=r"(r3)
                 : "r"(addr));
}
__device__ __forceinline__ void ldsm_x4_trans(uint32_t addr, uint32_t &r0, uint32_t &r1, uint32_t &r2, uint32_t &r3) {
    asm volatile("ldmatrix.sync.aligned.m8n8.x4.trans.shared.b16 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r0), "=r"(r1), "=r"(r2), "=r"(r3)
                 : "r"(addr));
}
// D(16x8,f32) += A(16x16,f16,row) * B(16x8,f16,col)
__device__ __forceinline__ void mma16816(float (&c)[4], uint32_t a0, uint32_t a1, uint32_t a2, uint32_t a3, uint32_t b0,
                                         uint32_t b1) {
    asm volatile(
        "mma.sync.aligned.m16n8k16.row.col.f32.f16.f16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
        : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
        : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1));
}
// transpose an 8x8 matrix of 16-bit elements held as one C / A-style fragment register per lane
__device__ __forceinline__ uint32_t movmatrix_trans(uint32_t x) {
    uint32_t y;
    asm volatile("movmatrix.sync.aligned.m8n8.trans.b16 %0, %1;" : "=r"(y) : "r"(x));
    return y;
}
__device__ __forceinline__ float fast_exp2(float x) {
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ uint32_t pack_half2(float lo, float hi) {
    const __half2 h = __floats2half2_rn(lo, hi);
    return *reinterpret_cast<const uint32_t *>(&h);
}
__device__ __forceinline__ long long global_ns() {
    long long t;
    asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t));
    return t;
}
__device__ __forceinline__ int sm_id() {
    int v;
    asm volatile("mov.u32 %0, %smid;" : "=r"(v));
    return v;
}
__device__ __forceinline__ Unit load_unit(const Unit *units, int u) {
    const int4 *p = reinterpret_cast<const int4 *>(units + u);
    const int4 a = __ldg(p), b = __ldg(p + 1);
    Unit un;
    un.req = a.x;
    un.range = a.y;
    un.part = a.z;
    un.slot = a.w;
    un.cnt = b.x;
    un.tail = b.y;
    un.piece_begin = b.z;
    un.n_pieces = b.w;
    return un;
}


// Ring slot handed from a worker's load cursor to its compute cursor: the chunk's record with the live tile / token
// counts filled in.  Word layout = ChunkRec; pad[0] = 1 when the chunk's q rows were staged into the warp's q slot.
constexpr int kQRowBytes = kHeadDim * 2 + 16;  // q rows in shared memory, padded: B-fragment loads hit 32 distinct banks
constexpr int kPfStart = 3;                    // the next chunk is requested when this many tiles of the current one are left

template <int WARPS, int STAGES>
__global__ void __launch_bounds__(WARPS * 32, 1) attend_tma_kernel(const AttendParams p) {
    constexpr int kWarpSmem = STAGES * kStageBytes;
    extern __shared__ unsigned char smem_raw[];
    __shared__ __align__(8) uint64_t bars[WARPS][STAGES];
    __shared__ __align__(16) int4 ring[WARPS][kRing][4];
    __shared__ __align__(16) unsigned char q_stage[WARPS][kMaxGroup * kQRowBytes];
    const Dev &d = p.d;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int W = gridDim.x * WARPS;
    const int w = warp * gridDim.x + blockIdx.x;  // warp-major: the first chunks of a small launch spread over all SMs
    const int n_chunks = __ldg(&d.plan->n_pieces);
    const long long t_start = d.diag ? global_ns() : 0;
    long long t_first = 0, t_stream = 0;
    Counters ctr;
    int m_first = -1;  // lane 0: pre-taken first merge ticket

    if (w < n_chunks) {
        const uint32_t wbase = ((smem_u32(smem_raw) + 1023u) & ~1023u) + warp * kWarpSmem;
        const uint32_t bar0 = smem_u32(&bars[warp][0]);
        if (lane == 0) {
#pragma unroll
            for (int s = 0; s < STAGES; ++s) mbar_init(bar0 + 8 * s, 1);
            asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        }
        __syncwarp();

        const int G = d.G, Hkv = d.Hkv;
        uint64_t policy = 0;  // K/V is read once per launch: evict-first keeps the partials resident in L2
        asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(policy));
        const unsigned char *tmaps = reinterpret_cast<const unsigned char *>(d.tmaps);
        const int layer_row = p.layer * d.slots * Hkv * d.R;
        const uint32_t q_s = smem_u32(&q_stage[warp][0]);

        // ---- load cursor: runs up to STAGES tiles ahead of the compute cursor, across chunk boundaries.  The NEXT
        //      chunk is fetched in the background, one step per issued tile: ticket (atomic) -> 64-byte record (one
        //      coalesced load by lanes 0..3) -> ring slot in shared memory; by the time the current chunk runs out,
        //      its successor is a shared-memory read away. ----
        int issued = 0, consumed = 0;
        int l_left = 0, l_row = 0, l_part = 0;
        int ring_w = 0, ring_r = 0;
        int pf_state = 1, pf_id = w;  // 0 idle | 1 ticket requested (pf_id valid: the first chunk is static) | 2 record requested | 3 record in the ring
        int pf_tk = 0;                // lane 0: the ticket
        bool pf_static = true;        // pf_id already holds the chunk id (worker w starts with chunk w: no atomic storm)
        int4 pf_rec = make_int4(0, 0, 0, 0);
        bool l_done = false, q_busy = false;
        auto pf_step = [&]() {
            if (pf_state == 0) {
                if (lane == 0) pf_tk = atomicAdd(d.sched, 1);
                pf_state = 1;
            } else if (pf_state == 1) {
                if (!pf_static) pf_id = W + __shfl_sync(0xffffffffu, pf_tk, 0);
                pf_static = false;
                if (pf_id < n_chunks) {
                    if (lane < 4) pf_rec = __ldg(reinterpret_cast<const int4 *>(d.recs + pf_id) + lane);
                } else if (p.fused && lane == 0 && m_first < 0) {
                    m_first = merge_first_ticket(d, W);  // nothing left to load: reserve the first merge tasks now
                }
                pf_state = 2;
            } else if (pf_state == 2) {
                if (pf_id < n_chunks && lane < 4) ring[warp][ring_w & (kRing - 1)][lane] = pf_rec;
                __syncwarp();
                pf_state = 3;
            }
        };
        // next chunk -> load cursor; false when the list is exhausted
        auto advance = [&]() -> bool {
            for (;;) {
                while (pf_state < 3) pf_step();
                pf_state = 0;
                if (pf_id >= n_chunks) {
                    l_done = true;
                    return false;
                }
                int4 *slot = ring[warp][ring_w & (kRing - 1)];
                const int4 a = slot[0], b = slot[1], c = slot[2];  // {unit, tile_begin, n_tiles, piece} {part, row0, req, range} {cnt, flags, n_pieces, J}
                if (!((p.part_mask >> b.x) & 1ull)) continue;     // partition not selected: nothing to load
                int n_tiles = a.z, cnt = c.x, app = -1;
                if (c.y & kRecTail) {  // the plan may be older than this step: a tail unit has grown since
                    const int raw = __ldg(d.len + b.z) + 1 - slot[3].z;  // tokens of the tail range, this step's included
                    cnt = min(d.R, raw);
                    if (c.y & kRecStretch) {
                        n_tiles = (cnt + kTileTokens - 1) / kTileTokens - a.y;
                        if (p.k_new) {  // fused (a2): this chunk ends with the tile that receives the new token
                            if (raw <= d.R)
                                app = raw - 1;
                            else if (lane == 0)
                                set_error(d, KF_ESTATE);  // no route for the tail position (the request waits for a slot)
                        }
                    }
                }
                // q rows of the chunk's head group -> the warp's q slot (if the previous chunk has picked its q up)
                const bool stage_q = !q_busy;
                if (stage_q) {
                    const unsigned char *qg =
                        reinterpret_cast<const unsigned char *>(p.q + ((size_t)b.z * d.Hq + (size_t)(a.x % Hkv) * G) * kHeadDim);
                    for (int i = lane; i < G * 16; i += 32) {
                        const uint32_t dst = q_s + (i >> 4) * kQRowBytes + (i & 15) * 16;
                        asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(qg + (size_t)i * 16) : "memory");
                    }
                    asm volatile("cp.async.commit_group;" ::: "memory");
                    q_busy = true;
                }
                __syncwarp();  // every lane has read the slot
                if (lane == 0) {
                    slot[0].z = n_tiles;
                    slot[2].x = cnt;
                    slot[3].x = stage_q ? 1 : 0;
                    slot[3].y = app;
                }
                l_left = n_tiles;
                l_part = b.x;
                l_row = layer_row + b.y;
                ++ring_w;
                return true;
            }
        };
        auto try_issue = [&]() {
            if (l_done) return;
            if (l_left == 0 && !advance()) return;
            if (lane == 0) {
                const int stage = issued % STAGES;
                const uint32_t sb = wbase + stage * kStageBytes, bar = bar0 + 8 * stage;
                const unsigned char *tk = tmaps + (size_t)l_part * 256;
                mbar_expect_tx(bar, kStageBytes);
                if (d.l2_hint) {
                    tma_load_2d_hint(sb, tk, 0, l_row, bar, policy);
                    tma_load_2d_hint(sb + kSubTile, tk, 64, l_row, bar, policy);
                    tma_load_2d_hint(sb + 2 * kSubTile, tk + 128, 0, l_row, bar, policy);
                    tma_load_2d_hint(sb + 3 * kSubTile, tk + 128, 64, l_row, bar, policy);
                } else {
                    tma_load_2d(sb, tk, 0, l_row, bar);
                    tma_load_2d(sb + kSubTile, tk, 64, l_row, bar);
                    tma_load_2d(sb + 2 * kSubTile, tk + 128, 0, l_row, bar);
                    tma_load_2d(sb + 3 * kSubTile, tk + 128, 64, l_row, bar);
                }
            }
            l_row += kTileTokens;
            --l_left;
            ++issued;
            // late enough that a slow worker does not reserve work long before it can start it, early enough to hide
            // the round trips of the atomic and of the record
            if (l_left < kPfStart && pf_state < 3) pf_step();
        };
#pragma unroll
        for (int s = 0; s < STAGES; ++s) try_issue();
        ctr = launch_prologue(d, w, W, lane);  // one more L2 round trip, now in the shadow of the first tiles

        // ---- fragment addressing.  TOKENS are the M rows of both MMAs (S^T = K Q^T, O^T = V^T P^T), the <= 8 query
        //      heads of the group are the N = 8 columns: no padding rows for G = 8, half as many HMMAs and accumulator
        //      registers as heads-as-M.  128B hardware swizzle: 16-byte chunk index ^= row & 7. ----
        const int l7 = lane & 7;
        const uint32_t ka_row = (l7 + ((lane >> 3) & 1) * 8) * 128;  // K as A operand (ldmatrix x4: matrix lane / 8)
        const int ka_kc = lane >> 4;                                  // which 8-half chunk of the 16-wide k-step
        const uint32_t va_row = (l7 + (lane >> 4) * 8) * 128;         // V as A operand through ldmatrix.trans
        const int va_dc = (lane >> 3) & 1;                            // which 8-wide half of the 16 output dims
        const int tq = lane >> 2;                                     // C fragments: token rows tq, tq + 8; B: head
        const int hp = (lane & 3) * 2;                                // C fragments: heads hp, hp + 1

        // ---- compute cursor ------------------------------------------------------------------------------
        int cu = 0, ct = 0, c_left = 0, piece = 0, c_cnt = 0, c_req = 0, c_range = 0, c_np = 0, c_J = 0;
        int c_app = -1, c_part = 0, c_row = 0;  // fused append: token offset of the new row in the unit (-1: none)
        uint32_t qb[8][2];  // B fragments of Q^T: [k-step][b0, b1] = Q[head tq][16 ks + hp, +1] and [.. + 8, +9]
        float o[8][4];      // O^T: [16-dim tile][c0..c3] = (dim 16 mt + tq, heads hp, hp+1), (dim + 8, heads hp, hp+1)
        float m0 = -INFINITY, m1 = -INFINITY, l0 = 0.f, l1 = 0.f;  // reference maximum (base 2) and row sum of heads hp, hp+1
        // completion signal of the piece written last, deferred by one tile: the release fence then finds the partial's
        // stores already performed instead of waiting ~1 us for them
        int32_t *sig_ptr = nullptr;  // lane 0
        int sig_val = 0;
        bool sig_pending = false;    // warp-uniform
        auto flush_signal = [&]() {
            // release: barrier first, THEN lane 0 fences and publishes -- the fence is cumulative over the stores of
            // the other lanes that the barrier ordered before it
            __syncwarp();
            if (lane == 0 && sig_pending) {
                release_fence();
                atomicAdd(sig_ptr, sig_val);
            }
            sig_pending = false;
        };

        while (consumed < issued) {
            if (c_left == 0) {
                // ---- next chunk (= one piece of one unit) ----
                __syncwarp();
                const int4 *slot = ring[warp][ring_r & (kRing - 1)];
                const int4 a = slot[0], b = slot[1], c = slot[2];
                const int staged = slot[3].x;
                c_app = slot[3].y;
                c_part = b.x;
                c_row = layer_row + b.y - a.y * kTileTokens;  // pool row of the unit's first token
                ++ring_r;
                cu = a.x;
                ct = a.y;
                c_left = a.z;
                piece = a.w;
                c_req = b.z;
                c_range = b.w;
                c_cnt = c.x;
                c_np = c.z;
                c_J = c.w;
                if (staged) {
                    asm volatile("cp.async.wait_all;" ::: "memory");
                    __syncwarp();
                    const uint32_t qa = q_s + tq * kQRowBytes + hp * 2;
#pragma unroll
                    for (int ks = 0; ks < 8; ++ks) {
                        uint32_t x0 = 0u, x1 = 0u;
                        if (tq < G) {
                            asm volatile("ld.shared.b32 %0, [%1];" : "=r"(x0) : "r"(qa + ks * 32));
                            asm volatile("ld.shared.b32 %0, [%1];" : "=r"(x1) : "r"(qa + ks * 32 + 16));
                        }
                        qb[ks][0] = x0;
                        qb[ks][1] = x1;
                    }
                    __syncwarp();  // every lane has its fragments: the slot may be refilled
                    q_busy = false;
                } else {
                    const __half *qg = p.q + ((size_t)c_req * d.Hq + (size_t)(cu % Hkv) * G + tq) * kHeadDim + hp;
#pragma unroll
                    for (int ks = 0; ks < 8; ++ks) {
                        qb[ks][0] = tq < G ? __ldg(reinterpret_cast<const uint32_t *>(qg + ks * 16)) : 0u;
                        qb[ks][1] = tq < G ? __ldg(reinterpret_cast<const uint32_t *>(qg + ks * 16 + 8)) : 0u;
                    }
                }
                m0 = m1 = -INFINITY;
                l0 = l1 = 0.f;
#pragma unroll
                for (int n = 0; n < 8; ++n) o[n][0] = o[n][1] = o[n][2] = o[n][3] = 0.f;
            }
            const int stage = consumed % STAGES;
            const uint32_t sb = wbase + stage * kStageBytes;
            mbar_wait(bar0 + 8 * stage, (consumed / STAGES) & 1);
            if (d.diag && consumed == 0) t_first = global_ns();

            const int valid = min(kTileTokens, c_cnt - ct * kTileTokens);
            const bool patched = c_app >= 0 && ct == (c_app >> 4);
            const bool ragged = valid < kTileTokens || patched;
            if (patched) {
                // (a2) this tile receives the step's new token: lanes 0..15 carry the 16-byte chunks of its K row,
                // lanes 16..31 those of its V row -- into the pool (what kf_kv_append does) and into this tile's
                // shared-memory copy, whatever the TMA load found at that position
                const int row = c_app & 15, is_v = lane >> 4, ch = lane & 15;
                const int4 val = __ldg(reinterpret_cast<const int4 *>((is_v ? p.v_new : p.k_new) +
                                                                      ((size_t)c_req * Hkv + cu % Hkv) * kHeadDim) + ch);
                const uint32_t a = sb + (2 * is_v + (ch >> 3)) * kSubTile + row * 128 + (((ch & 7) ^ (row & 7)) << 4);
                asm volatile("st.shared.v4.b32 [%0], {%1,%2,%3,%4};" ::"r"(a), "r"(val.x), "r"(val.y), "r"(val.z), "r"(val.w) : "memory");
                unsigned char *dst = d.pool[c_part] + (is_v ? d.v_off : 0) + ((size_t)c_row + c_app) * (kHeadDim * 2) + ch * 16;
                *reinterpret_cast<int4 *>(dst) = val;
                __syncwarp();
            }
            if (valid < kTileTokens) {
                // rows >= valid hold whatever the pool holds (maybe NaN patterns): zero them in V so 0 * V = 0
                for (int idx = lane; idx < (kTileTokens - valid) * 16; idx += 32) {
                    const int row = valid + (idx >> 4), rem = idx & 15;
                    const uint32_t a = sb + 2 * kSubTile + (rem >> 3) * kSubTile + row * 128 + (rem & 7) * 16;
                    asm volatile("st.shared.v4.b32 [%0], {%1,%1,%1,%1};" ::"r"(a), "r"(0u) : "memory");
                }
                __syncwarp();
            }

            // ---- S^T = K Q^T : 16 tokens x 8 heads; two accumulators (even / odd k-steps) halve the HMMA chain ----
            float sa[4] = {0.f, 0.f, 0.f, 0.f}, sc[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
            for (int ks = 0; ks < 8; ++ks) {
                uint32_t a0, a1, a2, a3;
                ldsm_x4(sb + (ks >> 2) * kSubTile + ka_row + (((((ks & 3) << 1) + ka_kc) ^ l7) << 4), a0, a1, a2, a3);
                mma16816(ks & 1 ? sc : sa, a0, a1, a2, a3, qb[ks][0], qb[ks][1]);
            }

            // ---- online softmax, base 2, per head column; the reference maximum is LAZY: it only moves (and the
            //      accumulators are only rescaled) when a score exceeds it by more than 2^kLazy, so the cross-lane
            //      maximum and the rescale cost nothing on most tiles; p = exp2(s - m + kPShift) <= 2^(kLazy + kPShift)
#pragma unroll
            for (int i = 0; i < 4; ++i) sc[i] = (sa[i] + sc[i]) * d.scale_log2;
            if (ragged) {
                if (tq >= valid) sc[0] = sc[1] = -INFINITY;
                if (tq + 8 >= valid) sc[2] = sc[3] = -INFINITY;
            }
            const float t0 = fmaxf(sc[0], sc[2]), t1 = fmaxf(sc[1], sc[3]);
            if (__any_sync(0xffffffffu, t0 > m0 + kLazy || t1 > m1 + kLazy)) {
                float x0 = t0, x1 = t1;
#pragma unroll
                for (int sh = 4; sh < 32; sh <<= 1) {
                    x0 = fmaxf(x0, __shfl_xor_sync(0xffffffffu, x0, sh));
                    x1 = fmaxf(x1, __shfl_xor_sync(0xffffffffu, x1, sh));
                }
                const float n0 = fmaxf(m0, x0), n1 = fmaxf(m1, x1);
                const float al0 = fast_exp2(m0 - n0), al1 = fast_exp2(m1 - n1);
                m0 = n0;
                m1 = n1;
                l0 *= al0;
                l1 *= al1;
#pragma unroll
                for (int n = 0; n < 8; ++n) {
                    o[n][0] *= al0;
                    o[n][1] *= al1;
                    o[n][2] *= al0;
                    o[n][3] *= al1;
                }
            }
            const float f0 = m0 - kPShift, f1 = m1 - kPShift;
            const float p0 = fast_exp2(sc[0] - f0), p1 = fast_exp2(sc[1] - f1);
            const float p2 = fast_exp2(sc[2] - f0), p3 = fast_exp2(sc[3] - f1);
            l0 += p0 + p2;
            l1 += p1 + p3;
            // P (tokens x heads, C-fragment layout) -> B fragments of P^T... of the product O^T = V^T P: movmatrix
            const uint32_t pb0 = movmatrix_trans(pack_half2(p0, p1)), pb1 = movmatrix_trans(pack_half2(p2, p3));

            // ---- O^T += V^T P : 128 dims x 8 heads -----------------------------------------------------------
#pragma unroll
            for (int mt = 0; mt < 8; ++mt) {
                uint32_t a0, a1, a2, a3;
                ldsm_x4_trans(sb + (2 + (mt >> 2)) * kSubTile + va_row + (((((mt & 3) << 1) + va_dc) ^ l7) << 4), a0, a1, a2,
                              a3);
                mma16816(o[mt], a0, a1, a2, a3, pb0, pb1);
            }

            // the zero-stores above went through the generic proxy: every lane that wrote orders them before the
            // async-proxy (TMA) refill of this stage, then the barrier, then the elected lane issues
            if (ragged) asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            __syncwarp();  // every lane is done reading this stage
            try_issue();   // refills this very stage: issued == consumed + STAGES whenever it issues
            if (sig_pending) flush_signal();

            ++consumed;
            ++ct;
            --c_left;
            if (c_left == 0) {
                // ---- end of the piece: emit its partial (o, lse) -------------------------------------------
                const int g = cu % Hkv;
                float lt0 = l0, lt1 = l1;
#pragma unroll
                for (int sh = 4; sh < 32; sh <<= 1) {
                    lt0 += __shfl_xor_sync(0xffffffffu, lt0, sh);
                    lt1 += __shfl_xor_sync(0xffffffffu, lt1, sh);
                }
                PieceDest pd;
                pd.o2 = nullptr;
                pd.lse2 = nullptr;
                if (c_np == 1) {
                    const size_t row = range_row(d, c_req, c_range, g * G);
                    pd.o = p.o_part + row * kHeadDim;
                    pd.lse = p.lse_part + row;
                    if (p.fused && c_J == 1) {  // this piece is the final result
                        const size_t frow = (size_t)c_req * d.Hq + g * G;
                        pd.o2 = p.o + frow * kHeadDim;
                        pd.lse2 = p.lse + frow;
                    }
                } else {
                    pd.o = d.piece_o + (size_t)piece * G * kHeadDim;
                    pd.lse = d.piece_lse + (size_t)piece * G;
                }
                const float inv0 = 1.f / lt0, inv1 = 1.f / lt1;
                const float lse0 = (m0 + log2f(lt0) - kPShift) * 0.6931471805599453f;
                const float lse1 = (m1 + log2f(lt1) - kPShift) * 0.6931471805599453f;
#pragma unroll
                for (int e = 0; e < 2; ++e) {
                    if (hp + e < G) {
                        const float inv = e ? inv1 : inv0;
                        float *dst = pd.o + (size_t)(hp + e) * kHeadDim + tq;
#pragma unroll
                        for (int n = 0; n < 8; ++n) {
                            dst[16 * n] = o[n][e] * inv;
                            dst[16 * n + 8] = o[n][2 + e] * inv;
                        }
                        if (tq == 0) pd.lse[hp + e] = e ? lse1 : lse0;
                        if (pd.o2) {
                            float *dst2 = pd.o2 + (size_t)(hp + e) * kHeadDim + tq;
#pragma unroll
                            for (int n = 0; n < 8; ++n) {
                                dst2[16 * n] = o[n][e] * inv;
                                dst2[16 * n + 8] = o[n][2 + e] * inv;
                            }
                            if (tq == 0) pd.lse2[hp + e] = e ? lse1 : lse0;
                        }
                    }
                }
                if (p.fused) {
                    // publish: pieces of a cut unit count on the unit, a whole range partial counts G heads on its group
                    if (c_np > 1) {
                        sig_ptr = &ctr.unit[cu];
                        sig_val = 1;
                        sig_pending = true;
                    } else if (c_J > 1) {
                        sig_ptr = &ctr.group[c_req * Hkv + g];
                        sig_val = G;
                        sig_pending = true;
                    }
                    if (sig_pending && consumed == issued) flush_signal();  // nothing left to hide it behind
                }
            }
        }
        if (sig_pending) flush_signal();
        if (d.diag) t_stream = global_ns();
    } else {
        ctr = launch_prologue(d, w, W, lane);
    }
    if (p.fused) merge_phase(p, ctr, W, lane, m_first);

    if (d.diag && lane == 0) {
        // diagnostics: {SM | stream-end offset << 8, start, first tile ready (0 = no chunk), end}
        d.worker_times[4 * w] = sm_id() | ((w < n_chunks ? t_stream - t_start : 0) << 8);
        d.worker_times[4 * w + 1] = t_start;
        d.worker_times[4 * w + 2] = t_first;
        d.worker_times[4 * w + 3] = global_ns();
    }
    launch_epilogue(d, W, lane, p.commit);
}

template <int WARPS, int STAGES>
static int setup_one() {
    const int smem = WARPS * STAGES * kStageBytes + 1024;
    return cudaFuncSetAttribute(attend_tma_kernel<WARPS, STAGES>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem) ==
                   cudaSuccess
               ? 0
               : KF_ECUDA;
}

template <int WARPS, int STAGES>
static int launch_one(const AttendParams &p, int n_ctas, cudaStream_t s) {
    const int smem = WARPS * STAGES * kStageBytes + 1024;
    // Cooperative launch: the fused merge makes workers wait for partials of other workers of the SAME launch, so
    // every CTA must be resident at once.  The grid never exceeds the SM count, but only a cooperative launch makes
    // the hardware gang-schedule it when other work shares the GPU (it fails instead of deadlocking otherwise).
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(n_ctas);
    cfg.blockDim = dim3(WARPS * 32);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = s;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeCooperative;
    attr[0].val.cooperative = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    cudaLaunchKernelEx(&cfg, attend_tma_kernel<WARPS, STAGES>, p);
    return 1;
}

#define KF_TMA_SHAPES(X) X(4, 2) X(4, 3) X(4, 4) X(4, 5) X(4, 6) X(8, 2) X(8, 3) X(12, 2) X(16, 1)

bool attend_tma_shape_ok(int warps, int stages) {
#define X(Wp, St) \
    if (warps == Wp && stages == St) return true;
    KF_TMA_SHAPES(X)
#undef X
    return false;
}

int attend_tma_setup() {
    int rc = 0;
#define X(Wp, St) rc |= setup_one<Wp, St>();
    KF_TMA_SHAPES(X)
#undef X
    return rc == 0 ? 0 : KF_ECUDA;
}

int launch_attend_tma(const AttendParams &p, int n_ctas, cudaStream_t s) {
#define X(Wp, St) \
    if (p.d.warps_per_cta == Wp && p.d.stages == St) return launch_one<Wp, St>(p, n_ctas, s);
    KF_TMA_SHAPES(X)
#undef X
    return KF_EINVAL;
}

}  // namespace kf
