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

// Release side of the partial hand-off: orders this thread's stores of a partial before the counter increment that
// publishes it.  acq_rel at gpu scope is all the message-passing pattern needs; __threadfence() is the sequentially
// consistent fence (MEMBAR.SC + L1 invalidate), several hundred ns more per hop of the merge tail.
__device__ __forceinline__ void release_fence() { asm volatile("fence.acq_rel.gpu;" ::: "memory"); }

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

// A unit cut into several pieces keeps them in the piece buffer at their global piece index (consecutive for
// one unit, tile order); a unit that is one piece writes its range partial directly.
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
        pd.o = d.piece_o + (size_t)piece * d.G * kHeadDim;
        pd.lse = d.piece_lse + (size_t)piece * d.G;
    }
    return pd;
}

// One warp merges n partials of ONE query head: partial j has its o row at src_o + j*o_stride and its lse at
// src_lse[j*lse_stride].  Lane l owns columns [4l, 4l+4).  Loads bypass L1 (__ldcg): the partials were written
// by other SMs, possibly in this same launch.  The lse values and the first batch of rows are requested before
// anything is computed, so a merge of <= 16 partials costs one L2 round trip.  The accumulation order is j
// ascending, whoever calls this, so every path (fused tail, stand-alone kernels) produces the same bits.
constexpr int kMergeBatch = 32;

// __noinline__: this code runs once or twice per worker at the very end of a launch, with a cold instruction
// cache -- one shared copy of it costs far fewer instruction-fetch misses than an inlined copy per call site.
static __device__ __noinline__ void merge_rows(const float *src_o, size_t o_stride, const float *src_lse,
                                           size_t lse_stride, int n, float *dst_o, float *dst_lse, float *dst2_o,
                                           float *dst2_lse, int lane) {
    float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
    float lse = -INFINITY;
    if (n == 1) {  // exact copy
        lse = __ldcg(src_lse);
        acc = __ldcg(reinterpret_cast<const float4 *>(src_o) + lane);
    } else {
        // lse values: lane l caches partials l, l+32, l+64, l+96; beyond that they are re-read
        float lc[4];
#pragma unroll
        for (int c = 0; c < 4; ++c) {
            const int j = lane + 32 * c;
            lc[c] = j < n ? __ldcg(src_lse + (size_t)j * lse_stride) : -INFINITY;
        }
        float4 v[kMergeBatch];
#pragma unroll
        for (int k = 0; k < kMergeBatch; ++k)
            v[k] = k < n ? __ldcg(reinterpret_cast<const float4 *>(src_o + (size_t)k * o_stride) + lane)
                         : make_float4(0.f, 0.f, 0.f, 0.f);
        float M = fmaxf(fmaxf(lc[0], lc[1]), fmaxf(lc[2], lc[3]));
        for (int j = lane + 128; j < n; j += 32) M = fmaxf(M, __ldcg(src_lse + (size_t)j * lse_stride));
        M = warp_max(M);
        if (M != -INFINITY) {
            float sum = 0.f;
#pragma unroll
            for (int c = 0; c < 4; ++c) sum += expf(lc[c] - M);  // exp(-inf) = 0 for the padding
            for (int j = lane + 128; j < n; j += 32) sum += expf(__ldcg(src_lse + (size_t)j * lse_stride) - M);
            sum = warp_sum(sum);
            lse = M + logf(sum);
        }
        for (int jb = 0; jb < n; jb += 32) {
            float wl = 0.f;  // this lane's weight of partial jb + lane
            if (jb + lane < n && lse != -INFINITY) {
                const int c = jb >> 5;
                const float lj = c == 0 ? lc[0] : c == 1 ? lc[1] : c == 2 ? lc[2] : c == 3 ? lc[3]
                                        : __ldcg(src_lse + (size_t)(jb + lane) * lse_stride);
                wl = expf(lj - lse);
            }
            const int cnt = min(32, n - jb);
            for (int j0 = 0; j0 < cnt; j0 += kMergeBatch) {
                if (jb + j0 > 0) {
#pragma unroll
                    for (int k = 0; k < kMergeBatch; ++k)
                        v[k] = j0 + k < cnt ? __ldcg(reinterpret_cast<const float4 *>(
                                                         src_o + (size_t)(jb + j0 + k) * o_stride) + lane)
                                            : make_float4(0.f, 0.f, 0.f, 0.f);
                }
#pragma unroll
                for (int k = 0; k < kMergeBatch; ++k) {
                    const float w = __shfl_sync(0xffffffffu, wl, (j0 + k) & 31);
                    if (j0 + k < cnt && w != 0.f) {  // w == 0 (lse_j = -inf): ignore its o_j, whatever it holds
                        acc.x = fmaf(w, v[k].x, acc.x);
                        acc.y = fmaf(w, v[k].y, acc.y);
                        acc.z = fmaf(w, v[k].z, acc.z);
                        acc.w = fmaf(w, v[k].w, acc.w);
                    }
                }
            }
        }
    }
    reinterpret_cast<float4 *>(dst_o)[lane] = acc;
    if (lane == 0) *dst_lse = lse;
    if (dst2_o) {
        reinterpret_cast<float4 *>(dst2_o)[lane] = acc;
        if (lane == 0) *dst2_lse = lse;
    }
}

// The same reduction for up to HC = min(8, 32 / N2) CONSECUTIVE query heads at once, n <= N2 partials each (N2 a power
// of two): all HC * N2 <= 32 rows are requested before anything is computed, so a warp merges HC heads in the ONE L2
// round trip that merge_rows spends on one.  The fused merge tail is a chain of dependent round trips per task (unit
// record, counter, rows, store, fence, signal); with G = 8 heads and 4 ranges per request it was 25 us of a 645 us
// launch at one head per task.  Head h reads src_o + h * 128 / src_lse + h and writes dst + h * 128 / dst_lse + h.
// Same arithmetic, same order (j ascending; the lse sum is the same shuffle tree, restricted to the N2 lanes of the
// head), so the result is bit-identical to merge_rows.
template <int N2>
static __device__ __noinline__ void merge_heads(const float *src_o, size_t o_stride, const float *src_lse, size_t lse_stride,
                                            int n, int heads, float *dst_o, float *dst_lse, float *dst2_o,
                                            float *dst2_lse, int lane) {
    constexpr int HC = 32 / N2 < 8 ? 32 / N2 : 8;
    const int hl = lane / N2, jl = lane % N2;  // this lane's (head, partial) in the lse phase
    const bool have = hl < heads && hl < HC && jl < n;
    const float lj = have ? __ldcg(src_lse + hl + (size_t)jl * lse_stride) : -INFINITY;
    float4 v[HC * N2];
#pragma unroll
    for (int k = 0; k < HC * N2; ++k) {
        const int h = k / N2, j = k % N2;
        v[k] = (h < heads && j < n)
                   ? __ldcg(reinterpret_cast<const float4 *>(src_o + (size_t)h * kHeadDim + (size_t)j * o_stride) + lane)
                   : make_float4(0.f, 0.f, 0.f, 0.f);
    }
    float M = lj;
#pragma unroll
    for (int o = N2 / 2; o > 0; o >>= 1) M = fmaxf(M, __shfl_xor_sync(0xffffffffu, M, o));
    float sum = M != -INFINITY ? expf(lj - M) : 0.f;  // exp(-inf) = 0 for the padding
#pragma unroll
    for (int o = N2 / 2; o > 0; o >>= 1) sum += __shfl_xor_sync(0xffffffffu, sum, o);
    const float lse = M != -INFINITY ? M + logf(sum) : -INFINITY;
    const float wl = (have && lse != -INFINITY) ? expf(lj - lse) : 0.f;
    float4 acc[HC];
#pragma unroll
    for (int h = 0; h < HC; ++h) acc[h] = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
    for (int k = 0; k < HC * N2; ++k) {
        const int h = k / N2, j = k % N2;
        const float w = __shfl_sync(0xffffffffu, wl, k);
        if (h < heads && j < n && w != 0.f) {  // w == 0 (lse_j = -inf): ignore its o_j, whatever it holds
            acc[h].x = fmaf(w, v[k].x, acc[h].x);
            acc[h].y = fmaf(w, v[k].y, acc[h].y);
            acc[h].z = fmaf(w, v[k].z, acc[h].z);
            acc[h].w = fmaf(w, v[k].w, acc[h].w);
        }
    }
#pragma unroll
    for (int h = 0; h < HC; ++h) {
        if (h < heads) {
            reinterpret_cast<float4 *>(dst_o + (size_t)h * kHeadDim)[lane] = acc[h];
            if (dst2_o) reinterpret_cast<float4 *>(dst2_o + (size_t)h * kHeadDim)[lane] = acc[h];
        }
    }
    if (have && jl == 0) {
        dst_lse[hl] = lse;
        if (dst2_o) dst2_lse[hl] = lse;
    }
}

// heads merged per task when no head has more than n_max partials; the padded partial count N2 that goes with it
__device__ __forceinline__ int merge_n2(int n_max) { return n_max <= 8 ? 8 : n_max <= 16 ? 16 : 32; }
__device__ __forceinline__ int merge_hc(int n2, int G) { return min(G, 32 / n2); }  // 4, 2 or 1 heads per task

// `heads` consecutive heads, n partials each: one merge_heads call when n fits its N2, else head by head
__device__ __forceinline__ void merge_group(int n2, const float *src_o, size_t o_stride, const float *src_lse,
                                            size_t lse_stride, int n, int heads, float *dst_o, float *dst_lse,
                                            float *dst2_o, float *dst2_lse, int lane) {
    if (n > n2 || n2 > 16) {  // more partials than one round trip of merge_heads holds: head by head
        for (int h = 0; h < heads; ++h)
            merge_rows(src_o + (size_t)h * kHeadDim, o_stride, src_lse + h, lse_stride, n, dst_o + (size_t)h * kHeadDim,
                       dst_lse + h, dst2_o ? dst2_o + (size_t)h * kHeadDim : nullptr, dst2_o ? dst2_lse + h : nullptr, lane);
        return;
    }
    // two instantiations only: this code runs at the very end of a launch with a cold instruction cache
    if (n2 <= 8)
        merge_heads<8>(src_o, o_stride, src_lse, lse_stride, n, heads, dst_o, dst_lse, dst2_o, dst2_lse, lane);
    else
        merge_heads<16>(src_o, o_stride, src_lse, lse_stride, n, heads, dst_o, dst_lse, dst2_o, dst2_lse, lane);
}

__device__ __forceinline__ Unit load_unit_g(const Unit *units, int u) {
    const int4 *q = reinterpret_cast<const int4 *>(units + u);
    const int4 a = __ldg(q), b = __ldg(q + 1);
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

// merge the pieces of unit u, query head i of its group, into the range partial (and into the final output if
// the request has a single range and `to_final`)
__device__ __forceinline__ void merge_unit_head(const AttendParams &p, const Unit &un, int g, int i, bool to_final,
                                                int lane) {
    const Dev &d = p.d;
    const int head = g * d.G + i;
    const size_t row = range_row(d, un.req, un.range, head);
    float *o2 = nullptr, *l2 = nullptr;
    if (to_final && d.scratch[un.req] == 1) {
        const size_t frow = (size_t)un.req * d.Hq + head;
        o2 = p.o + frow * kHeadDim;
        l2 = p.lse + frow;
    }
    merge_rows(d.piece_o + ((size_t)un.piece_begin * d.G + i) * kHeadDim, (size_t)d.G * kHeadDim,
               d.piece_lse + (size_t)un.piece_begin * d.G + i, d.G, un.n_pieces, p.o_part + row * kHeadDim,
               p.lse_part + row, o2, l2, lane);
}

// merge the J range partials of (req, query head h) into the final output
__device__ __forceinline__ void merge_request_head(const Dev &d, const float *o_part, const float *lse_part,
                                                   float *o, float *lse, int req, int h, int J, int lane) {
    const size_t row = range_row(d, req, 0, h);
    const size_t frow = (size_t)req * d.Hq + h;
    merge_rows(o_part + row * kHeadDim, (size_t)d.Hq * kHeadDim, lse_part + row, d.Hq, J, o + frow * kHeadDim,
               lse + frow, nullptr, nullptr, lane);
}

// ---- scheduler words and completion counters of one attend launch -----------------------------------------
// sched[0] chunk ticket, [1] finished workers, [2] merge-task ticket, [3] unused, [4] epoch.
// The completion counters are double-buffered by launch parity: a launch counts in buffer (epoch & 1) and
// zeroes the other one for the next launch, so nothing has to be reset on the critical path.
struct Counters {
    int32_t *unit;   // [U]      pieces of unit u finished
    int32_t *group;  // [B*Hkv]  range partials of (request, kv head) finished, counted per query head
};

__device__ __forceinline__ Counters launch_prologue(const Dev &d, int w, int W, int lane) {
    const int epoch = *reinterpret_cast<volatile int32_t *>(d.sched + 4);
    const int Ucap = d.B * d.Jmax * d.Hkv, Gcap = d.B * d.Hkv;
    Counters c, o;
    c.unit = d.unit_counter + (size_t)(epoch & 1) * Ucap;
    c.group = d.group_counter + (size_t)(epoch & 1) * Gcap;
    o.unit = d.unit_counter + (size_t)((epoch + 1) & 1) * Ucap;
    o.group = d.group_counter + (size_t)((epoch + 1) & 1) * Gcap;
    for (int i = w * 32 + lane; i < Ucap; i += W * 32) o.unit[i] = 0;
    for (int i = w * 32 + lane; i < Gcap; i += W * 32) o.group[i] = 0;
    return c;
}

// the last worker to finish rewinds the tickets and flips the epoch for the next launch; with `commit` (the last
// layer-step of a static step graph) it also performs the step commit a5 -- len_r += 1 -- which no worker of this
// launch reads any more: each of them read len before its own release below
__device__ __forceinline__ void launch_epilogue(const Dev &d, int W, int lane, int commit = 0) {
    int last = 0;
    __syncwarp();  // the other lanes' stores (merge outputs) and loads (len) are ordered before lane 0's release
    if (lane == 0) {
        release_fence();
        const int old = atomicAdd(d.sched + 1, 1);
        if (old == W - 1) {
            d.sched[0] = 0;
            d.sched[1] = 0;
            d.sched[2] = 0;
            d.sched[3] = 0;
            d.sched[4] = d.sched[4] + 1;
            last = 1;
        }
    }
    if (commit) {
        last = __shfl_sync(0xffffffffu, last, 0);
        if (last) {
            asm volatile("fence.acq_rel.gpu;" ::: "memory");  // acquire side: every worker's reads of len are done
            for (int r = lane; r < d.B; r += 32)
                if (commits(d, r)) d.len[r] += 1;
        }
    }
}

// called by the whole warp after it has written the partial of one piece of unit u (fused mode)
__device__ __forceinline__ void piece_done(const AttendParams &p, const Counters &c, int u, const Unit &un, int g,
                                           int lane) {
    const Dev &d = p.d;
    // release: barrier first, THEN lane 0 fences and publishes -- the fence is cumulative over the stores of the
    // other lanes that the barrier ordered before it (a fence in every lane before the barrier would not cover them)
    __syncwarp();
    if (lane == 0) {
        release_fence();
        if (un.n_pieces > 1)
            atomicAdd(&c.unit[u], 1);
        else if (d.scratch[un.req] > 1)
            atomicAdd(&c.group[un.req * d.Hkv + g], d.G);  // the range partial of all G heads is complete
    }
}

__device__ __forceinline__ void wait_counter(const int32_t *ctr, int target, int lane) {
    if (lane == 0) {
        int v;
        for (;;) {
            asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(ctr) : "memory");
            if (v >= target) break;
            __nanosleep(64);
        }
    }
    __syncwarp();  // lane 0's acquire happens-before the other lanes' loads of the partials (L2 loads, __ldcg)
}

// Fused tail: once the chunk list is exhausted every worker turns into a merge worker.
// One ticket stream covers both levels: tasks [0, nA) = (unit, chunk of heads of its group): pieces -> range partial;
// tasks [nA, total) = (request, kv head, chunk of heads): range partials -> output.  A chunk holds as many heads as
// fit one round trip of merge_heads, given the launch's largest piece count / range count (plan header).  A task
// waits until its inputs are
// complete; its producers are either chunks (taken by resident workers of this launch: the grid never exceeds
// the SM count) or tasks with a LOWER ticket, and every worker serves its tickets in ascending order, so the
// waits cannot deadlock.  Tickets are taken in batches (bounded atomic traffic on one word) and the next batch
// is requested before the current one is processed, which keeps the atomic's round trip off the critical path.
// `first` is lane 0's pre-taken first ticket (merge_first_ticket) or -1.
struct MergeShape {
    int n2A, hcA, caA;  // A level (pieces -> range partial): padded partials per head, heads per task, tasks per unit
    int n2B, hcB, caB;  // B level (range partials -> output): ditto per (request, kv head)
    int nA, total;
};
__device__ __forceinline__ MergeShape merge_shape(const Dev &d) {
    MergeShape m;
    // ONE N2 for both levels: the tail of a launch runs this code with a cold instruction cache, and a second
    // instantiation of merge_heads costs more in instruction fetches than the heads it would add per task
    m.n2A = m.n2B = merge_n2(max(__ldg(&d.plan->max_unit_pieces), __ldg(&d.plan->max_J)));
    m.hcA = merge_hc(m.n2A, d.G);
    m.caA = (d.G + m.hcA - 1) / m.hcA;
    m.hcB = merge_hc(m.n2B, d.G);
    m.caB = (d.G + m.hcB - 1) / m.hcB;
    m.nA = __ldg(&d.plan->n_units) * m.caA;
    m.total = m.nA + d.B * d.Hkv * m.caB;
    return m;
}
__device__ __forceinline__ int merge_batch(const Dev &d, int W) {
    return max(1, merge_shape(d).total / (4 * W));
}
__device__ __forceinline__ int merge_first_ticket(const Dev &d, int W) {  // call from ONE lane
    return atomicAdd(d.sched + 2, merge_batch(d, W));
}

__device__ __forceinline__ void merge_phase(const AttendParams &p, const Counters &c, int W, int lane, int first = -1) {
    const Dev &d = p.d;
    const int G = d.G, Hkv = d.Hkv;
    const MergeShape ms = merge_shape(d);
    const int batch = max(1, ms.total / (4 * W));
    int next = first;
    if (lane == 0 && next < 0) next = atomicAdd(d.sched + 2, batch);
    for (;;) {
        const int t0 = __shfl_sync(0xffffffffu, next, 0);
        if (t0 >= ms.total) break;
        if (lane == 0) next = atomicAdd(d.sched + 2, batch);  // in flight while this batch is processed
        const int t1 = min(ms.total, t0 + batch);
        for (int t = t0; t < t1; ++t) {
            if (t < ms.nA) {
                // task = (unit, chunk of hcA heads of its group): pieces -> range partial (and the output if J_r = 1)
                const int u = t / ms.caA, i0 = (t - u * ms.caA) * ms.hcA;
                const int heads = min(ms.hcA, G - i0);
                const Unit un = load_unit_g(d.units, u);
                if (un.n_pieces <= 1) continue;
                const int g = u % Hkv, head = g * G + i0;
                const int J = d.scratch[un.req];
                wait_counter(&c.unit[u], un.n_pieces, lane);
                const size_t row = range_row(d, un.req, un.range, head);
                const size_t frow = (size_t)un.req * d.Hq + head;
                merge_group(ms.n2A, d.piece_o + ((size_t)un.piece_begin * G + i0) * kHeadDim, (size_t)G * kHeadDim,
                            d.piece_lse + (size_t)un.piece_begin * G + i0, G, un.n_pieces, heads,
                            p.o_part + row * kHeadDim, p.lse_part + row, J == 1 ? p.o + frow * kHeadDim : nullptr,
                            J == 1 ? p.lse + frow : nullptr, lane);
                if (J > 1) {
                    __syncwarp();
                    if (lane == 0) {
                        release_fence();
                        atomicAdd(&c.group[un.req * Hkv + g], heads);
                    }
                }
            } else {
                // task = (request, kv head, chunk of hcB heads): range partials -> output
                const int tb = t - ms.nA;
                const int grp = tb / ms.caB, i0 = (tb - grp * ms.caB) * ms.hcB;
                const int heads = min(ms.hcB, G - i0);
                const int req = grp / Hkv, g = grp - req * Hkv;
                const int J = d.scratch[req];  // 0 for closed requests
                if (J <= 1) continue;          // a single range: its partial was also written to the output
                wait_counter(&c.group[grp], J * G, lane);
                const int h = g * G + i0;
                const size_t row = range_row(d, req, 0, h);
                const size_t frow = (size_t)req * d.Hq + h;
                merge_group(ms.n2B, p.o_part + row * kHeadDim, (size_t)d.Hq * kHeadDim, p.lse_part + row, d.Hq, J, heads,
                            p.o + frow * kHeadDim, p.lse + frow, nullptr, nullptr, lane);
            }
        }
    }
}

}  // namespace kf
