// kf_api.cu -- the C ABI of libkflume (include/kflume.h): argument checking, workspace layout, TMA descriptor
// creation and kernel launches.  No arithmetic of the method happens on the host.
#include <cuda.h>
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <new>

#include "kf_ctx.h"

using namespace kf;

namespace kf {
int cuda_fail(kf_ctx *ctx, cudaError_t e) {
    if (ctx) snprintf(ctx->cuda_err, sizeof(ctx->cuda_err), "%s: %s", cudaGetErrorName(e), cudaGetErrorString(e));
    return KF_ECUDA;
}
// true if the GPU can dereference this host pointer as it is (pinned memory under unified addressing)
bool device_can_read(const void *host_ptr) {
    cudaPointerAttributes a;
    if (cudaPointerGetAttributes(&a, host_ptr) != cudaSuccess) {
        cudaGetLastError();
        return false;
    }
    return a.type == cudaMemoryTypeHost && a.devicePointer == host_ptr;
}
// device_can_read() with a small per-ctx cache: the pinned buffers of an end-to-end loop are the same few pointers
// every layer-step, and cudaPointerGetAttributes costs ~1 us each.  (A cached pointer is trusted for the lifetime of
// the ctx: un-pinning a buffer that is still in use is the caller's error either way.)
bool host_ptr_ok(kf_ctx *ctx, const void *p) {
    const size_t slot = ((uintptr_t)p >> 6) % kf_ctx::kPinnedCache;  // direct-mapped
    if (ctx->pinned[slot] == p) return true;
    if (!device_can_read(p)) return false;
    ctx->pinned[slot] = p;
    return true;
}
}  // namespace kf

namespace {

constexpr size_t kAlign = 256;
constexpr int kDefaultWarps = 8, kDefaultStages = 3;
constexpr int kDefaultFirstPct = 100, kDefaultDecayPct = 50;
constexpr int kDefaultPlanRefresh = 128;

size_t max_chunks_of(const kf_config *c) {
    return (size_t)c->max_requests * c->max_ranges_per_request * c->n_kv_heads + kChunkSlack;
}
inline size_t align_up(size_t x, size_t a = kAlign) { return (x + a - 1) / a * a; }

struct Layout {
    size_t len, n_ranges, route_part, route_slot, range_begin, redirect, rr_cursor, rr_last, req_active, active, part_tokens, part_tails, free_head, free_cnt, free_stack, error, plan, units, chunks, recs, plan_age, sched,
        scratch, unit_counter, group_counter, piece_o, piece_lse, range_o, range_lse, stage_q, stage_k, stage_v,
        stage_o, stage_lse, tmaps, gates, worker_times, total;
};

bool valid_config(const kf_config *c) {
    if (!c) return false;
    if (c->head_dim != kHeadDim) return false;
    if (c->n_q_heads < 1 || c->n_kv_heads < 1 || c->n_q_heads % c->n_kv_heads) return false;
    const int G = c->n_q_heads / c->n_kv_heads;
    if (G < 1 || G > kMaxGroup) return false;
    if (c->n_q_heads > 128) return false;
    if (c->n_layers < 1) return false;
    if (c->range_tokens < 1 || (c->range_tokens & (c->range_tokens - 1))) return false;
    if (c->n_partitions < 1 || c->n_partitions > kMaxPartitions) return false;
    if (c->max_requests < 1 || c->max_requests > 4096) return false;
    if (c->max_ranges_per_request < 1 || c->slots_per_partition < 1) return false;
    if (!(c->softmax_scale >= 0.f) || !isfinite(c->softmax_scale)) return false;
    if (c->attend_impl < KF_IMPL_AUTO || c->attend_impl > KF_IMPL_TMA) return false;
    if (c->min_tiles_per_worker < 0) return false;
    if (c->workers_per_sm != 0 && c->workers_per_sm != 4 && c->workers_per_sm != 8 && c->workers_per_sm != 12 &&
        c->workers_per_sm != 16)
        return false;
    if (c->pipeline_stages != 0 &&
        !attend_tma_shape_ok(c->workers_per_sm ? c->workers_per_sm : kDefaultWarps, c->pipeline_stages))
        return false;
    if (c->sched_first_pct < 0 || c->sched_first_pct > 100) return false;
    if (c->sched_decay_pct < 0 || c->sched_decay_pct > 99) return false;
    if (c->plan_refresh_steps < 0) return false;
    if (c->kv_l2_policy < 0 || c->kv_l2_policy > 2) return false;
    if (c->diagnostics < 0 || c->attend_sms < 0) return false;
    // rows of one K (or V) half-pool must fit the int32 TMA coordinate
    const double rows = (double)c->n_layers * c->slots_per_partition * c->n_kv_heads * c->range_tokens;
    if (rows >= 2147483647.0) return false;
    if ((double)c->max_requests * c->max_ranges_per_request * c->n_kv_heads >= 1e9) return false;
    return true;
}

Layout make_layout(const kf_config *c) {
    Layout L;
    const size_t B = c->max_requests, J = c->max_ranges_per_request, P = c->n_partitions, Hq = c->n_q_heads,
                 Hkv = c->n_kv_heads, G = Hq / Hkv, S = c->slots_per_partition;
    const size_t E = B * J, U = E * Hkv, max_piece_slots = max_chunks_of(c);
    size_t off = 0;
    auto take = [&](size_t bytes) {
        const size_t o = off;
        off = align_up(off + bytes);
        return o;
    };
    L.len = take(B * 4);
    L.n_ranges = take(B * 4);
    L.route_part = take(E * 4);
    L.route_slot = take(E * 4);
    L.range_begin = take(E * 4);
    L.redirect = take(P * 4);
    L.rr_cursor = take(4);
    L.rr_last = take(4);
    L.req_active = take(B * 4);
    L.active = take(P * 4);
    L.part_tokens = take(P * 8);
    L.part_tails = take(P * 4);
    L.free_head = take(P * 4);
    L.free_cnt = take(P * 4);
    L.free_stack = take(P * S * 4);
    L.error = take(4);
    L.plan = take(sizeof(PlanHeader));
    L.units = take(U * sizeof(Unit));
    L.chunks = take(max_piece_slots * sizeof(Chunk));
    L.recs = take(max_piece_slots * sizeof(ChunkRec));
    L.plan_age = take(4);
    L.sched = take(8 * 4);
    L.scratch = take((B + B + (B + 1) + E + (E + 1) + (E + 1) + 3 * ((size_t)kMaxLevels * E + 1)) * 4);
    L.unit_counter = take(2 * U * 4);        // double-buffered by launch parity
    L.group_counter = take(2 * B * Hkv * 4);
    L.piece_o = take(max_piece_slots * G * kHeadDim * 4);
    L.piece_lse = take(max_piece_slots * G * 4);
    L.range_o = take(E * Hq * kHeadDim * 4);
    L.range_lse = take(E * Hq * 4);
    L.stage_q = take(B * Hq * kHeadDim * 2);
    L.stage_k = take(B * Hkv * kHeadDim * 2);
    L.stage_v = take(B * Hkv * kHeadDim * 2);
    L.stage_o = take(B * Hq * kHeadDim * 4);
    L.stage_lse = take(B * Hq * 4);
    L.tmaps = take(P * 2 * 128);
    L.gates = take(((size_t)kMaxGraphLayerSteps + 1) * 4);  // + 1: the word kf_signal_roundtrip plays with
    L.worker_times = take((size_t)kMaxWorkers * 4 * 8);
    L.total = off;
    return L;
}

size_t half_pool_bytes(const kf_config *c) {
    return (size_t)c->n_layers * c->slots_per_partition * c->n_kv_heads * c->range_tokens * (size_t)(kHeadDim * 2);
}


// after a launch: count it, surface launch errors
int after_launch(kf_ctx *ctx, int n) {
    if (n < 0) return n;
    ctx->launches += n;
    const cudaError_t e = cudaPeekAtLastError();
    if (e != cudaSuccess) {
        cudaGetLastError();
        return cuda_fail(ctx, e);
    }
    return KF_OK;
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

// One 2-D map per partition and per K / V half: [rows][128] fp16, box 16 rows x 64 halfs, 128B swizzle.
int encode_tmaps(kf_ctx *ctx, void *const *pools) {
    void *fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    cudaError_t e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres);
    if (e != cudaSuccess) return cuda_fail(ctx, e);
    if (!fn || qres != cudaDriverEntryPointSuccess) {
        snprintf(ctx->cuda_err, sizeof(ctx->cuda_err), "cuTensorMapEncodeTiled entry point unavailable");
        return KF_ECUDA;
    }
    EncodeTiledFn encode = (EncodeTiledFn)fn;
    const kf_config &c = ctx->cfg;
    const cuuint64_t rows = (cuuint64_t)c.n_layers * c.slots_per_partition * c.n_kv_heads * c.range_tokens;
    alignas(64) CUtensorMap maps[2 * kMaxPartitions];
    for (int p = 0; p < c.n_partitions; ++p) {
        for (int v = 0; v < 2; ++v) {
            void *base = (unsigned char *)pools[p] + (v ? ctx->dev.v_off : 0);
            const cuuint64_t dims[2] = {(cuuint64_t)kHeadDim, rows};
            const cuuint64_t strides[1] = {(cuuint64_t)kHeadDim * 2};
            const cuuint32_t box[2] = {64, (cuuint32_t)kTileTokens};
            const cuuint32_t estr[2] = {1, 1};
            const CUresult r = encode(&maps[2 * p + v], CU_TENSOR_MAP_DATA_TYPE_FLOAT16, 2, base, dims, strides, box,
                                      estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                                      CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
            if (r != CUDA_SUCCESS) {
                snprintf(ctx->cuda_err, sizeof(ctx->cuda_err), "cuTensorMapEncodeTiled failed: CUresult %d", (int)r);
                return KF_ECUDA;
            }
        }
    }
    static_assert(sizeof(CUtensorMap) == 128, "tensor map stride");
    e = cudaMemcpy((void *)ctx->dev.tmaps, maps, (size_t)c.n_partitions * 2 * sizeof(CUtensorMap),
                   cudaMemcpyHostToDevice);
    if (e != cudaSuccess) return cuda_fail(ctx, e);
    return KF_OK;
}

int ensure_plan(kf_ctx *ctx, cudaStream_t s) {
    if (!ctx->plan_dirty) return KF_OK;
    const int rc = after_launch(ctx, launch_plan(ctx->dev, 0, s));
    if (rc == KF_OK) ctx->plan_dirty = false;
    return rc;
}

int run_attend(kf_ctx *ctx, const AttendParams &ap, cudaStream_t s) {
    if (ctx->impl == KF_IMPL_SIMPLE) return after_launch(ctx, launch_attend_simple(ap, ctx->n_ctas, s));
    return after_launch(ctx, launch_attend_tma(ap, ctx->n_ctas, s));
}

bool bad_layer(const kf_ctx *ctx, int layer) { return layer < 0 || layer >= ctx->cfg.n_layers; }

}  // namespace

extern "C" {

int kf_version(void) { return KF_VERSION; }

const char *kf_strerror(int code) {
    switch (code) {
        case KF_OK: return "ok";
        case KF_EINVAL: return "invalid argument";
        case KF_ESTATE: return "call not valid in this state";
        case KF_ENOSPC: return "no free KV slot / range entry";
        case KF_ECUDA: return "CUDA error";
        default: return "unknown error";
    }
}

const char *kf_last_cuda_error(const kf_ctx *ctx) { return ctx ? ctx->cuda_err : ""; }

size_t kf_pool_bytes(const kf_config *cfg) { return valid_config(cfg) ? 2 * half_pool_bytes(cfg) : 0; }

size_t kf_workspace_bytes(const kf_config *cfg) { return valid_config(cfg) ? make_layout(cfg).total : 0; }

size_t kf_pool_offset(const kf_config *c, int32_t layer, int32_t slot, int32_t kv_head, int32_t token, int32_t is_v) {
    if (!valid_config(c) || layer < 0 || layer >= c->n_layers || slot < 0 || slot >= c->slots_per_partition ||
        kv_head < 0 || kv_head >= c->n_kv_heads || token < 0 || token >= c->range_tokens)
        return (size_t)-1;
    const size_t row = (((size_t)layer * c->slots_per_partition + slot) * c->n_kv_heads + kv_head) * c->range_tokens + token;
    return row * (size_t)(kHeadDim * 2) + (is_v ? half_pool_bytes(c) : 0);
}

int kf_create(kf_ctx **out, const kf_config *cfg, void *const *pool_ptrs, void *workspace, size_t workspace_bytes) {
    if (!out) return KF_EINVAL;
    *out = nullptr;
    if (!valid_config(cfg) || !pool_ptrs || !workspace) return KF_EINVAL;
    const Layout L = make_layout(cfg);
    if (workspace_bytes < L.total || ((uintptr_t)workspace & (kAlign - 1))) return KF_EINVAL;
    for (int p = 0; p < cfg->n_partitions; ++p)
        if (!pool_ptrs[p] || ((uintptr_t)pool_ptrs[p] & 1023)) return KF_EINVAL;

    kf_ctx *ctx = new (std::nothrow) kf_ctx();
    if (!ctx) return KF_EINVAL;
    memset(ctx, 0, sizeof(*ctx));
    ctx->cfg = *cfg;
    *out = ctx;  // returned even on KF_ECUDA so that kf_last_cuda_error() can be read; caller destroys it

    int dev_id = 0;
    cudaError_t e = cudaGetDevice(&dev_id);
    if (e != cudaSuccess) return cuda_fail(ctx, e);
    cudaDeviceProp prop;
    e = cudaGetDeviceProperties(&prop, dev_id);
    if (e != cudaSuccess) return cuda_fail(ctx, e);
    ctx->sm_count = prop.multiProcessorCount;
    ctx->impl = cfg->attend_impl == KF_IMPL_AUTO ? KF_IMPL_TMA : cfg->attend_impl;
    // the CUDA-core kernel always runs 8 warps per CTA; the TMA kernel's shape is tunable
    const int warps = ctx->impl == KF_IMPL_SIMPLE ? kWarpsPerCta : (cfg->workers_per_sm ? cfg->workers_per_sm : kDefaultWarps);
    ctx->n_ctas = cfg->attend_sms > 0 && cfg->attend_sms < ctx->sm_count ? cfg->attend_sms : ctx->sm_count;
    if (ctx->n_ctas * warps > kMaxWorkers) ctx->n_ctas = kMaxWorkers / warps;
    ctx->plan_dirty = true;

    unsigned char *ws = (unsigned char *)workspace;
    e = cudaMemset(ws, 0, L.total);
    if (e != cudaSuccess) return cuda_fail(ctx, e);
    // len = -1 (closed), routes = -1 (unused)
    e = cudaMemset(ws + L.len, 0xFF, (size_t)cfg->max_requests * 4);
    if (e == cudaSuccess) e = cudaMemset(ws + L.route_part, 0xFF, (size_t)cfg->max_requests * cfg->max_ranges_per_request * 4);
    if (e == cudaSuccess) e = cudaMemset(ws + L.route_slot, 0xFF, (size_t)cfg->max_requests * cfg->max_ranges_per_request * 4);
    if (e == cudaSuccess) e = cudaMemset(ws + L.range_begin, 0xFF, (size_t)cfg->max_requests * cfg->max_ranges_per_request * 4);
    if (e != cudaSuccess) return cuda_fail(ctx, e);
    e = cudaMemset(ws + L.rr_last, 0xFF, 4);  // -1: nothing allocated yet
    if (e == cudaSuccess) {
        int32_t ones[kMaxPartitions];
        for (int p = 0; p < kMaxPartitions; ++p) ones[p] = 1;  // every partition starts active
        e = cudaMemcpy(ws + L.active, ones, (size_t)cfg->n_partitions * 4, cudaMemcpyHostToDevice);
    }
    if (e != cudaSuccess) return cuda_fail(ctx, e);
    const int32_t stale = kPlanStale;  // no plan yet: the first plan kernel builds one
    e = cudaMemcpy(ws + L.plan_age, &stale, 4, cudaMemcpyHostToDevice);
    if (e != cudaSuccess) return cuda_fail(ctx, e);

    Dev &d = ctx->dev;
    d.Hq = cfg->n_q_heads;
    d.Hkv = cfg->n_kv_heads;
    d.G = d.Hq / d.Hkv;
    d.L = cfg->n_layers;
    d.R = cfg->range_tokens;
    d.P = cfg->n_partitions;
    d.B = cfg->max_requests;
    d.Jmax = cfg->max_ranges_per_request;
    d.slots = cfg->slots_per_partition;
    d.max_workers = ctx->n_ctas * warps;
    d.min_tiles = cfg->min_tiles_per_worker;  // 0 = chosen by the plan kernel from the amount of work
    d.warps_per_cta = warps;
    d.stages = cfg->pipeline_stages ? cfg->pipeline_stages : kDefaultStages;
    d.max_chunks = (int32_t)max_chunks_of(cfg);
    d.l2_hint = cfg->kv_l2_policy == 2 ? 0 : 1;  // K/V is read once per launch: evict-first by default
    d.diag = cfg->diagnostics ? 1 : 0;
    d.plan_refresh = cfg->plan_refresh_steps > 0 ? cfg->plan_refresh_steps : kDefaultPlanRefresh;
    d.sched_first = 0.01f * (cfg->sched_first_pct ? cfg->sched_first_pct : kDefaultFirstPct);
    d.sched_decay = 0.01f * (cfg->sched_decay_pct ? cfg->sched_decay_pct : kDefaultDecayPct);
    const float scale = cfg->softmax_scale > 0.f ? cfg->softmax_scale : 1.0f / sqrtf((float)kHeadDim);
    d.scale_log2 = scale * 1.4426950408889634f;
    d.len = (int32_t *)(ws + L.len);
    d.n_ranges = (int32_t *)(ws + L.n_ranges);
    d.route_part = (int32_t *)(ws + L.route_part);
    d.route_slot = (int32_t *)(ws + L.route_slot);
    d.range_begin = (int32_t *)(ws + L.range_begin);
    d.redirect = (int32_t *)(ws + L.redirect);
    d.rr_cursor = (int32_t *)(ws + L.rr_cursor);
    d.rr_last = (int32_t *)(ws + L.rr_last);
    d.req_active = (int32_t *)(ws + L.req_active);
    d.active = (int32_t *)(ws + L.active);
    d.part_tokens = (long long *)(ws + L.part_tokens);
    d.part_tails = (int32_t *)(ws + L.part_tails);
    d.free_head = (int32_t *)(ws + L.free_head);
    d.free_cnt = (int32_t *)(ws + L.free_cnt);
    d.free_stack = (int32_t *)(ws + L.free_stack);
    d.error = (int32_t *)(ws + L.error);
    d.plan = (PlanHeader *)(ws + L.plan);
    d.units = (Unit *)(ws + L.units);
    d.chunks = (Chunk *)(ws + L.chunks);
    d.recs = (ChunkRec *)(ws + L.recs);
    d.plan_age = (int32_t *)(ws + L.plan_age);
    d.sched = (int32_t *)(ws + L.sched);
    d.scratch = (int32_t *)(ws + L.scratch);
    d.unit_counter = (int32_t *)(ws + L.unit_counter);
    d.group_counter = (int32_t *)(ws + L.group_counter);
    d.piece_o = (float *)(ws + L.piece_o);
    d.piece_lse = (float *)(ws + L.piece_lse);
    d.range_o = (float *)(ws + L.range_o);
    d.range_lse = (float *)(ws + L.range_lse);
    d.stage_q = (__half *)(ws + L.stage_q);
    d.stage_k = (__half *)(ws + L.stage_k);
    d.stage_v = (__half *)(ws + L.stage_v);
    d.stage_o = (float *)(ws + L.stage_o);
    d.stage_lse = (float *)(ws + L.stage_lse);
    d.tmaps = ws + L.tmaps;
    d.gates = (uint32_t *)(ws + L.gates);
    d.worker_times = (long long *)(ws + L.worker_times);
    d.v_off = half_pool_bytes(cfg);
    for (int p = 0; p < cfg->n_partitions; ++p) d.pool[p] = (unsigned char *)pool_ptrs[p];

    launch_set_req_active(ctx->dev, nullptr, 0);  // every request takes part in decode steps until told otherwise
    if (plan_setup() != 0) return cuda_fail(ctx, cudaGetLastError());
    if (ctx->impl == KF_IMPL_TMA) {
        int rc = encode_tmaps(ctx, pool_ptrs);
        if (rc != KF_OK) return rc;
        if (attend_tma_setup() != 0) return cuda_fail(ctx, cudaGetLastError());
    }
    e = cudaDeviceSynchronize();
    if (e != cudaSuccess) return cuda_fail(ctx, e);
    return KF_OK;
}

int kf_destroy(kf_ctx *ctx) {
    if (!ctx) return KF_EINVAL;
    delete ctx;
    return KF_OK;
}

int kf_open_request(kf_ctx *ctx, int32_t req, int32_t n_tokens, kf_stream stream) {
    if (!ctx || req < 0 || req >= ctx->cfg.max_requests || n_tokens < 0) return KF_EINVAL;
    ctx->plan_dirty = true;
    return after_launch(ctx, launch_open_request(ctx->dev, req, n_tokens, (cudaStream_t)stream));
}

int kf_close_request(kf_ctx *ctx, int32_t req, kf_stream stream) {
    if (!ctx || req < 0 || req >= ctx->cfg.max_requests) return KF_EINVAL;
    ctx->plan_dirty = true;
    return after_launch(ctx, launch_close_request(ctx->dev, req, (cudaStream_t)stream));
}

int kf_load_context(kf_ctx *ctx, int32_t layer, int32_t req, int32_t tok_begin, int32_t n_tokens, const void *k,
                    const void *v, kf_stream stream) {
    if (!ctx || bad_layer(ctx, layer) || req < 0 || req >= ctx->cfg.max_requests || tok_begin < 0 || n_tokens < 0)
        return KF_EINVAL;
    if (n_tokens == 0) return KF_OK;
    if (!k || !v || ((uintptr_t)k & 15) || ((uintptr_t)v & 15)) return KF_EINVAL;
    if ((int64_t)tok_begin + n_tokens > (int64_t)ctx->cfg.max_ranges_per_request * ctx->cfg.range_tokens) return KF_EINVAL;
    return after_launch(ctx, launch_load_context(ctx->dev, layer, req, tok_begin, n_tokens, (const __half *)k,
                                                 (const __half *)v, (cudaStream_t)stream));
}

int kf_token_boundary(kf_ctx *ctx, kf_stream stream) {
    if (!ctx) return KF_EINVAL;
    // route update and work plan in ONE launch (the plan depends on the routes the update appends)
    // (the plan is kept when no route changed and it is younger than plan_refresh_steps boundaries)
    // open / close / create invalidate the plan on the DEVICE (plan_age), so this launch is the same whatever
    // happened before it -- a CUDA graph that contains it stays valid (kf_step_graph_*).
    const int rc = after_launch(ctx, launch_plan(ctx->dev, 1, (cudaStream_t)stream));
    if (rc == KF_OK) ctx->plan_dirty = false;
    return rc;
}

int kf_kv_append(kf_ctx *ctx, int32_t layer, const void *k_new, const void *v_new, kf_stream stream) {
    if (!ctx || bad_layer(ctx, layer) || !k_new || !v_new || ((uintptr_t)k_new & 15) || ((uintptr_t)v_new & 15))
        return KF_EINVAL;
    return after_launch(ctx, launch_kv_append(ctx->dev, layer, (const __half *)k_new, (const __half *)v_new,
                                              (cudaStream_t)stream));
}

int kf_partial_attend(kf_ctx *ctx, int32_t layer, const void *q, const uint8_t *partition_mask, float *o_part,
                      float *lse_part, kf_stream stream) {
    if (!ctx || bad_layer(ctx, layer) || !q || !o_part || !lse_part || ((uintptr_t)q & 15) || ((uintptr_t)o_part & 15))
        return KF_EINVAL;
    cudaStream_t s = (cudaStream_t)stream;
    int rc = ensure_plan(ctx, s);
    if (rc != KF_OK) return rc;
    AttendParams ap;
    ap.d = ctx->dev;
    ap.layer = layer;
    ap.q = (const __half *)q;
    ap.o_part = o_part;
    ap.lse_part = lse_part;
    ap.o = nullptr;
    ap.lse = nullptr;
    ap.fused = 0;
    ap.commit = 0;
    ap.k_new = nullptr;
    ap.v_new = nullptr;
    ap.part_mask = 0;
    for (int p = 0; p < ctx->cfg.n_partitions; ++p)
        if (!partition_mask || partition_mask[p]) ap.part_mask |= 1ull << p;
    rc = run_attend(ctx, ap, s);
    if (rc != KF_OK) return rc;
    return after_launch(ctx, launch_merge_units(ap, ctx->n_ctas, s));
}

int kf_merge_partials(kf_ctx *ctx, const float *o_part, const float *lse_part, float *o, float *lse, kf_stream stream) {
    if (!ctx || !o_part || !lse_part || !o || !lse || ((uintptr_t)o_part & 15) || ((uintptr_t)o & 15)) return KF_EINVAL;
    cudaStream_t s = (cudaStream_t)stream;
    int rc = ensure_plan(ctx, s);
    if (rc != KF_OK) return rc;
    return after_launch(ctx, launch_merge_ranges(ctx->dev, o_part, lse_part, o, lse, s));
}

int kf_attend_impl(kf_ctx *ctx, int32_t layer, const void *q, float *o, float *lse, float *o_part, float *lse_part,
                   int commit, const void *k_new, const void *v_new, kf_stream stream) {
    if (!ctx || bad_layer(ctx, layer) || !q || !o || !lse || ((uintptr_t)q & 15) || ((uintptr_t)o & 15)) return KF_EINVAL;
    if ((k_new == nullptr) != (v_new == nullptr) || ((uintptr_t)k_new & 15) || ((uintptr_t)v_new & 15)) return KF_EINVAL;
    if (k_new && ctx->impl != KF_IMPL_TMA) return KF_EINVAL;  // only the TMA kernel carries the fused append
    if ((o_part == nullptr) != (lse_part == nullptr) || ((uintptr_t)o_part & 15)) return KF_EINVAL;
    cudaStream_t s = (cudaStream_t)stream;
    int rc = ensure_plan(ctx, s);
    if (rc != KF_OK) return rc;
    AttendParams ap;
    ap.d = ctx->dev;
    ap.layer = layer;
    ap.q = (const __half *)q;
    ap.o_part = o_part ? o_part : ctx->dev.range_o;
    ap.lse_part = lse_part ? lse_part : ctx->dev.range_lse;
    ap.o = o;
    ap.lse = lse;
    ap.fused = 1;
    ap.commit = commit;
    ap.part_mask = ~0ull;
    ap.k_new = (const __half *)k_new;
    ap.v_new = (const __half *)v_new;
    rc = run_attend(ctx, ap, s);
    if (rc == KF_OK && commit) ctx->plan_dirty = true;  // lengths moved
    return rc;
}

int kf_attend(kf_ctx *ctx, int32_t layer, const void *q, float *o, float *lse, float *o_part, float *lse_part,
              kf_stream stream) {
    return kf_attend_impl(ctx, layer, q, o, lse, o_part, lse_part, 0, nullptr, nullptr, stream);
}

int kf_step_commit(kf_ctx *ctx, kf_stream stream) {
    if (!ctx) return KF_EINVAL;
    ctx->plan_dirty = true;
    return after_launch(ctx, launch_step_commit(ctx->dev, (cudaStream_t)stream));
}


int kf_layer_step_host_impl(kf_ctx *ctx, int32_t layer, const void *q_host, const void *k_new_host,
                            const void *v_new_host, float *o_host, float *lse_host, int commit, kf_stream stream) {
    if (!ctx || bad_layer(ctx, layer) || !q_host || !k_new_host || !v_new_host || !o_host || !lse_host) return KF_EINVAL;
    cudaStream_t s = (cudaStream_t)stream;
    const Dev &d = ctx->dev;
    const bool aligned = !(((uintptr_t)q_host | (uintptr_t)k_new_host | (uintptr_t)v_new_host | (uintptr_t)o_host) & 15);
    if (aligned && host_ptr_ok(ctx, q_host) && host_ptr_ok(ctx, k_new_host) && host_ptr_ok(ctx, v_new_host) &&
        host_ptr_ok(ctx, o_host) && host_ptr_ok(ctx, lse_host)) {
        // zero-copy: the append kernel reads k_new / v_new over the bus and stages q; the attend kernel's merge
        // tail writes o / lse straight into the host buffers.  No copy engine work at all.
        int rc = after_launch(ctx, launch_kv_append_stage(d, layer, (const __half *)k_new_host, (const __half *)v_new_host,
                                                          (const __half *)q_host, d.stage_q, s));
        if (rc != KF_OK) return rc;
        return kf_attend_impl(ctx, layer, d.stage_q, o_host, lse_host, nullptr, nullptr, commit, nullptr, nullptr, stream);
    }
    const size_t qb = (size_t)d.B * d.Hq * kHeadDim * 2, kb = (size_t)d.B * d.Hkv * kHeadDim * 2;
    cudaError_t e = cudaMemcpyAsync(d.stage_q, q_host, qb, cudaMemcpyHostToDevice, s);
    if (e == cudaSuccess) e = cudaMemcpyAsync(d.stage_k, k_new_host, kb, cudaMemcpyHostToDevice, s);
    if (e == cudaSuccess) e = cudaMemcpyAsync(d.stage_v, v_new_host, kb, cudaMemcpyHostToDevice, s);
    if (e != cudaSuccess) return cuda_fail(ctx, e);
    const bool fused = ctx->impl == KF_IMPL_TMA;  // the append rides in the attend launch
    int rc = fused ? KF_OK : kf_kv_append(ctx, layer, d.stage_k, d.stage_v, stream);
    if (rc != KF_OK) return rc;
    rc = kf_attend_impl(ctx, layer, d.stage_q, d.stage_o, d.stage_lse, nullptr, nullptr, commit,
                        fused ? d.stage_k : nullptr, fused ? d.stage_v : nullptr, stream);
    if (rc != KF_OK) return rc;
    e = cudaMemcpyAsync(o_host, d.stage_o, (size_t)d.B * d.Hq * kHeadDim * 4, cudaMemcpyDeviceToHost, s);
    if (e == cudaSuccess) e = cudaMemcpyAsync(lse_host, d.stage_lse, (size_t)d.B * d.Hq * 4, cudaMemcpyDeviceToHost, s);
    if (e != cudaSuccess) return cuda_fail(ctx, e);
    return KF_OK;
}

int kf_layer_step(kf_ctx *ctx, int32_t layer, const void *q, const void *k_new, const void *v_new, float *o, float *lse,
                  float *o_part, float *lse_part, kf_stream stream) {
    if (!ctx || !k_new || !v_new) return KF_EINVAL;
    if (ctx->impl == KF_IMPL_TMA) return kf_attend_impl(ctx, layer, q, o, lse, o_part, lse_part, 0, k_new, v_new, stream);
    const int rc = kf_kv_append(ctx, layer, k_new, v_new, stream);
    if (rc != KF_OK) return rc;
    return kf_attend_impl(ctx, layer, q, o, lse, o_part, lse_part, 0, nullptr, nullptr, stream);
}

int kf_layer_step_host(kf_ctx *ctx, int32_t layer, const void *q_host, const void *k_new_host, const void *v_new_host,
                       float *o_host, float *lse_host, kf_stream stream) {
    return kf_layer_step_host_impl(ctx, layer, q_host, k_new_host, v_new_host, o_host, lse_host, 0, stream);
}

int kf_route_snapshot(kf_ctx *ctx, int32_t *len, int32_t *n_ranges, int32_t *part, int32_t *slot, int32_t *free_head,
                      int32_t *rr_cursor, kf_stream stream) {
    if (!ctx) return KF_EINVAL;
    cudaStream_t s = (cudaStream_t)stream;
    const Dev &d = ctx->dev;
    const size_t B = d.B, E = (size_t)d.B * d.Jmax;
    cudaError_t e = cudaSuccess;
    if (len && e == cudaSuccess) e = cudaMemcpyAsync(len, d.len, B * 4, cudaMemcpyDeviceToHost, s);
    if (n_ranges && e == cudaSuccess) e = cudaMemcpyAsync(n_ranges, d.n_ranges, B * 4, cudaMemcpyDeviceToHost, s);
    if (part && e == cudaSuccess) e = cudaMemcpyAsync(part, d.route_part, E * 4, cudaMemcpyDeviceToHost, s);
    if (slot && e == cudaSuccess) e = cudaMemcpyAsync(slot, d.route_slot, E * 4, cudaMemcpyDeviceToHost, s);
    if (free_head && e == cudaSuccess) e = cudaMemcpyAsync(free_head, d.free_head, (size_t)d.P * 4, cudaMemcpyDeviceToHost, s);
    if (rr_cursor && e == cudaSuccess) e = cudaMemcpyAsync(rr_cursor, d.rr_cursor, 4, cudaMemcpyDeviceToHost, s);
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);
    if (e != cudaSuccess) return cuda_fail(ctx, e);
    return KF_OK;
}

int kf_set_active_partitions(kf_ctx *ctx, const uint8_t *active, kf_stream stream) {
    if (!ctx || !active) return KF_EINVAL;
    unsigned long long mask = 0;
    for (int p = 0; p < ctx->cfg.n_partitions; ++p)
        if (active[p]) mask |= 1ull << p;
    if (mask == 0) return KF_EINVAL;
    return after_launch(ctx, launch_set_active(ctx->dev, mask, (cudaStream_t)stream));
}

int kf_redirect_tails(kf_ctx *ctx, const uint8_t *partitions, kf_stream stream) {
    if (!ctx || !partitions) return KF_EINVAL;
    unsigned long long mask = 0;
    for (int p = 0; p < ctx->cfg.n_partitions; ++p)
        if (partitions[p]) mask |= 1ull << p;
    return after_launch(ctx, launch_redirect(ctx->dev, mask, (cudaStream_t)stream));
}

int kf_route_begins(kf_ctx *ctx, int32_t *begin, kf_stream stream) {
    if (!ctx || !begin) return KF_EINVAL;
    cudaStream_t s = (cudaStream_t)stream;
    cudaError_t e = cudaMemcpyAsync(begin, ctx->dev.range_begin, (size_t)ctx->dev.B * ctx->dev.Jmax * 4, cudaMemcpyDeviceToHost, s);
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);
    if (e != cudaSuccess) return cuda_fail(ctx, e);
    return KF_OK;
}

int kf_set_active_requests(kf_ctx *ctx, const uint8_t *active_dev, kf_stream stream) {
    if (!ctx) return KF_EINVAL;
    ctx->plan_dirty = true;
    return after_launch(ctx, launch_set_req_active(ctx->dev, active_dev, (cudaStream_t)stream));
}

int kf_partition_state(kf_ctx *ctx, int32_t *active, int64_t *tokens, int32_t *tails, kf_stream stream) {
    if (!ctx) return KF_EINVAL;
    cudaStream_t s = (cudaStream_t)stream;
    const Dev &d = ctx->dev;
    const size_t P = d.P;
    cudaError_t e = cudaMemsetAsync(d.part_tokens, 0, P * 8, s);
    if (e == cudaSuccess) e = cudaMemsetAsync(d.part_tails, 0, P * 4, s);
    if (e != cudaSuccess) return cuda_fail(ctx, e);
    const int rc = after_launch(ctx, launch_partition_state(d, d.part_tokens, d.part_tails, s));
    if (rc != KF_OK) return rc;
    if (active && e == cudaSuccess) e = cudaMemcpyAsync(active, d.active, P * 4, cudaMemcpyDeviceToHost, s);
    if (tokens && e == cudaSuccess) e = cudaMemcpyAsync(tokens, d.part_tokens, P * 8, cudaMemcpyDeviceToHost, s);
    if (tails && e == cudaSuccess) e = cudaMemcpyAsync(tails, d.part_tails, P * 4, cudaMemcpyDeviceToHost, s);
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);
    if (e != cudaSuccess) return cuda_fail(ctx, e);
    return KF_OK;
}

int kf_status(kf_ctx *ctx, kf_stream stream) {
    if (!ctx) return KF_EINVAL;
    cudaStream_t s = (cudaStream_t)stream;
    int32_t word = 0;
    cudaError_t e = cudaMemcpyAsync(&word, ctx->dev.error, 4, cudaMemcpyDeviceToHost, s);
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);
    if (e != cudaSuccess) return cuda_fail(ctx, e);
    if (word != 0) {
        e = cudaMemsetAsync(ctx->dev.error, 0, 4, s);
        if (e == cudaSuccess) e = cudaStreamSynchronize(s);
        if (e != cudaSuccess) return cuda_fail(ctx, e);
    }
    return word;
}

int kf_plan_info(kf_ctx *ctx, int32_t *out, kf_stream stream) {
    if (!ctx || !out) return KF_EINVAL;
    cudaStream_t s = (cudaStream_t)stream;
    int rc = ensure_plan(ctx, s);
    if (rc != KF_OK) return rc;
    cudaError_t e = cudaMemcpyAsync(out, ctx->dev.plan, 8 * sizeof(int32_t), cudaMemcpyDeviceToHost, s);
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);
    if (e != cudaSuccess) return cuda_fail(ctx, e);
    return KF_OK;
}

int64_t kf_launch_count(const kf_ctx *ctx) { return ctx ? ctx->launches : 0; }

int kf_worker_times(kf_ctx *ctx, int64_t *out, int32_t *n_workers, kf_stream stream) {
    if (!ctx || !out || !n_workers) return KF_EINVAL;
    if (!ctx->dev.diag) return KF_ESTATE;  // the kernel records nothing unless kf_config.diagnostics asked for it
    cudaStream_t s = (cudaStream_t)stream;
    *n_workers = ctx->dev.max_workers;
    cudaError_t e = cudaMemcpyAsync(out, ctx->dev.worker_times, (size_t)ctx->dev.max_workers * 4 * 8,
                                    cudaMemcpyDeviceToHost, s);
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);
    if (e != cudaSuccess) return cuda_fail(ctx, e);
    return KF_OK;
}

}  // extern "C"
