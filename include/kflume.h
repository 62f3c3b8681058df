/*
 * kflume.h -- C ABI of libkflume: KernelFlume's data-parallel hot path on one B200 (sm_100a).
 *
 * What the library computes (arxiv/paper_2606_29207, text in PAPER.md):
 *   a decode query for one new token runs GQA attention over each token-range KV partition that a
 *   routing table assigns to a (here: emulated) weightless attention node; every range emits a partial
 *   output and its log-sum-exp; the partials are merged into the exact softmax result
 *   (PAPER.md:137, :143-147, :254).  A KV-append / route-update step feeds it: the new token's K/V
 *   is appended to the request's tail range, and a new range is opened -- the routing table extended --
 *   at the token boundary where the tail range is full.
 *
 * Conventions
 *   - Plain C, no CUDA or torch types.  A `kf_stream` is a `cudaStream_t` cast to `void*` (NULL = the
 *     legacy default stream).  Pointers are marked [device] or [host].
 *   - fp16 tensors are passed as `const void*` to IEEE binary16 data.
 *   - Every call returns an int: KF_OK (0) or a negative KF_E* code.  No exceptions, no aborts, nothing
 *     is printed.  Errors found ON THE DEVICE (capacity, state) are latched in a device error word and
 *     surfaced by kf_status() / kf_route_snapshot(); the launch that found them skips the faulty item.
 *   - OWNERSHIP: the caller owns all device memory (KV pools, workspace, q/k/v/o buffers) and all
 *     streams for the lifetime of the ctx.  The library owns only the host-side `kf_ctx`.  Hot calls
 *     (token_boundary, kv_append, partial_attend, merge_partials, attend, step_commit) are asynchronous
 *     on the caller's stream, never synchronise, never allocate, launch fixed grids and read all variable
 *     state (lengths, routes, work plan) from device memory -- so a CUDA Graph captured around them stays
 *     valid across route updates (the single-GPU analogue of PAPER.md:165-179, requirement R1 at :127).
 *   - One ctx = one stream order: the calls of a ctx share device-side scheduler words and completion counters, so
 *     they must be issued so that they execute one after another (one stream, or streams ordered by events).  Use
 *     separate ctxs (with separate workspaces) for concurrent batches.  Host-side entry points are not thread-safe
 *     per ctx.
 *   - There is NO CPU fallback: without a CUDA device kf_create() returns KF_ECUDA.
 *
 * Notation: B = max_requests, H_q / H_kv = query / KV heads, G = H_q / H_kv, d = head_dim = 128,
 *   R = range_tokens, P = n_partitions, Jmax = max_ranges_per_request, L = n_layers (physical).
 *   len_r = tokens of request r committed so far; a decode step attends over len_r + 1 tokens (the token
 *   appended in this step included: the tail node "appends, then computes attention").
 *
 * KV pool layout (one pool per partition = per emulated attention node; fp16):
 *   K element (p, layer, slot, g, t, i) lives at byte
 *       pool[p] + ((((layer*slots_per_partition + slot)*H_kv + g)*R + t)*128 + i)*2
 *   and the V element at the same offset + kf_pool_bytes()/2.  A slot holds one token range of one
 *   request for all physical layers ("[range][kv_head][token][128]" innermost order).
 */
#ifndef KFLUME_H
#define KFLUME_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define KF_VERSION 220 /* 0.2.2: + kf_route_install_latency (0.2.1: kf_attend_static; 0.2.0: kf_layer_step, redirects, graph flags, W-node stages) */

#define KF_OK 0
#define KF_EINVAL (-1) /* bad argument / shape / alignment / null pointer */
#define KF_ESTATE (-2) /* call not valid in this state (request closed/already open, no route for the tail) */
#define KF_ENOSPC (-3) /* no free slot in the round-robin partition, or Jmax ranges exceeded (device-detected) */
#define KF_ECUDA (-4)  /* a CUDA runtime/driver call failed (kf_last_cuda_error() has the text) */

#define KF_IMPL_AUTO 0   /* fastest available attend kernel (TMA + tensor-core path) */
#define KF_IMPL_SIMPLE 1 /* CUDA-core reference kernel (coalesced 128-bit loads, warp shuffles) */
#define KF_IMPL_TMA 2    /* TMA-staged, mma.sync tensor-core kernel */

typedef void *kf_stream;

typedef struct kf_config {
    int32_t n_q_heads;              /* H_q                                                        */
    int32_t n_kv_heads;             /* H_kv; H_q % H_kv == 0 and G = H_q/H_kv in 1..8             */
    int32_t head_dim;               /* must be 128                                                */
    int32_t n_layers;               /* physical layer pools L >= 1                                */
    int32_t range_tokens;           /* R, a power of two >= 1                                     */
    int32_t n_partitions;           /* P in 1..64: emulated attention nodes        */
    int32_t max_requests;           /* B in 1..4096                                               */
    int32_t max_ranges_per_request; /* Jmax >= 1                                                  */
    int32_t slots_per_partition;    /* token-range slots in each partition pool                   */
    float softmax_scale;            /* 0 => 1/sqrt(head_dim); scores are scale * q.k              */
    int32_t attend_impl;            /* KF_IMPL_*                                                  */
    int32_t min_tiles_per_worker;   /* smallest chunk of the work plan, in 16-token tiles; 0 => 12 when the step has at
                                     * least 16 tiles per worker, else 4 */
    /* tuning of the attend kernel and its work plan; 0 => default.  Results are bit-identical for a given
     * (min_tiles_per_worker, workers_per_sm, sched_*) because the plan's cuts depend only on these. */
    int32_t workers_per_sm;         /* warps (independent workers) per SM: 4 or 8                  */
    int32_t pipeline_stages;        /* 8 KB TMA stages in flight per worker: 2..6 (2..3 for 8 workers) */
    int32_t sched_first_pct;        /* 1..100 (0 => 100): guided self-scheduling factor: chunk <= pct% of (remaining tiles / workers) */
    int32_t sched_decay_pct;        /* 1..99: share of a unit's remaining tiles that each scheduling level takes */
    int32_t plan_refresh_steps;     /* the work plan is rebuilt when a route changes or after this many token boundaries
                                     * (0 => 128; 1 => every step); in between, tail ranges grow inside the kept plan */
    int32_t kv_l2_policy;           /* L2 policy of the K/V tile loads: 0 => default (1); 1 = evict-first (K/V is read once
                                     * per launch; keeps q, partials and the plan resident: +1..5% measured); 2 = normal */
    int32_t attend_sms;             /* SM budget of the attend kernels: CTAs (one per SM) of their persistent grid; 0 => all
                                     * SMs.  A narrower grid leaves SMs to kernels of other streams (kf_pipeline_step) */
    int32_t diagnostics;            /* non-zero: the attend kernel records per-worker timestamps (kf_worker_times);
                                     * 0 (default): it reads no timer and writes nothing beyond the method's outputs */
} kf_config;

typedef struct kf_ctx kf_ctx;

/* ---- library ------------------------------------------------------------------------------------ */
int kf_version(void);
const char *kf_strerror(int code);
/* Text of the last CUDA error seen by this ctx ("" if none).  [host] string owned by the ctx. */
const char *kf_last_cuda_error(const kf_ctx *ctx);

/* ---- sizes (pure host arithmetic, no GPU needed) --------------------------------------------------
 * kf_pool_bytes: bytes of ONE partition pool (K + V, all physical layers) =
 *   2 * L * slots_per_partition * H_kv * R * 128 * 2   (per-layer bytes per token 2*H_kv*d*2B).
 * kf_workspace_bytes: bytes of the device workspace (routing table, work plan, partial buffers, staging).
 * Both return 0 for an invalid config. */
size_t kf_pool_bytes(const kf_config *cfg);
size_t kf_workspace_bytes(const kf_config *cfg);
/* Byte offset inside a partition pool of element (layer, slot, kv_head, token, 0) of K (is_v=0) or V (is_v=1).
 * Returns (size_t)-1 on bad arguments. */
size_t kf_pool_offset(const kf_config *cfg, int32_t layer, int32_t slot, int32_t kv_head, int32_t token,
                      int32_t is_v);

/* ---- lifetime ------------------------------------------------------------------------------------
 * pool_ptrs: [host] array of P [device] pointers, each kf_pool_bytes() long, 1024-byte aligned.
 * workspace: [device], kf_workspace_bytes() long, 256-byte aligned; zero-initialised by kf_create.
 * Uses the current CUDA device.  All requests start closed; the routing table is empty. */
int kf_create(kf_ctx **out, const kf_config *cfg, void *const *pool_ptrs, void *workspace,
              size_t workspace_bytes);
int kf_destroy(kf_ctx *ctx);

/* ---- routing table --------------------------------------------------------------
 * kf_open_request: "post-prefill initialisation": marks request `req` open with
 *   len = n_tokens and allocates ceil(n_tokens/R) ranges j = 0.. in order.  The k-th range ever allocated
 *   goes to partition k mod P (one global round-robin cursor over the active set, see
 *   kf_set_active_partitions); the slot comes from that partition's LIFO
 *   free list if non-empty, else from its bump allocator.  Routes are layer-independent: an attention
 *   node holds all L layers of a range.  Device errors: ESTATE (already open), ENOSPC.
 * kf_close_request: returns the request's slots to the free lists (ascending j) and marks it closed. */
int kf_open_request(kf_ctx *ctx, int32_t req, int32_t n_tokens, kf_stream stream);
int kf_close_request(kf_ctx *ctx, int32_t req, kf_stream stream);

/* kf_set_active_partitions -- publish a new ACTIVE SET of attention nodes (a scale-up or scale-down event of the
 *   paper's policy: PAPER.md:216-219 "at the next token boundary, publish the route", :240 "future appends use the
 *   new A node, while existing KV ranges remain in place").  active: [host] uint8[P], non-zero = the partition
 *   receives new ranges; at least one must be set.  Takes effect for every range allocated after this call in stream
 *   order (kf_token_boundary, kf_open_request); existing routes never change, partitions that leave the set keep
 *   serving the ranges they hold.  Allocation order: the first active partition after the one used last, cyclically
 *   (with all P active: the k-th range ever allocated goes to partition k mod P).  All partitions start active.
 *   This call is the critical-path "route install" (paper: 7.2 us on the CPU): one tiny kernel.
 *   On its own it moves a tail only when its current range fills (reading 20): a node that left the set can
 *   still grow by (its tails) * R tokens.  Algorithm 1 l.16-17 ("publish the route and redirect active tails on i to
 *   prewarm[i]") is this call FOLLOWED BY kf_redirect_tails for node i.
 * kf_redirect_tails -- partitions: [host] uint8[P], non-zero = marked.  At the NEXT kf_token_boundary every active request
 *   whose tail range lives on a marked partition and holds at least one token closes that range at its current length
 *   and continues in a new range, beginning at position len_r, on the next active partition (PAPER.md:216-219, :240:
 *   "at the next token boundary ... future appends use the new A node, while existing KV ranges remain in place";
 *   DESIGN.md reading 28).  Ranges are therefore [begin_j, begin_j+1) with at most R tokens each (kf_route_begins);
 *   begin_j = j * R as long as no tail was redirected.  A redirect that finds no free slot or route entry is not carried
 *   out (no error).  The marks are consumed by that one boundary.  One tiny kernel, like the route install.
 * kf_partition_state -- occupancy that the policy monitors (Algorithm 1, l.6-9): [host] active[P] (0/1),
 *   tokens[P] = committed tokens resident on each partition (x 2*H_kv*d*2 B*L = KV bytes),
 *   tails[P] = open requests whose tail range lives there.  Any pointer may be NULL.  Synchronises `stream`. */
int kf_set_active_partitions(kf_ctx *ctx, const uint8_t *active, kf_stream stream);
int kf_redirect_tails(kf_ctx *ctx, const uint8_t *partitions, kf_stream stream);
/* kf_set_active_requests -- which OPEN requests take part in the following decode steps (continuous batching: a
 *   request may sit out steps without being closed; Algorithm 1 counts only "r active", l.7).  active: [device]
 *   uint8[B], non-zero = active, or NULL = all (the initial state).  A paused request keeps its routes and KV;
 *   kf_token_boundary opens no range for it, kf_kv_append ignores its row, the attend / merge calls produce no
 *   output for it (its rows of o / lse / partials are left untouched), kf_step_commit leaves its len alone, and
 *   kf_partition_state does not count it as a tail.  The buffer is read asynchronously on `stream`. */
int kf_set_active_requests(kf_ctx *ctx, const uint8_t *active, kf_stream stream);
int kf_partition_state(kf_ctx *ctx, int32_t *active, int64_t *tokens, int32_t *tails, kf_stream stream);

/* kf_load_context: copies tokens [tok_begin, tok_begin + n_tokens) of request `req`, layer `layer`, into the
 * routed slots.  k, v: [device] fp16 [H_kv][n_tokens][128].  Every position must already have a route
 * (position < n_ranges*R), else device error ESTATE.  Does not change len. */
int kf_load_context(kf_ctx *ctx, int32_t layer, int32_t req, int32_t tok_begin, int32_t n_tokens,
                    const void *k, const void *v, kf_stream stream);

/* ---- the decode step -----------------------------------------------------------------------------
 * (a1) kf_token_boundary -- route update at the token boundary (Fig. 5 at :173).
 *   For every open, active request, ascending, whose tail position len has no route (its tail range is full:
 *   len % R == 0 -- or an earlier boundary found no slot for it): allocate (partition, slot) as above and APPEND the
 *   route entry; earlier entries never change.  Then rebuilds the device-side work plan for a step over len+1
 *   tokens (or keeps it, plan_refresh_steps).  Call once per decode step, before the per-layer calls.
 *   Device errors: ENOSPC (no active partition has a free slot, or Jmax reached).  Such a request WAITS: kf_kv_append
 *   drops its row (ESTATE), the attend calls produce its output over the len committed tokens only, kf_step_commit
 *   does not advance it, and every later kf_token_boundary re-tries -- so it resumes at the same position once
 *   kf_close_request frees a slot or kf_set_active_partitions adds a node (reading 24). */
int kf_token_boundary(kf_ctx *ctx, kf_stream stream);

/* (a2) kf_kv_append -- the tail node appends (K_new, V_new).
 *   k_new, v_new: [device] fp16 [B][H_kv][128]; row r is written at token offset len_r - begin_j of the tail range
 *   j = n_ranges_r - 1 of open request r (begin_j = j*R unless a tail was redirected; rows of closed requests are ignored).  Does NOT advance len (all
 *   layers of a step append at the same position).  Device error ESTATE if that range has no route. */
int kf_kv_append(kf_ctx *ctx, int32_t layer, const void *k_new, const void *v_new, kf_stream stream);

/* (a3) kf_partial_attend -- local core attention per token range:
 *   for every open request r, range j < J_r (= ceil((len_r+1)/R) unless a tail was redirected) whose partition is selected, and query
 *   head h (KV head h / G):  s_t = scale * q_h . K_t over the range's tokens,
 *       lse_part[r][j][h] = ln sum_t exp(s_t),   o_part[r][j][h][:] = sum_t exp(s_t - lse) V_t.
 *   q: [device] fp16 [B][H_q][128].  partition_mask: [host] uint8 [P] (non-zero = selected) or NULL = all.
 *   o_part: [device] fp32 [B][Jmax][H_q][128];  lse_part: [device] fp32 [B][Jmax][H_q].
 *   Rows of unselected / non-existent ranges are left untouched. */
int kf_partial_attend(kf_ctx *ctx, int32_t layer, const void *q, const uint8_t *partition_mask, float *o_part,
                      float *lse_part, kf_stream stream);

/* (a4) kf_merge_partials -- online-softmax (log-sum-exp) reduction of the partials:
 *   lse[r][h] = ln sum_j exp(lse_part[r][j][h]);  o[r][h] = sum_j exp(lse_part[r][j][h] - lse[r][h]) o_part[r][j][h]
 *   over j < J_r.  J_r == 1 is an exact copy; a partial with lse = -inf has weight 0.
 *   o: [device] fp32 [B][H_q][128]; lse: [device] fp32 [B][H_q].  Rows of closed requests untouched. */
int kf_merge_partials(kf_ctx *ctx, const float *o_part, const float *lse_part, float *o, float *lse,
                      kf_stream stream);

/* (a3+a4) kf_attend -- both in ONE launch: the merge is fused into the tail of the attend kernel (the last
 *   work item to finish a range / a request performs the reduction, in a fixed order, so results are
 *   run-to-run identical and equal to the unfused path).  o_part / lse_part may be NULL (internal scratch). */
int kf_attend(kf_ctx *ctx, int32_t layer, const void *q, float *o, float *lse, float *o_part, float *lse_part,
              kf_stream stream);

/* (a3+a4, no allocation anywhere) kf_attend_static -- kf_attend for a caller that cannot supply memory for the range
 *   partials and cannot allocate any.  Who that is: an attention node whose HBM is already handed out to KV pools down to
 *   the last slot (the paper's A nodes hold nothing but KV) and that is pulled into a running decode loop;
 *   a thread that must stay out of the CUDA allocator because cudaMalloc / cudaFree synchronise the device and would
 *   stall the step graphs other streams are replaying; code living under a framework that owns all device memory through
 *   its own caching allocator.  Same arguments and results as kf_attend(ctx, layer, q, o, lse, NULL, NULL, stream) --
 *   bit for bit: the same plan, kernel and merge order -- but the range partials (o_j, lse_j of PAPER.md:147, :254) go to
 *   a fixed array of KF_STATIC_SCRATCH_BYTES that is part of the library image (a file-scope __device__ array) instead
 *   of to the workspace.  The call never calls cudaMalloc / cudaFree or any routine that allocates device or host memory.
 *   LIMIT: max_requests * max_ranges_per_request * n_q_heads * (128 + 1) * 4 bytes (+ up to 255 of padding) must fit in
 *     KF_STATIC_SCRATCH_BYTES, else KF_EINVAL and kf_last_cuda_error() says how many bytes were needed.
 *   COST: every GPU on which this process uses the library holds those KF_STATIC_SCRATCH_BYTES from the moment the
 *     library's code is loaded onto it until the process exits, used or not.
 *   FIRST CALL PER GPU: looks the array's device address up (cudaGetSymbolAddress, with the ctx's device current) and
 *     keeps it; that look-up is a set-up step which may make the runtime load code onto the GPU, so make the first call
 *     on each GPU before starting any stream capture.  Later calls only launch.
 *   SHARING: there is ONE array per GPU for all ctxs and threads.  It keeps whatever the previous call left; the kernel
 *     never reads a partial it has not written in the same launch, so nothing needs clearing between calls.  Two calls
 *     whose kernels may run at the same time on one GPU (different streams, different ctxs) write the same bytes and
 *     corrupt each other's results: order them on one stream or with events, like the calls of one ctx. */
#define KF_STATIC_SCRATCH_BYTES (16u << 20)
int kf_attend_static(kf_ctx *ctx, int32_t layer, const void *q, float *o, float *lse, kf_stream stream);

/* (a5) kf_step_commit -- len_r += 1 for every open, active request whose tail position had a route in this step
 *   (the step boundary; a request waiting for a slot stays where it is, see kf_token_boundary). */
int kf_step_commit(kf_ctx *ctx, kf_stream stream);

/* (a2+a3+a4) kf_layer_step -- one layer-step in ONE launch: kf_kv_append(k_new, v_new) followed by kf_attend(q, ...),
 *   same arguments, same results, same device errors.  With the TMA kernel the append rides in the attend launch: the
 *   worker that attends the tail tile of (request, kv head) writes the new K/V row to the pool and patches it into its
 *   shared-memory copy of that tile (the tail node "appends (K_new, V_new), then computes attention");
 *   the static step graph uses the same launch.  With KF_IMPL_SIMPLE it is the two launches one after the other. */
int kf_layer_step(kf_ctx *ctx, int32_t layer, const void *q, const void *k_new, const void *v_new, float *o, float *lse,
                  float *o_part, float *lse_part, kf_stream stream);

/* One layer-step with HOST buffers (end-to-end path): q / k_new / v_new [host, fp16, shapes as above] in,
 * o [B][H_q][128] and lse [B][H_q] (fp32) out [host].  With PINNED host memory (16-byte aligned) nothing is copied
 * by a copy engine: the append kernel reads k_new / v_new over the bus and stages q, kf_attend writes o / lse
 * straight into the host buffers.  Otherwise the buffers go through device staging with cudaMemcpyAsync.
 * Asynchronous on `stream`; the caller synchronises the stream before reading o / lse or rewriting the inputs. */
int kf_layer_step_host(kf_ctx *ctx, int32_t layer, const void *q_host, const void *k_new_host,
                       const void *v_new_host, float *o_host, float *lse_host, kf_stream stream);

/* ---- one decode step as a static CUDA graph ----------------------------------------------------------
 * The paper keeps the W-node computation in one static CUDA Graph and confines elasticity to a routing table the
 * graph never sees (PAPER.md:127 requirement R1, :165-179).  The same holds here: every hot kernel launches a
 * fixed grid and reads lengths, routes and the work plan from device memory, so ONE captured graph of
 *     kf_token_boundary -> for i < n: { kf_kv_append(layers[i], k_new[i], v_new[i]);
 *                                       kf_attend(layers[i], q[i], o[i], lse[i]) } -> kf_step_commit
 * (device buffers + TMA kernel: n + 1 kernel nodes -- each layer-step is the single launch of kf_layer_step, the commit
 * rides in the last one)
 * is replayed for every decode step, across range fills, route updates and kf_open/close_request, without
 * re-capture.  A replay also removes the submission latency between the small kernels of a step.
 * kf_step_graph_create: captures on `stream` (must not be the legacy default stream; nothing executes) and
 *   instantiates.  layers: [host] int32[n], physical layer of each layer-step.  q, k_new, v_new, o, lse: [host]
 *   arrays of n pointers, shapes as in kf_kv_append / kf_attend.  host_io == 0: they are [device] pointers and may
 *   be re-bound at every launch.  host_io != 0: they are PINNED [host] buffers (the end-to-end path of
 *   kf_layer_step_host: zero-copy reads of q / k_new / v_new, o / lse written straight to the host).  Pinned,
 *   16-byte aligned buffers may be re-bound at every launch as well; buffers that had to go through copy nodes
 *   (not device-accessible) are bound for the graph's lifetime -- the caller rewrites their contents between
 *   launches (pre-registered buffers).
 * kf_step_graph_launch: one decode step.  q .. lse: all NULL = keep the bound pointers; else all five arrays
 *   [host, n pointers each] re-bind the pointers (host-side node update; no re-instantiation; KF_EINVAL for a
 *   host-io graph with copy nodes or for host pointers the GPU cannot dereference).
 *   Asynchronous on `stream`.  Errors as the calls it contains (device errors via kf_status).
 * kf_step_graph_destroy: frees the graph; the ctx must still be alive. */
typedef struct kf_graph kf_graph;
int kf_step_graph_create(kf_ctx *ctx, int32_t n_layer_steps, const int32_t *layers, int32_t host_io,
                         const void *const *q, const void *const *k_new, const void *const *v_new, float *const *o,
                         float *const *lse, kf_stream stream, kf_graph **out);
int kf_step_graph_launch(kf_graph *graph, const void *const *q, const void *const *k_new, const void *const *v_new,
                         float *const *o, float *const *lse, kf_stream stream);
int kf_step_graph_destroy(kf_graph *graph);

/* ---- graph progress signalling ---------------------------------------------------------
 * The paper's static graph "contains only local compute and signal writes": where an outbound buffer becomes ready a
 * WriteValue32-style write sets a flag in host-visible memory, "allowing the CPU to observe graph progress without
 * ending replay" (:167); the other way round a ReadValue32-style wait inside the graph holds a stage back until the CPU
 * has written a completion flag to GPU memory -- on "a dedicated signaling stream rather than the graph's execution
 * stream: the execution stream is already blocked on that wait, so enqueuing the flag write on the same stream would
 * place it behind the wait and deadlock" (:175).  The single-GPU analogue: a host thread (the paper's CPU routing
 * loop) can hand the inputs of layer-step i to a RUNNING step graph and pick its outputs up, layer-step by
 * layer-step, with no re-capture -- e.g. while it edits the routing table for the next step.
 *
 * kf_step_graph_flags: adds the signal nodes to a step graph that has not been launched yet (it is re-captured on
 *   `stream`; nothing executes).  ready_host: [host] PINNED uint32[n] or NULL: after layer-step i of launch L the graph
 *   writes seq(L, i) = (L - 1) * n + i + 1 to ready_host[i]; every write of that layer-step (o[i] / lse[i], also when
 *   they are host buffers) is visible to a host thread that has read the value.  gates != 0: before layer-step i of
 *   launch L (before its kf_kv_append reads k_new[i] / v_new[i] / q[i]) the graph waits until gate word i -- device
 *   memory inside the workspace -- is >= seq(L, i) (cyclic 32-bit comparison).  Both values are re-written into the
 *   graph's mem-op nodes at every launch (host-side update, no re-instantiation).  With gates != 0 the call zeroes the
 *   gate words and SYNCHRONISES `stream` before it returns, so a release issued right afterwards -- on any stream, while
 *   `stream` still has other work queued -- cannot be overwritten.  KF_ESTATE after the first launch;
 *   KF_EINVAL if ready_host is not pinned memory the GPU can address.
 * kf_step_graph_seq: the sequence number layer-step i will carry in the NEXT launch (0 on bad arguments).
 * kf_step_graph_release: writes `seq` to gate word i with a stream memory operation on `signal_stream`.  Everything the
 *   host stored into the layer-step's pinned input buffers before this call is visible to the kernels behind the
 *   gate.  KF_ESTATE if `signal_stream` is the stream of the graph's last launch (the deadlock of PAPER.md:175 is
 *   refused instead of entered) or the graph has no gates.  A gate may be released before the launch that waits on it. */
int kf_step_graph_flags(kf_graph *graph, uint32_t *ready_host, int32_t gates, kf_stream stream);
uint32_t kf_step_graph_seq(const kf_graph *graph, int32_t layer_step);
int kf_step_graph_release(kf_graph *graph, int32_t layer_step, uint32_t seq, kf_stream signal_stream);

/* ---- inspection (tests) ---------------------------------------------------------------------------
 * kf_route_snapshot: downloads the routing state into [host] arrays (any may be NULL):
 *   len[B] (-1 = closed), n_ranges[B], part[B][Jmax], slot[B][Jmax] (-1 where unused), free_head[P],
 *   rr_cursor[1].  Synchronises `stream`.
 * kf_status: synchronises `stream`, returns the device error word (KF_OK or the FIRST latched KF_E*) and
 *   clears it.
 * kf_launch_count: number of CUDA kernels this ctx has launched so far (host-side counter). */
int kf_route_snapshot(kf_ctx *ctx, int32_t *len, int32_t *n_ranges, int32_t *part, int32_t *slot,
                      int32_t *free_head, int32_t *rr_cursor, kf_stream stream);
/* kf_route_begins: begin[B][Jmax] [host] = first token position of every range (-1 where unused).  Synchronises. */
int kf_route_begins(kf_ctx *ctx, int32_t *begin, kf_stream stream);
int kf_status(kf_ctx *ctx, kf_stream stream);
int64_t kf_launch_count(const kf_ctx *ctx);

/* ---- Algorithm 1: the A-node scaling policy, host-side controller ----------------------------
 * Pure host arithmetic (double), no GPU work.  Feed it kf_partition_state(); act on it with
 * kf_set_active_partitions().  The paper gives no values for beta_mem, beta_slo, gamma: they are inputs.
 *   kf_policy_bytes_per_token: 2 * H_kv * d_h * L * 2 B.
 *   kf_policy_threshold:       Eq. (1)  C_thresh = min(beta_mem * C_kv_cap, beta_slo * T_A^max * BW_HBM).
 *   kf_policy_initial_nodes:   l.2-3    N_A = ceil(sum_i s_i * bytes_per_token / C_thresh); s: [host] int64[n]; -1 on bad input.
 *   kf_policy_step:            l.6-19   for every node i holding at least one tail (tails[i] > 0):
 *        g_i = tails[i] * bytes_per_token;  b_i = tokens[i] * bytes_per_token;
 *        tau_fill = (C_thresh - b_i) / g_i                                   (Eq. 2; +inf for nodes without tails)
 *        want_prewarm = tau_fill * T_step < T_prewarm and no prewarm pending or ready for i
 *        want_publish = b_i >= gamma * C_thresh and the prewarm for i is ready
 *      (acting on want_publish = kf_set_active_partitions without node i, then kf_redirect_tails for node i)
 *      tokens, tails: [host] [P] as kf_partition_state returns them; prewarm_pending / prewarm_ready: [host] uint8[P]
 *      kept by the caller (a prewarm is the background bring-up of a fresh node); out: [host] [P]. */
typedef struct kf_policy_config {
    double beta_mem, beta_slo, gamma; /* in (0, 1] */
    double t_a_max_s;                 /* largest admissible routed-attention time per layer, seconds (from the TPOT SLO) */
    double bw_hbm;                    /* effective HBM bandwidth of one attention node, bytes / s */
    double c_kv_cap;                  /* usable KV capacity of one attention node, bytes */
    double t_step_s, t_prewarm_s;     /* predicted decode-step time; measured time to prepare a new route */
    int32_t n_kv_heads, head_dim, n_layers;
} kf_policy_config;
typedef struct kf_policy_decision {
    double tau_fill;
    int32_t want_prewarm, want_publish;
} kf_policy_decision;
double kf_policy_bytes_per_token(const kf_policy_config *cfg);
double kf_policy_threshold(const kf_policy_config *cfg);
int64_t kf_policy_initial_nodes(const kf_policy_config *cfg, const int64_t *s, int32_t n_requests);
int kf_policy_step(const kf_policy_config *cfg, int32_t n_partitions, const int64_t *tokens, const int32_t *tails,
                   const uint8_t *prewarm_pending, const uint8_t *prewarm_ready, kf_policy_decision *out);

/* ---- W-node stages and the inter-layer kernel pipeline ----------------------------------
 * The stages of a decode layer that run on the paper's weight-bearing W nodes, around core attention:
 *   T_p  projection (step 1):  q = x Wq^T, then (k_new, v_new) = x Wkv^T -- "Q first": two
 *        launches, so that everything which depends only on q can be released before the K/V projection is done;
 *   T_f  post-attention (step 5): y = o Wo^T;  h = silu(y Wg^T) * (y Wu^T) (SwiGLU, the FFN of the
 *        Llama models the paper serves);  x' = h Wd^T.
 * Every contraction is the hand-written tcgen05 GEMM of kf_wgemm.cu (weights streamed once by TMA, accumulators in
 * TMEM).  Tensors stored between kernels are fp16, accumulation is fp32.  No residuals, norms or rotary embedding:
 * the weights are synthetic and this part exists to measure the pipeline of PAPER.md:266-280 (reading 26).
 *
 * Weights: ONE [device] buffer, 1024-byte aligned, kf_wside_weight_bytes() long; matrix `which` of layer l starts at
 *   kf_wside_weight_offset() and is stored [out_features][in_features] fp16, rows contiguous:
 *   KF_W_Q [H_q*d][hidden], KF_W_KV [2*H_kv*d][hidden] (K rows, then V rows), KF_W_O [hidden][H_q*d],
 *   KF_W_GATE [ffn][hidden], KF_W_UP [ffn][hidden] (directly behind the gate), KF_W_DOWN [hidden][ffn].
 * Workspace: [device], 256-byte aligned, kf_wside_workspace_bytes(); holds the fp16 copy of o, y, h and the split-K
 *   partial sums.  The caller owns both buffers; the library owns the host-side handle.  The calls of one kf_wside must
 *   execute one after another (they share the workspace): one stream, or streams ordered by events.
 * Shapes: x, x_next [batch][hidden] fp16; q [batch][H_q][128], k_new / v_new [batch][H_kv][128] fp16 (the layouts
 *   kf_kv_append / kf_attend take); o [batch][H_q][128] fp32 (what kf_attend writes).  1 <= batch <= max_batch <= 128.
 *   hidden and ffn are multiples of 128, head_dim is 128.  Every tensor pointer must be 16-byte aligned (KF_EINVAL
 *   otherwise: rows are read and written with vector accesses).  All calls are asynchronous on `stream`, never synchronise,
 *   never allocate, and can be captured into a CUDA graph. */
#define KF_W_Q 0
#define KF_W_KV 1
#define KF_W_O 2
#define KF_W_GATE 3
#define KF_W_UP 4
#define KF_W_DOWN 5
typedef struct kf_wside_config {
    int32_t hidden, n_q_heads, n_kv_heads, head_dim /* 128 */, ffn, n_layers, max_batch /* <= 128 */;
} kf_wside_config;
typedef struct kf_wside kf_wside;
size_t kf_wside_weight_bytes(const kf_wside_config *cfg);
size_t kf_wside_weight_offset(const kf_wside_config *cfg, int32_t layer, int32_t which);
size_t kf_wside_workspace_bytes(const kf_wside_config *cfg);
int kf_wside_create(kf_wside **out, const kf_wside_config *cfg, void *weights, void *workspace, size_t workspace_bytes);
int kf_wside_destroy(kf_wside *w);
/* kf_wside_set_sms: SM budget of the GEMM kernels = CTAs of their persistent grid (0 => all SMs); takes effect for the
 *   calls that follow.  Together with kf_config.attend_sms it partitions the GPU between the W side and the A side. */
int kf_wside_set_sms(kf_wside *w, int32_t n_sms);
const char *kf_wside_last_error(const kf_wside *w);
int64_t kf_wside_launch_count(const kf_wside *w);
int kf_w_project_q(kf_wside *w, int32_t layer, const void *x, int32_t batch, void *q, kf_stream stream);
int kf_w_project_kv(kf_wside *w, int32_t layer, const void *x, int32_t batch, void *k_new, void *v_new, kf_stream stream);
int kf_w_post_attention(kf_wside *w, int32_t layer, const float *o, int32_t batch, void *x_next, kf_stream stream);

/* kf_pipeline_step -- ONE decode step of n_micro microbatches through n_layers layers, W-side stages included
 *   (Fig. 7).  Microbatch m is the batch of ctxs[m] (its own requests, routing table and KV pools;
 *   max_requests <= the kf_wside's max_batch, same head shape).  layers: [host] int32[n_layers] W-side layer of each
 *   layer of the step (its KV layer is layers[l] % the ctx's physical layers).  x: [host] n_micro [device] pointers
 *   [B_m][hidden] fp16: the hidden state entering layer 0, overwritten in place by every layer (x' of the last layer on
 *   return).  q, k_new, v_new, o, lse: [host] arrays of n_micro [device] scratch buffers (shapes as in kf_attend).
 *   Per microbatch and layer: kf_w_project_q, kf_w_project_kv, kf_kv_append, kf_attend, kf_w_post_attention; one
 *   kf_token_boundary per microbatch at the start, the step commit with the last layer's attend.
 *   pipelined == 0: everything on w_stream, microbatch after microbatch -- the serial schedule, T_p + T_A + T_f per
 *   microbatch and layer.  pipelined != 0: projections and post-attention on w_stream, append + attention on a_stream
 *   (must differ), ordered by events exactly as Fig. 7: while the A side attends one microbatch the W side finishes the
 *   previous one and projects the next; a filled pipeline completes a microbatch every max(T_p + T_f, T_A) and
 *   G_pipe = (T_p + T_A + T_f) / max(T_p + T_f, T_A).  On ONE GPU both sides share the SMs and the HBM,
 *   so kf_config.attend_sms is the knob that leaves SMs to the GEMMs.  Results are identical in both modes.
 *   Asynchronous; when w_stream has drained the step is complete. */
int kf_pipeline_step(kf_wside *w, kf_ctx *const *ctxs, int32_t n_micro, int32_t n_layers, const int32_t *layers,
                     void *const *x, void *const *q, void *const *k_new, void *const *v_new, float *const *o,
                     float *const *lse, int32_t pipelined, kf_stream w_stream, kf_stream a_stream);

/* ---- diagnostics (not part of the method; nothing here runs on the hot path) -------------------------------------
 * kf_plan_info: downloads the work-plan header into out[8] [host]: {n_units, n_tiles, n_workers_active,
 *   n_pieces, n_range_entries, tile_tokens, max_workers, n_levels}.  Synchronises `stream`.  Like kf_attend it first
 *   rebuilds the plan if a kf_step_commit happened since the last kf_token_boundary (device error ESTATE if the new
 *   tail position has no route yet): call it between kf_token_boundary and kf_step_commit.
 * kf_worker_times: per-worker timestamps of the LAST attend launch, out[max_workers][4] [host] =
 *   {SM id | (time spent streaming chunks, ns) << 8, t_start, t_first_tile_ready (0: took no chunk), t_end} in
 *   globaltimer nanoseconds; *n_workers = max_workers.  Synchronises `stream`.  KF_ESTATE unless the ctx was created
 *   with kf_config.diagnostics != 0 (only then does the attend kernel read the timer and write these words).
 * kf_probe_read (measurement aid): streams all P KV pools of the ctx once, in one launch, with plain 128-bit loads on
 *   a persistent grid and discards the data -- the read-only HBM bandwidth this box delivers to a trivial kernel, the
 *   third roofline denominator next to the nominal 8 TB/s and the measured copy bandwidth.
 *   sink: [device] 4 bytes, scratch.  *bytes_read [host, may be NULL] = P * kf_pool_bytes().  Asynchronous on `stream`;
 *   time it with events.  Not counted in kf_launch_count.
 * kf_signal_roundtrip: latency of the signalling path above, `iters` times: a two-node graph [wait gate >= seq] ->
 *   [write seq to a pinned host word] is launched on exec_stream, the host releases the gate on signal_stream and
 *   spins on the host word.  *median_us / *min_us [host] = host enqueue + GPU reaction + write visible to the host: an
 *   upper bound on "GPU store -> host sees it".  Synchronises both streams.
 * kf_route_install_latency: what a route install costs when issued from C (the paper's CPU routing loop installs a route
 *   in 7.2 us): `iters` times the active set is replaced by a neighbouring one with the kernel
 *   kf_set_active_partitions launches.  *enqueue_us_median [host] = host time of the launch call alone;
 *   *complete_us_median [host] = launch + stream synchronise (the set is in device memory, every later kernel sees it).
 *   The active set found at entry is re-published before the call returns.  Synchronises `stream`. */
int kf_route_install_latency(kf_ctx *ctx, int32_t iters, kf_stream stream, double *enqueue_us_median,
                             double *complete_us_median);
int kf_plan_info(kf_ctx *ctx, int32_t *out, kf_stream stream);
int kf_signal_roundtrip(kf_ctx *ctx, int32_t iters, kf_stream exec_stream, kf_stream signal_stream, double *median_us,
                        double *min_us);
int kf_worker_times(kf_ctx *ctx, int64_t *out, int32_t *n_workers, kf_stream stream);
int kf_probe_read(kf_ctx *ctx, void *sink, size_t *bytes_read, kf_stream stream);

#ifdef __cplusplus
}
#endif
#endif /* KFLUME_H */
