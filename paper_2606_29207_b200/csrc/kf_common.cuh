// kf_common.cuh -- device-side state, work plan and launch parameters shared by the kernels of libkflume.
// Product code: shares nothing with oracle/.
#pragma once

#include <cuda_fp16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/kflume.h"

namespace kf {

constexpr int kHeadDim = 128;
constexpr int kTileTokens = 16;       // work-plan granule = one MMA k-step of tokens
constexpr int kWarpsPerCta = 8;       // default workers (warps) per CTA; one worker = one warp
constexpr int kMaxWarpsPerCta = 16;
constexpr int kMaxWorkers = 2560;     // >= SMs * kMaxWarpsPerCta on any Blackwell part (148 * 16 = 2368)
constexpr int kMaxLevels = 16;        // levels of the guided self-scheduling chunk list
constexpr int kChunkSlack = 16 * kMaxWorkers;  // chunk capacity = units + kChunkSlack
constexpr int kMaxGroup = 8;          // G = H_q / H_kv
constexpr int kMaxPartitions = 64;
constexpr int kMaxGraphLayerSteps = 4096;  // layer-steps per step graph = gate words in the workspace
constexpr int kPlanStale = 1 << 30;    // plan_age value that forces a rebuild at the next token boundary

// One unit of attention work: (request, token range, kv head).  Built by the plan kernel.
struct Unit {
    int32_t req;
    int32_t range;
    int32_t part;
    int32_t slot;
    int32_t cnt;         // tokens of this range when the plan was built (1..R); see live_extent() for tail units
    int32_t tail;        // != 0: this is the request's LAST range (it grows by one token per step); value = range_begin + 1
    int32_t piece_begin; // first global piece index of this unit (pieces of a unit are consecutive, tile order)
    int32_t n_pieces;    // pieces = chunks this unit is cut into
};

// One chunk of work = one piece: a contiguous run of 16-token tiles inside ONE unit.  The chunk list is
// ordered by scheduling level (big chunks first, small chunks last: guided self-scheduling) and consumed
// through an atomic counter, so fast SMs take more chunks; the cuts themselves are static, which keeps the
// reduction order -- and therefore the result bits -- independent of which worker ran which chunk.
struct Chunk {
    int32_t unit;
    int32_t tile_begin; // first tile inside the unit
    int32_t n_tiles;    // >= 1
    int32_t piece;      // global piece index (unit-major)
};

// The same chunk as the TMA kernel wants it: ONE 64-byte record holds everything its load cursor (route, first pool
// row, tile count) and its compute cursor (request, head group, token count, piece bookkeeping, J_r) need, so a
// worker that has a ticket is one L2 load away from its first TMA -- no dependent chunk -> unit -> length chain.
struct alignas(64) ChunkRec {
    int32_t unit, tile_begin, n_tiles, piece;  // as in Chunk
    int32_t part;      // partition that holds the unit's range
    int32_t row0;      // pool row of the chunk's first token in physical layer 0: (slot * H_kv + g) * R + tile_begin * 16
    int32_t req, range;
    int32_t cnt;       // tokens of the unit when the plan was built
    int32_t flags;     // kRecTail: the unit is its request's last range; kRecStretch: this chunk holds the planned
                       // last tile of a tail unit -- the one chunk that grows while the plan is kept (live_tiles())
    int32_t n_pieces;  // pieces of the unit
    int32_t J;         // ranges of the request in this plan
    int32_t pad[4];    // [2] = range_begin of the unit; [0], [1] are filled in by the worker (q staged, append offset)
};
constexpr int kRecTail = 1, kRecStretch = 2;

struct PlanHeader {
    int32_t n_units;
    int32_t n_tiles;
    int32_t n_workers; // workers that get at least one chunk = min(max_workers, n_chunks)
    int32_t n_pieces;  // = number of chunks
    int32_t n_entries; // (request, range) entries = n_units / H_kv
    int32_t tile_tokens;
    int32_t max_workers;
    int32_t n_levels;
    int32_t max_unit_pieces;  // largest n_pieces of any unit / largest J_r of any request: the fused merge sizes its
    int32_t max_J;            // tasks from them (how many heads one warp merges per round trip, kf_merge.cuh)
};

// Device pointers into the caller's workspace + immutable config.  Passed BY VALUE to every kernel.
struct Dev {
    // config
    int32_t Hq, Hkv, G, L, R, P, B, Jmax, slots;
    int32_t max_workers, min_tiles;
    int32_t warps_per_cta, stages;      // launch shape of the attend kernels
    int32_t l2_hint;                    // 1: K/V tiles are loaded with an L2 evict-first policy
    int32_t diag;                       // 1: the attend kernel records per-worker timestamps (worker_times)
    int32_t max_chunks;                 // capacity of chunks[] and of the piece buffers
    int32_t plan_refresh;               // a plan is rebuilt after this many token boundaries (or when routes change)
    float sched_first, sched_decay;     // GSS factor rho (chunk <= rho * remaining / workers); share of a unit's remaining tiles per level
    float scale_log2;  // softmax_scale * log2(e)
    // routing state
    int32_t *len;        // [B]   -1 = closed
    int32_t *n_ranges;   // [B]
    int32_t *route_part; // [B][Jmax]
    int32_t *route_slot; // [B][Jmax]
    int32_t *range_begin; // [B][Jmax] first token position of range j (j * R unless a tail was redirected, reading 28)
    int32_t *redirect;   // [P]   1: tails on this partition move to a new range at the next token boundary (one-shot)
    int32_t *rr_cursor;  // [1]   ranges allocated so far
    int32_t *rr_last;    // [1]   partition of the last allocation (-1: none yet)
    int32_t *req_active; // [B]   1: the request takes part in decode steps (kf_set_active_requests); 0: paused
    int32_t *active;     // [P]   1: partition receives new ranges (the published active set)
    long long *part_tokens;  // [P] scratch of kf_partition_state
    int32_t *part_tails;     // [P]
    int32_t *free_head;  // [P]
    int32_t *free_cnt;   // [P]
    int32_t *free_stack; // [P][slots]
    int32_t *error;      // [1]
    // work plan
    PlanHeader *plan;
    Unit *units;            // [B*Jmax*Hkv]
    Chunk *chunks;          // [max_chunks]
    ChunkRec *recs;         // [max_chunks]  the chunk list again, self-contained records for the TMA kernel
    int32_t *plan_age;      // [0] token boundaries served by the current plan
    int32_t *sched;         // [0] chunk counter (dynamic part of the list), [1] finished-worker counter
    int32_t *scratch;       // plan scratch: [B] J, [B] S, [B+1] entry prefix, [E] tiles, [E+1] tile prefix,
                            //               [E+1] piece prefix, [kMaxLevels*E+1] chunk prefix
    int32_t *unit_counter;  // [B*Jmax*Hkv]  last-arriver counters (self-resetting)
    int32_t *group_counter; // [B*Hkv]
    // partial buffers
    float *piece_o;   // [max_chunks][G][128]
    float *piece_lse; // [max_chunks][G]
    float *range_o;   // [B][Jmax][Hq][128]  scratch when the caller passes no o_part
    float *range_lse; // [B][Jmax][Hq]
    // staging for kf_layer_step_host
    __half *stage_q, *stage_k, *stage_v; // [B][Hq][128], [B][Hkv][128] x2
    float *stage_o, *stage_lse;          // [B][Hq][128], [B][Hq]
    // pools
    unsigned char *pool[kMaxPartitions];
    size_t v_off;        // byte offset of the V half of a pool
    const void *tmaps;   // [P][2] CUtensorMap (K, V) in device memory, 128-byte stride
    uint32_t *gates;     // [kMaxGraphLayerSteps] gate words of the signalled step graph (kf_step_graph_flags)
    long long *worker_times;  // [kMaxWorkers][4]: {smid, t_start, t_first_tile, t_end} (globaltimer ns), diagnostics
};

struct AttendParams {
    Dev d;
    int32_t layer;
    const __half *q; // [B][Hq][128]
    float *o_part;   // [B][Jmax][Hq][128]
    float *lse_part; // [B][Jmax][Hq]
    float *o;        // [B][Hq][128] (fused only)
    float *lse;      // [B][Hq]
    uint64_t part_mask;
    int32_t fused;
    int32_t commit;  // 1: the last worker of this launch performs the step commit (static step graph only)
    // (a2) fused into the launch (static step graph, TMA kernel): [B][H_kv][128] or nullptr.  The worker that attends
    // the tail tile of (request, kv head) writes the new K/V row to the pool and patches it into its shared-memory
    // copy of that tile, so the step needs no separate kf_kv_append launch in front of the attention.
    const __half *k_new, *v_new;
};

__device__ __forceinline__ void set_error(const Dev &d, int code) { atomicCAS(d.error, 0, code); }

// A work plan outlives the step it was built in (it is rebuilt when a route changes or after plan_refresh
// boundaries): the only thing that moves in between is the length of each request's TAIL range, +1 token per step.
// So the token count of a tail unit is re-derived from len at run time, and the chunk that covers the planned end
// of a tail unit (always the last chunk of scheduling level 0: one of the first and largest chunks) is stretched
// to the live end.  Every other chunk is exactly as planned.
__device__ __forceinline__ int live_cnt(const Dev &d, const Unit &un) {
    return un.tail ? min(d.R, __ldg(d.len + un.req) + 1 - (un.tail - 1)) : un.cnt;
}
__device__ __forceinline__ int live_tiles(const Unit &un, int cnt_live, int tile_begin, int n_tiles) {
    const int planned = (un.cnt + kTileTokens - 1) / kTileTokens;
    return (un.tail && tile_begin + n_tiles == planned) ? (cnt_live + kTileTokens - 1) / kTileTokens - tile_begin
                                                        : n_tiles;
}

// (a5) does request r advance at the step commit?  Open, taking part in the step, and its tail position had a route:
// a request whose boundary could not get a slot (ENOSPC) appended nothing, so it must not move on -- the next
// kf_token_boundary re-tries the allocation at the same position (reading 24).
__device__ __forceinline__ bool commits(const Dev &d, int r) {
    const int len = d.len[r], nr = d.n_ranges[r];
    return len >= 0 && d.req_active[r] && nr > 0 && len - d.range_begin[(size_t)r * d.Jmax + nr - 1] < d.R;
}

// byte offset (within a partition pool) of K row (layer, slot, g, t)
__device__ __forceinline__ size_t row_offset(const Dev &d, int layer, int slot, int g, int t) {
    return ((((size_t)layer * d.slots + slot) * d.Hkv + g) * d.R + t) * (size_t)(kHeadDim * 2);
}

// host-side launchers (definitions in the respective .cu files); each returns the number of kernels launched
// or a negative KF_E* code.
int launch_open_request(const Dev &d, int req, int n_tokens, cudaStream_t s);
int launch_close_request(const Dev &d, int req, cudaStream_t s);
int launch_plan(const Dev &d, int do_boundary, cudaStream_t s);  // (a1, optional) + work plan, one launch
int plan_setup();        // cudaFuncSetAttribute for the plan kernel's dynamic shared memory; 0 or KF_ECUDA
int launch_step_commit(const Dev &d, cudaStream_t s);
int launch_set_active(const Dev &d, unsigned long long mask, cudaStream_t s);
int launch_redirect(const Dev &d, unsigned long long mask, cudaStream_t s);
int launch_set_req_active(const Dev &d, const unsigned char *mask_dev, cudaStream_t s);
int launch_partition_state(const Dev &d, long long *tokens, int *tails, cudaStream_t s);
int launch_load_context(const Dev &d, int layer, int req, int tok_begin, int n_tokens, const __half *k,
                        const __half *v, cudaStream_t s);
int launch_kv_append(const Dev &d, int layer, const __half *k_new, const __half *v_new, cudaStream_t s);
int launch_kv_append_stage(const Dev &d, int layer, const __half *k_new, const __half *v_new, const __half *q_src,
                           __half *q_dst, cudaStream_t s);
int launch_attend_simple(const AttendParams &p, int n_ctas, cudaStream_t s);
int launch_attend_tma(const AttendParams &p, int n_ctas, cudaStream_t s);
bool attend_tma_shape_ok(int warps, int stages);
int attend_tma_setup();  // cudaFuncSetAttribute for the dynamic shared memory; 0 or KF_ECUDA
int launch_merge_units(const AttendParams &p, int n_ctas, cudaStream_t s);
int launch_merge_ranges(const Dev &d, const float *o_part, const float *lse_part, float *o, float *lse,
                        cudaStream_t s);

}  // namespace kf
