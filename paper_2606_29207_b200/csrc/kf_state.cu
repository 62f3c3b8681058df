// kf_state.cu -- device-side routing table, route update at the token boundary
// (PAPER.md:149, :240), step commit, and the work plan that splits a step's attention work evenly over
// the persistent workers (warps) of the attend kernels.
#include "kf_common.cuh"

namespace kf {

// ------------------------------------------------------------------------------------------------
// allocation: one global round-robin cursor, per-partition LIFO free list then bump allocator
// (reading 9).  Called by a single thread.
// ------------------------------------------------------------------------------------------------
// `begin` = first token position of the new range; `quiet`: a failure is not an error (a tail redirect that finds no
// room is simply not carried out, reading 28).
__device__ bool alloc_range(const Dev &d, int req, int begin, bool quiet = false) {
    const int j = d.n_ranges[req];
    if (j >= d.Jmax) {
        if (!quiet) set_error(d, KF_ENOSPC);
        return false;
    }
    // round-robin over the ACTIVE partitions: the first active one after the partition used last, cyclically
    // (with every partition active this is "the k-th range ever allocated goes to partition k mod P").  A full
    // partition is passed over (reading 24): ENOSPC is latched only when NO active partition has a free
    // slot -- e.g. after a scale-down left fewer nodes than the pools were sized for.
    const int k = *d.rr_cursor;
    const int last = *d.rr_last;
    int p = -1;
    for (int i = 1; i <= d.P; ++i) {
        const int c = (last + i) % d.P;
        if (d.active[c] && (d.free_cnt[c] > 0 || d.free_head[c] < d.slots)) {
            p = c;
            break;
        }
    }
    if (p < 0) {
        if (!quiet) set_error(d, KF_ENOSPC);
        return false;
    }
    const int nfree = d.free_cnt[p];
    const int slot = nfree > 0 ? d.free_stack[(size_t)p * d.slots + nfree - 1] : d.free_head[p];
    *d.rr_cursor = k + 1;
    *d.rr_last = p;
    if (nfree > 0)
        d.free_cnt[p] = nfree - 1;
    else
        d.free_head[p] = slot + 1;
    d.route_part[(size_t)req * d.Jmax + j] = p;
    d.route_slot[(size_t)req * d.Jmax + j] = slot;
    d.range_begin[(size_t)req * d.Jmax + j] = begin;
    d.n_ranges[req] = j + 1;
    return true;
}

__global__ void open_request_kernel(Dev d, int req, int n_tokens) {
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    if (d.len[req] >= 0) {
        set_error(d, KF_ESTATE);
        return;
    }
    *d.plan_age = kPlanStale;  // routes edited: the next plan kernel must rebuild
    d.len[req] = n_tokens;
    d.n_ranges[req] = 0;
    const int J = (int)(((int64_t)n_tokens + d.R - 1) / d.R);
    for (int j = 0; j < J; ++j)
        if (!alloc_range(d, req, j * d.R)) break;
}

__global__ void close_request_kernel(Dev d, int req) {
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    if (d.len[req] < 0) {
        set_error(d, KF_ESTATE);
        return;
    }
    *d.plan_age = kPlanStale;
    const int J = d.n_ranges[req];
    for (int j = 0; j < J; ++j) {
        const int p = d.route_part[(size_t)req * d.Jmax + j];
        const int s = d.route_slot[(size_t)req * d.Jmax + j];
        d.free_stack[(size_t)p * d.slots + d.free_cnt[p]] = s;
        d.free_cnt[p] += 1;
        d.route_part[(size_t)req * d.Jmax + j] = -1;
        d.route_slot[(size_t)req * d.Jmax + j] = -1;
        d.range_begin[(size_t)req * d.Jmax + j] = -1;
    }
    d.n_ranges[req] = 0;
    d.len[req] = -1;
}

// (a1) route update: one warp scans the requests 32 at a time; lane 0 allocates in ascending order.
// returns (in every lane) the number of ranges opened, i.e. of route entries appended
__device__ int token_boundary_warp(const Dev &d, int lane) {
    int opened = 0;
    for (int base = 0; base < d.B; base += 32) {
        const int r = base + lane;
        bool need = false, redir = false;
        if (r < d.B) {
            const int len = d.len[r];
            if (len >= 0 && d.req_active[r]) {
                const int nr = d.n_ranges[r];
                const int bt = nr > 0 ? d.range_begin[(size_t)r * d.Jmax + nr - 1] : 0;
                // the tail position has no route yet: the tail range is full (len - begin == R; len % R == 0 without
                // redirects) -- or an earlier boundary could not get a slot for it (ENOSPC) and the request has been
                // waiting since (reading 24)
                need = nr == 0 || len - bt >= d.R;
                // reading 28 (Algorithm 1 l.16-17): the tail lives on a node whose tails are being redirected and holds
                // at least one token: close it here, continue in a new range that begins at position len
                redir = !need && len > bt && d.redirect[d.route_part[(size_t)r * d.Jmax + nr - 1]] != 0;
            }
        }
        const unsigned mr = __ballot_sync(0xffffffffu, redir);
        unsigned m = __ballot_sync(0xffffffffu, need) | mr;
        // only allocations that SUCCEEDED change a route (and with it the work plan): a request that waits for a slot
        // (reading 24) asks again at every boundary, and a redirect that finds no slot is dropped quietly -- neither may
        // force a plan rebuild step after step
        int done = 0;
        if (lane == 0) {
            while (m) {
                const int b = __ffs(m) - 1;
                m &= m - 1;
                done += alloc_range(d, base + b, d.len[base + b], (mr >> b) & 1u) ? 1 : 0;
            }
        }
        opened += __shfl_sync(0xffffffffu, done, 0);
        __syncwarp();
    }
    if (lane < d.P) d.redirect[lane] = 0;  // the marks are consumed by this boundary (P <= 64: two passes)
    if (lane + 32 < d.P) d.redirect[lane + 32] = 0;
    return opened;
}

// publish a new active set (scale-up / scale-down event): affects FUTURE ranges only
__global__ void set_active_kernel(Dev d, unsigned long long mask) {
    const int p = threadIdx.x;
    if (p < d.P) d.active[p] = (int)((mask >> p) & 1ull);
}

// mark partitions whose tails move at the next token boundary (Algorithm 1 l.17, reading 28)
__global__ void redirect_kernel(Dev d, unsigned long long mask) {
    const int p = threadIdx.x;
    if (p < d.P) d.redirect[p] = (int)((mask >> p) & 1ull);
}

// which open requests take part in the following decode steps (continuous batching: a request may pause);
// mask == nullptr: all.  The plan depends on it: aged to stale.
__global__ void set_req_active_kernel(Dev d, const unsigned char *mask) {
    const int r = blockIdx.x * blockDim.x + threadIdx.x;
    if (r < d.B) d.req_active[r] = mask ? (mask[r] ? 1 : 0) : 1;
    if (r == 0) *d.plan_age = kPlanStale;
}

// per-partition occupancy for the scaling policy (Algorithm 1, l.6-9): committed tokens resident on partition p
// and the number of open requests whose tail range lives there.  One thread per request, atomics on [P] words.
__global__ void partition_state_kernel(Dev d, long long *tokens, int *tails) {
    const int r = blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= d.B) return;
    const int len = d.len[r];
    if (len < 0) return;
    const int J = d.n_ranges[r];
    for (int j = 0; j < J; ++j) {
        const int p = d.route_part[(size_t)r * d.Jmax + j];
        const int bj = d.range_begin[(size_t)r * d.Jmax + j];
        const long long cnt = j + 1 < J ? d.range_begin[(size_t)r * d.Jmax + j + 1] - bj : max(0, min(d.R, len - bj));
        atomicAdd(reinterpret_cast<unsigned long long *>(tokens + p), (unsigned long long)cnt);
        if (j == J - 1 && d.req_active[r]) atomicAdd(tails + p, 1);  // "r active" (Alg. 1 l.7)
    }
}

__global__ void step_commit_kernel(Dev d) {
    const int r = blockIdx.x * blockDim.x + threadIdx.x;
    if (r < d.B && commits(d, r)) d.len[r] += 1;
}

// ------------------------------------------------------------------------------------------------
// work plan
// ------------------------------------------------------------------------------------------------
// in-place exclusive scan of data[0..n) by the whole block; returns the total (valid in all threads)
__device__ int block_exclusive_scan(int *data, int n) {
    __shared__ int warp_sums[32];
    __shared__ int carry_s;
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5, nw = blockDim.x >> 5;
    if (tid == 0) carry_s = 0;
    __syncthreads();
    for (int base = 0; base < n; base += blockDim.x) {
        const int i = base + tid;
        const int v = i < n ? data[i] : 0;
        int x = v;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int y = __shfl_up_sync(0xffffffffu, x, o);
            if (lane >= o) x += y;
        }
        if (lane == 31) warp_sums[wid] = x;
        __syncthreads();
        if (wid == 0) {
            int s = lane < nw ? warp_sums[lane] : 0;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int y = __shfl_up_sync(0xffffffffu, s, o);
                if (lane >= o) s += y;
            }
            warp_sums[lane] = s;
        }
        __syncthreads();
        const int carry = carry_s;
        const int prefix = carry + (wid > 0 ? warp_sums[wid - 1] : 0) + x - v;
        if (i < n) data[i] = prefix;
        __syncthreads();
        if (tid == 0) carry_s = carry + warp_sums[nw - 1];
        __syncthreads();
    }
    return carry_s;
}

// largest i in [0, n) with a[i] <= x   (a non-decreasing, a[0] <= x)
__device__ __forceinline__ int last_le(const int *a, int n, int x) {
    int lo = 0, hi = n - 1;
    while (lo < hi) {
        const int mid = (lo + hi + 1) >> 1;
        if (a[mid] <= x)
            lo = mid;
        else
            hi = mid - 1;
    }
    return lo;
}

// ---- guided self-scheduling ----------------------------------------------------------------------------
// Chunk sizes follow guided self-scheduling: a chunk that starts at position `pos` of the step's tile sequence
// (Nt tiles, W workers) holds at most  rho * (Nt - pos) / W  tiles, never fewer than min_tiles -- so whichever
// worker takes it, and however slow its SM, it finishes before the rest of the work can run out.
// The tile sequence is LEVEL-major: every unit (n tiles) is cut at the same relative positions -- level 0 takes
// the first `decay` of its tiles, every later level `decay` of what is left, the last level the rest -- and
// the sequence visits the level-0 portions of all units, then the level-1 portions, ...  So the small chunks at
// the end of the launch are spread over all units (each unit ends up with a few pieces per level) instead of
// shredding the last units into hundreds of pieces.
struct Levels {
    int K;
    int end16[kMaxLevels];  // cumulative fraction at the end of level k, 16-bit fixed point (last = 65536)
};

__device__ void make_levels(Levels &lv, long long Nt, int W, int m, float f) {
    const double base = (double)Nt / (double)W;
    double cum = 0.0;
    int K = 0;
    for (;;) {
        const double phi = (1.0 - cum) * f;
        // stop when what is left per worker is about two minimum chunks
        if ((1.0 - cum) * base <= 2.0 * m || K == kMaxLevels - 1 || f > 0.9995f) {
            lv.end16[K++] = 65536;
            break;
        }
        cum += phi;
        lv.end16[K++] = (int)(cum * 65536.0);
    }
    lv.K = K;
}

// tiles [b0, b0 + len) of a unit with n tiles belong to level k.  Levels run from the END of the unit towards its
// start and round up, so level 0 -- the first and largest chunks of the launch -- always holds the unit's last
// tile: the one place where a tail unit grows between plan rebuilds (live_tiles(), kf_common.cuh).
__device__ __forceinline__ void level_span(const Levels &lv, int n, int k, int m, int &b0, int &len) {
    // a level that would leave fewer than m (the smallest chunk) tiles to the later ones takes them too: small
    // units end up as one or two pieces instead of one sliver per level
    int lo = k == 0 ? 0 : (int)(((long long)n * lv.end16[k - 1] + 65535) >> 16);
    int hi = (int)(((long long)n * lv.end16[k] + 65535) >> 16);
    if (k > 0 && n - lo < m) lo = n;
    if (n - hi < m) hi = n;
    b0 = n - hi;
    len = hi - lo;
}

// scratch (ints): J[B] (always global: the attend kernels read it) | S[B] | epre[B+1] | etiles[E] | tpre[E+1] |
//                 ppre[E+1] | pos[K*E+1] | ccnt[K*E] | lpre[K*E+1]
// Every array other than J lives in shared memory when it fits (it does for all BASELINE configs) and in the
// global scratch area otherwise: the plan is a chain of ~15 dependent phases, and a global round trip per phase
// is what made this kernel cost 30 us.  With do_boundary != 0 the kernel first performs the route update (a1).
constexpr int kPlanSmemInts = 48 * 1024;  // 192 KB of dynamic shared memory

__global__ void __launch_bounds__(1024, 1) plan_kernel(Dev d, int do_boundary) {
    extern __shared__ int plan_smem[];
    __shared__ Levels lv;
    __shared__ int s_m, s_keep, s_max_pieces, s_max_J;
    const int tid = threadIdx.x, nt = blockDim.x;
    const int B = d.B, Emax = d.B * d.Jmax, T = kTileTokens, Hkv = d.Hkv;
    if (do_boundary) {
        // keep the current plan if no range was opened and it is younger than plan_refresh boundaries
        // (kf_open_request / kf_close_request / kf_create age it to kPlanStale: always rebuilt)
        if (tid < 32) {
            const int opened = token_boundary_warp(d, tid);
            if (tid == 0) {
                const int age = *d.plan_age;
                const bool keep = opened == 0 && age + 1 < d.plan_refresh;
                *d.plan_age = keep ? age + 1 : 0;
                s_keep = keep ? 1 : 0;
            }
        }
        __syncthreads();
    } else if (tid == 0) {
        *d.plan_age = 0;
    }
    if (do_boundary && s_keep) return;
    int used = 0;
    auto take = [&](int n, int *fallback) -> int * {
        if (used + n <= kPlanSmemInts) {
            int *p = plan_smem + used;
            used += n;
            return p;
        }
        return fallback;
    };
    int *Jr = d.scratch;
    int *g_Sr = Jr + B, *g_epre = g_Sr + B, *g_etiles = g_epre + (B + 1), *g_tpre = g_etiles + Emax;
    int *g_ppre = g_tpre + (Emax + 1), *g_pos = g_ppre + (Emax + 1);
    int *g_ccnt = g_pos + ((size_t)kMaxLevels * Emax + 1), *g_lpre = g_ccnt + (size_t)kMaxLevels * Emax;
    int *Sr = take(B, g_Sr);
    int *epre = take(B + 1, g_epre);
    int *etiles = nullptr, *tpre = nullptr, *ppre = nullptr, *pos = nullptr, *ccnt = nullptr, *lpre = nullptr;

    if (tid == 0) s_max_pieces = s_max_J = 0;
    __syncthreads();
    // 1. per request: tokens attended this step S = len + 1, ranges J = ceil(S / R)
    for (int r = tid; r < B; r += nt) {
        const int len = d.len[r];
        int64_t S = (len >= 0 && d.req_active[r]) ? (int64_t)len + 1 : 0;  // closed or paused: no work this step
        const int nr = d.n_ranges[r];
        int J = S > 0 ? nr : 0;
        if (S > 0) {
            const int bt = nr > 0 ? d.range_begin[(size_t)r * d.Jmax + nr - 1] : 0;
            if (nr == 0 || len - bt >= d.R) {  // no route for the tail position: kf_token_boundary was not called
                set_error(d, KF_ESTATE);
                S = nr == 0 ? 0 : (int64_t)bt + d.R;
            }
        }
        Jr[r] = J;
        Sr[r] = (int)S;
        epre[r] = J;
        if (J > 1) atomicMax(&s_max_J, J);
    }
    __syncthreads();
    const int E = block_exclusive_scan(epre, B);
    if (tid == 0) epre[B] = E;
    etiles = take(E, g_etiles);
    tpre = take(E + 1, g_tpre);
    ppre = take(E + 1, g_ppre);
    __syncthreads();

    // 2. per (request, range) entry: token count and tiles (identical for the H_kv units of the entry)
    for (int e = tid; e < E; e += nt) {
        const int r = last_le(epre, B + 1, e);
        const int j = e - epre[r];
        const int *bg = d.range_begin + (size_t)r * d.Jmax;
        const int cnt = (j + 1 < Jr[r] ? bg[j + 1] : Sr[r]) - bg[j];  // ranges are [begin_j, begin_j+1); the tail ends at S
        const int tiles = (cnt + T - 1) / T;
        etiles[e] = tiles;
        tpre[e] = tiles * Hkv;
    }
    __syncthreads();
    const int Nt = block_exclusive_scan(tpre, E);
    if (tid == 0) {
        tpre[E] = Nt;
        // smallest chunk: fewer, larger pieces pay off once every worker has real work (measured: 8..12 beat 4 by
        // 1-7% from 64K context tokens up), while a latency-bound launch wants all the parallelism it can get
        s_m = d.min_tiles > 0 ? d.min_tiles : (Nt >= 16 * d.max_workers ? 12 : 4);
    }
    __syncthreads();

    // 3. levels, positions in the level-major tile sequence, chunk counts per (level, entry);
    //    coarsen (double min_tiles) until the chunk list fits its buffer
    const int W = d.max_workers;
    const float rho = d.sched_first;
    int n_chunks = 0;
    for (int iter = 0; iter < 32; ++iter) {
        if (tid == 0) make_levels(lv, Nt, W, s_m, d.sched_decay);
        __syncthreads();
        const int KE = lv.K * E, m = s_m;
        if (iter == 0) {  // K only shrinks when min_tiles is coarsened
            pos = take(KE + 1, g_pos);
            ccnt = take(KE, g_ccnt);
            lpre = take(KE + 1, g_lpre);
        }
        for (int idx = tid; idx < KE; idx += nt) {
            const int k = idx / E, e = idx - k * E;
            int b0, len;
            level_span(lv, etiles[e], k, m, b0, len);
            pos[idx] = len * Hkv;
        }
        __syncthreads();
        block_exclusive_scan(pos, KE);
        __syncthreads();
        for (int idx = tid; idx < KE; idx += nt) {
            const int k = idx / E, e = idx - k * E;
            int b0, len;
            level_span(lv, etiles[e], k, m, b0, len);
            const float left = (float)(Nt - pos[idx]);
            const int size = max(m, (int)ceilf(rho * left / (float)W));
            const int c = (len + size - 1) / size;
            ccnt[idx] = c;
            lpre[idx] = c * Hkv;
        }
        __syncthreads();
        n_chunks = block_exclusive_scan(lpre, KE);
        if (tid == 0) lpre[KE] = n_chunks;
        __syncthreads();
        if (n_chunks <= d.max_chunks) break;
        if (tid == 0) s_m = s_m >= (1 << 28) ? s_m : s_m * 2;
        __syncthreads();
    }
    const int K = lv.K;

    // 4. pieces per entry (per kv head) -> piece prefix
    for (int e = tid; e < E; e += nt) {
        int pu = 0;
        for (int k = 0; k < K; ++k) pu += ccnt[k * E + e];
        ppre[e] = pu;
        if (pu > 1) atomicMax(&s_max_pieces, pu);
    }
    __syncthreads();
    const int pieces_per_head = block_exclusive_scan(ppre, E);
    if (tid == 0) ppre[E] = pieces_per_head;
    __syncthreads();

    // 5. chunk descriptors in level-major order; piece index = unit-major, (level, tile) order inside the unit
    const int items = K * E * Hkv;
    for (int idx = tid; idx < items; idx += nt) {
        const int k = idx / (E * Hkv);
        const int rem = idx - k * (E * Hkv);
        const int e = rem / Hkv, g = rem - e * Hkv;
        const int c = ccnt[k * E + e];
        if (c == 0) continue;
        int b0, len;
        level_span(lv, etiles[e], k, s_m, b0, len);
        int before = 0;
        for (int kk = 0; kk < k; ++kk) before += ccnt[kk * E + e];
        const int pu = ppre[e + 1] - ppre[e];
        const int piece0 = ppre[e] * Hkv + g * pu + before;
        const int chunk0 = lpre[k * E + e] + g * c;
        const int cq = len / c, cr = len - cq * c;  // the first cr chunks hold cq + 1 tiles
        const int r = last_le(epre, B + 1, e);
        const int j = e - epre[r];
        ChunkRec rec;
        rec.unit = e * Hkv + g;
        rec.part = d.route_part[(size_t)r * d.Jmax + j];
        const int slot = d.route_slot[(size_t)r * d.Jmax + j];
        rec.req = r;
        rec.range = j;
        const int *bg = d.range_begin + (size_t)r * d.Jmax;
        rec.cnt = (j + 1 < Jr[r] ? bg[j + 1] : Sr[r]) - bg[j];
        rec.n_pieces = pu;
        rec.J = Jr[r];
        rec.pad[0] = rec.pad[1] = rec.pad[3] = 0;
        rec.pad[2] = bg[j];
        const int tail = j == Jr[r] - 1 ? kRecTail : 0;
        for (int i = 0; i < c; ++i) {
            const int t0 = b0 + i * cq + min(i, cr);
            const int t1 = b0 + (i + 1) * cq + min(i + 1, cr);
            Chunk ch;
            ch.unit = e * Hkv + g;
            ch.tile_begin = t0;
            ch.n_tiles = t1 - t0;
            ch.piece = piece0 + i;
            d.chunks[chunk0 + i] = ch;
            rec.tile_begin = t0;
            rec.n_tiles = t1 - t0;
            rec.piece = piece0 + i;
            rec.row0 = (slot * Hkv + g) * d.R + t0 * T;
            rec.flags = tail | (tail && t1 == etiles[e] ? kRecStretch : 0);
            d.recs[chunk0 + i] = rec;
        }
    }

    // 6. units
    const int U = E * Hkv;
    for (int u = tid; u < U; u += nt) {
        const int e = u / Hkv, g = u - e * Hkv;
        const int r = last_le(epre, B + 1, e);
        const int j = e - epre[r];
        const int pu = ppre[e + 1] - ppre[e];
        Unit un;
        un.req = r;
        un.range = j;
        un.part = d.route_part[(size_t)r * d.Jmax + j];
        un.slot = d.route_slot[(size_t)r * d.Jmax + j];
        const int *bg = d.range_begin + (size_t)r * d.Jmax;
        un.cnt = (j + 1 < Jr[r] ? bg[j + 1] : Sr[r]) - bg[j];
        un.tail = j == Jr[r] - 1 ? bg[j] + 1 : 0;
        un.piece_begin = ppre[e] * Hkv + g * pu;
        un.n_pieces = pu;
        d.units[u] = un;
    }
    if (tid == 0) {
        PlanHeader h;
        h.n_units = U;
        h.n_tiles = Nt;
        h.n_workers = min(W, n_chunks);
        h.n_pieces = n_chunks;
        h.n_entries = E;
        h.tile_tokens = T;
        h.max_workers = W;
        h.n_levels = K;
        h.max_unit_pieces = s_max_pieces;
        h.max_J = s_max_J;
        *d.plan = h;
    }
}

// ------------------------------------------------------------------------------------------------
int launch_open_request(const Dev &d, int req, int n_tokens, cudaStream_t s) {
    open_request_kernel<<<1, 32, 0, s>>>(d, req, n_tokens);
    return 1;
}
int launch_close_request(const Dev &d, int req, cudaStream_t s) {
    close_request_kernel<<<1, 32, 0, s>>>(d, req);
    return 1;
}
// do_boundary != 0: route update (a1) followed by the work plan, in one launch
int launch_plan(const Dev &d, int do_boundary, cudaStream_t s) {
    plan_kernel<<<1, 1024, kPlanSmemInts * sizeof(int), s>>>(d, do_boundary);
    return 1;
}
int plan_setup() {
    return cudaFuncSetAttribute(plan_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                (int)(kPlanSmemInts * sizeof(int))) == cudaSuccess
               ? 0
               : KF_ECUDA;
}
int launch_set_active(const Dev &d, unsigned long long mask, cudaStream_t s) {
    set_active_kernel<<<1, kMaxPartitions, 0, s>>>(d, mask);
    return 1;
}
int launch_redirect(const Dev &d, unsigned long long mask, cudaStream_t s) {
    redirect_kernel<<<1, kMaxPartitions, 0, s>>>(d, mask);
    return 1;
}
int launch_set_req_active(const Dev &d, const unsigned char *mask_dev, cudaStream_t s) {
    set_req_active_kernel<<<(d.B + 127) / 128, 128, 0, s>>>(d, mask_dev);
    return 1;
}
int launch_partition_state(const Dev &d, long long *tokens, int *tails, cudaStream_t s) {
    partition_state_kernel<<<(d.B + 127) / 128, 128, 0, s>>>(d, tokens, tails);
    return 1;
}
int launch_step_commit(const Dev &d, cudaStream_t s) {
    step_commit_kernel<<<(d.B + 255) / 256, 256, 0, s>>>(d);
    return 1;
}

}  // namespace kf
