// kf_state.cu -- device-side routing table, route update at the token boundary
// (PAPER.md:149, :240), step commit, and the work plan that splits a step's attention work evenly over
// the persistent workers (warps) of the attend kernels.
#include "kf_common.cuh"

namespace kf {

// ------------------------------------------------------------------------------------------------
// allocation: one global round-robin cursor, per-partition LIFO free list then bump allocator
// (reading 9).  Called by a single thread.
// ------------------------------------------------------------------------------------------------
__device__ bool alloc_range(const Dev &d, int req) {
    const int j = d.n_ranges[req];
    if (j >= d.Jmax) {
        set_error(d, KF_ENOSPC);
        return false;
    }
    const int k = *d.rr_cursor;
    const int p = k % d.P;
    const int nfree = d.free_cnt[p];
    int slot;
    if (nfree > 0) {
        slot = d.free_stack[(size_t)p * d.slots + nfree - 1];
    } else {
        slot = d.free_head[p];
        if (slot >= d.slots) {
            set_error(d, KF_ENOSPC);
            return false;
        }
    }
    *d.rr_cursor = k + 1;
    if (nfree > 0)
        d.free_cnt[p] = nfree - 1;
    else
        d.free_head[p] = slot + 1;
    d.route_part[(size_t)req * d.Jmax + j] = p;
    d.route_slot[(size_t)req * d.Jmax + j] = slot;
    d.n_ranges[req] = j + 1;
    return true;
}

__global__ void open_request_kernel(Dev d, int req, int n_tokens) {
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    if (d.len[req] >= 0) {
        set_error(d, KF_ESTATE);
        return;
    }
    d.len[req] = n_tokens;
    d.n_ranges[req] = 0;
    const int J = (int)(((int64_t)n_tokens + d.R - 1) / d.R);
    for (int j = 0; j < J; ++j)
        if (!alloc_range(d, req)) break;
}

__global__ void close_request_kernel(Dev d, int req) {
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    if (d.len[req] < 0) {
        set_error(d, KF_ESTATE);
        return;
    }
    const int J = d.n_ranges[req];
    for (int j = 0; j < J; ++j) {
        const int p = d.route_part[(size_t)req * d.Jmax + j];
        const int s = d.route_slot[(size_t)req * d.Jmax + j];
        d.free_stack[(size_t)p * d.slots + d.free_cnt[p]] = s;
        d.free_cnt[p] += 1;
        d.route_part[(size_t)req * d.Jmax + j] = -1;
        d.route_slot[(size_t)req * d.Jmax + j] = -1;
    }
    d.n_ranges[req] = 0;
    d.len[req] = -1;
}

// (a1) route update: one warp scans the requests 32 at a time; lane 0 allocates in ascending order.
__global__ void token_boundary_kernel(Dev d) {
    const int lane = threadIdx.x;
    for (int base = 0; base < d.B; base += 32) {
        const int r = base + lane;
        bool need = false;
        if (r < d.B) {
            const int len = d.len[r];
            need = len >= 0 && (len % d.R) == 0 && d.n_ranges[r] == len / d.R;
        }
        unsigned m = __ballot_sync(0xffffffffu, need);
        if (lane == 0) {
            while (m) {
                const int b = __ffs(m) - 1;
                m &= m - 1;
                alloc_range(d, base + b);
            }
        }
        __syncwarp();
    }
}

__global__ void step_commit_kernel(Dev d) {
    const int r = blockIdx.x * blockDim.x + threadIdx.x;
    if (r < d.B && d.len[r] >= 0) d.len[r] += 1;
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

// scratch layout (ints): J[B] | S[B] | epre[B+1] | etiles[Emax] | tpre[Emax+1] | cuts[kMaxWorkers]
__global__ void __launch_bounds__(1024, 1) plan_kernel(Dev d) {
    const int tid = threadIdx.x, nt = blockDim.x;
    const int B = d.B, Emax = d.B * d.Jmax, T = kTileTokens;
    int *Jr = d.scratch;
    int *Sr = Jr + B;
    int *epre = Sr + B;
    int *etiles = epre + (B + 1);
    int *tpre = etiles + Emax;
    int *cuts = tpre + (Emax + 1);

    // 1. per request: tokens attended this step S = len + 1, ranges J = ceil(S / R)
    for (int r = tid; r < B; r += nt) {
        const int len = d.len[r];
        int64_t S = len >= 0 ? (int64_t)len + 1 : 0;
        int J = (int)((S + d.R - 1) / d.R);
        const int nr = d.n_ranges[r];
        if (J > nr) {  // no route for the tail position: kf_token_boundary was not called
            set_error(d, KF_ESTATE);
            J = nr;
            S = (int64_t)nr * d.R;
        }
        Jr[r] = J;
        Sr[r] = (int)S;
        epre[r] = J;
    }
    __syncthreads();
    const int E = block_exclusive_scan(epre, B);
    if (tid == 0) epre[B] = E;
    __syncthreads();

    // 2. per (request, range) entry: token count and tiles
    for (int e = tid; e < E; e += nt) {
        const int r = last_le(epre, B + 1, e);
        const int j = e - epre[r];
        const int cnt = min(d.R, Sr[r] - j * d.R);
        const int tiles = (cnt + T - 1) / T;
        etiles[e] = tiles;
        tpre[e] = tiles * d.Hkv;
    }
    __syncthreads();
    const int Nt = block_exclusive_scan(tpre, E);
    if (tid == 0) tpre[E] = Nt;
    __syncthreads();

    // 3. equal split of the global tile sequence over A workers
    int A = 0;
    if (Nt > 0) A = max(1, min(d.max_workers, Nt / d.min_tiles));
    for (int w = tid; w < d.max_workers; w += nt) {
        Span sp = {0, 0, 0, 0};
        int cut = 0;
        if (w < A) {
            const int start = (int)(((int64_t)w * Nt) / A);
            const int end = (int)(((int64_t)(w + 1) * Nt) / A);
            const int e = last_le(tpre, E + 1, start);
            const int rel = start - tpre[e];
            const int g = rel / etiles[e];
            sp.unit = e * d.Hkv + g;
            sp.tile_in_unit = rel - g * etiles[e];
            sp.n_tiles = end - start;
            cut = sp.tile_in_unit != 0;
        }
        d.spans[w] = sp;
        cuts[w] = cut;
    }
    __syncthreads();
    const int total_cuts = block_exclusive_scan(cuts, A);
    for (int w = tid; w < A; w += nt) {
        const int own = d.spans[w].tile_in_unit != 0;
        d.spans[w].piece = d.spans[w].unit + cuts[w] + own;
    }
    __syncthreads();

    // 4. units, with the pieces (worker spans) that intersect them
    const int U = E * d.Hkv;
    for (int u = tid; u < U; u += nt) {
        const int e = u / d.Hkv, g = u - e * d.Hkv;
        const int r = last_le(epre, B + 1, e);
        const int j = e - epre[r];
        const int tb = tpre[e] + g * etiles[e];
        const int te = tb + etiles[e];
        // number of workers whose span starts before tile x: ceil(x * A / Nt)
        const int wb = (int)(((int64_t)tb * A + Nt - 1) / Nt);
        const int we = (int)(((int64_t)te * A + Nt - 1) / Nt);
        const int cb = wb > 0 ? cuts[wb - 1] + (d.spans[wb - 1].tile_in_unit != 0) : 0;
        const int ce = we > 0 ? cuts[we - 1] + (d.spans[we - 1].tile_in_unit != 0) : 0;
        Unit un;
        un.req = r;
        un.range = j;
        un.part = d.route_part[(size_t)r * d.Jmax + j];
        un.slot = d.route_slot[(size_t)r * d.Jmax + j];
        un.cnt = min(d.R, Sr[r] - j * d.R);
        un.tile_begin = tb;
        un.piece_begin = u + cb;
        un.n_pieces = (u + 1 + ce) - (u + cb);
        d.units[u] = un;
    }
    if (tid == 0) {
        PlanHeader h;
        h.n_units = U;
        h.n_tiles = Nt;
        h.n_workers = A;
        h.n_pieces = U + total_cuts;
        h.n_entries = E;
        h.tile_tokens = T;
        h.max_workers = d.max_workers;
        h.pad = 0;
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
int launch_token_boundary(const Dev &d, cudaStream_t s) {
    token_boundary_kernel<<<1, 32, 0, s>>>(d);
    return 1;
}
int launch_plan(const Dev &d, cudaStream_t s) {
    plan_kernel<<<1, 1024, 0, s>>>(d);
    return 1;
}
int launch_step_commit(const Dev &d, cudaStream_t s) {
    step_commit_kernel<<<(d.B + 255) / 256, 256, 0, s>>>(d);
    return 1;
}

}  // namespace kf
