// Trigger and event counts — the paper's own outputs on top of the edge diff.
//   PAPER.md:215-221 (§III.B.3): every row of the translated past adjacency list is compared with its
//   isomorphic row of the present one; a vertex whose rows differ gets local_trigger = 1 and
//   global_trigger tells whether any did.  Rows differ exactly for the endpoints of the created and
//   destroyed edges, which vor_diff already produced, so the trigger is a scatter over those lists.
//   PAPER.md:229 (§III.B.4): the triggering indices go to eventsIndices, their number to eventsNumber
//   (an order-preserving compaction of the trigger array).
//   eventsCount = for every active vertex, how many active vertices are connected to it,
//   in each of the two triangulations (the paper's triple loop; here one pass over each edge list with
//   two atomics per edge whose endpoints are both active).
// All lists live in ONE index space (site path: persistent identity; field path: the translated /
// filtered lists).
#include "common.cuh"

namespace {

constexpr int kEvThreads = 512;
constexpr int kEvItems = 8;
constexpr int kEvBatch = kEvThreads * kEvItems;

__global__ void ev_mark_kernel(const uint64_t* __restrict__ created, const int64_t* __restrict__ n_created,
                               const uint64_t* __restrict__ destroyed, const int64_t* __restrict__ n_destroyed,
                               int64_t cap_created, int64_t cap_destroyed, int32_t n,
                               int32_t* __restrict__ trigger) {
    const int64_t nc = min(*n_created, cap_created), nd = min(*n_destroyed, cap_destroyed);
    for (int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; k < nc + nd; k += (int64_t)gridDim.x * blockDim.x) {
        const uint64_t e = k < nc ? created[k] : destroyed[k - nc];
        const uint32_t i = (uint32_t)(e >> 32), j = (uint32_t)e;
        if (i >= (uint32_t)n || j >= (uint32_t)n) continue;     // keys with a label >= n_labels are ignored
        trigger[i] = 1;
        trigger[j] = 1;
    }
}

__device__ __forceinline__ void ev_chunk(int64_t n, int64_t* beg, int64_t* end) {
    int64_t C = (n + gridDim.x - 1) / gridDim.x;
    C = (C + 32 * kEvItems - 1) / (32 * kEvItems) * (32 * kEvItems);     // whole warp tiles
    const int64_t s = (int64_t)blockIdx.x * C;
    *beg = s < n ? s : n;
    *end = s + C < n ? s + C : n;
}

__device__ __forceinline__ int64_t ev_block_sum(int64_t v, int64_t* sh) {
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    if (lane == 0) sh[wid] = v;
    __syncthreads();
    int64_t t = lane < (int)(blockDim.x >> 5) ? sh[lane] : 0;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
    __syncthreads();
    return t;
}

__global__ void __launch_bounds__(kEvThreads) ev_count_kernel(const int32_t* __restrict__ trigger, int32_t n,
                                                              int64_t* __restrict__ partial) {
    __shared__ int64_t sh[32];
    int64_t beg, end;
    ev_chunk(n, &beg, &end);
    int64_t c = 0;
    for (int64_t i = beg + threadIdx.x; i < end; i += kEvThreads) c += trigger[i] != 0;
    c = ev_block_sum(c, sh);
    if (threadIdx.x == 0) partial[blockIdx.x] = c;
}

// eventsIndices = ascending indices of the active vertices; eventsNumber; global_trigger
__global__ void __launch_bounds__(kEvThreads) ev_write_kernel(const int32_t* __restrict__ trigger, int32_t n,
                                                              const int64_t* __restrict__ partial,
                                                              int32_t* __restrict__ events_indices,
                                                              int32_t* __restrict__ events_number,
                                                              int32_t* __restrict__ global_trigger) {
    __shared__ int64_t sh[32];
    __shared__ int32_t wtot[kEvThreads / 32];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    int64_t beg, end;
    ev_chunk(n, &beg, &end);
    int64_t before = 0, all = 0;
    for (int b = threadIdx.x; b < (int)gridDim.x; b += kEvThreads) {
        const int64_t v = partial[b];
        all += v;
        if (b < (int)blockIdx.x) before += v;
    }
    before = ev_block_sum(before, sh);
    all = ev_block_sum(all, sh);
    if (blockIdx.x == 0 && threadIdx.x == 0) { *events_number = (int32_t)all; *global_trigger = all > 0; }
    int64_t run = before;
    for (int64_t sub = beg; sub < end; sub += kEvBatch) {
        const int64_t wb = sub + (int64_t)wid * (32 * kEvItems) + lane;      // item = wb + 32 k
        unsigned ball[kEvItems];
        int32_t mine = 0;
#pragma unroll
        for (int k = 0; k < kEvItems; ++k) {
            const int64_t i = wb + 32 * k;
            ball[k] = __ballot_sync(0xffffffffu, i < end && trigger[i] != 0);
            mine += __popc(ball[k]);
        }
        if (lane == 0) wtot[wid] = mine;
        __syncthreads();
        int32_t wbase = 0, total = 0;
        for (int w = 0; w < kEvThreads / 32; ++w) {
            const int32_t t = wtot[w];
            if (w < wid) wbase += t;
            total += t;
        }
        int64_t pos = run + wbase;
#pragma unroll
        for (int k = 0; k < kEvItems; ++k) {
            if (ball[k] >> lane & 1u) events_indices[pos + __popc(ball[k] & ((1u << lane) - 1u))] = (int32_t)(wb + 32 * k);
            pos += __popc(ball[k]);
        }
        run += total;
        __syncthreads();
    }
}

// blocks [0, gridDim/2): past list -> count_prev; the rest: present list -> count_now
__global__ void ev_degree_kernel(const uint64_t* __restrict__ prev, const int64_t* __restrict__ n_prev,
                                 const uint64_t* __restrict__ now, const int64_t* __restrict__ n_now,
                                 int64_t cap_prev, int64_t cap_now, const int32_t* __restrict__ trigger, int32_t n,
                                 int32_t* __restrict__ count_prev, int32_t* __restrict__ count_now) {
    const int half = gridDim.x >> 1;
    const bool second = (int)blockIdx.x >= half;
    const uint64_t* __restrict__ E = second ? now : prev;
    const int64_t m = second ? min(*n_now, cap_now) : min(*n_prev, cap_prev);
    int32_t* __restrict__ cnt = second ? count_now : count_prev;
    const int b = second ? blockIdx.x - half : blockIdx.x;
    for (int64_t k = (int64_t)b * blockDim.x + threadIdx.x; k < m; k += (int64_t)half * blockDim.x) {
        const uint64_t e = __ldcs(E + k);
        const uint32_t i = (uint32_t)(e >> 32), j = (uint32_t)e;
        if (i >= (uint32_t)n || j >= (uint32_t)n) continue;
        if (trigger[i] && trigger[j]) { atomicAdd(cnt + i, 1); atomicAdd(cnt + j, 1); }
    }
}

}  // namespace

extern "C" int vor_events(vor_ctx* ctx, const uint64_t* d_prev, const int64_t* d_n_prev,
                          const uint64_t* d_now, const int64_t* d_n_now, int64_t cap_prev, int64_t cap_now,
                          const uint64_t* d_created, const int64_t* d_n_created,
                          const uint64_t* d_destroyed, const int64_t* d_n_destroyed, int64_t cap_created,
                          int64_t cap_destroyed,
                          int32_t n_labels,
                          int32_t* d_trigger, int32_t* d_events_indices, int32_t* d_events_number,
                          int32_t* d_global_trigger, int32_t* d_count_prev, int32_t* d_count_now,
                          void* stream_) {
    if (!ctx) return VOR_EINVAL;
    if (int drc_ = vor_check_device(ctx)) return drc_;
    if (!d_prev || !d_n_prev || !d_now || !d_n_now || !d_created || !d_n_created || !d_destroyed ||
        !d_n_destroyed || !d_trigger || !d_events_indices || !d_events_number || !d_global_trigger ||
        !d_count_prev || !d_count_now)
        return vor_fail(ctx, VOR_EINVAL, "vor_events: null pointer");
    if (n_labels < 1 || cap_prev < 0 || cap_now < 0 || cap_created < 0 || cap_destroyed < 0)
        return vor_fail(ctx, VOR_EINVAL, "vor_events: n_labels must be >= 1, capacities >= 0");
    cudaStream_t stream = (cudaStream_t)stream_;
    const size_t bytes = (size_t)n_labels * sizeof(int32_t);
    VOR_CUDA(cudaMemsetAsync(d_trigger, 0, bytes, stream));
    VOR_CUDA(cudaMemsetAsync(d_count_prev, 0, bytes, stream));
    VOR_CUDA(cudaMemsetAsync(d_count_now, 0, bytes, stream));
    const int grid = min(4 * ctx->num_sms, kMaxCoopBlocks);   // d_blk_count holds 2 * kMaxCoopBlocks partials
    VOR_LAUNCH(ev_mark_kernel, grid, 256, 0, stream, d_created, d_n_created, d_destroyed, d_n_destroyed,
               cap_created, cap_destroyed, n_labels, d_trigger);
    VOR_LAUNCH(ev_count_kernel, grid, kEvThreads, 0, stream, d_trigger, n_labels, ctx->d_blk_count);
    VOR_LAUNCH(ev_write_kernel, grid, kEvThreads, 0, stream, d_trigger, n_labels, ctx->d_blk_count,
               d_events_indices, d_events_number, d_global_trigger);
    VOR_LAUNCH(ev_degree_kernel, 2 * grid, 256, 0, stream, d_prev, d_n_prev, d_now, d_n_now, cap_prev, cap_now,
               d_trigger, n_labels, d_count_prev, d_count_now);
    return VOR_OK;
}

// ------------------------------------------------------------------------------------------------------------
// Couples of active vertices and T1 pairing (§III.B.4: the active
// points that are connected are stored as couples, permutations dropped, each couple connected in only one
// configuration is "breaking" (D_P) or "arising" (D_N); end points sharing two neighbours
// = bulk edge, one = boundary edge; PAPER.md:238 and Fig. 8: a T1 event replaces the breaking link by the
// arising link between its two common neighbours).
//
// Data structures (all context scratch):
//   adjacency lists of BOTH triangulations in compressed symmetric form - the paper's adjacency matrix with
//   sorted rows, row v = all neighbours of v ascending: off[n+1], adj[2E].  Built from the
//   i<j key lists by degree count -> exclusive scan -> atomic fill -> rank within the row (keys are unique,
//   so the rank of a neighbour is the number of smaller ones in its row).
//   union list U = now ∪ destroyed in key order (a key's slot = its own index + its lower bound in the other
//   list), class in the two bits that a packed key never uses (bit 63: breaking, bit 31: arising), or kDrop
//   when an end point is inactive or >= n_labels.  Couples = order-preserving compaction of U.
namespace {

constexpr uint64_t kDrop = ~(uint64_t)0;
constexpr uint64_t kBitBreak = (uint64_t)1 << 63, kBitArise = (uint64_t)1 << 31;

struct T1Graph {
    const uint64_t* keys;
    const int64_t* n_dev;
    int64_t cap;
    uint32_t* deg;      // [n + 1] degrees, then fill cursors
    uint32_t* off;      // [n + 1]
    uint32_t* adj_u;    // unsorted rows
    uint32_t* adj_s;    // sorted rows
};

__device__ __forceinline__ int64_t t1_len(const T1Graph& g) { return min(max(*g.n_dev, (int64_t)0), g.cap); }

__device__ __forceinline__ bool t1_edge(const T1Graph& g, int64_t k, int32_t n, uint32_t* i, uint32_t* j) {
    const uint64_t e = g.keys[k];
    *i = (uint32_t)(e >> 32); *j = (uint32_t)e;
    return *i < (uint32_t)n && *j < (uint32_t)n;
}

// blockIdx.y selects the triangulation
__global__ void t1_degree_kernel(T1Graph gp, T1Graph gn, int32_t n) {
    const T1Graph& g = blockIdx.y ? gn : gp;
    const int64_t m = t1_len(g);
    for (int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; k < m; k += (int64_t)gridDim.x * blockDim.x) {
        uint32_t i, j;
        if (!t1_edge(g, k, n, &i, &j)) continue;
        atomicAdd(g.deg + i, 1u);
        atomicAdd(g.deg + j, 1u);
    }
}

__device__ __forceinline__ void t1_chunk(int64_t n, int batch, int64_t* beg, int64_t* end) {
    int64_t C = (n + gridDim.x - 1) / gridDim.x;
    C = (C + batch - 1) / batch * batch;
    const int64_t s = (int64_t)blockIdx.x * C;
    *beg = s < n ? s : n;
    *end = s + C < n ? s + C : n;
}

// exclusive scan of deg[0..n) -> off[0..n], in two kernels: per-chunk sums, then every block adds the sums of
// the chunks before it and scans its own chunk; deg is zeroed for its second life as fill cursor
__global__ void __launch_bounds__(kEvThreads) t1_scan_sum_kernel(T1Graph gp, T1Graph gn, int32_t n,
                                                                 int64_t* __restrict__ partial) {
    __shared__ int64_t sh[32];
    const T1Graph& g = blockIdx.y ? gn : gp;
    int64_t beg, end;
    t1_chunk(n, kEvThreads, &beg, &end);
    int64_t c = 0;
    for (int64_t i = beg + threadIdx.x; i < end; i += kEvThreads) c += g.deg[i];
    c = ev_block_sum(c, sh);
    if (threadIdx.x == 0) partial[blockIdx.y * gridDim.x + blockIdx.x] = c;
}

__global__ void __launch_bounds__(kEvThreads) t1_scan_apply_kernel(T1Graph gp, T1Graph gn, int32_t n,
                                                                   const int64_t* __restrict__ partial) {
    __shared__ int64_t sh[32];
    __shared__ uint32_t wsum[kEvThreads / 32];
    const T1Graph& g = blockIdx.y ? gn : gp;
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    int64_t beg, end;
    t1_chunk(n, kEvThreads, &beg, &end);
    int64_t before = 0, all = 0;
    for (int b = threadIdx.x; b < (int)gridDim.x; b += kEvThreads) {
        const int64_t v = partial[blockIdx.y * gridDim.x + b];
        all += v;
        if (b < (int)blockIdx.x) before += v;
    }
    before = ev_block_sum(before, sh);
    all = ev_block_sum(all, sh);
    if (blockIdx.x == 0 && threadIdx.x == 0) g.off[n] = (uint32_t)all;
    uint32_t run = (uint32_t)before;
    for (int64_t sub = beg; sub < end; sub += kEvThreads) {
        const int64_t i = sub + threadIdx.x;
        const uint32_t v = i < end ? g.deg[i] : 0u;
        uint32_t inc = v;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t t = __shfl_up_sync(0xffffffffu, inc, o);
            if (lane >= o) inc += t;
        }
        if (lane == 31) wsum[wid] = inc;
        __syncthreads();
        uint32_t wbase = 0, total = 0;
        for (int w = 0; w < kEvThreads / 32; ++w) {
            const uint32_t t = wsum[w];
            if (w < wid) wbase += t;
            total += t;
        }
        if (i < end) { g.off[i] = run + wbase + inc - v; g.deg[i] = 0u; }
        run += total;
        __syncthreads();
    }
}

__global__ void t1_fill_kernel(T1Graph gp, T1Graph gn, int32_t n) {
    const T1Graph& g = blockIdx.y ? gn : gp;
    const int64_t m = t1_len(g);
    for (int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; k < m; k += (int64_t)gridDim.x * blockDim.x) {
        uint32_t i, j;
        if (!t1_edge(g, k, n, &i, &j)) continue;
        g.adj_u[g.off[i] + atomicAdd(g.deg + i, 1u)] = j;
        g.adj_u[g.off[j] + atomicAdd(g.deg + j, 1u)] = i;
    }
}

__device__ __forceinline__ void t1_place(const T1Graph& g, uint32_t v, uint32_t e) {
    const uint32_t b = g.off[v], end = g.off[v + 1];
    uint32_t r = 0;
    for (uint32_t p = b; p < end; ++p) r += g.adj_u[p] < e;
    g.adj_s[b + r] = e;
}

__global__ void t1_rank_kernel(T1Graph gp, T1Graph gn, int32_t n) {
    const T1Graph& g = blockIdx.y ? gn : gp;
    const int64_t m = t1_len(g);
    for (int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; k < m; k += (int64_t)gridDim.x * blockDim.x) {
        uint32_t i, j;
        if (!t1_edge(g, k, n, &i, &j)) continue;
        t1_place(g, i, j);
        t1_place(g, j, i);
    }
}

__device__ __forceinline__ int64_t t1_lower_bound(const uint64_t* __restrict__ a, int64_t n, uint64_t key) {
    int64_t lo = 0, hi = n;
    while (lo < hi) {
        const int64_t mid = (lo + hi) >> 1;
        if (a[mid] < key) lo = mid + 1; else hi = mid;
    }
    return lo;
}

struct T1Lists {
    const uint64_t* now; const int64_t* n_now; int64_t cap_now;
    const uint64_t* created; const int64_t* n_created; int64_t cap_created;
    const uint64_t* destroyed; const int64_t* n_destroyed; int64_t cap_destroyed;
};

// Union list by merge path: every thread owns kT1Merge consecutive slots of the union, finds where they start in
// the two lists (one co-rank search per thread instead of one search per key), then merges sequentially; the
// class of a present key follows a cursor in `created` (one lower bound per thread).  The block also counts
// the couples of its chunk (the chunks are those of the compaction that follows).
constexpr int kT1Merge = 8;

__global__ void __launch_bounds__(kEvThreads) t1_union_kernel(T1Lists l, const int32_t* __restrict__ trigger, int32_t n,
                                                              uint64_t* __restrict__ U, int64_t* __restrict__ partial) {
    __shared__ int64_t sh[32];
    const int64_t nn = min(max(*l.n_now, (int64_t)0), l.cap_now), nc = min(max(*l.n_created, (int64_t)0), l.cap_created),
                  nd = min(max(*l.n_destroyed, (int64_t)0), l.cap_destroyed);
    const uint64_t* __restrict__ A = l.now;
    const uint64_t* __restrict__ B = l.destroyed;
    int64_t beg, end;
    t1_chunk(nn + nd, 32 * kEvItems, &beg, &end);
    int64_t kept = 0;
    for (int64_t d0 = beg + (int64_t)threadIdx.x * kT1Merge; d0 < end; d0 += (int64_t)kEvThreads * kT1Merge) {
        const int64_t d1 = min(d0 + kT1Merge, end);
        // co-rank of slot d0: i keys of `now` and d0 - i keys of `destroyed` precede it (the lists are disjoint)
        int64_t lo = max((int64_t)0, d0 - nd), hi = min(d0, nn);
        while (lo < hi) {
            const int64_t mid = (lo + hi) >> 1, j = d0 - mid;
            if (j > 0 && B[j - 1] > A[mid]) lo = mid + 1; else hi = mid;
        }
        int64_t i = lo, j = d0 - lo;
        int64_t c = i < nn ? t1_lower_bound(l.created, nc, A[i]) : nc;      // cursor in `created`
        for (int64_t d = d0; d < d1; ++d) {
            uint64_t key, bits;
            if (j >= nd || (i < nn && A[i] < B[j])) {
                key = A[i++];
                while (c < nc && l.created[c] < key) ++c;
                bits = (c < nc && l.created[c] == key) ? kBitArise : 0;
            } else {
                key = B[j++];
                bits = kBitBreak;
            }
            const uint32_t a = (uint32_t)(key >> 32), b = (uint32_t)key;
            const bool keep = a < (uint32_t)n && b < (uint32_t)n && trigger[a] != 0 && trigger[b] != 0;
            U[d] = keep ? (key | bits) : kDrop;
            kept += keep;
        }
    }
    kept = ev_block_sum(kept, sh);
    if (threadIdx.x == 0) partial[blockIdx.x] = kept;
}

__global__ void __launch_bounds__(kEvThreads) t1_write_kernel(const uint64_t* __restrict__ U, T1Lists l,
                                                              const int64_t* __restrict__ partial,
                                                              uint64_t* __restrict__ couples, int32_t* __restrict__ cls,
                                                              int64_t cap, int64_t* __restrict__ n_couples,
                                                              int32_t* __restrict__ flags) {
    __shared__ int64_t sh[32];
    __shared__ int32_t wtot[kEvThreads / 32];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int64_t m = min(max(*l.n_now, (int64_t)0), l.cap_now) + min(max(*l.n_destroyed, (int64_t)0), l.cap_destroyed);
    int64_t beg, end;
    t1_chunk(m, 32 * kEvItems, &beg, &end);
    int64_t before = 0, all = 0;
    for (int b = threadIdx.x; b < (int)gridDim.x; b += kEvThreads) {
        const int64_t v = partial[b];
        all += v;
        if (b < (int)blockIdx.x) before += v;
    }
    before = ev_block_sum(before, sh);
    all = ev_block_sum(all, sh);
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        *n_couples = all;
        if (all > cap) atomicOr(flags, FLAG_DIFF_CAP);
    }
    int64_t run = before;
    for (int64_t sub = beg; sub < end; sub += kEvBatch) {
        const int64_t wb = sub + (int64_t)wid * (32 * kEvItems) + lane;
        unsigned ball[kEvItems];
        uint64_t u[kEvItems];
        int32_t mine = 0;
#pragma unroll
        for (int k = 0; k < kEvItems; ++k) {
            const int64_t i = wb + 32 * k;
            u[k] = i < end ? U[i] : kDrop;
            ball[k] = __ballot_sync(0xffffffffu, u[k] != kDrop);
            mine += __popc(ball[k]);
        }
        if (lane == 0) wtot[wid] = mine;
        __syncthreads();
        int32_t wbase = 0, total = 0;
        for (int w = 0; w < kEvThreads / 32; ++w) {
            const int32_t t = wtot[w];
            if (w < wid) wbase += t;
            total += t;
        }
        int64_t pos = run + wbase;
#pragma unroll
        for (int k = 0; k < kEvItems; ++k) {
            const int64_t at = pos + __popc(ball[k] & ((1u << lane) - 1u));
            if ((ball[k] >> lane & 1u) && at < cap) {
                couples[at] = u[k] & ~(kBitBreak | kBitArise);
                cls[at] = (u[k] & kBitBreak) ? 1 : ((u[k] & kBitArise) ? 2 : 0);
            }
            pos += __popc(ball[k]);
        }
        run += total;
        __syncthreads();
    }
}

// common neighbours of i and j (rows ascending): their number, the first two in c2
__device__ __forceinline__ int32_t t1_common(const T1Graph& g, uint32_t i, uint32_t j, uint32_t* c2) {
    uint32_t a = g.off[i], ae = g.off[i + 1], b = g.off[j], be = g.off[j + 1];
    int32_t cnt = 0;
    if (a == ae || b == be) return 0;
    uint32_t x = g.adj_s[a], y = g.adj_s[b];
    for (;;) {
        if (x == y) {
            if (cnt < 2) c2[cnt] = x;
            ++cnt;
        }
        const bool sa = x <= y, sb = y <= x;
        if (sa) { if (++a == ae) break; x = g.adj_s[a]; }
        if (sb) { if (++b == be) break; y = g.adj_s[b]; }
    }
    return cnt;
}

__device__ __forceinline__ bool t1_linked(const T1Graph& g, uint32_t v, uint32_t e) {
    uint32_t lo = g.off[v], hi = g.off[v + 1];
    while (lo < hi) {
        const uint32_t mid = (lo + hi) >> 1;
        if (g.adj_s[mid] < e) lo = mid + 1; else hi = mid;
    }
    return lo < g.off[v + 1] && g.adj_s[lo] == e;
}

__global__ void t1_pair_kernel(T1Graph gp, T1Graph gn, const uint64_t* __restrict__ couples,
                               const int32_t* __restrict__ cls, const int64_t* __restrict__ n_couples, int64_t cap,
                               int32_t* __restrict__ common_prev, int32_t* __restrict__ common_now,
                               uint64_t* __restrict__ partner) {
    const int64_t m = min(*n_couples, cap);
    for (int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; k < m; k += (int64_t)gridDim.x * blockDim.x) {
        const uint64_t key = couples[k];
        const uint32_t i = (uint32_t)(key >> 32), j = (uint32_t)key;
        const int32_t c = cls[k];
        uint32_t c2[2] = {0, 0};
        uint64_t pt = kDrop;
        int32_t cp = -1, cn = -1;
        if (c != 2) {
            cp = t1_common(gp, i, j, c2);
            if (c == 1 && cp == 2 && t1_linked(gn, c2[0], c2[1]) && !t1_linked(gp, c2[0], c2[1]))
                pt = ((uint64_t)c2[0] << 32) | c2[1];
        }
        if (c != 1) {
            cn = t1_common(gn, i, j, c2);
            if (c == 2 && cn == 2 && t1_linked(gp, c2[0], c2[1]) && !t1_linked(gn, c2[0], c2[1]))
                pt = ((uint64_t)c2[0] << 32) | c2[1];
        }
        common_prev[k] = cp;
        common_now[k] = cn;
        partner[k] = pt;
    }
}

int t1_scratch(vor_ctx* ctx, int slot, size_t bytes, void** out) {
    if (ctx->t1_bytes[slot] < bytes) {
        if (ctx->d_t1[slot]) VOR_CUDA(cudaFree(ctx->d_t1[slot]));   // cudaFree waits for the work that uses it
        ctx->d_t1[slot] = nullptr; ctx->t1_bytes[slot] = 0;
        VOR_CUDA(cudaMalloc(&ctx->d_t1[slot], bytes));
        ctx->t1_bytes[slot] = bytes;
    }
    *out = ctx->d_t1[slot];
    return VOR_OK;
}

}  // namespace

// Both triangulations as symmetric adjacency lists with sorted rows in the context's scratch.
static int t1_graphs(vor_ctx* ctx, const uint64_t* d_prev, const int64_t* d_n_prev, const uint64_t* d_now,
                     const int64_t* d_n_now, int64_t cap_prev, int64_t cap_now, int32_t n_labels, T1Graph* gp,
                     T1Graph* gn) {
    const size_t n1 = (size_t)n_labels + 1;
    uint32_t *deg, *off, *adj_u, *adj_s;
    int rc;
    const size_t n_adj = 2 * (size_t)(cap_prev + cap_now) + 1;
    if ((rc = t1_scratch(ctx, 0, 2 * n1 * sizeof(uint32_t), (void**)&deg)) != VOR_OK) return rc;
    if ((rc = t1_scratch(ctx, 1, 2 * n1 * sizeof(uint32_t), (void**)&off)) != VOR_OK) return rc;
    if ((rc = t1_scratch(ctx, 2, n_adj * sizeof(uint32_t), (void**)&adj_u)) != VOR_OK) return rc;
    if ((rc = t1_scratch(ctx, 3, n_adj * sizeof(uint32_t), (void**)&adj_s)) != VOR_OK) return rc;
    *gp = T1Graph{d_prev, d_n_prev, cap_prev, deg, off, adj_u, adj_s};
    *gn = T1Graph{d_now, d_n_now, cap_now, deg + n1, off + n1, adj_u + 2 * cap_prev, adj_s + 2 * cap_prev};
    return VOR_OK;
}

static int t1_build_graphs(vor_ctx* ctx, const T1Graph& gp, const T1Graph& gn, int32_t n_labels, cudaStream_t stream) {
    const size_t n1 = (size_t)n_labels + 1;
    VOR_CUDA(cudaMemsetAsync(gp.deg, 0, 2 * n1 * sizeof(uint32_t), stream));
    const int grid = min(4 * ctx->num_sms, kMaxCoopBlocks);
    const dim3 both(grid, 2);
    VOR_LAUNCH(t1_degree_kernel, both, 256, 0, stream, gp, gn, n_labels);
    VOR_LAUNCH(t1_scan_sum_kernel, both, kEvThreads, 0, stream, gp, gn, n_labels, ctx->d_blk_count);
    VOR_LAUNCH(t1_scan_apply_kernel, both, kEvThreads, 0, stream, gp, gn, n_labels, ctx->d_blk_count);
    VOR_LAUNCH(t1_fill_kernel, both, 256, 0, stream, gp, gn, n_labels);
    VOR_LAUNCH(t1_rank_kernel, both, 256, 0, stream, gp, gn, n_labels);
    return VOR_OK;
}

extern "C" int vor_t1_events(vor_ctx* ctx, const uint64_t* d_prev, const int64_t* d_n_prev,
                             const uint64_t* d_now, const int64_t* d_n_now, int64_t cap_prev, int64_t cap_now,
                             const uint64_t* d_created, const int64_t* d_n_created,
                             const uint64_t* d_destroyed, const int64_t* d_n_destroyed, int64_t cap_created,
                             int64_t cap_destroyed, const int32_t* d_trigger, int32_t n_labels,
                             uint64_t* d_couples, int32_t* d_class, int32_t* d_common_prev, int32_t* d_common_now,
                             uint64_t* d_partner, int64_t cap, int64_t* d_n_couples, void* stream_) {
    if (!ctx) return VOR_EINVAL;
    if (int drc_ = vor_check_device(ctx)) return drc_;
    if (!d_prev || !d_n_prev || !d_now || !d_n_now || !d_created || !d_n_created || !d_destroyed || !d_n_destroyed ||
        !d_trigger || !d_couples || !d_class || !d_common_prev || !d_common_now || !d_partner || !d_n_couples)
        return vor_fail(ctx, VOR_EINVAL, "vor_t1_events: null pointer");
    if (n_labels < 1 || cap_prev < 0 || cap_now < 0 || cap_created < 0 || cap_destroyed < 0 || cap < 0)
        return vor_fail(ctx, VOR_EINVAL, "vor_t1_events: n_labels must be >= 1, capacities >= 0");
    if (2 * (cap_prev + cap_now) >= ((int64_t)1 << 32))
        return vor_fail(ctx, VOR_EINVAL, "vor_t1_events: cap_prev + cap_now must be below 2^31");
    cudaStream_t stream = (cudaStream_t)stream_;
    uint64_t* U;
    int rc;
    T1Graph gp, gn;
    if ((rc = t1_graphs(ctx, d_prev, d_n_prev, d_now, d_n_now, cap_prev, cap_now, n_labels, &gp, &gn)) != VOR_OK) return rc;
    if ((rc = t1_scratch(ctx, 4, ((size_t)(cap_now + cap_destroyed) + 1) * sizeof(uint64_t), (void**)&U)) != VOR_OK) return rc;
    T1Lists l{d_now, d_n_now, cap_now, d_created, d_n_created, cap_created, d_destroyed, d_n_destroyed, cap_destroyed};

    const int grid = min(4 * ctx->num_sms, kMaxCoopBlocks);   // 2 * grid partials in d_blk_count
    if ((rc = t1_build_graphs(ctx, gp, gn, n_labels, stream)) != VOR_OK) return rc;
    VOR_LAUNCH(t1_union_kernel, grid, kEvThreads, 0, stream, l, d_trigger, n_labels, U, ctx->d_blk_count);
    VOR_LAUNCH(t1_write_kernel, grid, kEvThreads, 0, stream, U, l, ctx->d_blk_count, d_couples, d_class, cap,
               d_n_couples, ctx->d_flags);
    VOR_LAUNCH(t1_pair_kernel, 16 * grid, 256, 0, stream, gp, gn, d_couples, d_class, d_n_couples, cap,
               d_common_prev, d_common_now, d_partner);
    return VOR_OK;
}

// ------------------------------------------------------------------------------------------------------------
// Bulk / boundary edges: "if two connected points share two neighbours, then the edge is in
// the bulk; if two connected points share only one neighbour, then the edge is on the boundary".  One thread
// per edge intersects the two sorted adjacency rows built as for vor_t1_events.
namespace {

__global__ void edge_commons_kernel(T1Graph g, int32_t n, int32_t* __restrict__ commons) {
    const int64_t m = t1_len(g);
    for (int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; k < m; k += (int64_t)gridDim.x * blockDim.x) {
        uint32_t i, j, c2[2];
        commons[k] = t1_edge(g, k, n, &i, &j) ? t1_common(g, i, j, c2) : -1;
    }
}

}  // namespace

extern "C" int vor_edge_commons(vor_ctx* ctx, const uint64_t* d_edges, const int64_t* d_n_edges, int64_t cap_edges,
                                int32_t n_labels, int32_t* d_commons, void* stream_) {
    if (!ctx) return VOR_EINVAL;
    if (int drc_ = vor_check_device(ctx)) return drc_;
    if (!d_edges || !d_n_edges || !d_commons) return vor_fail(ctx, VOR_EINVAL, "vor_edge_commons: null pointer");
    if (n_labels < 1 || cap_edges < 0 || 2 * cap_edges >= ((int64_t)1 << 32))
        return vor_fail(ctx, VOR_EINVAL, "vor_edge_commons: n_labels >= 1, 0 <= cap_edges < 2^31");
    cudaStream_t stream = (cudaStream_t)stream_;
    const size_t n1 = (size_t)n_labels + 1;
    uint32_t *deg, *off, *adj_u, *adj_s;
    int rc;
    const size_t n_adj = 2 * (size_t)cap_edges + 1;
    if ((rc = t1_scratch(ctx, 0, 2 * n1 * sizeof(uint32_t), (void**)&deg)) != VOR_OK) return rc;
    if ((rc = t1_scratch(ctx, 1, 2 * n1 * sizeof(uint32_t), (void**)&off)) != VOR_OK) return rc;
    if ((rc = t1_scratch(ctx, 2, n_adj * sizeof(uint32_t), (void**)&adj_u)) != VOR_OK) return rc;
    if ((rc = t1_scratch(ctx, 3, n_adj * sizeof(uint32_t), (void**)&adj_s)) != VOR_OK) return rc;
    T1Graph g{d_edges, d_n_edges, cap_edges, deg, off, adj_u, adj_s};
    VOR_CUDA(cudaMemsetAsync(deg, 0, n1 * sizeof(uint32_t), stream));
    const int grid = min(4 * ctx->num_sms, kMaxCoopBlocks);
    const dim3 one(grid, 1);                                 // blockIdx.y == 0: the kernels read only the first graph
    VOR_LAUNCH(t1_degree_kernel, one, 256, 0, stream, g, g, n_labels);
    VOR_LAUNCH(t1_scan_sum_kernel, one, kEvThreads, 0, stream, g, g, n_labels, ctx->d_blk_count);
    VOR_LAUNCH(t1_scan_apply_kernel, one, kEvThreads, 0, stream, g, g, n_labels, ctx->d_blk_count);
    VOR_LAUNCH(t1_fill_kernel, one, 256, 0, stream, g, g, n_labels);
    VOR_LAUNCH(t1_rank_kernel, one, 256, 0, stream, g, g, n_labels);
    VOR_LAUNCH(edge_commons_kernel, 4 * grid, 256, 0, stream, g, n_labels, d_commons);
    return VOR_OK;
}

// ------------------------------------------------------------------------------------------------------------
// Bulk and boundary vertices of an event: boundary vertices = end points of an edge with
// exactly one common neighbour; an active vertex takes part in a bulk event of a triangulation if at least
// three of its neighbours there are active, in a boundary event if at least one of them is an active boundary
// vertex.
namespace {

// blockIdx.y selects the triangulation; every boundary edge marks its two end points
__global__ void ev_boundary_kernel(T1Graph gp, T1Graph gn, int32_t n, int32_t* __restrict__ boundary_prev,
                                   int32_t* __restrict__ boundary_now) {
    const T1Graph& g = blockIdx.y ? gn : gp;
    int32_t* __restrict__ out = blockIdx.y ? boundary_now : boundary_prev;
    const int64_t m = t1_len(g);
    for (int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; k < m; k += (int64_t)gridDim.x * blockDim.x) {
        uint32_t i, j, c2[2];
        if (!t1_edge(g, k, n, &i, &j)) continue;
        if (t1_common(g, i, j, c2) == 1) { out[i] = 1; out[j] = 1; }
    }
}

__global__ void ev_vclass_kernel(T1Graph gp, T1Graph gn, const int32_t* __restrict__ trigger, int32_t n,
                                 const int32_t* __restrict__ boundary_prev, const int32_t* __restrict__ boundary_now,
                                 int32_t* __restrict__ vclass) {
    for (int32_t v = blockIdx.x * blockDim.x + threadIdx.x; v < n; v += gridDim.x * blockDim.x) {
        int32_t c = 0;
        if (trigger[v]) {
#pragma unroll
            for (int t = 0; t < 2; ++t) {
                const T1Graph& g = t ? gn : gp;
                const int32_t* __restrict__ bnd = t ? boundary_now : boundary_prev;
                int32_t act = 0, ab = 0;
                for (uint32_t p = g.off[v]; p < g.off[v + 1]; ++p) {
                    const uint32_t u = g.adj_s[p];
                    if (trigger[u]) { ++act; ab += bnd[u]; }
                }
                if (act >= 3) c |= 1 << (2 * t);
                if (ab >= 1) c |= 2 << (2 * t);
            }
        }
        vclass[v] = c;
    }
}

}  // namespace

extern "C" int vor_event_vertices(vor_ctx* ctx, const uint64_t* d_prev, const int64_t* d_n_prev,
                                  const uint64_t* d_now, const int64_t* d_n_now, int64_t cap_prev, int64_t cap_now,
                                  const int32_t* d_trigger, int32_t n_labels, int32_t* d_boundary_prev,
                                  int32_t* d_boundary_now, int32_t* d_vclass, void* stream_) {
    if (!ctx) return VOR_EINVAL;
    if (int drc_ = vor_check_device(ctx)) return drc_;
    if (!d_prev || !d_n_prev || !d_now || !d_n_now || !d_trigger || !d_boundary_prev || !d_boundary_now || !d_vclass)
        return vor_fail(ctx, VOR_EINVAL, "vor_event_vertices: null pointer");
    if (n_labels < 1 || cap_prev < 0 || cap_now < 0 || 2 * (cap_prev + cap_now) >= ((int64_t)1 << 32))
        return vor_fail(ctx, VOR_EINVAL, "vor_event_vertices: n_labels >= 1, capacities >= 0, cap_prev + cap_now < 2^31");
    cudaStream_t stream = (cudaStream_t)stream_;
    int rc;
    T1Graph gp, gn;
    if ((rc = t1_graphs(ctx, d_prev, d_n_prev, d_now, d_n_now, cap_prev, cap_now, n_labels, &gp, &gn)) != VOR_OK) return rc;
    if ((rc = t1_build_graphs(ctx, gp, gn, n_labels, stream)) != VOR_OK) return rc;
    VOR_CUDA(cudaMemsetAsync(d_boundary_prev, 0, (size_t)n_labels * sizeof(int32_t), stream));
    VOR_CUDA(cudaMemsetAsync(d_boundary_now, 0, (size_t)n_labels * sizeof(int32_t), stream));
    const int grid = min(4 * ctx->num_sms, kMaxCoopBlocks);
    VOR_LAUNCH(ev_boundary_kernel, dim3(4 * grid, 2), 256, 0, stream, gp, gn, n_labels, d_boundary_prev, d_boundary_now);
    VOR_LAUNCH(ev_vclass_kernel, 4 * grid, 256, 0, stream, gp, gn, d_trigger, n_labels, d_boundary_prev, d_boundary_now,
               d_vclass);
    return VOR_OK;
}
