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
        if (i < (uint32_t)n) trigger[i] = 1;
        if (j < (uint32_t)n) trigger[j] = 1;
    }
}

__device__ __forceinline__ void ev_chunk(int64_t n, int64_t* beg, int64_t* end) {
    int64_t C = (n + gridDim.x - 1) / gridDim.x;
    C = (C + kEvBatch - 1) / kEvBatch * kEvBatch;
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
    const int grid = 4 * ctx->num_sms;                      // <= 2 * kMaxCoopBlocks partials
    VOR_LAUNCH(ev_mark_kernel, grid, 256, 0, stream, d_created, d_n_created, d_destroyed, d_n_destroyed,
               cap_created, cap_destroyed, n_labels, d_trigger);
    VOR_LAUNCH(ev_count_kernel, grid, kEvThreads, 0, stream, d_trigger, n_labels, ctx->d_blk_count);
    VOR_LAUNCH(ev_write_kernel, grid, kEvThreads, 0, stream, d_trigger, n_labels, ctx->d_blk_count,
               d_events_indices, d_events_number, d_global_trigger);
    VOR_LAUNCH(ev_degree_kernel, 2 * grid, 256, 0, stream, d_prev, d_n_prev, d_now, d_n_now, cap_prev, cap_now,
               d_trigger, n_labels, d_count_prev, d_count_now);
    return VOR_OK;
}
