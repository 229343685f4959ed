// a5 — frame-to-frame comparison of two edge sets.
// Paper: translate the past adjacency list into "now" labels with the isomorphism,
// sort, compare row by row, exclude appearing / disappearing bubbles
// and classify the couples connected in only one triangulation as "breaking" (in
// D_P only) or "arising" (in D_N only).  Here both sets are ascending unique key
// lists, so breaking = prev \ now (destroyed) and arising = now \ prev (created) are sorted set
// differences: each key is binary-searched in the other list (both lists are L2-resident), then an
// order-preserving compaction writes the survivors.
#include "common.cuh"

namespace {

constexpr int kDiffThreads = kSortThreads;

__device__ __forceinline__ bool contains(const uint64_t* __restrict__ a, int64_t n, uint64_t key) {
    int64_t lo = 0, hi = n;
    while (lo < hi) {
        const int64_t mid = (lo + hi) >> 1;
        if (a[mid] < key) lo = mid + 1; else hi = mid;
    }
    return lo < n && a[lo] == key;
}

__device__ __forceinline__ void chunk_of(int64_t n, int nblocks, int b, int64_t* beg, int64_t* end) {
    int64_t C = (n + nblocks - 1) / nblocks;
    C = (C + kDiffThreads - 1) / kDiffThreads * kDiffThreads;
    int64_t s = (int64_t)b * C;
    *beg = s < n ? s : n;
    *end = s + C < n ? s + C : n;
}

__device__ __forceinline__ int64_t block_sum(int64_t v, int64_t* sh) {
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

// grid = 2 * nb blocks: blocks [0, nb) handle created = now \ prev, [nb, 2nb) destroyed = prev \ now
__global__ void __launch_bounds__(kDiffThreads) diff_count_kernel(
        const uint64_t* __restrict__ prev, const int64_t* __restrict__ n_prev_p,
        const uint64_t* __restrict__ now, const int64_t* __restrict__ n_now_p,
        int64_t* __restrict__ blk_count) {
    __shared__ int64_t sh[32];
    const int nb = gridDim.x >> 1;
    const bool second = (int)blockIdx.x >= nb;
    const uint64_t* A = second ? prev : now;        // elements of A not in B
    const uint64_t* B = second ? now : prev;
    const int64_t nA = second ? *n_prev_p : *n_now_p, nB = second ? *n_now_p : *n_prev_p;
    int64_t beg, end;
    chunk_of(nA, nb, second ? blockIdx.x - nb : blockIdx.x, &beg, &end);
    int64_t c = 0;
    for (int64_t i = beg + threadIdx.x; i < end; i += kDiffThreads) c += !contains(B, nB, A[i]);
    c = block_sum(c, sh);
    if (threadIdx.x == 0) blk_count[blockIdx.x] = c;
}

__global__ void __launch_bounds__(kDiffThreads) diff_write_kernel(
        const uint64_t* __restrict__ prev, const int64_t* __restrict__ n_prev_p,
        const uint64_t* __restrict__ now, const int64_t* __restrict__ n_now_p,
        const int64_t* __restrict__ blk_count, uint64_t* __restrict__ created,
        uint64_t* __restrict__ destroyed, int64_t cap, int64_t* __restrict__ n_created,
        int64_t* __restrict__ n_destroyed, int32_t* __restrict__ flags) {
    __shared__ int64_t sh[32];
    __shared__ int32_t wtot[kDiffThreads / 32];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int nb = gridDim.x >> 1;
    const bool second = (int)blockIdx.x >= nb;
    const int me = second ? blockIdx.x - nb : blockIdx.x;
    const uint64_t* A = second ? prev : now;
    const uint64_t* B = second ? now : prev;
    const int64_t nA = second ? *n_prev_p : *n_now_p, nB = second ? *n_now_p : *n_prev_p;
    uint64_t* out = second ? destroyed : created;
    int64_t beg, end;
    chunk_of(nA, nb, me, &beg, &end);
    int64_t before = 0, all = 0;
    for (int b = threadIdx.x; b < nb; b += kDiffThreads) {
        const int64_t v = blk_count[(second ? nb : 0) + b];
        all += v;
        if (b < me) before += v;
    }
    before = block_sum(before, sh);
    all = block_sum(all, sh);
    if (me == 0 && threadIdx.x == 0) {
        *(second ? n_destroyed : n_created) = all;
        if (all > cap) atomicOr(flags, FLAG_DIFF_CAP);
    }
    int64_t run = before;
    for (int64_t sub = beg; sub < end; sub += kDiffThreads) {
        const int64_t i = sub + threadIdx.x;
        uint64_t k = 0;
        bool keep = false;
        if (i < end) {
            k = A[i];
            keep = !contains(B, nB, k);
        }
        const unsigned ball = __ballot_sync(0xffffffffu, keep);
        if (lane == 0) wtot[wid] = __popc(ball);
        __syncthreads();
        int32_t wbase = 0, total = 0;
        for (int w = 0; w < kDiffThreads / 32; ++w) {
            const int32_t t = wtot[w];
            if (w < wid) wbase += t;
            total += t;
        }
        if (keep) {
            const int64_t pos = run + wbase + __popc(ball & ((1u << lane) - 1u));
            if (pos < cap) out[pos] = k;
        }
        run += total;
        __syncthreads();
    }
}

// prev edge (i,j) -> (p2n[i], p2n[j]); dropped if an endpoint is -1 or both collapse (R22);
// unordered append (sorted afterwards).
__global__ void translate_prev_kernel(const uint64_t* __restrict__ prev, const int64_t* __restrict__ n_prev_p,
                                      const int32_t* __restrict__ p2n, int32_t n_prev_labels,
                                      uint64_t* __restrict__ out, int64_t cap,
                                      unsigned long long* __restrict__ n_out, int32_t* __restrict__ flags) {
    const int64_t n = *n_prev_p;
    for (int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; k < n; k += (int64_t)gridDim.x * blockDim.x) {
        const uint64_t e = prev[k];
        const uint32_t a = (uint32_t)(e >> 32), b = (uint32_t)e;
        if (a >= (uint32_t)n_prev_labels || b >= (uint32_t)n_prev_labels) continue;
        const int32_t i = p2n[a], j = p2n[b];
        if (i < 0 || j < 0 || i == j) continue;
        const unsigned long long pos = atomicAdd(n_out, 1ull);
        if ((int64_t)pos < cap) out[pos] = ((uint64_t)(uint32_t)min(i, j) << 32) | (uint32_t)max(i, j);
        else atomicOr(flags, FLAG_RAWKEY_OVERFLOW);
    }
}

// now edge kept iff both endpoints have a partner in the previous frame
__global__ void filter_now_kernel(const uint64_t* __restrict__ now, const int64_t* __restrict__ n_now_p,
                                  const int32_t* __restrict__ n2p, int32_t n_now_labels,
                                  uint64_t* __restrict__ out, int64_t cap,
                                  unsigned long long* __restrict__ n_out, int32_t* __restrict__ flags) {
    const int64_t n = *n_now_p;
    for (int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; k < n; k += (int64_t)gridDim.x * blockDim.x) {
        const uint64_t e = now[k];
        const uint32_t a = (uint32_t)(e >> 32), b = (uint32_t)e;
        if (a >= (uint32_t)n_now_labels || b >= (uint32_t)n_now_labels) continue;
        if (n2p[a] < 0 || n2p[b] < 0) continue;
        const unsigned long long pos = atomicAdd(n_out, 1ull);
        if ((int64_t)pos < cap) out[pos] = e;
        else atomicOr(flags, FLAG_RAWKEY_OVERFLOW);
    }
}

int bits_for(int32_t n) {
    int bits = 1;
    while (bits < 31 && ((int64_t)1 << bits) < (int64_t)n) ++bits;
    return bits;
}

}  // namespace

extern "C" int vor_diff(vor_ctx* ctx, const uint64_t* d_prev, const int64_t* d_n_prev,
                        const uint64_t* d_now, const int64_t* d_n_now,
                        const int32_t* d_p2n, const int32_t* d_n2p,
                        int32_t n_prev_labels, int32_t n_now_labels,
                        uint64_t* d_created, uint64_t* d_destroyed, int64_t cap,
                        int64_t* d_n_created, int64_t* d_n_destroyed, void* stream_) {
    if (!ctx) return VOR_EINVAL;
    if (!d_prev || !d_n_prev || !d_now || !d_n_now || !d_created || !d_destroyed || !d_n_created ||
        !d_n_destroyed || cap < 0)
        return vor_fail(ctx, VOR_EINVAL, "vor_diff: null pointer or negative capacity");
    if ((d_p2n == nullptr) != (d_n2p == nullptr))
        return vor_fail(ctx, VOR_EINVAL, "vor_diff: give both maps or neither");
    cudaStream_t stream = (cudaStream_t)stream_;
    const uint64_t* P = d_prev;
    const int64_t* nP = d_n_prev;
    const uint64_t* N = d_now;
    const int64_t* nN = d_n_now;
    if (d_p2n) {
        if (n_prev_labels < 1 || n_now_labels < 1)
            return vor_fail(ctx, VOR_EINVAL, "vor_diff: label counts required with maps");
        if (!ctx->d_tr_prev) {
            VOR_CUDA(cudaMalloc((void**)&ctx->d_tr_prev, ctx->max_raw_keys * sizeof(uint64_t)));
            VOR_CUDA(cudaMalloc((void**)&ctx->d_tr_now, ctx->max_raw_keys * sizeof(uint64_t)));
        }
        const int bits = bits_for(n_now_labels);
        // translated prev -> d_keys_a -> sort/unique -> d_tr_prev
        VOR_CUDA(cudaMemsetAsync(ctx->d_n_raw, 0, sizeof(int64_t), stream));
        VOR_LAUNCH(translate_prev_kernel, 4 * kNumSMs, 256, 0, stream, d_prev, d_n_prev, d_p2n,
                   n_prev_labels, ctx->d_keys_a, ctx->max_raw_keys,
                   (unsigned long long*)ctx->d_n_raw, ctx->d_flags);
        int rc = vor_sort_unique_keys(ctx, ctx->d_keys_a, ctx->d_n_raw, bits, ctx->d_tr_prev,
                                      ctx->max_raw_keys, &ctx->d_tr_counts[0], FLAG_RAWKEY_OVERFLOW, stream);
        if (rc != VOR_OK) return rc;
        // filtered now -> d_keys_a -> sort/unique -> d_tr_now
        VOR_CUDA(cudaMemsetAsync(ctx->d_n_raw, 0, sizeof(int64_t), stream));
        VOR_LAUNCH(filter_now_kernel, 4 * kNumSMs, 256, 0, stream, d_now, d_n_now, d_n2p, n_now_labels,
                   ctx->d_keys_a, ctx->max_raw_keys, (unsigned long long*)ctx->d_n_raw, ctx->d_flags);
        rc = vor_sort_unique_keys(ctx, ctx->d_keys_a, ctx->d_n_raw, bits, ctx->d_tr_now,
                                  ctx->max_raw_keys, &ctx->d_tr_counts[1], FLAG_RAWKEY_OVERFLOW, stream);
        if (rc != VOR_OK) return rc;
        P = ctx->d_tr_prev; nP = &ctx->d_tr_counts[0];
        N = ctx->d_tr_now;  nN = &ctx->d_tr_counts[1];
    }
    VOR_LAUNCH(diff_count_kernel, 2 * kSortBlocks, kDiffThreads, 0, stream, P, nP, N, nN,
               ctx->d_blk_count);
    VOR_LAUNCH(diff_write_kernel, 2 * kSortBlocks, kDiffThreads, 0, stream, P, nP, N, nN,
               ctx->d_blk_count, d_created, d_destroyed, cap, d_n_created, d_n_destroyed, ctx->d_flags);
    return VOR_OK;
}
