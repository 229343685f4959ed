// a5 — frame-to-frame comparison of two edge sets.
// Paper: translate the past adjacency list into "now" labels with the isomorphism,
// sort, compare row by row, exclude appearing / disappearing bubbles
// and classify the couples connected in only one triangulation as "breaking" (in
// D_P only) or "arising" (in D_N only).  Here both sets are ascending unique key
// lists, so breaking = prev \ now (destroyed) and arising = now \ prev (created) are sorted set
// differences.  ONE cooperative kernel: half of the blocks take each direction; a block owns a
// contiguous chunk of its list A; every thread takes kDiffKeys consecutive keys of A, finds the
// position of the first one in the other list B with one binary search (the top levels of the search
// tree stay in L1) and walks B from there.  The per-thread membership masks stay in shared memory
// across the grid sync that separates counting from the order-preserving write.
#include <cooperative_groups.h>

#include "common.cuh"

namespace cg = cooperative_groups;

namespace {

constexpr int kDiffThreads = 512;
constexpr int kDiffKeys = 8;                       // consecutive keys of A per thread per batch
constexpr int kDiffBatch = kDiffThreads * kDiffKeys;
constexpr int kDiffMaxBatches = 48;                // batches per block whose masks are cached

struct DiffShared {
    uint8_t mask[kDiffMaxBatches][kDiffThreads];
    int64_t red[32];
    int32_t wtot[kDiffThreads / 32];
};

__device__ __forceinline__ int64_t lower_bound(const uint64_t* __restrict__ a, int64_t lo, int64_t hi,
                                               uint64_t key) {
    while (lo < hi) {
        const int64_t mid = (lo + hi) >> 1;
        if (__ldg(a + mid) < key) lo = mid + 1; else hi = mid;
    }
    return lo;
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

// Bit k of the result: A[i0 + k] (i0 + k < end) is absent from B.
__device__ __forceinline__ uint32_t absent_mask(const uint64_t* __restrict__ A, int64_t i0, int64_t end,
                                                const uint64_t* __restrict__ B, int64_t nB) {
    if (i0 >= end) return 0u;
    uint32_t m = 0;
    int64_t j = lower_bound(B, 0, nB, __ldg(A + i0));
    uint64_t bj = j < nB ? __ldg(B + j) : ~0ull;       // ~0 is never a key (i < j < 2^32)
#pragma unroll
    for (int k = 0; k < kDiffKeys; ++k) {
        if (i0 + k < end) {
            const uint64_t key = __ldg(A + i0 + k);
            while (bj < key) { ++j; bj = j < nB ? __ldg(B + j) : ~0ull; }
            m |= (uint32_t)(bj != key) << k;
        }
    }
    return m;
}

struct DiffParams {
    const uint64_t* prev; const int64_t* n_prev;
    const uint64_t* now;  const int64_t* n_now;
    uint64_t* created; uint64_t* destroyed; int64_t cap;
    int64_t* n_created; int64_t* n_destroyed;
    int64_t* partial;          // [gridDim]
    int32_t* flags;
};

// grid = 2 * nb blocks: blocks [0, nb) handle created = now \ prev, [nb, 2nb) destroyed = prev \ now
__global__ void __launch_bounds__(kDiffThreads, 3) diff_kernel(const DiffParams p) {
    __shared__ DiffShared sh;
    cg::grid_group grid = cg::this_grid();
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int nb = gridDim.x >> 1;
    const bool second = (int)blockIdx.x >= nb;
    const int me = second ? blockIdx.x - nb : blockIdx.x;
    const uint64_t* __restrict__ A = second ? p.prev : p.now;        // elements of A not in B
    const uint64_t* __restrict__ B = second ? p.now : p.prev;
    const int64_t nA = second ? *p.n_prev : *p.n_now, nB = second ? *p.n_now : *p.n_prev;
    uint64_t* __restrict__ out = second ? p.destroyed : p.created;
    int64_t C = (nA + nb - 1) / nb;
    C = (C + 32 * kDiffKeys - 1) / (32 * kDiffKeys) * (32 * kDiffKeys);    // whole warps of full threads
    const int64_t beg = (int64_t)me * C < nA ? (int64_t)me * C : nA;
    const int64_t end = beg + C < nA ? beg + C : nA;
    const int64_t nbatch = (end - beg + kDiffBatch - 1) / kDiffBatch;

    // ---- pass 1: membership + count
    int64_t c = 0;
    for (int64_t k = 0; k < nbatch; ++k) {
        const uint32_t m = absent_mask(A, beg + k * kDiffBatch + (int64_t)threadIdx.x * kDiffKeys, end, B, nB);
        if (k < kDiffMaxBatches) sh.mask[k][threadIdx.x] = (uint8_t)m;
        c += __popc(m);
    }
    c = block_sum(c, sh.red);
    if (threadIdx.x == 0) p.partial[blockIdx.x] = c;
    grid.sync();

    // ---- pass 2: order-preserving write
    int64_t before = 0, all = 0;
    for (int b = threadIdx.x; b < nb; b += kDiffThreads) {
        const int64_t v = __ldcg(p.partial + (second ? nb : 0) + b);
        all += v;
        if (b < me) before += v;
    }
    before = block_sum(before, sh.red);
    all = block_sum(all, sh.red);
    if (me == 0 && threadIdx.x == 0) {
        *(second ? p.n_destroyed : p.n_created) = all;
        if (all > p.cap) atomicOr(p.flags, FLAG_DIFF_CAP);
    }
    int64_t run = before;
    for (int64_t k = 0; k < nbatch; ++k) {
        const int64_t i0 = beg + k * kDiffBatch + (int64_t)threadIdx.x * kDiffKeys;
        const uint32_t m = k < kDiffMaxBatches ? (uint32_t)sh.mask[k][threadIdx.x] : absent_mask(A, i0, end, B, nB);
        const int n = __popc(m);
        int inc = n;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int t = __shfl_up_sync(0xffffffffu, inc, o);
            if (lane >= o) inc += t;
        }
        if (lane == 31) sh.wtot[wid] = inc;
        __syncthreads();
        int32_t wbase = 0, total = 0;
#pragma unroll
        for (int w = 0; w < kDiffThreads / 32; ++w) {
            const int32_t t = sh.wtot[w];
            if (w < wid) wbase += t;
            total += t;
        }
        int64_t pos = run + wbase + inc - n;
#pragma unroll
        for (int q = 0; q < kDiffKeys; ++q) {
            if (m >> q & 1u) {
                if (pos < p.cap) out[pos] = __ldg(A + i0 + q);
                ++pos;
            }
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
                                      ctx->max_raw_keys, &ctx->d_tr_counts[0], FLAG_RAWKEY_OVERFLOW,
                                      4 * (int64_t)n_prev_labels, stream);
        if (rc != VOR_OK) return rc;
        // filtered now -> d_keys_a -> sort/unique -> d_tr_now
        VOR_CUDA(cudaMemsetAsync(ctx->d_n_raw, 0, sizeof(int64_t), stream));
        VOR_LAUNCH(filter_now_kernel, 4 * kNumSMs, 256, 0, stream, d_now, d_n_now, d_n2p, n_now_labels,
                   ctx->d_keys_a, ctx->max_raw_keys, (unsigned long long*)ctx->d_n_raw, ctx->d_flags);
        rc = vor_sort_unique_keys(ctx, ctx->d_keys_a, ctx->d_n_raw, bits, ctx->d_tr_now,
                                  ctx->max_raw_keys, &ctx->d_tr_counts[1], FLAG_RAWKEY_OVERFLOW,
                                  4 * (int64_t)n_now_labels, stream);
        if (rc != VOR_OK) return rc;
        P = ctx->d_tr_prev; nP = &ctx->d_tr_counts[0];
        N = ctx->d_tr_now;  nN = &ctx->d_tr_counts[1];
    }
    DiffParams dp{P, nP, N, nN, d_created, d_destroyed, cap, d_n_created, d_n_destroyed,
                  ctx->d_blk_count, ctx->d_flags};
    int grid = vor_coop_grid(ctx, 2, (const void*)diff_kernel, kDiffThreads, 3);
    grid &= ~1;                                         // one half per direction
    if (grid < 2) return vor_fail(ctx, VOR_ECUDA, "vor_diff: device too small for the cooperative grid");
    VOR_LAUNCH_COOP(diff_kernel, grid, kDiffThreads, stream, (void*)&dp);
    return VOR_OK;
}
