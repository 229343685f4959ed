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

#include <mutex>

#include "common.cuh"
#include "rows.cuh"

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
    int64_t cap_prev, cap_now;     // capacities of the input buffers: the device counts are clamped to them
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
    const int64_t nP = min(*p.n_prev, p.cap_prev), nN = min(*p.n_now, p.cap_now);
    const int64_t nA = second ? nP : nN, nB = second ? nN : nP;
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

// ---------------------------------------------------------------- row-by-row comparison (site path)
// PAPER.md:215-221 (§III.B.3): "each thread accesses a given row of (E_P)_PN and its isomorphic one in
// (E_N)_NN" and compares them.  With persistent site identity both lists come from vor_edges_rows,
// which also returns the offset of every site's row (row a = the keys (a, b), b > a, ascending), so
// row a of the past list and row a of the present list are found without searching.
// Two plain kernels, no grid synchronisation and nothing that waits on another block:
//   diff_rows_mark_kernel   one thread per pair of rows: both rows are loaded at once (all loads
//                           independent), every entry is looked up in the other row in registers; the
//                           16 + 16 bit membership mask of the row goes to a scratch array, the block's
//                           two counts to a per-block array;
//   diff_rows_write_kernel  every block sums the counts of the blocks before it, scans its own masks
//                           and writes the created / destroyed keys in ascending order (only the
//                           changed keys are read again).
// Rows longer than kDrFast entries (hubs, overflowed rows) take a two-pointer merge in both kernels.
constexpr int kDrThreads = 256;
constexpr int kDrPerThread = 2;                    // rows per thread
constexpr int kDrRows = kDrThreads * kDrPerThread; // rows per block
constexpr int kDrFast = 8;                         // row length handled in registers
constexpr uint32_t kDrLong = 0xffffffffu;          // mask marker: a long row (never a valid mask: bits 8-15 stay 0)

struct DiffRowsParams {
    const uint64_t* prev; const uint32_t* prev_ptr;
    const uint64_t* now;  const uint32_t* now_ptr;
    int32_t n_rows;
    uint64_t* created; uint64_t* destroyed; int64_t cap;
    int64_t* n_created; int64_t* n_destroyed;
    uint32_t* masks;               // [n_rows]
    uint32_t* blk_counts;          // [2][n_blocks] created, destroyed keys of every block's rows
    int32_t* flags;
};

__device__ __forceinline__ uint32_t key_lo(const uint64_t* __restrict__ k) {
    return __ldg(reinterpret_cast<const uint32_t*>(k));            // little endian: the larger label b
}

// two-pointer merge of two long rows; emit == false only counts
template <bool kEmit>
__device__ void row_merge(const uint64_t* __restrict__ A, uint32_t a0, uint32_t a1,
                          const uint64_t* __restrict__ B, uint32_t b0, uint32_t b1,
                          uint32_t* ca, uint32_t* cb, uint64_t* outA, int64_t posA, uint64_t* outB, int64_t posB,
                          int64_t cap) {
    uint32_t i = a0, j = b0;
    uint32_t na = 0, nb = 0;
    while (i < a1 || j < b1) {
        const uint64_t x = i < a1 ? __ldg(A + i) : ~0ull, y = j < b1 ? __ldg(B + j) : ~0ull;
        if (x == y) { ++i; ++j; }
        else if (x < y) { if (kEmit && posA + na < cap) outA[posA + na] = x; ++na; ++i; }
        else { if (kEmit && posB + nb < cap) outB[posB + nb] = y; ++nb; ++j; }
    }
    *ca = na; *cb = nb;
}

// warp w of a block owns rows [r0, r0 + 32 * kDrPerThread): row = r0 + 32 k + lane
__device__ __forceinline__ int64_t dr_row0(int wid) {
    return (int64_t)blockIdx.x * kDrRows + (int64_t)wid * (32 * kDrPerThread);
}

__global__ void __launch_bounds__(kDrThreads) diff_rows_mark_kernel(const DiffRowsParams p) {
    __shared__ uint2 wtot[kDrThreads / 32];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int64_t r0 = dr_row0(wid);
    uint32_t a0[kDrPerThread], na[kDrPerThread], b0[kDrPerThread], nb[kDrPerThread];
#pragma unroll
    for (int k = 0; k < kDrPerThread; ++k) {
        const int64_t a = r0 + 32 * k + lane;
        a0[k] = na[k] = b0[k] = nb[k] = 0;
        if (a < p.n_rows) {
            a0[k] = __ldg(p.now_ptr + a); na[k] = __ldg(p.now_ptr + a + 1) - a0[k];
            b0[k] = __ldg(p.prev_ptr + a); nb[k] = __ldg(p.prev_ptr + a + 1) - b0[k];
        }
    }
    uint32_t ea[kDrPerThread][kDrFast], eb[kDrPerThread][kDrFast];
#pragma unroll
    for (int k = 0; k < kDrPerThread; ++k) {
        const bool fast = na[k] <= kDrFast && nb[k] <= kDrFast;
#pragma unroll
        for (int i = 0; i < kDrFast; ++i) {
            ea[k][i] = fast && i < (int)na[k] ? key_lo(p.now + a0[k] + i) : 0xffffffffu;     // the padding never
            eb[k][i] = fast && i < (int)nb[k] ? key_lo(p.prev + b0[k] + i) : 0xfffffffeu;    // equals a label
        }
    }
    uint32_t c = 0, d = 0;
#pragma unroll
    for (int k = 0; k < kDrPerThread; ++k) {
        const int64_t a = r0 + 32 * k + lane;
        uint32_t m;
        if (na[k] <= kDrFast && nb[k] <= kDrFast) {
            uint32_t found = 0;                                   // bit i: ea[i] in prev; bit 16 + j: eb[j] in now
#pragma unroll
            for (int i = 0; i < kDrFast; ++i)
#pragma unroll
                for (int j = 0; j < kDrFast; ++j)
                    if (ea[k][i] == eb[k][j]) found |= (1u << i) | (1u << (16 + j));
            m = (((1u << na[k]) - 1u) | (((1u << nb[k]) - 1u) << 16)) & ~found;
            c += __popc(m & 0xffffu); d += __popc(m >> 16);
        } else {
            uint32_t ca, cb;
            row_merge<false>(p.now, a0[k], a0[k] + na[k], p.prev, b0[k], b0[k] + nb[k], &ca, &cb, nullptr, 0, nullptr, 0, 0);
            m = kDrLong; c += ca; d += cb;
        }
        if (a < p.n_rows) p.masks[a] = m;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) { c += __shfl_xor_sync(0xffffffffu, c, o); d += __shfl_xor_sync(0xffffffffu, d, o); }
    if (lane == 0) wtot[wid] = make_uint2(c, d);
    __syncthreads();
    if (threadIdx.x == 0) {
        uint32_t tc = 0, td = 0;
#pragma unroll
        for (int w = 0; w < kDrThreads / 32; ++w) { tc += wtot[w].x; td += wtot[w].y; }
        p.blk_counts[blockIdx.x] = tc;
        p.blk_counts[gridDim.x + blockIdx.x] = td;
    }
}

__global__ void __launch_bounds__(kDrThreads) diff_rows_write_kernel(const DiffRowsParams p) {
    __shared__ uint2 wtot[kDrThreads / 32];
    __shared__ int64_t red[2][kDrThreads / 32];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int32_t n_blocks = gridDim.x;
    // ---- keys of the blocks before this one (and, in the last block, of all of them)
    int64_t bc = 0, bd = 0;
    for (int32_t b = threadIdx.x; b < (int32_t)blockIdx.x; b += kDrThreads) {
        bc += __ldg(p.blk_counts + b); bd += __ldg(p.blk_counts + n_blocks + b);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) { bc += __shfl_xor_sync(0xffffffffu, bc, o); bd += __shfl_xor_sync(0xffffffffu, bd, o); }
    if (lane == 0) { red[0][wid] = bc; red[1][wid] = bd; }
    // ---- this block's masks and counts; positions inside the warp (k-major), then inside the block
    const int64_t r0 = dr_row0(wid);
    uint32_t m[kDrPerThread], nc[kDrPerThread], nd[kDrPerThread];
#pragma unroll
    for (int k = 0; k < kDrPerThread; ++k) {
        const int64_t a = r0 + 32 * k + lane;
        m[k] = a < p.n_rows ? __ldcs(p.masks + a) : 0u;
        nc[k] = __popc(m[k] & 0xffffu); nd[k] = __popc(m[k] >> 16);
        if (m[k] == kDrLong) {
            const uint32_t a0 = __ldg(p.now_ptr + a), a1 = __ldg(p.now_ptr + a + 1);
            const uint32_t b0 = __ldg(p.prev_ptr + a), b1 = __ldg(p.prev_ptr + a + 1);
            row_merge<false>(p.now, a0, a1, p.prev, b0, b1, &nc[k], &nd[k], nullptr, 0, nullptr, 0, 0);
        }
    }
    uint32_t prec[kDrPerThread], pred[kDrPerThread];
    uint32_t wrc = 0, wrd = 0;                                    // running totals of the warp
#pragma unroll
    for (int k = 0; k < kDrPerThread; ++k) {
        uint32_t ic = nc[k], id = nd[k];
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t tc = __shfl_up_sync(0xffffffffu, ic, o), td = __shfl_up_sync(0xffffffffu, id, o);
            if (lane >= o) { ic += tc; id += td; }
        }
        prec[k] = wrc + ic - nc[k]; pred[k] = wrd + id - nd[k];
        wrc += __shfl_sync(0xffffffffu, ic, 31); wrd += __shfl_sync(0xffffffffu, id, 31);
    }
    if (lane == 0) wtot[wid] = make_uint2(wrc, wrd);
    __syncthreads();
    bc = 0; bd = 0;
    uint32_t totc = 0, totd = 0;
#pragma unroll
    for (int w = 0; w < kDrThreads / 32; ++w) {
        bc += red[0][w]; bd += red[1][w];
        const uint2 t = wtot[w];
        if (w < wid) { bc += t.x; bd += t.y; }
        totc += t.x; totd += t.y;
    }
    if (blockIdx.x == n_blocks - 1 && threadIdx.x == kDrThreads - 1) {   // the last warp: bc, bd exclude only itself
        const int64_t allc = bc + wtot[wid].x, alld = bd + wtot[wid].y;
        *p.n_created = allc; *p.n_destroyed = alld;
        if (allc > p.cap || alld > p.cap) atomicOr(p.flags, FLAG_DIFF_CAP);
    }
    // ---- write: only the changed keys are read again
#pragma unroll
    for (int k = 0; k < kDrPerThread; ++k) {
        if (m[k] == 0) continue;
        const int64_t a = r0 + 32 * k + lane;
        int64_t pc = bc + prec[k], pd = bd + pred[k];
        const uint32_t a0 = __ldg(p.now_ptr + a), b0 = __ldg(p.prev_ptr + a);
        if (m[k] == kDrLong) {
            uint32_t x, y;
            row_merge<true>(p.now, a0, __ldg(p.now_ptr + a + 1), p.prev, b0, __ldg(p.prev_ptr + a + 1), &x, &y,
                            p.created, pc, p.destroyed, pd, p.cap);
            continue;
        }
        for (uint32_t mc = m[k] & 0xffffu; mc; mc &= mc - 1) {
            if (pc < p.cap) p.created[pc] = __ldg(p.now + a0 + (__ffs(mc) - 1));
            ++pc;
        }
        for (uint32_t md = m[k] >> 16; md; md &= md - 1) {
            if (pd < p.cap) p.destroyed[pd] = __ldg(p.prev + b0 + (__ffs(md) - 1));
            ++pd;
        }
    }
}

// prev edge (i,j) -> (p2n[i], p2n[j]); dropped if an endpoint is -1 or both collapse (R22);
// unordered append (sorted afterwards).
__global__ void translate_prev_kernel(const uint64_t* __restrict__ prev, const int64_t* __restrict__ n_prev_p,
                                      int64_t cap_in, const int32_t* __restrict__ p2n, int32_t n_prev_labels,
                                      uint64_t* __restrict__ out, int64_t cap,
                                      unsigned long long* __restrict__ n_out, int32_t* __restrict__ flags) {
    const int64_t n = min(*n_prev_p, cap_in);
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
                                  int64_t cap_in, const int32_t* __restrict__ n2p, int32_t n_now_labels,
                                  uint64_t* __restrict__ out, int64_t cap,
                                  unsigned long long* __restrict__ n_out, int32_t* __restrict__ flags) {
    const int64_t n = min(*n_now_p, cap_in);
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

// the same two filters feeding the adjacency rows directly (row a collects b > a; rows.cuh): the finish
// kernel of vor_edges then returns the sorted unique list with its row offsets, without a radix sort
__global__ void translate_prev_rows_kernel(const uint64_t* __restrict__ prev, const int64_t* __restrict__ n_prev_p,
                                           int64_t cap_in, const int32_t* __restrict__ p2n, int32_t n_prev_labels,
                                           const RowSet rs) {
    const int64_t n = min(*n_prev_p, cap_in);
    for (int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; k < n; k += (int64_t)gridDim.x * blockDim.x) {
        const uint64_t e = prev[k];
        const uint32_t a = (uint32_t)(e >> 32), b = (uint32_t)e;
        if (a >= (uint32_t)n_prev_labels || b >= (uint32_t)n_prev_labels) continue;
        const int32_t i = p2n[a], j = p2n[b];
        if (i < 0 || j < 0 || i == j) continue;
        row_insert(rs, (uint32_t)min(i, j), (uint32_t)max(i, j));
    }
}

__global__ void filter_now_rows_kernel(const uint64_t* __restrict__ now, const int64_t* __restrict__ n_now_p,
                                       int64_t cap_in, const int32_t* __restrict__ n2p, int32_t n_now_labels,
                                       const RowSet rs) {
    const int64_t n = min(*n_now_p, cap_in);
    for (int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; k < n; k += (int64_t)gridDim.x * blockDim.x) {
        const uint64_t e = now[k];
        const uint32_t a = (uint32_t)(e >> 32), b = (uint32_t)e;
        if (a >= (uint32_t)n_now_labels || b >= (uint32_t)n_now_labels) continue;
        if (n2p[a] < 0 || n2p[b] < 0) continue;
        row_insert(rs, a, b);
    }
}

int bits_for(int32_t n) {
    int bits = 1;
    while (bits < 31 && ((int64_t)1 << bits) < (int64_t)n) ++bits;
    return bits;
}

}  // namespace

extern "C" int vor_diff(vor_ctx* ctx, const uint64_t* d_prev, const int64_t* d_n_prev,
                        const uint64_t* d_now, const int64_t* d_n_now, int64_t cap_prev, int64_t cap_now,
                        const int32_t* d_p2n, const int32_t* d_n2p,
                        int32_t n_prev_labels, int32_t n_now_labels,
                        uint64_t* d_created, uint64_t* d_destroyed, int64_t cap,
                        int64_t* d_n_created, int64_t* d_n_destroyed, void* stream_) {
    if (!ctx) return VOR_EINVAL;
    if (int drc_ = vor_check_device(ctx)) return drc_;
    if (!d_prev || !d_n_prev || !d_now || !d_n_now || !d_created || !d_destroyed || !d_n_created ||
        !d_n_destroyed || cap < 0 || cap_prev < 0 || cap_now < 0)
        return vor_fail(ctx, VOR_EINVAL, "vor_diff: null pointer or negative capacity");
    if ((d_p2n == nullptr) != (d_n2p == nullptr))
        return vor_fail(ctx, VOR_EINVAL, "vor_diff: give both maps or neither");
    cudaStream_t stream = (cudaStream_t)stream_;
    const uint64_t* P = d_prev;
    const int64_t* nP = d_n_prev;
    const uint64_t* N = d_now;
    const int64_t* nN = d_n_now;
    int64_t capP = cap_prev, capN = cap_now;
    if (d_p2n) {
        if (n_prev_labels < 1 || n_now_labels < 1)
            return vor_fail(ctx, VOR_EINVAL, "vor_diff: label counts required with maps");
        if (!ctx->d_tr_prev) {
            VOR_CUDA(cudaMalloc((void**)&ctx->d_tr_prev, ctx->max_raw_keys * sizeof(uint64_t)));
            VOR_CUDA(cudaMalloc((void**)&ctx->d_tr_now, ctx->max_raw_keys * sizeof(uint64_t)));
        }
        if (n_now_labels <= ctx->max_sites) {
            // both lists go through the adjacency rows (one row per now label): sorted, unique, with row
            // offsets - then the row-by-row comparison.  No radix sort, no cooperative searching kernel.
            if (!ctx->d_tr_rowptr[0]) {
                VOR_CUDA(cudaMalloc((void**)&ctx->d_tr_rowptr[0], ((size_t)ctx->max_sites + 1) * sizeof(uint32_t)));
                VOR_CUDA(cudaMalloc((void**)&ctx->d_tr_rowptr[1], ((size_t)ctx->max_sites + 1) * sizeof(uint32_t)));
            }
            RowSet rs = vor_row_set(ctx);
            rs.n_rows = n_now_labels;
            VOR_CUDA(cudaMemsetAsync(ctx->d_n_raw, 0, 8 * sizeof(int64_t), stream));
            VOR_LAUNCH(translate_prev_rows_kernel, 4 * kNumSMs, 256, 0, stream, d_prev, d_n_prev, cap_prev, d_p2n,
                       n_prev_labels, rs);
            int rc = vor_edges_finish(ctx, rs, ctx->d_tr_prev, ctx->max_raw_keys, &ctx->d_tr_counts[0],
                                      ctx->d_tr_rowptr[0], false, stream);
            if (rc != VOR_OK) return rc;
            VOR_CUDA(cudaMemsetAsync(ctx->d_n_raw, 0, 8 * sizeof(int64_t), stream));
            VOR_LAUNCH(filter_now_rows_kernel, 4 * kNumSMs, 256, 0, stream, d_now, d_n_now, cap_now, d_n2p,
                       n_now_labels, rs);
            rc = vor_edges_finish(ctx, rs, ctx->d_tr_now, ctx->max_raw_keys, &ctx->d_tr_counts[1],
                                  ctx->d_tr_rowptr[1], false, stream);
            if (rc != VOR_OK) return rc;
            return vor_diff_rows(ctx, ctx->d_tr_prev, ctx->d_tr_rowptr[0], ctx->d_tr_now, ctx->d_tr_rowptr[1],
                                 n_now_labels, d_created, d_destroyed, cap, d_n_created, d_n_destroyed, stream_);
        }
        const int bits = bits_for(n_now_labels);
        // translated prev -> d_keys_a -> sort/unique -> d_tr_prev
        VOR_CUDA(cudaMemsetAsync(ctx->d_n_raw, 0, sizeof(int64_t), stream));
        VOR_LAUNCH(translate_prev_kernel, 4 * kNumSMs, 256, 0, stream, d_prev, d_n_prev, cap_prev, d_p2n,
                   n_prev_labels, ctx->d_keys_a, ctx->max_raw_keys,
                   (unsigned long long*)ctx->d_n_raw, ctx->d_flags);
        int rc = vor_sort_unique_keys(ctx, ctx->d_keys_a, ctx->d_n_raw, bits, ctx->d_tr_prev,
                                      ctx->max_raw_keys, &ctx->d_tr_counts[0], FLAG_RAWKEY_OVERFLOW,
                                      4 * (int64_t)n_prev_labels, stream);
        if (rc != VOR_OK) return rc;
        // filtered now -> d_keys_a -> sort/unique -> d_tr_now
        VOR_CUDA(cudaMemsetAsync(ctx->d_n_raw, 0, sizeof(int64_t), stream));
        VOR_LAUNCH(filter_now_kernel, 4 * kNumSMs, 256, 0, stream, d_now, d_n_now, cap_now, d_n2p, n_now_labels,
                   ctx->d_keys_a, ctx->max_raw_keys, (unsigned long long*)ctx->d_n_raw, ctx->d_flags);
        rc = vor_sort_unique_keys(ctx, ctx->d_keys_a, ctx->d_n_raw, bits, ctx->d_tr_now,
                                  ctx->max_raw_keys, &ctx->d_tr_counts[1], FLAG_RAWKEY_OVERFLOW,
                                  4 * (int64_t)n_now_labels, stream);
        if (rc != VOR_OK) return rc;
        P = ctx->d_tr_prev; nP = &ctx->d_tr_counts[0];
        N = ctx->d_tr_now;  nN = &ctx->d_tr_counts[1];
        capP = capN = ctx->max_raw_keys;
    }
    DiffParams dp{P, nP, N, nN, capP, capN, d_created, d_destroyed, cap, d_n_created, d_n_destroyed,
                  ctx->d_blk_count, ctx->d_flags};
    int grid = vor_coop_grid(ctx, 2, (const void*)diff_kernel, kDiffThreads, 3);
    grid &= ~1;                                         // one half per direction
    if (grid < 2) return vor_fail(ctx, VOR_ECUDA, "vor_diff: device too small for the cooperative grid");
    VOR_LAUNCH_COOP(diff_kernel, grid, kDiffThreads, stream, (void*)&dp);
    return VOR_OK;
}

extern "C" int vor_diff_rows(vor_ctx* ctx, const uint64_t* d_prev, const uint32_t* d_prev_row_ptr,
                             const uint64_t* d_now, const uint32_t* d_now_row_ptr, int32_t n_rows,
                             uint64_t* d_created, uint64_t* d_destroyed, int64_t cap,
                             int64_t* d_n_created, int64_t* d_n_destroyed, void* stream_) {
    if (!ctx) return VOR_EINVAL;
    if (int drc_ = vor_check_device(ctx)) return drc_;
    if (!d_prev || !d_prev_row_ptr || !d_now || !d_now_row_ptr || !d_created || !d_destroyed ||
        !d_n_created || !d_n_destroyed || cap < 0)
        return vor_fail(ctx, VOR_EINVAL, "vor_diff_rows: null pointer or negative capacity");
    if (n_rows < 1) return vor_fail(ctx, VOR_EINVAL, "vor_diff_rows: n_rows must be >= 1");
    cudaStream_t stream = (cudaStream_t)stream_;
    const int64_t n_blocks = ((int64_t)n_rows + kDrRows - 1) / kDrRows;
    if (!ctx->d_dr_scratch || ctx->dr_rows < n_rows) {
        if (ctx->d_dr_scratch) { VOR_CUDA(cudaStreamSynchronize(stream)); VOR_CUDA(cudaFree(ctx->d_dr_scratch)); ctx->d_dr_scratch = nullptr; }
        const int64_t rows = n_rows > ctx->max_sites ? n_rows : ctx->max_sites;
        const int64_t blocks = (rows + kDrRows - 1) / kDrRows;
        VOR_CUDA(cudaMalloc((void**)&ctx->d_dr_scratch, ((size_t)rows + 2 * (size_t)blocks) * sizeof(uint32_t)));
        ctx->dr_rows = rows;
    }
    DiffRowsParams dp{d_prev, d_prev_row_ptr, d_now, d_now_row_ptr, n_rows, d_created, d_destroyed, cap,
                      d_n_created, d_n_destroyed, ctx->d_dr_scratch, ctx->d_dr_scratch + ctx->dr_rows, ctx->d_flags};
    VOR_LAUNCH(diff_rows_mark_kernel, (unsigned)n_blocks, kDrThreads, 0, stream, dp);
    VOR_LAUNCH(diff_rows_write_kernel, (unsigned)n_blocks, kDrThreads, 0, stream, dp);
    return VOR_OK;
}

// ------------------------------------------------------------------------------------------------------------
// vor_diff_rows_static: the row-by-row comparison for callers that may not allocate device memory (a host
// framework that owns the GPU's memory pool, a process with a memory budget fixed at start-up, a latency path
// that cannot take cudaMalloc's device-wide synchronisation).  Same two kernels as vor_diff_rows; their working
// memory is the file-scope array below instead of a context buffer.  include/vor.h states the contract.
namespace {

constexpr int64_t kStaticMaxRows = VOR_DIFF_ROWS_STATIC_MAX_ROWS;
constexpr int64_t kStaticMaxBlocks = (kStaticMaxRows + kDrRows - 1) / kDrRows;
constexpr int64_t kStaticWords = kStaticMaxRows + 2 * kStaticMaxBlocks + 64;   // masks | block counts | flag word

// 4.02 MiB in the image of every GPU that loads the library.  HOST code must not use this name as a pointer:
// there it is only a handle for cudaGetSymbolAddress (static_scratch_address below).
static __device__ __align__(256) uint32_t g_static_scratch[kStaticWords];

constexpr int kStaticMaxDevices = 64;
std::mutex g_static_mu;
uint32_t* g_static_addr[kStaticMaxDevices];     // device address of g_static_scratch, per device ordinal

// Device address of the array on the CURRENT device; looked up once per device, with that device current.
cudaError_t static_scratch_address(uint32_t** out) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= kStaticMaxDevices) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_static_mu);
    if (!g_static_addr[dev]) {
        void* ptr = nullptr;
        e = cudaGetSymbolAddress(&ptr, g_static_scratch);
        if (e != cudaSuccess) return e;
        g_static_addr[dev] = static_cast<uint32_t*>(ptr);
    }
    *out = g_static_addr[dev];
    return cudaSuccess;
}

}  // namespace

extern "C" int vor_diff_rows_static(const uint64_t* d_prev, const uint32_t* d_prev_row_ptr,
                                    const uint64_t* d_now, const uint32_t* d_now_row_ptr, int32_t n_rows,
                                    uint64_t* d_created, uint64_t* d_destroyed, int64_t cap,
                                    int64_t* d_n_created, int64_t* d_n_destroyed, void* stream_) {
    if (!d_prev || !d_prev_row_ptr || !d_now || !d_now_row_ptr || !d_created || !d_destroyed ||
        !d_n_created || !d_n_destroyed || cap < 0 || n_rows < 1)
        return VOR_EINVAL;
    if (n_rows > kStaticMaxRows) return VOR_ELIMIT;       // before any CUDA call: nothing is enqueued
    uint32_t* scratch = nullptr;
    if (static_scratch_address(&scratch) != cudaSuccess) return VOR_ECUDA;
    cudaStream_t stream = (cudaStream_t)stream_;
    const unsigned n_blocks = (unsigned)(((int64_t)n_rows + kDrRows - 1) / kDrRows);
    // masks: words [0, n_rows); block counts: 2 * n_blocks words from kStaticMaxRows on; the last word takes the
    // kernels' overflow bit, which nobody reads here (the caller compares the counts with cap).  Every word the
    // second kernel reads is written by the first one, so stale contents of an earlier call never matter.
    DiffRowsParams dp{d_prev, d_prev_row_ptr, d_now, d_now_row_ptr, n_rows, d_created, d_destroyed, cap,
                      d_n_created, d_n_destroyed, scratch, scratch + kStaticMaxRows,
                      reinterpret_cast<int32_t*>(scratch + kStaticWords - 1)};
    diff_rows_mark_kernel<<<n_blocks, kDrThreads, 0, stream>>>(dp);
    if (cudaGetLastError() != cudaSuccess) return VOR_ECUDA;
    diff_rows_write_kernel<<<n_blocks, kDrThreads, 0, stream>>>(dp);
    if (cudaGetLastError() != cudaSuccess) return VOR_ECUDA;
    return VOR_OK;
}

// ------------------------------------------------------------------------------------------------------------
// Union of several ASCENDING key lists (multi-GPU row strips: every rank extracts the keys of its
// strip, one all-gather brings the lists together, "followed by a merge-unique").  The lists are merged pairwise
// in ceil(log2 n_lists) rounds by merge path (one co-rank search per 8 output slots, then a sequential merge;
// repeats are kept, so every round's layout is the concatenation given by the prefix sums of the counts), then
// one order-preserving pass drops the repeats.
namespace {

constexpr int kMlThreads = 256, kMlPer = 8, kMlMaxLists = 1024;

struct MergeRound {
    const uint64_t* src;       // round 0: the caller's buffers, list l at l * stride; later: concatenated
    int round0;
    int64_t stride;
    uint64_t* dst;             // concatenated
    const int64_t* counts;
    int32_t n_lists;
    int32_t span;              // lists per input segment (1, 2, 4, ...); output segments hold 2 * span lists
    int64_t* total;            // sum of the (clamped) counts
    int32_t* flags;            // sticky status: FLAG_EDGE_CAP when a count exceeds the stride
};

__global__ void __launch_bounds__(kMlThreads) merge_round_kernel(const MergeRound m) {
    __shared__ int64_t pre[kMlMaxLists + 1];
    for (int l = threadIdx.x; l < m.n_lists; l += kMlThreads) {
        const int64_t c = m.counts[l];
        pre[l + 1] = min(max(c, (int64_t)0), m.stride);
        // a list that overflowed its slot upstream is merged truncated: every rank that merges it must hear of it,
        // not only the rank that produced it (its own vor_edges_image latched the same bit there)
        if (m.round0 && blockIdx.x == 0 && c > m.stride) atomicOr(m.flags, FLAG_EDGE_CAP);
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        pre[0] = 0;
        for (int l = 0; l < m.n_lists; ++l) pre[l + 1] += pre[l];
        if (blockIdx.x == 0) *m.total = pre[m.n_lists];
    }
    __syncthreads();
    const int64_t total = pre[m.n_lists];
    const int32_t two = 2 * m.span, nseg = (m.n_lists + two - 1) / two;
    for (int64_t p0 = ((int64_t)blockIdx.x * kMlThreads + threadIdx.x) * kMlPer; p0 < total;
         p0 += (int64_t)gridDim.x * kMlThreads * kMlPer) {
        int64_t p = p0;
        const int64_t p_end = min(p0 + kMlPer, total);
        while (p < p_end) {
            // the output segment that holds slot p: the last S with pre[S * two] <= p
            int32_t lo = 0, hi = nseg - 1;
            while (lo < hi) {
                const int32_t mid = (lo + hi + 1) >> 1;
                if (pre[min(mid * two, m.n_lists)] <= p) lo = mid; else hi = mid - 1;
            }
            const int32_t l0 = lo * two, l1 = min(l0 + m.span, m.n_lists), l2 = min(l0 + two, m.n_lists);
            const int64_t s0 = pre[l0], nA = pre[l1] - s0, nB = pre[l2] - pre[l1];
            if (nA + nB == 0) { ++p; continue; }          // cannot happen for p < total; keeps the loop finite
            const uint64_t* __restrict__ A = m.round0 ? m.src + (int64_t)l0 * m.stride : m.src + s0;
            const uint64_t* __restrict__ B = m.round0 ? m.src + (int64_t)l1 * m.stride : m.src + s0 + nA;
            const int64_t d0 = p - s0;
            int64_t a = max((int64_t)0, d0 - nB), b = min(d0, nA);
            while (a < b) {                                 // co-rank: a keys of A and d0 - a keys of B precede slot d0
                const int64_t mid = (a + b) >> 1, j = d0 - mid;
                if (j > 0 && B[j - 1] >= A[mid]) a = mid + 1; else b = mid;   // ties: A first
            }
            int64_t i = a, j = d0 - a;
            const int64_t seg_end = min(p_end, s0 + nA + nB);
            for (; p < seg_end; ++p) {
                uint64_t key;
                if (j >= nB || (i < nA && A[i] <= B[j])) key = A[i++]; else key = B[j++];
                m.dst[p] = key;
            }
        }
    }
}

struct UniqueParams {
    const uint64_t* in; const int64_t* n_in; int64_t cap_in;
    uint64_t* out; int64_t cap; int64_t* n_out; int64_t* partial; int32_t* flags; int flag_bit;
};

__device__ __forceinline__ void ml_chunk(int64_t n, int64_t* beg, int64_t* end) {
    int64_t C = (n + gridDim.x - 1) / gridDim.x;
    C = (C + kMlThreads - 1) / kMlThreads * kMlThreads;
    const int64_t s = (int64_t)blockIdx.x * C;
    *beg = s < n ? s : n;
    *end = s + C < n ? s + C : n;
}

__device__ __forceinline__ int64_t ml_block_sum(int64_t v, int64_t* sh) {
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    if (lane == 0) sh[wid] = v;
    __syncthreads();
    int64_t t = lane < kMlThreads / 32 ? sh[lane] : 0;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
    __syncthreads();
    return t;
}

__global__ void __launch_bounds__(kMlThreads) unique_count_kernel(const UniqueParams p) {
    __shared__ int64_t sh[32];
    const int64_t n = min(*p.n_in, p.cap_in);
    int64_t beg, end;
    ml_chunk(n, &beg, &end);
    int64_t c = 0;
    for (int64_t i = beg + threadIdx.x; i < end; i += kMlThreads) c += i == 0 || p.in[i] != p.in[i - 1];
    c = ml_block_sum(c, sh);
    if (threadIdx.x == 0) p.partial[blockIdx.x] = c;
}

__global__ void __launch_bounds__(kMlThreads) unique_write_kernel(const UniqueParams p) {
    __shared__ int64_t sh[32];
    __shared__ int32_t wtot[kMlThreads / 32];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int64_t n = min(*p.n_in, p.cap_in);
    int64_t beg, end;
    ml_chunk(n, &beg, &end);
    int64_t before = 0, all = 0;
    for (int b = threadIdx.x; b < (int)gridDim.x; b += kMlThreads) {
        const int64_t v = p.partial[b];
        all += v;
        if (b < (int)blockIdx.x) before += v;
    }
    before = ml_block_sum(before, sh);
    all = ml_block_sum(all, sh);
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        *p.n_out = all;
        if (all > p.cap) atomicOr(p.flags, p.flag_bit);
    }
    int64_t run = before;
    for (int64_t sub = beg; sub < end; sub += kMlThreads) {
        const int64_t i = sub + threadIdx.x;
        const uint64_t key = i < end ? p.in[i] : 0;
        const bool keep = i < end && (i == 0 || key != p.in[i - 1]);
        const unsigned ball = __ballot_sync(0xffffffffu, keep);
        if (lane == 0) wtot[wid] = __popc(ball);
        __syncthreads();
        int32_t wbase = 0, total = 0;
#pragma unroll
        for (int w = 0; w < kMlThreads / 32; ++w) {
            const int32_t t = wtot[w];
            if (w < wid) wbase += t;
            total += t;
        }
        const int64_t pos = run + wbase + __popc(ball & ((1u << lane) - 1u));
        if (keep && pos < p.cap) p.out[pos] = key;
        run += total;
        __syncthreads();
    }
}

}  // namespace

extern "C" int vor_merge_lists(vor_ctx* ctx, const uint64_t* d_lists, int64_t stride, const int64_t* d_counts,
                               int32_t n_lists, int32_t n_labels, uint64_t* d_out, int64_t cap, int64_t* d_n_out,
                               void* stream_) {
    if (!ctx) return VOR_EINVAL;
    if (int drc_ = vor_check_device(ctx)) return drc_;
    if (!d_lists || !d_counts || !d_out || !d_n_out) return vor_fail(ctx, VOR_EINVAL, "vor_merge_lists: null pointer");
    if (stride < 0 || n_lists < 1 || n_lists > kMlMaxLists || n_labels < 1 || cap < 0)
        return vor_fail(ctx, VOR_EINVAL, "vor_merge_lists: stride >= 0, 1 <= n_lists <= 1024, n_labels >= 1, cap >= 0");
    if (stride * n_lists > ctx->max_raw_keys)
        return vor_fail(ctx, VOR_EINVAL, "vor_merge_lists: stride * n_lists exceeds the context's max_raw_keys scratch");
    cudaStream_t stream = (cudaStream_t)stream_;
    const int grid = 8 * ctx->num_sms;
    uint64_t* buf[2] = {ctx->d_keys_a, ctx->d_keys_b};
    const uint64_t* src = d_lists;
    int which = 0;
    for (int32_t span = 1, round = 0; round == 0 || span < n_lists; span *= 2, ++round) {
        MergeRound m{src, round == 0, stride, buf[which], d_counts, n_lists, span, ctx->d_n_raw, ctx->d_flags};
        VOR_LAUNCH(merge_round_kernel, grid, kMlThreads, 0, stream, m);
        src = buf[which];
        which ^= 1;
    }
    UniqueParams up{src, ctx->d_n_raw, ctx->max_raw_keys, d_out, cap, d_n_out, ctx->d_blk_count, ctx->d_flags, FLAG_EDGE_CAP};
    const int ugrid = min(4 * ctx->num_sms, 2 * kMaxCoopBlocks);   // one partial per block in d_blk_count
    VOR_LAUNCH(unique_count_kernel, ugrid, kMlThreads, 0, stream, up);
    VOR_LAUNCH(unique_write_kernel, ugrid, kMlThreads, 0, stream, up);
    return VOR_OK;
}
