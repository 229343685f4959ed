// a3 + a4 — site-adjacency (digital Delaunay) edge set.
// Paper: the Delaunay graph as an adjacency matrix (§III.B) filled from the coloured
// lattice and "compressed" by sort + unique.  This build's rule
// (R6, BASELINE.json): every 4-connected label discontinuity (right, down, periodic wrap)
// contributes the pair (min,max), packed as (min << 32 | max); the result is the ascending unique list.
//
//   emit:   stream the label image once (128-bit loads), compare right/down, de-duplicate keys in a
//           per-CTA shared-memory hash set, append the CTA's distinct keys to a global buffer with
//           one atomic per CTA.  ~40 raw discontinuities per site collapse to ~4 keys per site.
//   sort:   LSD radix sort, 8 bits per pass, only the 2*ceil(log2 N) significant bits; persistent
//           one-CTA-per-SM kernels, each CTA owns a contiguous chunk (stable by construction).
//   unique: head flags + order-preserving compaction (count kernel, write kernel).
#include "common.cuh"

namespace {

constexpr uint64_t kEmpty = ~0ull;

// ------------------------------------------------------------------------------------ emit
constexpr int kEmitThreads = 256;
constexpr int kEmitCols = 128;          // per CTA tile: 32 lanes x 4 labels
constexpr int kEmitRowsPerWarp = 8;
constexpr int kEmitRows = (kEmitThreads / 32) * kEmitRowsPerWarp;   // 64
constexpr int kHashSlots = 1024;
constexpr int kMaxProbe = 48;

__device__ __forceinline__ uint32_t hash_key(uint32_t a, uint32_t b) {
    uint32_t h = a * 0x9E3779B1u ^ (b * 0x85EBCA77u);
    h ^= h >> 15;
    return h;
}

struct EmitShared {
    unsigned long long table[kHashSlots];
    int32_t scan[kEmitThreads / 32];
    long long base;
};

__device__ __forceinline__ void emit_pair(int32_t a, int32_t b, EmitShared& sh,
                                          uint64_t* __restrict__ keys, int64_t cap,
                                          unsigned long long* __restrict__ n_raw, int32_t* flags) {
    const uint32_t lo = (uint32_t)min(a, b), hi = (uint32_t)max(a, b);
    const unsigned long long key = ((unsigned long long)lo << 32) | hi;
    uint32_t h = hash_key(lo, hi) & (kHashSlots - 1);
    for (int probe = 0; probe < kMaxProbe; ++probe) {
        const unsigned long long cur = sh.table[h];
        if (cur == key) return;
        if (cur == kEmpty) {
            const unsigned long long old = atomicCAS(&sh.table[h], kEmpty, key);
            if (old == kEmpty || old == key) return;
        }
        h = (h + 1) & (kHashSlots - 1);
    }
    // table crowded (very dense sites): emit straight to global, duplicates are removed later
    const unsigned long long pos = atomicAdd(n_raw, 1ull);
    if ((int64_t)pos < cap) keys[pos] = key;
    else atomicOr(flags, FLAG_RAWKEY_OVERFLOW);
}

template <bool VEC>
__global__ void __launch_bounds__(kEmitThreads) edges_emit_kernel(
        const int32_t* __restrict__ labels, int32_t L, uint64_t* __restrict__ keys, int64_t cap,
        unsigned long long* __restrict__ n_raw, int32_t* __restrict__ flags) {
    __shared__ EmitShared sh;
    for (int i = threadIdx.x; i < kHashSlots; i += kEmitThreads) sh.table[i] = kEmpty;
    __syncthreads();
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int32_t x0 = blockIdx.x * kEmitCols + lane * 4;
    const int32_t ybeg = blockIdx.y * kEmitRows + wid * kEmitRowsPerWarp;
    const bool active = x0 < L;                    // VEC: L % 4 == 0, so 4 columns are all in or out
    if (ybeg < L) {
        int32_t c[4], nx[4];
        auto load_row = [&](int32_t y, int32_t* v) {
            if (!active) { v[0] = v[1] = v[2] = v[3] = 0; return; }
            const int32_t* row = labels + (int64_t)y * L;
            if (VEC) {
                const int4 t = __ldg(reinterpret_cast<const int4*>(row + x0));
                v[0] = t.x; v[1] = t.y; v[2] = t.z; v[3] = t.w;
            } else {
#pragma unroll
                for (int k = 0; k < 4; ++k) v[k] = x0 + k < L ? __ldg(row + x0 + k) : -1;
            }
        };
        load_row(ybeg, c);
        const int32_t yend = min(ybeg + kEmitRowsPerWarp, L);
        for (int32_t y = ybeg; y < yend; ++y) {
            const int32_t yn = y + 1 == L ? 0 : y + 1;
            load_row(yn, nx);
            // right neighbour of my 4th column: next lane's first column, or a wrapped load
            int32_t r = __shfl_down_sync(0xffffffffu, c[0], 1);
            if (active) {
                const int32_t xr = x0 + 4;
                if (lane == 31 || xr >= L) r = __ldg(labels + (int64_t)y * L + (xr >= L ? xr - L : xr));
                if (VEC) {
                    if (c[0] != c[1]) emit_pair(c[0], c[1], sh, keys, cap, n_raw, flags);
                    if (c[1] != c[2]) emit_pair(c[1], c[2], sh, keys, cap, n_raw, flags);
                    if (c[2] != c[3]) emit_pair(c[2], c[3], sh, keys, cap, n_raw, flags);
                    if (c[3] != r) emit_pair(c[3], r, sh, keys, cap, n_raw, flags);
#pragma unroll
                    for (int k = 0; k < 4; ++k)
                        if (c[k] != nx[k]) emit_pair(c[k], nx[k], sh, keys, cap, n_raw, flags);
                } else {
                    // ragged row end: column k's right neighbour is k+1, or column 0 through the wrap
#pragma unroll
                    for (int k = 0; k < 4; ++k) {
                        if (x0 + k >= L) break;
                        int32_t rk;
                        if (x0 + k + 1 >= L) rk = __ldg(labels + (int64_t)y * L);
                        else rk = k < 3 ? c[k + 1] : r;
                        if (c[k] != rk) emit_pair(c[k], rk, sh, keys, cap, n_raw, flags);
                        if (c[k] != nx[k]) emit_pair(c[k], nx[k], sh, keys, cap, n_raw, flags);
                    }
                }
            }
#pragma unroll
            for (int k = 0; k < 4; ++k) c[k] = nx[k];
        }
    }
    __syncthreads();
    // compact the hash set: 4 slots per thread
    unsigned long long mine[kHashSlots / kEmitThreads];
    int32_t cnt = 0;
#pragma unroll
    for (int k = 0; k < kHashSlots / kEmitThreads; ++k) {
        mine[k] = sh.table[threadIdx.x * (kHashSlots / kEmitThreads) + k];
        cnt += mine[k] != kEmpty;
    }
    int32_t inc = cnt;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        int32_t t = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += t;
    }
    if (lane == 31) sh.scan[wid] = inc;
    __syncthreads();
    int32_t wbase = 0, total = 0;
#pragma unroll
    for (int k = 0; k < kEmitThreads / 32; ++k) {
        if (k < wid) wbase += sh.scan[k];
        total += sh.scan[k];
    }
    if (threadIdx.x == 0) sh.base = total ? (long long)atomicAdd(n_raw, (unsigned long long)total) : 0;
    __syncthreads();
    if (total == 0) return;
    const int64_t base = sh.base;
    if (base + total > cap) {
        if (threadIdx.x == 0) atomicOr(flags, FLAG_RAWKEY_OVERFLOW);
        return;
    }
    int64_t pos = base + wbase + inc - cnt;
#pragma unroll
    for (int k = 0; k < kHashSlots / kEmitThreads; ++k)
        if (mine[k] != kEmpty) keys[pos++] = mine[k];
}

// ------------------------------------------------------------------------------------ radix sort
constexpr int kKeysPerThread = 4;
constexpr int kSubTile = kSortThreads * kKeysPerThread;       // 4096 keys
constexpr int kSortWarps = kSortThreads / 32;

struct DigitSpec {
    int label_bits;    // significant bits of each 32-bit half
    int shift;         // 8 * pass
};

__device__ __forceinline__ uint32_t digit_of(uint64_t key, DigitSpec ds) {
    const uint64_t compact = ((key >> 32) << ds.label_bits) | (key & 0xffffffffull);
    return (uint32_t)(compact >> ds.shift) & 255u;
}

// chunk of block b: [b*C, min((b+1)*C, n)), C = ceil(n / gridDim) rounded up to the sub-tile size
__device__ __forceinline__ void block_chunk(int64_t n, int64_t* beg, int64_t* end) {
    int64_t C = (n + gridDim.x - 1) / gridDim.x;
    C = (C + kSubTile - 1) / kSubTile * kSubTile;
    int64_t b = (int64_t)blockIdx.x * C;
    *beg = b < n ? b : n;
    *end = b + C < n ? b + C : n;
}

__global__ void __launch_bounds__(kSortThreads) radix_hist_kernel(
        const uint64_t* __restrict__ in, const int64_t* __restrict__ n_ptr, int64_t n_cap,
        DigitSpec ds, uint32_t* __restrict__ hist) {
    __shared__ uint32_t h[256];
    if (threadIdx.x < 256) h[threadIdx.x] = 0;
    __syncthreads();
    const int64_t n = min(*n_ptr, n_cap);
    int64_t beg, end;
    block_chunk(n, &beg, &end);
    for (int64_t i = beg + threadIdx.x; i < end; i += kSortThreads) atomicAdd(&h[digit_of(in[i], ds)], 1u);
    __syncthreads();
    if (threadIdx.x < 256) hist[blockIdx.x * 256 + threadIdx.x] = h[threadIdx.x];
}

__global__ void __launch_bounds__(kSortThreads) radix_scatter_kernel(
        const uint64_t* __restrict__ in, uint64_t* __restrict__ out, const int64_t* __restrict__ n_ptr,
        int64_t n_cap, DigitSpec ds, const uint32_t* __restrict__ hist) {
    __shared__ uint32_t cnt[kSortWarps][256];      // per-warp digit counts, then per-warp bases
    __shared__ uint32_t running[256];
    __shared__ uint32_t wsum[8];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int64_t n = min(*n_ptr, n_cap);
    int64_t beg, end;
    block_chunk(n, &beg, &end);
    if (beg >= end) return;

    // global base of (digit d, this block) = sum over digits < d of all blocks + blocks < me of d
    if (threadIdx.x < 256) {
        const int d = threadIdx.x;
        uint32_t total = 0, before = 0;
        for (int b = 0; b < (int)gridDim.x; ++b) {
            const uint32_t v = hist[b * 256 + d];
            total += v;
            if (b < (int)blockIdx.x) before += v;
        }
        // exclusive scan of `total` over the 256 digits (8 warps)
        uint32_t inc = total;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            uint32_t t = __shfl_up_sync(0xffffffffu, inc, o);
            if (lane >= o) inc += t;
        }
        if (lane == 31) wsum[wid] = inc;
        running[d] = inc - total + before;          // completed below with the warp offsets
    }
    __syncthreads();
    if (threadIdx.x < 256) {
        uint32_t off = 0;
        for (int k = 0; k < wid; ++k) off += wsum[k];
        running[threadIdx.x] += off;
    }
    __syncthreads();

    for (int64_t sub = beg; sub < end; sub += kSubTile) {
        for (int i = threadIdx.x; i < kSortWarps * 256; i += kSortThreads) (&cnt[0][0])[i] = 0;
        __syncthreads();
        uint64_t key[kKeysPerThread];
        uint32_t dg[kKeysPerThread], rk[kKeysPerThread];
        const int64_t wbase = sub + (int64_t)wid * (32 * kKeysPerThread);
#pragma unroll
        for (int it = 0; it < kKeysPerThread; ++it) {
            const int64_t i = wbase + it * 32 + lane;
            const bool valid = i < end;
            key[it] = valid ? in[i] : 0;
            dg[it] = valid ? digit_of(key[it], ds) : 256u;
            const unsigned peers = __match_any_sync(0xffffffffu, dg[it]);
            const int leader = __ffs(peers) - 1;
            uint32_t old = 0;
            if (valid && lane == leader) {
                old = cnt[wid][dg[it]];
                cnt[wid][dg[it]] = old + __popc(peers);
            }
            old = __shfl_sync(0xffffffffu, old, leader);
            rk[it] = old + __popc(peers & ((1u << lane) - 1u));
            __syncwarp();
        }
        __syncthreads();
        if (threadIdx.x < 256) {
            const int d = threadIdx.x;
            uint32_t run = running[d];
#pragma unroll 4
            for (int w = 0; w < kSortWarps; ++w) {
                const uint32_t t = cnt[w][d];
                cnt[w][d] = run;
                run += t;
            }
            running[d] = run;
        }
        __syncthreads();
#pragma unroll
        for (int it = 0; it < kKeysPerThread; ++it)
            if (dg[it] < 256u) out[cnt[wid][dg[it]] + rk[it]] = key[it];
        __syncthreads();
    }
}

// ------------------------------------------------------------------------------------ unique
__device__ __forceinline__ int64_t block_sum_i64(int64_t v, int64_t* sh /* [32] */) {
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

__global__ void __launch_bounds__(kSortThreads) unique_count_kernel(
        const uint64_t* __restrict__ keys, const int64_t* __restrict__ n_ptr, int64_t n_cap,
        int64_t* __restrict__ blk_count) {
    __shared__ int64_t sh[32];
    const int64_t n = min(*n_ptr, n_cap);
    int64_t beg, end;
    block_chunk(n, &beg, &end);
    int64_t c = 0;
    for (int64_t i = beg + threadIdx.x; i < end; i += kSortThreads)
        c += (i == 0 || keys[i] != keys[i - 1]);
    c = block_sum_i64(c, sh);
    if (threadIdx.x == 0) blk_count[blockIdx.x] = c;
}

__global__ void __launch_bounds__(kSortThreads) unique_write_kernel(
        const uint64_t* __restrict__ keys, const int64_t* __restrict__ n_ptr, int64_t n_cap,
        const int64_t* __restrict__ blk_count, uint64_t* __restrict__ out, int64_t cap,
        int64_t* __restrict__ n_out, int32_t* __restrict__ flags, int flag_bit) {
    __shared__ int64_t sh[32];
    __shared__ int32_t wtot[kSortWarps];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int64_t n = min(*n_ptr, n_cap);
    int64_t beg, end;
    block_chunk(n, &beg, &end);
    int64_t before = 0, all = 0;
    for (int b = threadIdx.x; b < (int)gridDim.x; b += kSortThreads) {
        const int64_t v = blk_count[b];
        all += v;
        if (b < (int)blockIdx.x) before += v;
    }
    before = block_sum_i64(before, sh);
    all = block_sum_i64(all, sh);
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        *n_out = all;
        if (all > cap) atomicOr(flags, flag_bit);
    }
    int64_t run = before;
    for (int64_t sub = beg; sub < end; sub += kSortThreads) {
        const int64_t i = sub + threadIdx.x;
        uint64_t k = 0;
        bool head = false;
        if (i < end) {
            k = keys[i];
            head = (i == 0 || k != keys[i - 1]);
        }
        const unsigned ball = __ballot_sync(0xffffffffu, head);
        if (lane == 0) wtot[wid] = __popc(ball);
        __syncthreads();
        int32_t wbase = 0, total = 0;
        for (int w = 0; w < kSortWarps; ++w) {
            const int32_t t = wtot[w];
            if (w < wid) wbase += t;
            total += t;
        }
        if (head) {
            const int64_t pos = run + wbase + __popc(ball & ((1u << lane) - 1u));
            if (pos < cap) out[pos] = k;
        }
        run += total;
        __syncthreads();
    }
}

}  // namespace

// Sort the *d_n_in keys held in ctx->d_keys_a (d_keys_in_a must be that buffer) and write the
// ascending unique list to d_out[0..cap), its length to *d_n_out.  key_bits = significant bits of
// each 32-bit half.  Uses ctx->d_keys_b as the pong buffer.
int vor_sort_unique_keys(vor_ctx* ctx, uint64_t* d_keys_in_a, const int64_t* d_n_in, int key_bits,
                         uint64_t* d_out, int64_t cap, int64_t* d_n_out, int flag_bit,
                         cudaStream_t stream) {
    const int passes = (2 * key_bits + 7) / 8;
    uint64_t* src = d_keys_in_a;
    uint64_t* dst = ctx->d_keys_b;
    for (int pass = 0; pass < passes; ++pass) {
        DigitSpec ds{key_bits, 8 * pass};
        VOR_LAUNCH(radix_hist_kernel, kSortBlocks, kSortThreads, 0, stream, src, d_n_in,
                   ctx->max_raw_keys, ds, ctx->d_hist);
        VOR_LAUNCH(radix_scatter_kernel, kSortBlocks, kSortThreads, 0, stream, src, dst, d_n_in,
                   ctx->max_raw_keys, ds, ctx->d_hist);
        uint64_t* t = src; src = dst; dst = t;
    }
    VOR_LAUNCH(unique_count_kernel, kSortBlocks, kSortThreads, 0, stream, src, d_n_in,
               ctx->max_raw_keys, ctx->d_blk_count);
    VOR_LAUNCH(unique_write_kernel, kSortBlocks, kSortThreads, 0, stream, src, d_n_in,
               ctx->max_raw_keys, ctx->d_blk_count, d_out, cap, d_n_out, ctx->d_flags, flag_bit);
    return VOR_OK;
}

extern "C" int vor_edges(vor_ctx* ctx, const int32_t* d_labels, uint64_t* d_edges, int64_t cap,
                         int64_t* d_n_edges, void* stream_) {
    if (!ctx) return VOR_EINVAL;
    if (!d_labels || !d_edges || !d_n_edges || cap < 0)
        return vor_fail(ctx, VOR_EINVAL, "vor_edges: null pointer or negative capacity");
    cudaStream_t stream = (cudaStream_t)stream_;
    VOR_CUDA(cudaMemsetAsync(ctx->d_n_raw, 0, sizeof(int64_t), stream));
    const int32_t L = ctx->L;
    dim3 grid((L + kEmitCols - 1) / kEmitCols, (L + kEmitRows - 1) / kEmitRows);
    const bool vec = (L % 4 == 0) && (((uintptr_t)d_labels & 15) == 0);
    if (vec)
        VOR_LAUNCH(edges_emit_kernel<true>, grid, kEmitThreads, 0, stream, d_labels, L, ctx->d_keys_a,
                   ctx->max_raw_keys, (unsigned long long*)ctx->d_n_raw, ctx->d_flags);
    else
        VOR_LAUNCH(edges_emit_kernel<false>, grid, kEmitThreads, 0, stream, d_labels, L, ctx->d_keys_a,
                   ctx->max_raw_keys, (unsigned long long*)ctx->d_n_raw, ctx->d_flags);
    return vor_sort_unique_keys(ctx, ctx->d_keys_a, ctx->d_n_raw, vor_label_bits(ctx), d_edges, cap,
                                d_n_edges, FLAG_EDGE_CAP, stream);
}
