// a1 — counting-sort cell list of the sites (BASELINE.json north_star; the paper itself loops over
// all centres).  Buckets are squares of width w fixed-point units, nbx x nby of them with
// w * nbx == Px and w * nby == Py exactly, so that bucket arithmetic wraps consistently on the torus.
//
// Layout: d_bucket_start[nbx*nby + 1] (exclusive prefix), d_sorted[n] = int4(x, y, original index,
// bucket) in bucket order.  Order inside a bucket is arbitrary (atomic cursors); the label kernel
// never depends on it because ties are resolved by the original index explicitly.
#include <math.h>

#include "common.cuh"

namespace {

constexpr int kScanThreads = 1024;
constexpr int kScanItems = 4;
constexpr int kScanTile = kScanThreads * kScanItems;

// n_dev (optional): the number of sites as a device scalar, clamped to n (the grid covers n threads)
__global__ void count_sites_kernel(const int32_t* __restrict__ sx, const int32_t* __restrict__ sy,
                                   int32_t n, const int32_t* __restrict__ n_dev, int32_t w, int32_t nb,
                                   int32_t* __restrict__ fill) {
    int32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (n_dev) n = min(n, *n_dev);
    if (i >= n) return;
    int32_t b = (sy[i] / w) * nb + (sx[i] / w);
    atomicAdd(&fill[b], 1);
}

__device__ __forceinline__ int32_t block_exclusive_scan(int32_t v, int32_t* total) {
    __shared__ int32_t warp_sums[32];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    int32_t inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        int32_t t = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += t;
    }
    if (lane == 31) warp_sums[wid] = inc;
    __syncthreads();
    if (wid == 0) {
        int32_t s = warp_sums[lane];
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            int32_t t = __shfl_up_sync(0xffffffffu, s, o);
            if (lane >= o) s += t;
        }
        warp_sums[lane] = s;
    }
    __syncthreads();
    int32_t base = wid ? warp_sums[wid - 1] : 0;
    *total = warp_sums[31];
    __syncthreads();
    return base + inc - v;
}

// phase 1: per-tile sums
__global__ void __launch_bounds__(kScanThreads) scan_reduce_kernel(const int32_t* __restrict__ in,
                                                                    int64_t n,
                                                                    int32_t* __restrict__ part) {
    int64_t base = (int64_t)blockIdx.x * kScanTile + (int64_t)threadIdx.x * kScanItems;
    int32_t s = 0;
#pragma unroll
    for (int k = 0; k < kScanItems; ++k)
        if (base + k < n) s += in[base + k];
    int32_t total;
    block_exclusive_scan(s, &total);
    if (threadIdx.x == 0) part[blockIdx.x] = total;
}

// phase 2: exclusive scan of the tile sums (single block, <= 8192 tiles)
__global__ void __launch_bounds__(kScanThreads) scan_partials_kernel(int32_t* __restrict__ part,
                                                                      int32_t nparts) {
    int32_t carry = 0;
    for (int32_t base = 0; base < nparts; base += kScanThreads) {
        int32_t i = base + threadIdx.x;
        int32_t v = i < nparts ? part[i] : 0;
        int32_t total;
        int32_t ex = block_exclusive_scan(v, &total);
        if (i < nparts) part[i] = carry + ex;
        carry += total;
    }
}

// phase 3: in-tile exclusive scan + tile offset; also writes out[n] = grand total and clears `in`
__global__ void __launch_bounds__(kScanThreads) scan_apply_kernel(int32_t* __restrict__ in, int64_t n,
                                                                   const int32_t* __restrict__ part,
                                                                   int32_t* __restrict__ out) {
    int64_t base = (int64_t)blockIdx.x * kScanTile + (int64_t)threadIdx.x * kScanItems;
    int32_t v[kScanItems];
    int32_t s = 0;
#pragma unroll
    for (int k = 0; k < kScanItems; ++k) {
        v[k] = base + k < n ? in[base + k] : 0;
        s += v[k];
    }
    int32_t total;
    int32_t ex = block_exclusive_scan(s, &total) + part[blockIdx.x];
#pragma unroll
    for (int k = 0; k < kScanItems; ++k) {
        if (base + k < n) {
            out[base + k] = ex;
            in[base + k] = 0;
        }
        ex += v[k];
        if (base + k == n - 1) out[n] = ex;
    }
}

__global__ void scatter_sites_kernel(const int32_t* __restrict__ sx, const int32_t* __restrict__ sy,
                                     int32_t n, const int32_t* __restrict__ n_dev, int32_t w, int32_t nb,
                                     const int32_t* __restrict__ start, int32_t* __restrict__ fill,
                                     int4* __restrict__ sorted) {
    int32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (n_dev) n = min(n, *n_dev);
    if (i >= n) return;
    int32_t x = sx[i], y = sy[i];
    int32_t b = (y / w) * nb + (x / w);
    int32_t pos = start[b] + atomicAdd(&fill[b], 1);
    sorted[pos] = make_int4(x, y, i, b);
}

}  // namespace

// n_sites: number of sites, or their upper bound when d_n_dev (device scalar) holds the exact number;
// n_hint sizes the buckets (about one site per bucket)
static int build_cells(vor_ctx* ctx, const int32_t* d_sx, const int32_t* d_sy, int32_t n_sites,
                       const int32_t* d_n_dev, int32_t n_hint, cudaStream_t stream) {
    // bucket width w: the common divisor of Px and Py nearest (in ratio) to the width at which a bucket of
    // the DOMAIN holds `occupancy` sites on average; at least 2 cells, at most 4096 buckets per axis
    const double target = FP_ONE * sqrt((double)ctx->Lx * ctx->Ly * (double)ctx->bucket_occ_x100 / (100.0 * (double)n_hint));
    const int64_t g = ctx->w_gcd;
    int64_t best = 0;
    auto consider = [&](int64_t w) {
        if (w < ctx->w_min) return;
        const double r = w > target ? w / target : target / w;
        if (best == 0) { best = w; return; }
        const double rb = best > target ? best / target : target / best;
        if (r < rb || (r == rb && w < best)) best = w;
    };
    for (int64_t d = 1; d * d <= g; ++d) {
        if (g % d) continue;
        consider(d);
        consider(g / d);
    }
    if (best == 0) best = g;
    ctx->w = (int32_t)best;
    ctx->nbx = (int32_t)(ctx->Px / best);
    ctx->nby = (int32_t)(ctx->Py / best);
    ctx->n_sites = n_sites;
    ctx->n_hint = n_hint;
    ctx->d_n_dev = d_n_dev;
    const int64_t nbuckets = (int64_t)ctx->nbx * ctx->nby;

    VOR_CUDA(cudaMemsetAsync(ctx->d_bucket_fill, 0, nbuckets * sizeof(int32_t), stream));
    const int threads = 256;
    const int grid = (n_sites + threads - 1) / threads;
    VOR_LAUNCH(count_sites_kernel, grid, threads, 0, stream, d_sx, d_sy, n_sites, d_n_dev, ctx->w, ctx->nbx,
               ctx->d_bucket_fill);
    const int tiles = (int)((nbuckets + kScanTile - 1) / kScanTile);
    VOR_LAUNCH(scan_reduce_kernel, tiles, kScanThreads, 0, stream, ctx->d_bucket_fill, nbuckets,
               ctx->d_scan_part);
    VOR_LAUNCH(scan_partials_kernel, 1, kScanThreads, 0, stream, ctx->d_scan_part, tiles);
    VOR_LAUNCH(scan_apply_kernel, tiles, kScanThreads, 0, stream, ctx->d_bucket_fill, nbuckets,
               ctx->d_scan_part, ctx->d_bucket_start);
    VOR_LAUNCH(scatter_sites_kernel, grid, threads, 0, stream, d_sx, d_sy, n_sites, d_n_dev, ctx->w, ctx->nbx,
               ctx->d_bucket_start, ctx->d_bucket_fill, ctx->d_sorted);
    return VOR_OK;
}

extern "C" int vor_build_cells(vor_ctx* ctx, const int32_t* d_sx, const int32_t* d_sy,
                               int32_t n_sites, void* stream_) {
    if (!ctx) return VOR_EINVAL;
    if (int drc_ = vor_check_device(ctx)) return drc_;
    if (!d_sx || !d_sy) return vor_fail(ctx, VOR_EINVAL, "vor_build_cells: null site array");
    if (n_sites < 1 || n_sites > ctx->max_sites)
        return vor_fail(ctx, VOR_EINVAL, "vor_build_cells: n_sites out of range [1, max_sites]");
    return build_cells(ctx, d_sx, d_sy, n_sites, nullptr, n_sites, (cudaStream_t)stream_);
}

extern "C" int vor_build_cells_dev(vor_ctx* ctx, const int32_t* d_sx, const int32_t* d_sy,
                                   const int32_t* d_n_sites, int32_t cap, int32_t n_hint, void* stream_) {
    if (!ctx) return VOR_EINVAL;
    if (int drc_ = vor_check_device(ctx)) return drc_;
    if (!d_sx || !d_sy || !d_n_sites) return vor_fail(ctx, VOR_EINVAL, "vor_build_cells_dev: null pointer");
    if (cap < 1 || cap > ctx->max_sites)
        return vor_fail(ctx, VOR_EINVAL, "vor_build_cells_dev: cap out of range [1, max_sites]");
    if (n_hint < 1 || n_hint > cap) n_hint = cap;
    return build_cells(ctx, d_sx, d_sy, cap, d_n_sites, n_hint, (cudaStream_t)stream_);
}
