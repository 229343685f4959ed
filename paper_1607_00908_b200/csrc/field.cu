// a6..a8 — the field-derived front end: bubbles from a thresholded scalar field.
//  a6 field_threshold_ccl  PAPER.md:95 (§III.A): threshold -> two-valued variable -> cluster labelling
//                          (the paper adapts the label-equivalence method of its ref. [6]); here a
//                          lock-free union-find whose roots are the minimum linear index, run first
//                          per 64 x 32 tile in shared memory, then over the tile seams in HBM.
//  a7 field_centroids      PAPER.md:95-101: bubble size by atomic counting, centre of mass = sum of
//                          the lattice coordinates / size.  Integer sums (order independent), periodic
//                          unwrap relative to the root cell, one float64 divide.
//  a8 match_sites          PAPER.md:213, 223: isomorphism P->N from the two sets of centres; mutual
//                          nearest neighbour within a radius; unmatched = appeared / disappeared.
#include "common.cuh"

namespace {

// ------------------------------------------------------------------------------------ a6: CCL
__device__ __forceinline__ int32_t uf_find(const int32_t* parent, int32_t a) {
    int32_t p = parent[a];
    while (p != a) { a = p; p = parent[a]; }
    return a;
}

// roots are always the smallest index of their tree: link the larger root under the smaller one
__device__ __forceinline__ void uf_union(int32_t* parent, int32_t a, int32_t b) {
    for (;;) {
        a = uf_find(parent, a);
        b = uf_find(parent, b);
        if (a == b) return;
        if (a < b) { const int32_t t = a; a = b; b = t; }      // a > b
        const int32_t old = atomicMin(&parent[a], b);
        if (old == a) return;
        a = old;                                                // someone re-rooted a meanwhile
    }
}

// Tile stage: one CTA thresholds a kTileW x kTileH tile into shared memory, runs the same union-find
// on the tile's own right / down pairs there (roots = smallest local index = smallest global index of
// the tile-component, because local row-major order follows the global one), flattens, and writes
// parent[cell] = global index of its tile root.  HBM: 4 B/cell read, 4 B/cell written.
constexpr int kTileW = 64, kTileH = 32, kTileThreads = 256;
constexpr int kTileRows = kTileW * kTileH / kTileThreads;     // rows per thread (8)

__device__ __forceinline__ int32_t suf_find(const int32_t* parent, int32_t a) {
    int32_t p = parent[a];
    while (p != a) { a = p; p = parent[a]; }
    return a;
}
__device__ __forceinline__ void suf_union(int32_t* parent, int32_t a, int32_t b) {
    for (;;) {
        a = suf_find(parent, a);
        b = suf_find(parent, b);
        if (a == b) return;
        if (a < b) { const int32_t t = a; a = b; b = t; }
        const int32_t old = atomicMin(&parent[a], b);
        if (old == a) return;
        a = old;
    }
}

// conn8: cells that touch at a corner are connected too (the D2Q9 directions)
__global__ void __launch_bounds__(kTileThreads) ccl_tile_kernel(const float* __restrict__ field, float thr,
                                                                int above, int32_t Lx, int32_t Ly, int conn8,
                                                                int32_t* __restrict__ parent) {
    __shared__ int32_t lab[kTileH * kTileW];
    const int32_t X0 = blockIdx.x * kTileW, Y0 = blockIdx.y * kTileH;
    const int lane = threadIdx.x & 31;
    const int lx = threadIdx.x & (kTileW - 1), ly0 = (threadIdx.x / kTileW) * kTileRows;
    const int32_t x = X0 + lx;
    // a warp holds 32 consecutive columns of one row: every cell starts out pointing at the first
    // cell of its horizontal run inside those 32 columns, so no union is needed along rows
#pragma unroll
    for (int j = 0; j < kTileRows; ++j) {
        const int32_t y = Y0 + ly0 + j;
        bool m = false;
        if (x < Lx && y < Ly) {
            const float v = __ldcs(field + (int64_t)y * Lx + x);
            m = above ? (v > thr) : (v < thr);             // NaN compares false both ways
        }
        const unsigned bits = __ballot_sync(0xffffffffu, m);
        const int run = __clz((int)~(bits << (31 - lane)));   // set cells ending at this lane (>= 1 if m)
        const int li = (ly0 + j) * kTileW + lx;
        lab[li] = m ? li - run + 1 : -1;
    }
    __syncthreads();
    // unions: the two 32-column halves of a row, and vertically adjacent runs (once per overlap: at
    // the overlap's leftmost column the cell to the left is unset in one of the two rows)
#pragma unroll
    for (int j = 0; j < kTileRows; ++j) {
        const int li = (ly0 + j) * kTileW + lx;
        if (lab[li] < 0) continue;
        if (lx == 32 && lab[li - 1] >= 0) suf_union(lab, li, li - 1);
        if (ly0 + j + 1 < kTileH) {
            if (lab[li + kTileW] >= 0) {
                if (lx == 0 || lab[li - 1] < 0 || lab[li + kTileW - 1] < 0) suf_union(lab, li, li + kTileW);
            } else if (conn8) {
                // the cell below is background: a diagonal neighbour is reachable only through the corner
                // (were the cell below set, it would join both through its own row)
                if (lx + 1 < kTileW && lab[li + kTileW + 1] >= 0) suf_union(lab, li, li + kTileW + 1);
                if (lx > 0 && lab[li + kTileW - 1] >= 0) suf_union(lab, li, li + kTileW - 1);
            }
        }
    }
    __syncthreads();
#pragma unroll
    for (int j = 0; j < kTileRows; ++j) {
        const int32_t y = Y0 + ly0 + j;
        if (x >= Lx || y >= Ly) continue;
        const int li = (ly0 + j) * kTileW + lx;
        int32_t out = -1;
        if (lab[li] >= 0) {
            const int32_t r = suf_find(lab, li);
            out = (int32_t)((int64_t)(Y0 + r / kTileW) * Lx + X0 + (r & (kTileW - 1)));
        }
        parent[(int64_t)y * Lx + x] = out;
    }
}

// Seam stage: the pairs that straddle tile borders (including the periodic wrap and the ragged last
// tiles) are united in the global array.  Items [0, ntx * Ly): vertical seam lines (cell | right
// neighbour, with conn8 also its upper and lower right neighbour); items [ntx * Ly, ntx * Ly + nty * Lx):
// horizontal seam lines (cell | lower neighbour, with conn8 also lower left and lower right).  A neighbour
// beyond a walled axis does not exist.
__global__ void ccl_seam_kernel(int32_t Lx, int32_t Ly, int per_x, int per_y, int conn8, int32_t ntx, int32_t nty,
                                int32_t* __restrict__ parent) {
    const int64_t nv = (int64_t)ntx * Ly, n = nv + (int64_t)nty * Lx;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        int32_t x, y, dx0, dy0;                          // the cell and the direction of its plain neighbour
        if (i < nv) {
            y = (int32_t)(i % Ly);
            x = min((int32_t)(i / Ly + 1) * kTileW - 1, Lx - 1);
            dx0 = 1; dy0 = 0;
        } else {
            const int64_t r = i - nv;
            x = (int32_t)(r % Lx);
            y = min((int32_t)(r / Lx + 1) * kTileH - 1, Ly - 1);
            dx0 = 0; dy0 = 1;
        }
        const int64_t a = (int64_t)y * Lx + x;
        if (parent[a] < 0) continue;
        for (int t = -1; t <= 1; ++t) {
            if (t != 0 && !conn8) continue;
            int32_t u = x + (dx0 ? 1 : t), v = y + (dy0 ? 1 : t);
            if (u < 0 || u >= Lx) { if (!per_x) continue; u = u < 0 ? u + Lx : u - Lx; }
            if (v < 0 || v >= Ly) { if (!per_y) continue; v = v < 0 ? v + Ly : v - Ly; }
            const int64_t b = (int64_t)v * Lx + u;
            if (a != b && parent[b] >= 0) uf_union(parent, (int32_t)a, (int32_t)b);
        }
    }
}

__global__ void ccl_flatten_kernel(int64_t n, int32_t* __restrict__ parent) {
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        const int32_t q = parent[i];
        if (q < 0) continue;
        const int32_t r = uf_find(parent, q);
        if (r != q) parent[i] = r;                          // most cells already point at their root
    }
}

// ------------------------------------------------------------------------------------ compaction
// Order-preserving compaction of the items i in [0, n) that satisfy pred(i).  Every WARP owns one contiguous
// range of whole 256-item tiles; consecutive ranges go to different blocks, so that short lists spread over
// the SMs.  The count kernel leaves one count per warp; the write kernel derives every warp's offset from
// those (row sums over the blocks, in the block's prologue) and then each warp streams its range with
// ballots only - no barrier inside the loop.
constexpr int kCompThreads = 512;
constexpr int kCompWarps = kCompThreads / 32;
constexpr int kCompItems = 8;                      // items per lane per tile (warp-strided: coalesced)
constexpr int kCompTile = 32 * kCompItems;
constexpr int kCompGrid = 4 * kNumSMs;             // kCompWarps * kCompGrid warp counts in ctx->d_comp_wcount

// range of warp W = wid * gridDim.x + blockIdx.x among gridDim.x * kCompWarps warps
__device__ __forceinline__ void comp_range(int64_t n, int64_t* beg, int64_t* end) {
    const int64_t nw = (int64_t)gridDim.x * kCompWarps, W = (int64_t)(threadIdx.x >> 5) * gridDim.x + blockIdx.x;
    int64_t C = (n + nw - 1) / nw;
    C = (C + kCompTile - 1) / kCompTile * kCompTile;
    const int64_t s = W * C;
    *beg = s < n ? s : n;
    *end = s + C < n ? s + C : n;
}

template <typename Pred>
__global__ void __launch_bounds__(kCompThreads) comp_count_kernel(Pred pred, int32_t* __restrict__ wcount) {
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    int64_t beg, end;
    comp_range(pred.size(), &beg, &end);
    int32_t c = 0;
    for (int64_t i = beg + lane; i < end; i += 32) c += pred(i);
    c = __reduce_add_sync(0xffffffffu, c);
    if (lane == 0) wcount[wid * gridDim.x + blockIdx.x] = c;
}

template <typename Pred, typename Sink>
__global__ void __launch_bounds__(kCompThreads) comp_write_kernel(Pred pred, Sink sink,
                                                                  const int32_t* __restrict__ wcount) {
    __shared__ int64_t rowsum[kCompWarps];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int G = gridDim.x;
    // warp `wid` sums row `wid` of the counts: all of it, and the part that belongs to earlier blocks
    int64_t rs = 0, rp = 0;
    for (int b = lane; b < G; b += 32) {
        const int64_t v = wcount[wid * G + b];
        rs += v;
        if (b < (int)blockIdx.x) rp += v;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) { rs += __shfl_xor_sync(0xffffffffu, rs, o); rp += __shfl_xor_sync(0xffffffffu, rp, o); }
    if (lane == 0) rowsum[wid] = rs;
    __syncthreads();
    int64_t run = rp, all = 0;
#pragma unroll
    for (int w = 0; w < kCompWarps; ++w) {
        const int64_t t = rowsum[w];
        all += t;
        if (w < wid) run += t;
    }
    if (blockIdx.x == 0 && threadIdx.x == 0) sink.total(all);
    int64_t beg, end;
    comp_range(pred.size(), &beg, &end);
    for (int64_t sub = beg; sub < end; sub += kCompTile) {
        unsigned ball[kCompItems];
#pragma unroll
        for (int k = 0; k < kCompItems; ++k) {
            const int64_t i = sub + 32 * k + lane;
            ball[k] = __ballot_sync(0xffffffffu, i < end && pred(i));
        }
#pragma unroll
        for (int k = 0; k < kCompItems; ++k) {
            if (ball[k] >> lane & 1u) sink.put(run + __popc(ball[k] & ((1u << lane) - 1u)), sub + 32 * k + lane);
            run += __popc(ball[k]);
        }
    }
}

// ------------------------------------------------------------------------------------ a7: centroids
// floor(x / d) for 0 <= x < 2^32 with one multiply-high and two shifts (Granlund-Montgomery); the
// accumulation splits two linear indices per cell into (x, y).
struct FastDiv {
    uint32_t m, s1, s2, d;
    __device__ __forceinline__ uint32_t div(uint32_t x) const {
        const uint32_t t = __umulhi(m, x);
        return (t + ((x - t) >> s1)) >> s2;
    }
};
inline FastDiv make_fastdiv(uint32_t d) {
    uint32_t l = 0;
    while (((uint64_t)1 << l) < d) ++l;
    FastDiv f;
    f.m = (uint32_t)((((uint64_t)1 << 32) * (((uint64_t)1 << l) - d)) / d + 1);
    f.s1 = l < 1 ? l : 1;
    f.s2 = l > 0 ? l - 1 : 0;
    f.d = d;
    return f;
}

struct RootPred {
    const int32_t* ccl;
    int64_t n;
    __device__ int64_t size() const { return n; }
    __device__ bool operator()(int64_t i) const { return ccl[i] == (int32_t)i; }
};
struct RootSink {
    int32_t* comp_root;
    int32_t* rank;
    int32_t max_comp;
    int32_t* n_raw;
    int32_t* flags;
    long long* acc;            // accumulators of the components found are zeroed here (no full memset)
    int n_acc;
    __device__ void total(int64_t t) const {
        *n_raw = (int32_t)(t < max_comp ? t : max_comp);
        if (t > max_comp) atomicOr(flags, FLAG_COMP_CAP);
    }
    __device__ void put(int64_t pos, int64_t i) const {
        rank[i] = pos < max_comp ? (int32_t)pos : -1;
        if (pos < max_comp) {
            comp_root[pos] = (int32_t)i;
            for (int a = 0; a < n_acc; ++a) acc[(size_t)a * max_comp + pos] = 0;
        }
    }
};

// fixed-point density of a cell (the centre of mass weighted by rho): floor(rho * 65536)
// limited to [1, 2^24]; NaN -> 1.  Integer weights keep the sums independent of the accumulation order.
__device__ __forceinline__ int64_t cell_weight(float rho) {
    const float s = rho * 65536.0f;                             // exact: a power-of-two scale
    return s >= 16777216.0f ? 16777216 : (s >= 1.0f ? (int64_t)s : 1);
}

// acc: [0] cells, [1] sum of w dx, [2] sum of w dy, [3] sum of w (weighted only), each max_comp entries.
// A thread takes kAccCells consecutive cells of one row (Lx % kAccCells == 0: one 16-byte load), merges the ones
// that carry its first bubble label (inside a bubble and on its edge that is all of them), and the warp merges
// the threads that hold the same label (`match_any`; skipped when the whole warp agrees) before ONE lane adds
// to the component's accumulators.  Cells of a second bubble inside the same four (rare) add their own terms.
constexpr int kAccCells = 4;

template <bool kWeighted>
__device__ __forceinline__ void acc_add(unsigned long long* __restrict__ acc, int32_t max_comp, int32_t k,
                                        int64_t n, int64_t sx, int64_t sy, int64_t sw) {
    atomicAdd(&acc[k], (unsigned long long)n);
    atomicAdd(&acc[(size_t)max_comp + k], (unsigned long long)sx);
    atomicAdd(&acc[2 * (size_t)max_comp + k], (unsigned long long)sy);
    if constexpr (kWeighted) atomicAdd(&acc[3 * (size_t)max_comp + k], (unsigned long long)sw);
}

template <bool kWeighted, int kCells>
__global__ void __launch_bounds__(256) accumulate_kernel(const int32_t* __restrict__ ccl, const float* __restrict__ field,
                                                         const int32_t* __restrict__ rank, int32_t Lx, int32_t Ly,
                                                         int per_x, int per_y, FastDiv fd,
                                                         unsigned long long* __restrict__ acc, int32_t max_comp) {
    const unsigned full = 0xffffffffu;
    const int64_t n = (int64_t)Lx * Ly, groups = n / kCells;           // kCells divides Lx
    const int64_t ground = (groups + 31) / 32 * 32;                    // keep warps converged for the collectives
    for (int64_t g = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; g < ground; g += (int64_t)gridDim.x * blockDim.x) {
        int32_t r[kCells];
        float rho[kCells];
        if (g < groups) {
            if constexpr (kCells == 4) {
                const int4 v = __ldcs(reinterpret_cast<const int4*>(ccl) + g);
                r[0] = v.x; r[1] = v.y; r[2] = v.z; r[3] = v.w;
                if constexpr (kWeighted) {
                    const float4 f = __ldcs(reinterpret_cast<const float4*>(field) + g);
                    rho[0] = f.x; rho[1] = f.y; rho[2] = f.z; rho[3] = f.w;
                }
            } else {
                r[0] = ccl[g];
                if constexpr (kWeighted) rho[0] = field[g];
            }
        } else {
#pragma unroll
            for (int c = 0; c < kCells; ++c) r[c] = -1;
        }
        // the thread's label: the first bubble label among its cells
        int32_t key = -1;
#pragma unroll
        for (int c = kCells - 1; c >= 0; --c) key = r[c] >= 0 ? r[c] : key;
        const bool uniform = __all_sync(full, key == __shfl_sync(full, key, 0));
        const unsigned peers = uniform ? full : __match_any_sync(full, key);
        if (key < 0) continue;                                  // whole peer group leaves together
        const uint32_t i0 = (uint32_t)(g * kCells);
        const int32_t y = (int32_t)fd.div(i0), x0 = (int32_t)(i0 - (uint32_t)y * (uint32_t)Lx);
        const int32_t yr = (int32_t)fd.div((uint32_t)key), xr = key - yr * Lx;
        int32_t dy = y - yr;
        if (per_y) { if (2 * dy >= Ly) dy -= Ly; else if (2 * dy < -Ly) dy += Ly; }
        int64_t tn = 0, tsx = 0, tsy = 0, tsw = 0;
#pragma unroll
        for (int c = 0; c < kCells; ++c) {
            if (r[c] < 0) continue;
            int64_t w = 1;
            if constexpr (kWeighted) w = cell_weight(rho[c]);
            if (r[c] == key) {
                int32_t dx = x0 + c - xr;
                if (per_x) { if (2 * dx >= Lx) dx -= Lx; else if (2 * dx < -Lx) dx += Lx; }
                tn += 1; tsx += w * dx; tsy += w * dy; tsw += w;
            } else {                                            // a second bubble within the same cells
                const int32_t k2 = rank[r[c]];
                if (k2 >= 0) {
                    const int32_t yr2 = (int32_t)fd.div((uint32_t)r[c]), xr2 = r[c] - yr2 * Lx;
                    int32_t dx = x0 + c - xr2, dy2 = y - yr2;
                    if (per_x) { if (2 * dx >= Lx) dx -= Lx; else if (2 * dx < -Lx) dx += Lx; }
                    if (per_y) { if (2 * dy2 >= Ly) dy2 -= Ly; else if (2 * dy2 < -Ly) dy2 += Ly; }
                    acc_add<kWeighted>(acc, max_comp, k2, 1, w * dx, w * dy2, w);
                }
            }
        }
        // sums over the peer group; 32-bit reductions when nothing can overflow (no weights: |dx| < 2^22, 128 cells)
        if constexpr (!kWeighted) {
            const int32_t pn = __reduce_add_sync(peers, (int32_t)tn);
            const int32_t px = __reduce_add_sync(peers, (int32_t)tsx);
            const int32_t py = __reduce_add_sync(peers, (int32_t)tsy);
            if ((int)(__ffs(peers) - 1) == (int)(threadIdx.x & 31)) {
                const int32_t k = rank[key];
                if (k >= 0) acc_add<false>(acc, max_comp, k, pn, px, py, 0);
            }
        } else {
            if (uniform) {
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) {
                    tn += __shfl_xor_sync(full, tn, o);
                    tsx += __shfl_xor_sync(full, tsx, o);
                    tsy += __shfl_xor_sync(full, tsy, o);
                    tsw += __shfl_xor_sync(full, tsw, o);
                }
                if ((threadIdx.x & 31) == 0) {
                    const int32_t k = rank[key];
                    if (k >= 0) acc_add<true>(acc, max_comp, k, tn, tsx, tsy, tsw);
                }
            } else {
                const int32_t k = rank[key];
                if (k >= 0) acc_add<true>(acc, max_comp, k, tn, tsx, tsy, tsw);
            }
        }
    }
}

struct SizePred {
    const long long* acc;
    const int32_t* n_raw;
    int32_t min_size;
    __device__ int64_t size() const { return *n_raw; }
    __device__ bool operator()(int64_t k) const { return acc[k] >= (long long)min_size && acc[k] > 0; }
};
struct CentroidSink {
    const long long* acc;
    const int32_t* comp_root;
    int32_t max_comp, Lx, Ly, cap, weighted;
    double* cx; double* cy; int32_t* sx; int32_t* sy; int32_t* size; int32_t* root;
    int32_t* n_comp; int32_t* flags;
    __device__ void total(int64_t t) const {
        *n_comp = (int32_t)t;
        if (t > cap) atomicOr(flags, FLAG_COMP_CAP);
    }
    // floor(256 S / W), W > 0; 64-bit arithmetic whenever 256 |S| fits (always, without weights)
    __device__ static long long floor_div256(long long S, long long W) {
        if (S > -((long long)1 << 54) && S < ((long long)1 << 54)) {
            const long long a = FP_ONE * S;
            return a >= 0 ? a / W : -((-a + W - 1) / W);
        }
        const __int128 a = (__int128)FP_ONE * S, b = W;
        return (long long)(a >= 0 ? a / b : -((-a + b - 1) / b));
    }
    __device__ void put(int64_t pos, int64_t k) const {
        if (pos >= cap) return;
        const long long m = acc[k], Sx = acc[(size_t)max_comp + k], Sy = acc[2 * (size_t)max_comp + k];
        const long long W = weighted ? acc[3 * (size_t)max_comp + k] : m;     // total weight
        const int32_t r = comp_root[k];
        const long long xr = r % Lx, yr = r / Lx, Px = (long long)FP_ONE * Lx, Py = (long long)FP_ONE * Ly;
        const long long fx = floor_div256(Sx, W), fy = floor_div256(Sy, W);
        sx[pos] = (int32_t)((((FP_ONE * xr + FP_HALF + fx) % Px) + Px) % Px);
        sy[pos] = (int32_t)((((FP_ONE * yr + FP_HALF + fy) % Py) + Py) % Py);
        double ux = __dadd_rn(__dadd_rn((double)xr, 0.5), __ddiv_rn((double)Sx, (double)W));
        double uy = __dadd_rn(__dadd_rn((double)yr, 0.5), __ddiv_rn((double)Sy, (double)W));
        if (ux < 0) ux += Lx; else if (ux >= Lx) ux -= Lx;
        if (uy < 0) uy += Ly; else if (uy >= Ly) uy -= Ly;
        cx[pos] = ux; cy[pos] = uy;
        size[pos] = (int32_t)m;
        root[pos] = r;
    }
};

// ------------------------------------------------------------------------------------ a8: match
// Fast path: both point sets are hashed into a uniform grid of nbm x nbm buckets whose width is at
// least the matching radius, so that every partner within the radius lies in the 3 x 3 buckets around
// the query (with wrap).  A bucket holds kMatchSlots ids; if any bucket overflows a device flag makes
// the brute-force kernel below redo the search (same result by definition), so the outcome never
// depends on the grid.
constexpr int kMatchThreads = 256;

struct MatchGrid {
    int32_t* cnt[2];           // [nbm * nbm] per set (0 = prev, 1 = now)
    int32_t* ids[2];           // [nbm * nbm * kMatchSlots]
    int32_t nbm;
    int32_t* overflow;         // device flag
};

// periods of the two axes in fixed point and whether each axis wraps (a walled axis: plain distance)
struct MatchGeom {
    long long Px, Py;
    int per_x, per_y;
    __device__ __forceinline__ long long d2(long long ax, long long ay, long long vx, long long vy) const {
        long long dx = ax > vx ? ax - vx : vx - ax;
        if (per_x && Px - dx < dx) dx = Px - dx;
        long long dy = ay > vy ? ay - vy : vy - ay;
        if (per_y && Py - dy < dy) dy = Py - dy;
        return dx * dx + dy * dy;
    }
};

__device__ __forceinline__ int32_t mbucket(int32_t v, long long P, int32_t nbm) {
    return (int32_t)(((long long)v * nbm) / P);
}

__global__ void match_fill_kernel(const int32_t* __restrict__ px, const int32_t* __restrict__ py,
                                  const int32_t* __restrict__ n_prev_p, const int32_t* __restrict__ nx,
                                  const int32_t* __restrict__ ny, const int32_t* __restrict__ n_now_p,
                                  int32_t cap_prev, int32_t cap_now, MatchGeom geo, MatchGrid g) {
    const int32_t n_prev = min(*n_prev_p, cap_prev), n_now = min(*n_now_p, cap_now);
    for (int32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < n_prev + n_now; i += gridDim.x * blockDim.x) {
        const int set = i >= n_prev;
        const int32_t k = set ? i - n_prev : i;
        const int32_t x = set ? nx[k] : px[k], y = set ? ny[k] : py[k];
        const int32_t b = mbucket(y, geo.Py, g.nbm) * g.nbm + mbucket(x, geo.Px, g.nbm);
        const int32_t slot = atomicAdd(&g.cnt[set][b], 1);
        if (slot < kMatchSlots) g.ids[set][(size_t)b * kMatchSlots + slot] = k;
        else *g.overflow = 1;
    }
}

// best[q] for every query of both directions: nearest target within the radius (ties: smallest index)
__global__ void match_grid_kernel(const int32_t* __restrict__ px, const int32_t* __restrict__ py,
                                  const int32_t* __restrict__ n_prev_p, const int32_t* __restrict__ nx,
                                  const int32_t* __restrict__ ny, const int32_t* __restrict__ n_now_p,
                                  int32_t cap_prev, int32_t cap_now, MatchGeom geo, long long r2, MatchGrid g,
                                  int32_t* __restrict__ best) {
    const int32_t n_prev = min(*n_prev_p, cap_prev), n_now = min(*n_now_p, cap_now);
    for (int32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < n_prev + n_now; i += gridDim.x * blockDim.x) {
        const bool q_is_now = i >= n_prev;                  // now queries search the prev set
        const int32_t q = q_is_now ? i - n_prev : i;
        const int tset = q_is_now ? 0 : 1;
        const int32_t* __restrict__ tx = q_is_now ? px : nx;
        const int32_t* __restrict__ ty = q_is_now ? py : ny;
        const long long ax = q_is_now ? nx[q] : px[q], ay = q_is_now ? ny[q] : py[q];
        const int32_t bx = mbucket((int32_t)ax, geo.Px, g.nbm), by = mbucket((int32_t)ay, geo.Py, g.nbm);
        long long bd = INT64_MAX;
        int32_t bi = -1;
        const int span = g.nbm >= 3 ? 3 : g.nbm;             // tiny grids: every bucket once
        for (int oy = 0; oy < span; ++oy) {
            int32_t cy = g.nbm >= 3 ? by + oy - 1 : oy;      // beyond a walled axis there is no bucket
            if (cy < 0 || cy >= g.nbm) { if (!geo.per_y) continue; cy = cy < 0 ? cy + g.nbm : cy - g.nbm; }
            for (int ox = 0; ox < span; ++ox) {
                int32_t cx = g.nbm >= 3 ? bx + ox - 1 : ox;
                if (cx < 0 || cx >= g.nbm) { if (!geo.per_x) continue; cx = cx < 0 ? cx + g.nbm : cx - g.nbm; }
                const int32_t b = cy * g.nbm + cx;
                const int32_t c = min(g.cnt[tset][b], kMatchSlots);
                for (int32_t s = 0; s < c; ++s) {
                    const int32_t t = g.ids[tset][(size_t)b * kMatchSlots + s];
                    const long long d2 = geo.d2(ax, ay, tx[t], ty[t]);
                    if (d2 < bd || (d2 == bd && t < bi)) { bd = d2; bi = t; }
                }
            }
        }
        best[(q_is_now ? cap_prev : 0) + q] = (bi >= 0 && bd <= r2) ? bi : -1;
    }
}

// blocks [0, gq) : queries = now, targets = prev -> best[cap_prev + j];  blocks [gq, ..): the reverse
__global__ void __launch_bounds__(kMatchThreads) match_best_kernel(
        const int32_t* __restrict__ px, const int32_t* __restrict__ py, const int32_t* __restrict__ n_prev_p,
        const int32_t* __restrict__ nx, const int32_t* __restrict__ ny, const int32_t* __restrict__ n_now_p,
        int32_t cap_prev, int32_t cap_now, int32_t blocks_now, MatchGeom geo, long long r2,
        int32_t* __restrict__ best, int32_t* __restrict__ flags, const int32_t* __restrict__ needed) {
    __shared__ int32_t tx[kMatchThreads], ty[kMatchThreads];
    if (blockIdx.x == 0 && threadIdx.x == 0 && (*n_prev_p > cap_prev || *n_now_p > cap_now))
        atomicOr(flags, FLAG_MATCH_CAP);
    if (needed && *needed == 0) return;                   // the grid path answered every query
    const bool q_is_now = (int)blockIdx.x < blocks_now;
    const int32_t n_prev = min(*n_prev_p, cap_prev), n_now = min(*n_now_p, cap_now);
    const int32_t* qx = q_is_now ? nx : px; const int32_t* qy = q_is_now ? ny : py;
    const int32_t* sx = q_is_now ? px : nx; const int32_t* sy = q_is_now ? py : ny;
    const int32_t nq = q_is_now ? n_now : n_prev, nt = q_is_now ? n_prev : n_now;
    const int32_t q = (q_is_now ? blockIdx.x : blockIdx.x - blocks_now) * kMatchThreads + threadIdx.x;
    if ((q_is_now ? blockIdx.x : blockIdx.x - blocks_now) * kMatchThreads >= nq) return;
    const long long ax = q < nq ? qx[q] : 0, ay = q < nq ? qy[q] : 0;
    long long bd = INT64_MAX;
    int32_t bi = -1;
    for (int32_t base = 0; base < nt; base += kMatchThreads) {
        const int32_t t = base + threadIdx.x;
        __syncthreads();
        tx[threadIdx.x] = t < nt ? sx[t] : 0;
        ty[threadIdx.x] = t < nt ? sy[t] : 0;
        __syncthreads();
        const int32_t lim = min(kMatchThreads, nt - base);
        for (int32_t k = 0; k < lim; ++k) {
            const long long d2 = geo.d2(ax, ay, tx[k], ty[k]);
            if (d2 < bd) { bd = d2; bi = base + k; }
        }
    }
    if (q < nq) best[(q_is_now ? cap_prev : 0) + q] = (bi >= 0 && bd <= r2) ? bi : -1;
}

__global__ void match_combine_kernel(const int32_t* __restrict__ n_prev_p, const int32_t* __restrict__ n_now_p,
                                     int32_t cap_prev, int32_t cap_now, const int32_t* __restrict__ best,
                                     int32_t* __restrict__ p2n, int32_t* __restrict__ n2p) {
    const int32_t n_prev = min(*n_prev_p, cap_prev), n_now = min(*n_now_p, cap_now);
    const int32_t* bn = best;                 // best now for each prev
    const int32_t* bp = best + cap_prev;      // best prev for each now
    for (int32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < cap_prev + cap_now; i += gridDim.x * blockDim.x) {
        if (i < cap_prev) {
            int32_t v = -1;
            if (i < n_prev) { const int32_t j = bn[i]; if (j >= 0 && bp[j] == i) v = j; }
            p2n[i] = v;
        } else {
            const int32_t j = i - cap_prev;
            int32_t v = -1;
            if (j < n_now) { const int32_t k = bp[j]; if (k >= 0 && bn[k] == j) v = k; }
            n2p[j] = v;
        }
    }
}



// ------------------------------------------------------------------------------------ size histogram
__global__ void size_hist_kernel(const int32_t* __restrict__ size, const int32_t* __restrict__ n_comp, int32_t cap,
                                 int32_t bin_width, int32_t n_bins, unsigned long long* __restrict__ hist) {
    const int32_t n = min(*n_comp, cap);
    for (int32_t k = blockIdx.x * blockDim.x + threadIdx.x; k < n; k += gridDim.x * blockDim.x) {
        const int32_t s = size[k];
        if (s < 0) continue;
        const int32_t b = min(s / bin_width, n_bins - 1);
        atomicAdd(&hist[b], 1ull);
    }
}

}  // namespace

extern "C" int field_threshold_ccl(vor_ctx* ctx, const float* d_field, float thr, int above,
                                   int32_t* d_ccl, void* stream_) {
    return field_threshold_ccl_conn(ctx, d_field, thr, above, 4, d_ccl, stream_);
}

extern "C" int field_threshold_ccl_conn(vor_ctx* ctx, const float* d_field, float thr, int above,
                                        int32_t connectivity, int32_t* d_ccl, void* stream_) {
    if (!ctx) return VOR_EINVAL;
    if (int drc_ = vor_check_device(ctx)) return drc_;
    if (!d_field || !d_ccl) return vor_fail(ctx, VOR_EINVAL, "field_threshold_ccl: null pointer");
    if (connectivity != 4 && connectivity != 8)
        return vor_fail(ctx, VOR_EINVAL, "field_threshold_ccl: connectivity must be 4 or 8");
    const int64_t n = (int64_t)ctx->Lx * ctx->Ly;
    if (n > INT32_MAX) return vor_fail(ctx, VOR_EINVAL, "field_threshold_ccl: Lx * Ly must fit a 32-bit cell index");
    cudaStream_t stream = (cudaStream_t)stream_;
    const int conn8 = connectivity == 8;
    const int grid = (int)((n + 255) / 256 < 8 * kNumSMs ? (n + 255) / 256 : 8 * kNumSMs);
    const int32_t ntx = (ctx->Lx + kTileW - 1) / kTileW, nty = (ctx->Ly + kTileH - 1) / kTileH;
    VOR_LAUNCH(ccl_tile_kernel, dim3(ntx, nty), kTileThreads, 0, stream, d_field, thr, above ? 1 : 0, ctx->Lx, ctx->Ly,
               conn8, d_ccl);
    const int64_t seams = (int64_t)ntx * ctx->Ly + (int64_t)nty * ctx->Lx;
    const int sgrid = (int)((seams + 255) / 256 < 8 * kNumSMs ? (seams + 255) / 256 : 8 * kNumSMs);
    VOR_LAUNCH(ccl_seam_kernel, sgrid, 256, 0, stream, ctx->Lx, ctx->Ly, ctx->per_x, ctx->per_y, conn8, ntx, nty, d_ccl);
    VOR_LAUNCH(ccl_flatten_kernel, grid, 256, 0, stream, n, d_ccl);
    return VOR_OK;
}

extern "C" int field_centroids(vor_ctx* ctx, const int32_t* d_ccl, int32_t min_size,
                               double* d_cx, double* d_cy, int32_t* d_sx, int32_t* d_sy,
                               int32_t* d_size, int32_t* d_root, int32_t cap, int32_t* d_n_comp,
                               void* stream_) {
    return field_centroids_weighted(ctx, d_ccl, nullptr, min_size, d_cx, d_cy, d_sx, d_sy, d_size, d_root, cap,
                                    d_n_comp, stream_);
}

extern "C" int field_centroids_weighted(vor_ctx* ctx, const int32_t* d_ccl, const float* d_field, int32_t min_size,
                                        double* d_cx, double* d_cy, int32_t* d_sx, int32_t* d_sy,
                                        int32_t* d_size, int32_t* d_root, int32_t cap, int32_t* d_n_comp,
                                        void* stream_) {
    if (!ctx) return VOR_EINVAL;
    if (int drc_ = vor_check_device(ctx)) return drc_;
    if (!d_ccl || !d_cx || !d_cy || !d_sx || !d_sy || !d_size || !d_root || !d_n_comp || cap < 0)
        return vor_fail(ctx, VOR_EINVAL, "field_centroids: null pointer or negative capacity");
    cudaStream_t stream = (cudaStream_t)stream_;
    const int64_t n = (int64_t)ctx->Lx * ctx->Ly;
    if (n > INT32_MAX) return vor_fail(ctx, VOR_EINVAL, "field_centroids: Lx * Ly must fit a 32-bit cell index");
    if (!ctx->d_rank) {
        int64_t mc = (n + 1) / 2;
        if (mc > (1 << 22)) mc = 1 << 22;
        ctx->max_comp = (int32_t)mc;
        VOR_CUDA(cudaMalloc((void**)&ctx->d_rank, n * sizeof(int32_t)));
        VOR_CUDA(cudaMalloc((void**)&ctx->d_acc, 4 * (size_t)mc * sizeof(int64_t)));
        VOR_CUDA(cudaMalloc((void**)&ctx->d_comp_root, (size_t)mc * sizeof(int32_t)));
        VOR_CUDA(cudaMalloc((void**)&ctx->d_comp_wcount, (size_t)kCompWarps * kCompGrid * sizeof(int32_t)));
    }
    const int weighted = d_field != nullptr;
    RootPred rp{d_ccl, n};
    RootSink rs{ctx->d_comp_root, ctx->d_rank, ctx->max_comp, &ctx->d_comp_count[0], ctx->d_flags,
                (long long*)ctx->d_acc, weighted ? 4 : 3};
    VOR_LAUNCH(comp_count_kernel<RootPred>, kCompGrid, kCompThreads, 0, stream, rp, ctx->d_comp_wcount);
    VOR_LAUNCH((comp_write_kernel<RootPred, RootSink>), kCompGrid, kCompThreads, 0, stream, rp, rs,
               ctx->d_comp_wcount);
    {
        const bool vec = ctx->Lx % kAccCells == 0 && ((uintptr_t)d_ccl & 15) == 0 && (!weighted || ((uintptr_t)d_field & 15) == 0);
        const int64_t items = vec ? n / kAccCells : n;
        const int agrid = (int)((items + 255) / 256 < 8 * kNumSMs ? (items + 255) / 256 : 8 * kNumSMs);
        const FastDiv fd = make_fastdiv((uint32_t)ctx->Lx);
        unsigned long long* acc = (unsigned long long*)ctx->d_acc;
#define VOR_ACC(W, C)                                                                                            \
        VOR_LAUNCH((accumulate_kernel<W, C>), agrid, 256, 0, stream, d_ccl, d_field, ctx->d_rank, ctx->Lx, ctx->Ly, \
                   ctx->per_x, ctx->per_y, fd, acc, ctx->max_comp)
        if (weighted) { if (vec) VOR_ACC(true, 4); else VOR_ACC(true, 1); }
        else { if (vec) VOR_ACC(false, 4); else VOR_ACC(false, 1); }
#undef VOR_ACC
    }
    SizePred sp{(const long long*)ctx->d_acc, &ctx->d_comp_count[0], min_size};
    CentroidSink cs{(const long long*)ctx->d_acc, ctx->d_comp_root, ctx->max_comp, ctx->Lx, ctx->Ly, cap, weighted,
                    d_cx, d_cy, d_sx, d_sy, d_size, d_root, d_n_comp, ctx->d_flags};
    VOR_LAUNCH(comp_count_kernel<SizePred>, kCompGrid, kCompThreads, 0, stream, sp, ctx->d_comp_wcount);
    VOR_LAUNCH((comp_write_kernel<SizePred, CentroidSink>), kCompGrid, kCompThreads, 0, stream, sp, cs,
               ctx->d_comp_wcount);
    return VOR_OK;
}

extern "C" int field_size_histogram(vor_ctx* ctx, const int32_t* d_size, const int32_t* d_n_comp, int32_t cap,
                                    int32_t bin_width, int32_t n_bins, int64_t* d_hist, void* stream_) {
    if (!ctx) return VOR_EINVAL;
    if (int drc_ = vor_check_device(ctx)) return drc_;
    if (!d_size || !d_n_comp || !d_hist) return vor_fail(ctx, VOR_EINVAL, "field_size_histogram: null pointer");
    if (cap < 0 || bin_width < 1 || n_bins < 1)
        return vor_fail(ctx, VOR_EINVAL, "field_size_histogram: cap >= 0, bin_width >= 1, n_bins >= 1");
    cudaStream_t stream = (cudaStream_t)stream_;
    VOR_CUDA(cudaMemsetAsync(d_hist, 0, (size_t)n_bins * sizeof(int64_t), stream));
    VOR_LAUNCH(size_hist_kernel, 2 * ctx->num_sms, 256, 0, stream, d_size, d_n_comp, cap, bin_width, n_bins,
               (unsigned long long*)d_hist);
    return VOR_OK;
}

extern "C" int match_sites(vor_ctx* ctx, const int32_t* d_px, const int32_t* d_py,
                           const int32_t* d_n_prev, const int32_t* d_nx, const int32_t* d_ny,
                           const int32_t* d_n_now, int32_t cap_prev, int32_t cap_now,
                           int32_t radius_fp, int32_t* d_p2n, int32_t* d_n2p, void* stream_) {
    if (!ctx) return VOR_EINVAL;
    if (int drc_ = vor_check_device(ctx)) return drc_;
    if (!d_px || !d_py || !d_n_prev || !d_nx || !d_ny || !d_n_now || !d_p2n || !d_n2p)
        return vor_fail(ctx, VOR_EINVAL, "match_sites: null pointer");
    if (cap_prev < 1 || cap_now < 1 || radius_fp < 0)
        return vor_fail(ctx, VOR_EINVAL, "match_sites: capacities must be >= 1, radius >= 0");
    cudaStream_t stream = (cudaStream_t)stream_;
    const int64_t need = (int64_t)cap_prev + cap_now;
    if (!ctx->d_best || ctx->best_cap < need) {
        if (ctx->d_best) { VOR_CUDA(cudaStreamSynchronize(stream)); VOR_CUDA(cudaFree(ctx->d_best)); ctx->d_best = nullptr; }
        VOR_CUDA(cudaMalloc((void**)&ctx->d_best, need * sizeof(int32_t)));
        ctx->best_cap = need;
    }
    const int bn = (cap_now + kMatchThreads - 1) / kMatchThreads, bp = (cap_prev + kMatchThreads - 1) / kMatchThreads;
    const long long r2 = (long long)radius_fp * radius_fp;
    // grid path: bucket width P / nbm >= radius
    // the matching lives on the DOMAIN: periods 256 * Lx, 256 * Ly, a walled axis does not wrap
    const MatchGeom geo{(long long)FP_ONE * ctx->Lx, (long long)FP_ONE * ctx->Ly, ctx->per_x, ctx->per_y};
    const long long pmin = geo.Px < geo.Py ? geo.Px : geo.Py;
    int64_t nbm = radius_fp > 0 ? pmin / radius_fp : kMatchGrid;
    if (nbm > kMatchGrid) nbm = kMatchGrid;
    if (nbm < 1) nbm = 1;
    const size_t cells = (size_t)kMatchGrid * kMatchGrid;
    if (!ctx->d_mgrid)
        VOR_CUDA(cudaMalloc((void**)&ctx->d_mgrid, (2 * cells + 2 * cells * kMatchSlots + 1) * sizeof(int32_t)));
    MatchGrid g;
    g.cnt[0] = ctx->d_mgrid; g.cnt[1] = ctx->d_mgrid + cells;
    g.ids[0] = ctx->d_mgrid + 2 * cells; g.ids[1] = g.ids[0] + cells * kMatchSlots;
    g.overflow = g.ids[1] + cells * kMatchSlots;
    g.nbm = (int32_t)nbm;
    VOR_CUDA(cudaMemsetAsync(ctx->d_mgrid, 0, 2 * cells * sizeof(int32_t), stream));
    VOR_CUDA(cudaMemsetAsync(g.overflow, 0, sizeof(int32_t), stream));
    VOR_LAUNCH(match_fill_kernel, 2 * kNumSMs, 256, 0, stream, d_px, d_py, d_n_prev, d_nx, d_ny, d_n_now,
               cap_prev, cap_now, geo, g);
    VOR_LAUNCH(match_grid_kernel, 4 * kNumSMs, 128, 0, stream, d_px, d_py, d_n_prev, d_nx, d_ny, d_n_now,
               cap_prev, cap_now, geo, r2, g, ctx->d_best);
    VOR_LAUNCH(match_best_kernel, bn + bp, kMatchThreads, 0, stream, d_px, d_py, d_n_prev, d_nx, d_ny,
               d_n_now, cap_prev, cap_now, bn, geo, r2,
               ctx->d_best, ctx->d_flags, (const int32_t*)g.overflow);
    VOR_LAUNCH(match_combine_kernel, 2 * kNumSMs, 256, 0, stream, d_n_prev, d_n_now, cap_prev, cap_now,
               ctx->d_best, d_p2n, d_n2p);
    return VOR_OK;
}
