// a2 — digital Voronoi colouring: labels[cell] = argmin_i (min-image squared distance, i), exact.
// Definition: PAPER.md:35 (§II, Voronoi region) and PAPER.md:129-131 (§III.B.1: every lattice site
// colours itself with the label of the nearest centre; squared distance).  The paper's kernel is
// one thread per lattice site looping over ALL centres; this file computes the same argmin over a
// pruned candidate set that provably contains every cell's nearest site.
//
// Two code paths, both exact:
//  * tile path (fast): one warp per TW x TH tile of cells.
//      1. gather the sites of the cell-list buckets covering the tile's bounding box grown by a halo
//         H (bucket rows are contiguous in the bucket-ordered site array: coalesced loads);
//      2. dc = distance from the tile centre to its nearest gathered site.  The nearest-site
//         distance is 1-Lipschitz, so every cell of the tile has a site within U = dc + r_tile;
//         if the gathered region does not reach U beyond the box on every side, gather again with
//         H = U (at most once more);
//      3. keep only sites within U of the box (any other site is farther than U from every cell);
//      4. order the survivors by original index, so that a strict '<' scan resolves ties to the
//         smallest index;
//      5. every lane scans the survivors for its TW*TH/32 cells using
//         d2 = |c|^2 + (|s|^2 - 2 c.s): only t = |s|^2 - 2 cx sx - 2 cy sy is compared, in int32,
//         coordinates relative to the tile centre (|s| <= 23170 guarantees no overflow).
//  * general path: one thread per cell, ring search over cell-list buckets in int64 with the
//    minimum-image metric.  After scanning all buckets within Chebyshev bucket distance r of the
//    cell's own bucket every other site has |dx| or |dy| > r*w, so the search stops once
//    best_d2 <= (r*w)^2; when the ring would wrap onto itself it scans all sites.  Used for tiny
//    lattices, very dense or very sparse sites, and as per-tile fallback of the tile path.
#include "common.cuh"

namespace {

struct LabelParams {
    int32_t L;
    int32_t P;                 // 256 * L  (L <= 2^22 -> P <= 2^30)
    int32_t nb;
    int32_t w;
    int32_t n;
    const int32_t* __restrict__ bucket_start;
    const int4* __restrict__ sorted;
    int32_t tiles_x;
    int32_t tiles_y;
    int32_t halo0;             // initial halo, fixed point
    int32_t r_tile;            // ceil(sqrt(hx^2 + hy^2)), fixed point
};

constexpr int kWarpsPerCta = 8;
constexpr int kCapGather = 160;    // gathered sites per tile
constexpr int kCapCand = 64;       // surviving candidates per tile
constexpr int kMaxRel = 23170;     // |relative site coordinate| bound of the int32 path
constexpr int kMaxSeg = 32;

__device__ __forceinline__ int32_t floor_div(int32_t a, int32_t b) {
    int32_t q = a / b;
    return (a % b != 0 && ((a < 0) != (b < 0))) ? q - 1 : q;
}
__device__ __forceinline__ int32_t pos_mod(int32_t a, int32_t b) {
    int32_t r = a % b;
    return r < 0 ? r + b : r;
}

// ---------------------------------------------------------------- general path (exact, int64)
__device__ __forceinline__ void consider(const int4 s, int64_t cx, int64_t cy, int64_t P,
                                         int64_t& best, int32_t& besti) {
    int64_t ax = cx > s.x ? cx - s.x : s.x - cx;
    int64_t dx = ax < P - ax ? ax : P - ax;
    int64_t ay = cy > s.y ? cy - s.y : s.y - cy;
    int64_t dy = ay < P - ay ? ay : P - ay;
    int64_t d2 = dx * dx + dy * dy;
    if (d2 < best || (d2 == best && s.z < besti)) { best = d2; besti = s.z; }
}

__device__ int32_t label_cell_general(const LabelParams& p, int32_t x, int32_t y) {
    const int64_t P = p.P;
    const int64_t cx = (int64_t)FP_ONE * x + FP_HALF, cy = (int64_t)FP_ONE * y + FP_HALF;
    const int32_t bx = (int32_t)(cx / p.w), by = (int32_t)(cy / p.w);
    int64_t best = INT64_MAX;
    int32_t besti = INT32_MAX;
    for (int32_t r = 0;; ++r) {
        if (2 * r + 1 >= p.nb) {            // the ring would wrap onto itself: scan everything once
            best = INT64_MAX; besti = INT32_MAX;
            for (int32_t k = 0; k < p.n; ++k) consider(p.sorted[k], cx, cy, P, best, besti);
            return besti;
        }
        for (int32_t oy = -r; oy <= r; ++oy) {
            const int32_t qy = pos_mod(by + oy, p.nb);
            const bool edge_row = (oy == -r || oy == r);
            for (int32_t ox = -r; ox <= r; ox += (edge_row || r == 0) ? 1 : 2 * r) {
                const int32_t qx = pos_mod(bx + ox, p.nb);
                const int32_t b = qy * p.nb + qx;
                const int32_t e = p.bucket_start[b + 1];
                for (int32_t k = p.bucket_start[b]; k < e; ++k)
                    consider(p.sorted[k], cx, cy, P, best, besti);
            }
        }
        const int64_t rw = (int64_t)r * p.w;
        if (r >= 1 && best <= rw * rw) return besti;
    }
}

__global__ void __launch_bounds__(256) label_general_kernel(LabelParams p, int32_t* __restrict__ labels) {
    const int64_t cell = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    // 16 x 16 blocks of cells per CTA keep a warp's cells inside few buckets
    const int32_t bw = (p.L + 15) / 16;
    const int32_t blk = (int32_t)(cell >> 8), in = (int32_t)(cell & 255);
    const int32_t x = (blk % bw) * 16 + (in & 15), y = (blk / bw) * 16 + (in >> 4);
    if (x < p.L && y < p.L) labels[(int64_t)y * p.L + x] = label_cell_general(p, x, y);
}

// ---------------------------------------------------------------- tile path
struct WarpScratch {
    int32_t g_rx[kCapGather];
    int32_t g_ry[kCapGather];
    int32_t g_idx[kCapGather];
    int4 cand[kCapCand];           // (2*rx, 2*ry, rx^2+ry^2, original index), ascending index
};

// Gather the sites of all buckets overlapping [centre -/+ (h + H)] into ws.g_*, coordinates
// relative to the tile centre.  Returns the number gathered, or -1 if the region is not valid for
// the int32 path (too wide / too many rows / too many sites).  *margin = lower bound on the distance
// from the tile's cell-centre box to any site NOT gathered; *dc2 = min squared distance centre-site.
template <int HX, int HY>
__device__ __forceinline__ int32_t gather_region(const LabelParams& p, WarpScratch& ws, int lane,
                                                 int32_t cxm, int32_t cym, int32_t H,
                                                 int32_t* margin, int32_t* dc2) {
    const int32_t q0 = floor_div(cxm - HX - H, p.w), q1 = floor_div(cxm + HX + H, p.w);
    const int32_t r0 = floor_div(cym - HY - H, p.w), r1 = floor_div(cym + HY + H, p.w);
    const int32_t ncols = q1 - q0 + 1, nrows = r1 - r0 + 1;
    const int32_t RX0 = q0 * p.w, RX1 = (q1 + 1) * p.w, RY0 = r0 * p.w, RY1 = (r1 + 1) * p.w;
    const int32_t half = p.P >> 1;
    if (RX1 - RX0 > half || RY1 - RY0 > half) return -1;
    if (cxm - RX0 > kMaxRel || RX1 - cxm > kMaxRel || cym - RY0 > kMaxRel || RY1 - cym > kMaxRel) return -1;
    const int32_t a0 = pos_mod(q0, p.nb);
    const bool split = a0 + ncols > p.nb;
    const int32_t nseg = split ? 2 * nrows : nrows;
    if (nseg > kMaxSeg) return -1;
    {
        int32_t m = cxm - HX - RX0 + 1;
        m = min(m, RX1 - (cxm + HX));
        m = min(m, cym - HY - RY0 + 1);
        m = min(m, RY1 - (cym + HY));
        *margin = m;
    }
    // lane s describes segment s: a contiguous run of buckets in one bucket row
    int32_t beg = 0, cnt = 0;
    if (lane < nseg) {
        const int32_t row = split ? lane >> 1 : lane;
        const int32_t ay = pos_mod(r0 + row, p.nb);
        int32_t c0, c1;                                  // bucket columns [c0, c1)
        if (!split) { c0 = a0; c1 = a0 + ncols; }
        else if ((lane & 1) == 0) { c0 = a0; c1 = p.nb; }
        else { c0 = 0; c1 = a0 + ncols - p.nb; }
        beg = p.bucket_start[ay * p.nb + c0];
        cnt = p.bucket_start[ay * p.nb + c1] - beg;
    }
    int32_t inc = cnt;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        int32_t t = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += t;
    }
    const int32_t total = __shfl_sync(0xffffffffu, inc, 31);
    if (total > kCapGather) return -1;
    const int32_t exc = inc - cnt;
    int32_t best = INT32_MAX;
    for (int32_t base = 0; base < total; base += 32) {
        const int32_t i = base + lane;
        // segment of item i = number of segments whose inclusive prefix is <= i
        int32_t seg = 0;
        for (int32_t s = 0; s < nseg; ++s) seg += (__shfl_sync(0xffffffffu, inc, s) <= i);
        const int32_t sbeg = __shfl_sync(0xffffffffu, beg, seg & 31);
        const int32_t sexc = __shfl_sync(0xffffffffu, exc, seg & 31);
        if (i < total) {
            const int4 s = __ldg(&p.sorted[sbeg + (i - sexc)]);
            int32_t rx = s.x - cxm, ry = s.y - cym;
            rx = rx >= half ? rx - p.P : (rx < -half ? rx + p.P : rx);
            ry = ry >= half ? ry - p.P : (ry < -half ? ry + p.P : ry);
            ws.g_rx[i] = rx; ws.g_ry[i] = ry; ws.g_idx[i] = s.z;
            best = min(best, rx * rx + ry * ry);
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) best = min(best, __shfl_xor_sync(0xffffffffu, best, o));
    *dc2 = best;
    __syncwarp();
    return total;
}

template <int TW, int TH>
__global__ void __launch_bounds__(kWarpsPerCta * 32) label_tile_kernel(LabelParams p,
                                                                       int32_t* __restrict__ labels) {
    constexpr int HX = FP_HALF * (TW - 1), HY = FP_HALF * (TH - 1);
    constexpr int GROUPS = 32 / TW;            // lane groups stacked in y
    constexpr int ROWS = TH / GROUPS;          // rows per lane
    static_assert(TW * GROUPS == 32 && ROWS * GROUPS == TH, "tile shape");
    __shared__ WarpScratch scratch[kWarpsPerCta];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    WarpScratch& ws = scratch[wid];
    const int64_t tile = (int64_t)blockIdx.x * kWarpsPerCta + wid;
    if (tile >= (int64_t)p.tiles_x * p.tiles_y) return;
    const int32_t tx0 = (int32_t)(tile % p.tiles_x) * TW, ty0 = (int32_t)(tile / p.tiles_x) * TH;
    const int32_t cxm = FP_ONE * tx0 + FP_HALF + HX, cym = FP_ONE * ty0 + FP_HALF + HY;
    const int32_t lx = lane % TW, ly0 = (lane / TW) * ROWS;

    // ---- 1,2: gather with a halo that provably covers U
    int32_t total = -1, margin = 0, dc2 = 0, U = 0;
    int32_t H = p.halo0;
    bool fast = false;
    for (int attempt = 0; attempt < 4; ++attempt) {
        total = gather_region<HX, HY>(p, ws, lane, cxm, cym, H, &margin, &dc2);
        if (total < 0) break;
        if (total == 0) { H = 2 * H + p.w; continue; }
        U = __float2int_ru(sqrtf((float)dc2)) + 1 + p.r_tile;
        if (U < margin) { fast = true; break; }
        H = U;
    }

    if (fast) {
        // ---- 3: keep sites within U of the tile's cell-centre box (compaction in place)
        int32_t m = 0;
        const int32_t U2 = U * U;
        for (int32_t base = 0; base < total; base += 32) {
            const int32_t i = base + lane;
            int32_t rx = 0, ry = 0, idx = 0;
            bool keep = false;
            if (i < total) {
                rx = ws.g_rx[i]; ry = ws.g_ry[i]; idx = ws.g_idx[i];
                const int32_t ddx = max(abs(rx) - HX, 0), ddy = max(abs(ry) - HY, 0);
                keep = ddx * ddx + ddy * ddy <= U2;
            }
            const unsigned ball = __ballot_sync(0xffffffffu, keep);
            __syncwarp();
            if (keep) {
                const int32_t pos = m + __popc(ball & ((1u << lane) - 1u));
                ws.g_rx[pos] = rx; ws.g_ry[pos] = ry; ws.g_idx[pos] = idx;
            }
            m += __popc(ball);
            __syncwarp();
        }
        if (m > kCapCand) fast = false;
        else {
            // ---- 4: rank by original index (indices are distinct)
            for (int32_t j = lane; j < m; j += 32) {
                const int32_t idx = ws.g_idx[j];
                int32_t rank = 0;
                for (int32_t k = 0; k < m; ++k) rank += (ws.g_idx[k] < idx);
                const int32_t rx = ws.g_rx[j], ry = ws.g_ry[j];
                ws.cand[rank] = make_int4(2 * rx, 2 * ry, rx * rx + ry * ry, idx);
            }
            __syncwarp();
            // ---- 5: every lane scans the candidates for its ROWS cells (column lx)
            const int32_t cxr = FP_ONE * lx - HX;               // cell centre relative to tile centre
            int32_t best[ROWS], bi[ROWS];
#pragma unroll
            for (int j = 0; j < ROWS; ++j) { best[j] = INT32_MAX; bi[j] = 0; }
            const int32_t cyr0 = FP_ONE * ly0 - HY;
            for (int32_t k = 0; k < m; ++k) {
                const int4 c = ws.cand[k];
                const int32_t a = c.z - cxr * c.x;
#pragma unroll
                for (int j = 0; j < ROWS; ++j) {
                    const int32_t t = a - (cyr0 + FP_ONE * j) * c.y;
                    if (t < best[j]) { best[j] = t; bi[j] = k; }
                }
            }
            const int32_t x = tx0 + lx;
            if (x < p.L) {
#pragma unroll
                for (int j = 0; j < ROWS; ++j) {
                    const int32_t y = ty0 + ly0 + j;
                    if (y < p.L) labels[(int64_t)y * p.L + x] = ws.cand[bi[j]].w;
                }
            }
        }
    }
    if (!fast) {
        const int32_t x = tx0 + lx;
#pragma unroll 1
        for (int j = 0; j < ROWS; ++j) {
            const int32_t y = ty0 + ly0 + j;
            if (x < p.L && y < p.L) labels[(int64_t)y * p.L + x] = label_cell_general(p, x, y);
        }
    }
}

}  // namespace

extern "C" int vor_label(vor_ctx* ctx, int32_t* d_labels, void* stream_) {
    if (!ctx) return VOR_EINVAL;
    if (!d_labels) return vor_fail(ctx, VOR_EINVAL, "vor_label: null labels");
    if (ctx->nb <= 0) return vor_fail(ctx, VOR_ESTATE, "vor_label: call vor_build_cells first");
    cudaStream_t stream = (cudaStream_t)stream_;
    LabelParams p;
    p.L = ctx->L; p.P = (int32_t)ctx->P; p.nb = ctx->nb; p.w = ctx->w; p.n = ctx->n_sites;
    p.bucket_start = ctx->d_bucket_start; p.sorted = ctx->d_sorted;
    const double spacing = sqrt((double)ctx->L * ctx->L / (double)ctx->n_sites);   // cells
    int path = (int)ctx->label_path;    // 0 auto, 1 general, 2 tile 16x16, 3 tile 8x8
    if (path == 0) path = spacing >= 10.0 ? 2 : (spacing >= 4.0 ? 3 : 1);
    if (ctx->L < 16) path = 1;
    const int tw = path == 2 ? 16 : 8;
    if (path == 1) {
        const int64_t bw = (ctx->L + 15) / 16;
        const int64_t blocks = bw * bw;
        VOR_LAUNCH(label_general_kernel, (unsigned)blocks, 256, 0, stream, p, d_labels);
        return VOR_OK;
    }
    p.tiles_x = (ctx->L + tw - 1) / tw;
    p.tiles_y = p.tiles_x;
    const double hx = 128.0 * (tw - 1);
    p.r_tile = (int32_t)ceil(sqrt(2.0 * hx * hx));
    p.halo0 = p.r_tile + (int32_t)(0.75 * spacing * FP_ONE);
    const int64_t tiles = (int64_t)p.tiles_x * p.tiles_y;
    const unsigned grid = (unsigned)((tiles + kWarpsPerCta - 1) / kWarpsPerCta);
    if (path == 2)
        VOR_LAUNCH((label_tile_kernel<16, 16>), grid, kWarpsPerCta * 32, 0, stream, p, d_labels);
    else
        VOR_LAUNCH((label_tile_kernel<8, 8>), grid, kWarpsPerCta * 32, 0, stream, p, d_labels);
    return VOR_OK;
}
