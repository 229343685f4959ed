// a2 — digital Voronoi colouring: labels[cell] = argmin_i (min-image squared distance, i), exact.
// Definition: PAPER.md:35 (§II, Voronoi region) and PAPER.md:129-131 (§III.B.1: every lattice site
// colours itself with the label of the nearest centre; squared distance).  The paper's kernel is
// one thread per lattice site looping over ALL centres; this file computes the same argmin over a
// pruned candidate set that provably contains every cell's nearest site.
//
// Three code paths, all exact (vor_set_option "label_path"; 0 = the library picks):
//  * CTA path (3; the DEFAULT wherever the site density allows it, e.g. every BASELINE config): label_cta_kernel
//    further down - 64 threads per 32 x 32 cells, one shared gather, eight 16 x 8 quadrants with exact bisector
//    candidate lists, packed-key scan; label_fixup_kernel takes the quadrants it cannot prove.  Described at its
//    definition ("A CTA of 64 threads ...").
//  * tile path (2): one warp per TW x TH tile of cells - the round-1 design, kept for lattices the CTA path
//    does not take and as a parity cross-check.
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
//    The common case runs a leaner variant of the same argument (tile_fast): at most 32 gathered
//    sites (one per lane, kept in registers, sorted by index once), and the bound applied per
//    QUADRANT of the tile (probe = quadrant centre, r = quadrant radius), which halves the halo and
//    the candidates per cell; each lane's cells lie in one quadrant, so it scans that quadrant's list.
//    Anything the lean variant cannot prove (too many sites, halo too small) falls back to the
//    generic tile code above, and from there to the general path.
//  * general path (1): one thread per cell, ring search over cell-list buckets in int64 with the
//    minimum-image metric.  After scanning all buckets within Chebyshev bucket distance r of the
//    cell's own bucket every other site has |dx| or |dy| > r*w, so the search stops once
//    best_d2 <= (r*w)^2; when the ring would wrap onto itself it scans all sites.  Used for tiny
//    lattices, very dense or very sparse sites, and as per-tile fallback of the tile path.
#include <type_traits>

#include "common.cuh"
#include "rows.cuh"

namespace {

struct LabelParams {
    int32_t Px, Py;            // periods of the labelling lattice in fixed point (<= 2^30)
    int32_t nbx, nby;          // buckets per axis, w * nbx == Px, w * nby == Py
    int32_t w;
    // window of the lattice that is labelled: cells [wx0, wx1) x [wy0, wy1), stored row-major with `pitch`
    // columns starting at the window's first cell (the whole domain, or a strip of rows)
    int32_t wx0, wy0, wx1, wy1;
    int32_t pitch;
    int32_t n;                 // number of sites (upper bound if n_dev is given)
    const int32_t* __restrict__ n_dev;        // exact number as a device scalar, or NULL
    const int32_t* __restrict__ bucket_start;
    const int4* __restrict__ sorted;
    int32_t tiles_x;
    int32_t tiles_y;
    int32_t halo0;             // initial halo of the generic tile path, fixed point
    int32_t r_tile;            // ceil(sqrt(hx^2 + hy^2)), fixed point
    int32_t halo_fast;         // halo of the quadrant fast path, fixed point
    int32_t r_quad;            // ceil(radius of a quadrant's cell-centre box), fixed point
    uint32_t div_m, div_s1, div_s2;   // floor(x / w) for 0 <= x < 2^32 (Granlund-Montgomery)
    int2* fail_items;          // CTA path: quadrants left to label_fixup_kernel
    int32_t* fail_count;
    int32_t* fail_count_next;  // counter of the next call: zeroed by label_fixup_kernel
    int32_t fail_cap;
    // fused label -> edge path (vor_label_edges): left / right border column of every 32-cell tile column
    // in compact form, col[tile_x * L + y]
    int32_t* col_left;
    int32_t* col_right;
    int32_t* dirty_tiles;      // tiles with an unproven quadrant: their pairs are taken from the label image
    int32_t* dirty_count;
};

// fused path: a label written by the second pass also goes to the compact border columns
__device__ __forceinline__ void store_label(const LabelParams& p, int32_t* __restrict__ labels, int32_t x,
                                            int32_t y, int32_t v) {
    labels[(int64_t)(y - p.wy0) * p.pitch + (x - p.wx0)] = v;
    if (p.col_left) {                                    // fused path: the window is the whole lattice
        if ((x & 31) == 0) p.col_left[(int64_t)(x >> 5) * p.wy1 + y] = v;
        if ((x & 31) == 31) p.col_right[(int64_t)(x >> 5) * p.wy1 + y] = v;
    }
}

__device__ __forceinline__ int32_t div_w(const LabelParams& p, int32_t x /* >= 0 */) {
    const uint32_t t = __umulhi(p.div_m, (uint32_t)x);
    return (int32_t)((t + (((uint32_t)x - t) >> p.div_s1)) >> p.div_s2);
}

// Segment of item i: the number of segments s < nseg whose inclusive prefix inc_s (held by lane s, nondecreasing)
// is <= i.  Binary lifting over the lanes: five shuffles instead of one per segment.  Whole warp, converged.
__device__ __forceinline__ int32_t segment_of(int32_t inc, int32_t nseg, int32_t i) {
    int32_t seg = 0;
#pragma unroll
    for (int step = 16; step > 0; step >>= 1) {
        const int32_t v = __shfl_sync(0xffffffffu, inc, (seg + step - 1) & 31);
        if (seg + step <= nseg && v <= i) seg += step;
    }
    return seg;
}

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
__device__ __forceinline__ void consider(const int4 s, int64_t cx, int64_t cy, int64_t Px, int64_t Py,
                                         int64_t& best, int32_t& besti) {
    int64_t ax = cx > s.x ? cx - s.x : s.x - cx;
    int64_t dx = ax < Px - ax ? ax : Px - ax;
    int64_t ay = cy > s.y ? cy - s.y : s.y - cy;
    int64_t dy = ay < Py - ay ? ay : Py - ay;
    int64_t d2 = dx * dx + dy * dy;
    if (d2 < best || (d2 == best && s.z < besti)) { best = d2; besti = s.z; }
}

__device__ int32_t label_cell_general(const LabelParams& p, int32_t x, int32_t y) {
    const int64_t Px = p.Px, Py = p.Py;
    const int64_t cx = (int64_t)FP_ONE * x + FP_HALF, cy = (int64_t)FP_ONE * y + FP_HALF;
    const int32_t bx = (int32_t)(cx / p.w), by = (int32_t)(cy / p.w);
    int64_t best = INT64_MAX;
    int32_t besti = INT32_MAX;
    for (int32_t r = 0;; ++r) {
        if (2 * r + 1 >= min(p.nbx, p.nby)) {   // the ring would wrap onto itself: scan everything once
            best = INT64_MAX; besti = INT32_MAX;
            const int32_t n = p.n_dev ? min(p.n, *p.n_dev) : p.n;
            for (int32_t k = 0; k < n; ++k) consider(p.sorted[k], cx, cy, Px, Py, best, besti);
            return n > 0 ? besti : -1;       // no site at all: background
        }
        for (int32_t oy = -r; oy <= r; ++oy) {
            const int32_t qy = pos_mod(by + oy, p.nby);
            const bool edge_row = (oy == -r || oy == r);
            for (int32_t ox = -r; ox <= r; ox += (edge_row || r == 0) ? 1 : 2 * r) {
                const int32_t qx = pos_mod(bx + ox, p.nbx);
                const int32_t b = qy * p.nbx + qx;
                const int32_t e = p.bucket_start[b + 1];
                for (int32_t k = p.bucket_start[b]; k < e; ++k)
                    consider(p.sorted[k], cx, cy, Px, Py, best, besti);
            }
        }
        const int64_t rw = (int64_t)r * p.w;
        if (r >= 1 && best <= rw * rw) return besti;
    }
}

__global__ void __launch_bounds__(256) label_general_kernel(LabelParams p, int32_t* __restrict__ labels) {
    const int64_t cell = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    // 16 x 16 blocks of cells per CTA keep a warp's cells inside few buckets
    const int32_t bw = (p.wx1 - p.wx0 + 15) / 16;
    const int32_t blk = (int32_t)(cell >> 8), in = (int32_t)(cell & 255);
    const int32_t x = p.wx0 + (blk % bw) * 16 + (in & 15), y = p.wy0 + (blk / bw) * 16 + (in >> 4);
    if (x < p.wx1 && y < p.wy1) labels[(int64_t)(y - p.wy0) * p.pitch + (x - p.wx0)] = label_cell_general(p, x, y);
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
    const int32_t halfx = p.Px >> 1, halfy = p.Py >> 1;
    if (RX1 - RX0 > halfx || RY1 - RY0 > halfy) return -1;
    if (cxm - RX0 > kMaxRel || RX1 - cxm > kMaxRel || cym - RY0 > kMaxRel || RY1 - cym > kMaxRel) return -1;
    const int32_t a0 = pos_mod(q0, p.nbx);
    const bool split = a0 + ncols > p.nbx;
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
        const int32_t ay = pos_mod(r0 + row, p.nby);
        int32_t c0, c1;                                  // bucket columns [c0, c1)
        if (!split) { c0 = a0; c1 = a0 + ncols; }
        else if ((lane & 1) == 0) { c0 = a0; c1 = p.nbx; }
        else { c0 = 0; c1 = a0 + ncols - p.nbx; }
        beg = p.bucket_start[ay * p.nbx + c0];
        cnt = p.bucket_start[ay * p.nbx + c1] - beg;
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
        const int32_t seg = segment_of(inc, nseg, i);
        const int32_t sbeg = __shfl_sync(0xffffffffu, beg, seg & 31);
        const int32_t sexc = __shfl_sync(0xffffffffu, exc, seg & 31);
        if (i < total) {
            const int4 s = __ldg(&p.sorted[sbeg + (i - sexc)]);
            int32_t rx = s.x - cxm, ry = s.y - cym;
            rx = rx >= halfx ? rx - p.Px : (rx < -halfx ? rx + p.Px : rx);
            ry = ry >= halfy ? ry - p.Py : (ry < -halfy ? ry + p.Py : ry);
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

constexpr int kListCap = 16;       // candidates per quadrant list of the fast path

struct FastScratch {
    int32_t sx[32], sy[32], si[32];          // gathered sites in ascending original index
    int4 list[4][kListCap];                  // per quadrant: (2*rx, 2*ry, rx^2+ry^2, original index)
};
union TileScratch {
    WarpScratch generic;
    FastScratch fast;
};

// ceil(sqrt(f)) or slightly more, f >= 0: one MUFU.RSQ; relative error of the product < 2^-21
__device__ __forceinline__ int32_t isqrt_up(int32_t f) {
    const float x = fmaxf((float)f, 1.0f);
    float r;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return (int32_t)(x * r) + 2;
}

// Quadrant fast path.  Returns false (nothing written) when it cannot prove exactness cheaply.
template <int TW, int TH>
__device__ __forceinline__ bool tile_fast(const LabelParams& p, FastScratch& fs, int lane,
                                          int32_t tx0, int32_t ty0, int32_t cxm, int32_t cym,
                                          int32_t* __restrict__ labels) {
    constexpr int HX = FP_HALF * (TW - 1), HY = FP_HALF * (TH - 1);
    constexpr int QW = TW / 2, QH = TH / 2;
    constexpr int QCX = FP_HALF * QW, QCY = FP_HALF * QH;            // quadrant centre offsets
    constexpr int QHX = FP_HALF * (QW - 1), QHY = FP_HALF * (QH - 1); // quadrant box half extents
    constexpr int GROUPS = 32 / TW, ROWS = TH / GROUPS;
    static_assert(QH % ROWS == 0, "a lane's rows must lie in one quadrant");
    const unsigned full = 0xffffffffu;
    const int32_t H = p.halo_fast, Px = p.Px, Py = p.Py, halfx = p.Px >> 1, halfy = p.Py >> 1;

    // ---- bucket range of the region, relative bounds
    const int32_t q0 = div_w(p, cxm - HX - H + Px) - p.nbx, q1 = div_w(p, cxm + HX + H + Px) - p.nbx;
    const int32_t r0 = div_w(p, cym - HY - H + Py) - p.nby, r1 = div_w(p, cym + HY + H + Py) - p.nby;
    const int32_t ncols = q1 - q0 + 1, nrows = r1 - r0 + 1;
    if (ncols * p.w > halfx || nrows * p.w > halfy) return false;
    const int32_t RX0 = q0 * p.w - cxm, RX1 = (q1 + 1) * p.w - cxm;     // region [RX0, RX1) rel. to centre
    const int32_t RY0 = r0 * p.w - cym, RY1 = (r1 + 1) * p.w - cym;
    if (-RX0 > kMaxRel || RX1 > kMaxRel || -RY0 > kMaxRel || RY1 > kMaxRel) return false;
    const int32_t a0 = q0 < 0 ? q0 + p.nbx : (q0 >= p.nbx ? q0 - p.nbx : q0);
    const bool split = a0 + ncols > p.nbx;
    const int32_t nseg = split ? 2 * nrows : nrows;
    if (nseg > 32) return false;

    // ---- one lane per segment (contiguous run of buckets in one bucket row)
    int32_t beg = 0, cnt = 0;
    if (lane < nseg) {
        const int32_t row = split ? lane >> 1 : lane;
        int32_t ay = r0 + row;
        ay = ay < 0 ? ay + p.nby : (ay >= p.nby ? ay - p.nby : ay);
        int32_t c0, c1;
        if (!split) { c0 = a0; c1 = a0 + ncols; }
        else if ((lane & 1) == 0) { c0 = a0; c1 = p.nbx; }
        else { c0 = 0; c1 = a0 + ncols - p.nbx; }
        beg = __ldg(&p.bucket_start[ay * p.nbx + c0]);
        cnt = __ldg(&p.bucket_start[ay * p.nbx + c1]) - beg;
    }
    int32_t inc = cnt;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int32_t t = __shfl_up_sync(full, inc, o);
        if (lane >= o) inc += t;
    }
    const int32_t total = __shfl_sync(full, inc, 31);
    if (total == 0 || total > 32) return false;
    const int32_t exc = inc - cnt;

    // ---- one lane per site
    const int32_t seg = segment_of(inc, nseg, lane);
    const int32_t sbeg = __shfl_sync(full, beg, seg & 31), sexc = __shfl_sync(full, exc, seg & 31);
    const bool valid = lane < total;
    int32_t rx = 0, ry = 0, idx = INT32_MAX;
    if (valid) {
        const int4 s = __ldg(&p.sorted[sbeg + (lane - sexc)]);
        rx = s.x - cxm; ry = s.y - cym; idx = s.z;
        rx = rx >= halfx ? rx - Px : (rx < -halfx ? rx + Px : rx);
        ry = ry >= halfy ? ry - Py : (ry < -halfy ? ry + Py : ry);
    }
    // ---- sort by original index: rank = number of sites with a smaller index (indices distinct)
    int32_t rank = 0;
    for (int32_t b = 0; b < total; ++b) rank += (__shfl_sync(full, idx, b) < idx);
    if (valid) { fs.sx[rank] = rx; fs.sy[rank] = ry; fs.si[rank] = idx; }
    __syncwarp();
    if (valid) { rx = fs.sx[lane]; ry = fs.sy[lane]; idx = fs.si[lane]; }

    // ---- per-quadrant bound U_q = dist(quadrant centre, nearest site) + quadrant radius
    const int32_t ax = rx - QCX, bx = rx + QCX, ay_ = ry - QCY, by = ry + QCY;
    const int32_t ax2 = ax * ax, bx2 = bx * bx, ay2 = ay_ * ay_, by2 = by * by;
    int32_t d[4] = {bx2 + by2, ax2 + by2, bx2 + ay2, ax2 + ay2};   // q = 2*row + col, centre (-/+QCX, -/+QCY)
    int32_t U[4];
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        const int32_t f = __reduce_min_sync(full, valid ? d[q] : INT32_MAX);
        U[q] = __float2int_ru(sqrtf((float)f)) + 1 + p.r_quad;
    }
    // every site within U_q of quadrant q's box must lie inside the gathered region
    const int32_t mx0 = min(-QCX - QHX - RX0 + 1, RX1 - (-QCX + QHX));
    const int32_t mx1 = min(QCX - QHX - RX0 + 1, RX1 - (QCX + QHX));
    const int32_t my0 = min(-QCY - QHY - RY0 + 1, RY1 - (-QCY + QHY));
    const int32_t my1 = min(QCY - QHY - RY0 + 1, RY1 - (QCY + QHY));
    if (U[0] >= min(mx0, my0) || U[1] >= min(mx1, my0) || U[2] >= min(mx0, my1) || U[3] >= min(mx1, my1))
        return false;

    // ---- candidate list of quadrant q: sites within U_q of its box, in ascending index order
    const int32_t ex0 = max(abs(bx) - QHX, 0), ex1 = max(abs(ax) - QHX, 0);
    const int32_t ey0 = max(abs(by) - QHY, 0), ey1 = max(abs(ay_) - QHY, 0);
    const int32_t ex0s = ex0 * ex0, ex1s = ex1 * ex1, ey0s = ey0 * ey0, ey1s = ey1 * ey1;
    const bool k0 = valid && ex0s + ey0s <= U[0] * U[0], k1 = valid && ex1s + ey0s <= U[1] * U[1];
    const bool k2 = valid && ex0s + ey1s <= U[2] * U[2], k3 = valid && ex1s + ey1s <= U[3] * U[3];
    const unsigned K0 = __ballot_sync(full, k0), K1 = __ballot_sync(full, k1);
    const unsigned K2 = __ballot_sync(full, k2), K3 = __ballot_sync(full, k3);
    if (__popc(K0) > kListCap || __popc(K1) > kListCap || __popc(K2) > kListCap || __popc(K3) > kListCap)
        return false;
    const unsigned lt = (1u << lane) - 1u;
    const int4 entry = make_int4(2 * rx, 2 * ry, rx * rx + ry * ry, idx);
    if (k0) fs.list[0][__popc(K0 & lt)] = entry;
    if (k1) fs.list[1][__popc(K1 & lt)] = entry;
    if (k2) fs.list[2][__popc(K2 & lt)] = entry;
    if (k3) fs.list[3][__popc(K3 & lt)] = entry;
    __syncwarp();

    // ---- each lane scans its quadrant's list for its ROWS cells (column lx)
    const int32_t lx = lane % TW, ly0 = (lane / TW) * ROWS;
    const int myq = (ly0 / QH) * 2 + (lx / QW);
    const unsigned Kq = myq == 0 ? K0 : (myq == 1 ? K1 : (myq == 2 ? K2 : K3));
    const int32_t n = __popc(Kq);
    const int4* __restrict__ list = fs.list[myq];
    const int32_t cxr = FP_ONE * lx - HX, cyr0 = FP_ONE * ly0 - HY;
    int32_t best[ROWS], bi[ROWS];
#pragma unroll
    for (int j = 0; j < ROWS; ++j) { best[j] = INT32_MAX; bi[j] = 0; }
    for (int32_t k = 0; k < n; ++k) {
        const int4 c = list[k];
        const int32_t a = c.z - cxr * c.x;
#pragma unroll
        for (int j = 0; j < ROWS; ++j) {
            const int32_t t = a - (cyr0 + FP_ONE * j) * c.y;
            if (t < best[j]) { best[j] = t; bi[j] = k; }
        }
    }
    const int32_t x = tx0 + lx;
    if (x < p.wx1) {
        int32_t* __restrict__ out = labels + (int64_t)(ty0 + ly0 - p.wy0) * p.pitch + (x - p.wx0);
#pragma unroll
        for (int j = 0; j < ROWS; ++j)
            if (ty0 + ly0 + j < p.wy1) out[(int64_t)j * p.pitch] = list[bi[j]].w;
    }
    return true;
}

// Generic tile path (any number of gathered sites up to kCapGather, adaptive halo).
template <int TW, int TH>
__device__ __noinline__ bool tile_generic(const LabelParams& p, WarpScratch& ws, int lane,
                                          int32_t tx0, int32_t ty0, int32_t cxm, int32_t cym,
                                          int32_t* __restrict__ labels) {
    constexpr int HX = FP_HALF * (TW - 1), HY = FP_HALF * (TH - 1);
    constexpr int GROUPS = 32 / TW, ROWS = TH / GROUPS;
    const int32_t lx = lane % TW, ly0 = (lane / TW) * ROWS;
    int32_t total = -1, margin = 0, dc2 = 0, U = 0;
    int32_t H = p.halo0;
    bool ok = false;
    for (int attempt = 0; attempt < 4; ++attempt) {
        total = gather_region<HX, HY>(p, ws, lane, cxm, cym, H, &margin, &dc2);
        if (total < 0) break;
        if (total == 0) { H = 2 * H + p.w; continue; }
        U = __float2int_ru(sqrtf((float)dc2)) + 1 + p.r_tile;
        if (U < margin) { ok = true; break; }
        H = U;
    }
    if (!ok) return false;
    // keep sites within U of the tile's cell-centre box (compaction in place)
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
    if (m > kCapCand) return false;
    // rank by original index (indices are distinct)
    for (int32_t j = lane; j < m; j += 32) {
        const int32_t idx = ws.g_idx[j];
        int32_t rank = 0;
        for (int32_t k = 0; k < m; ++k) rank += (ws.g_idx[k] < idx);
        const int32_t rx = ws.g_rx[j], ry = ws.g_ry[j];
        ws.cand[rank] = make_int4(2 * rx, 2 * ry, rx * rx + ry * ry, idx);
    }
    __syncwarp();
    const int32_t cxr = FP_ONE * lx - HX, cyr0 = FP_ONE * ly0 - HY;
    int32_t best[ROWS], bi[ROWS];
#pragma unroll
    for (int j = 0; j < ROWS; ++j) { best[j] = INT32_MAX; bi[j] = 0; }
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
    if (x < p.wx1) {
#pragma unroll
        for (int j = 0; j < ROWS; ++j) {
            const int32_t y = ty0 + ly0 + j;
            if (y < p.wy1) store_label(p, labels, x, y, ws.cand[bi[j]].w);
        }
    }
    return true;
}

// |packed key| < 2^31 needs U_q <= kMaxUPacked (packed-key scan of the CTA path)
constexpr int kMaxUPacked = 6400;

// ---------------------------------------------------------------- CTA three-phase path (default)
// The per-quadrant candidate lists are inherently small, scalar work (a few dozen distance tests per
// quadrant), so they are built by a few threads per quadrant instead of one warp per tile.
// A CTA of 64 threads covers 32 x 32 cells = 2 x 4 quadrants of 16 x 8 cells:
//   phase G  the sites of the cell-list buckets covering the CTA's cells plus the halo are gathered
//            into shared memory (coalesced row segments, coordinates relative to the CTA centre);
//            every warp computes the segment prefix, warp w loads items [32w, 32w+32); only the sites
//            inside the exact rectangle box +/- halo are kept;
//   phase A  8 lanes per quadrant build its candidate list from the shared site list:
//            U_q = dist(quadrant centre, nearest gathered site) + quadrant radius; the gathered region
//            must reach U_q beyond the quadrant box on every side; candidates = gathered sites within
//            U_q of the box, ordered by original index;
//   phase B  every warp scans its 32 x 16 cells (lane = column) against its quadrants' lists with
//            packed keys 16 * (|o|^2 - 2 c.o) + position: one integer min per (cell, candidate)
//            gives the nearest site and the smallest-index tie-break; full 128-byte row stores.
// A quadrant whose bound cannot be proven this way is marked and its cells take the general search.
constexpr int kQW = 16, kQH = 8;                      // cells per quadrant (one candidate list each)
constexpr int kCtaQX = 2, kCtaQY = 4;                 // quadrants per CTA: 32 x 32 cells
constexpr int kCtaQ = kCtaQX * kCtaQY;
constexpr int kQHWX = FP_HALF * (kQW - 1), kQHWY = FP_HALF * (kQH - 1);   // half extents of a quadrant's box of cell centres
constexpr int kCtaThreads = 64;
constexpr int kCtaListCap = 12;                       // candidates per quadrant (the exact test leaves about 3)
constexpr int kCtaCapSites = 64;                      // = kCtaThreads: one gathered site per thread
constexpr int kCtaMaxExtent = 23000;                  // |relative site coordinate| bound
constexpr int kCtaMaxU = 20000;                       // |o| <= 896 + U <= 20896: t = |o|^2 - 2 c.o fits int32
constexpr int kUnpackedFlag = 1 << 16;

struct CtaShared {
    int2 sxy[kCtaCapSites];                              // site coordinates relative to the CTA centre (one 64-bit load)
    int32_t si[kCtaCapSites];
    int4 list[kCtaListCap][kCtaQ];                       // [k][quadrant]: conflict-free across quadrants
    int4 tmp[kCtaListCap][kCtaQ];                        // unsorted survivors (phase A scratch)
    int32_t count[kCtaQ];                             // survivors per quadrant (phase A), then list length | flags
    int32_t nkept;                                    // gathered sites kept (inside the exact rectangle)
    // which residues |o|^2 mod 256 a quadrant's survivors have taken, and whether two of them share one.
    // Cell centres are odd multiples of 128 units away from the quadrant centre, so the compared value
    // t = |o|^2 - 2 c.o is congruent to |o|^2 mod 256: candidates with different residues never tie on any cell
    // of the quadrant, and then the order of the list does not matter (no ranking by index needed).
    uint32_t res[kCtaQ][8];
    int32_t coll[kCtaQ];
};
// fused path: (label, slot of the site in sx/sy/si) of every list entry, fetched with one 64-bit load;
// the CTA's 64 x 64 bit matrix of adjacent slots; the first row of the lower warp
struct CtaFusedShared {
    int2 fin[kCtaListCap][kCtaQ];
    uint8_t tslot[kCtaListCap][kCtaQ];                   // slot of the unsorted survivors
    uint32_t bm[kCtaCapSites * kCtaCapSites / 32];
    uint32_t seam[32];                                // row 15 of the tile (last row of the upper warp)
};
struct CtaNoFused {};

// Returns the number of gathered sites (0 = region unusable).  Region bounds relative to the CTA
// centre are returned through R[4] = {RX0, RX1, RY0, RY1}.
__device__ __forceinline__ int32_t cta_gather(const LabelParams& p, CtaShared& sh, int lane, int wid,
                                              int32_t cxm, int32_t cym, int32_t H, int32_t* R) {
    constexpr int HX = FP_HALF * (kQW * kCtaQX - 1), HY = FP_HALF * (kQH * kCtaQY - 1);
    const unsigned full = 0xffffffffu;
    const int32_t Px = p.Px, Py = p.Py, halfx = p.Px >> 1, halfy = p.Py >> 1;
    // a region wider than half a period is unusable (the test on the bucket span below would say the same); asked
    // first, it keeps div_w's arguments >= 0 and the products below inside int32 on small lattices, where the halo
    // (the retry's above all) can exceed the period
    if (2 * (HX + H) > halfx || 2 * (HY + H) > halfy) return 0;
    const int32_t q0 = div_w(p, cxm - HX - H + Px) - p.nbx, q1 = div_w(p, cxm + HX + H + Px) - p.nbx;
    const int32_t r0 = div_w(p, cym - HY - H + Py) - p.nby, r1 = div_w(p, cym + HY + H + Py) - p.nby;
    const int32_t ncols = q1 - q0 + 1, nrows = r1 - r0 + 1;
    if ((int64_t)ncols * p.w > halfx || (int64_t)nrows * p.w > halfy) return 0;
    // the buckets cover more than asked for; only the sites inside the exact rectangle
    // [-HX-H, HX+H] x [-HY-H, HY+H] are kept (shorter lists for every quadrant), so that rectangle is
    // the region the coverage test may rely on: R = {x lower (inclusive), x upper (exclusive), y ...}
    R[0] = -(HX + H); R[1] = HX + H + 1;
    R[2] = -(HY + H); R[3] = HY + H + 1;
    if (R[1] > kCtaMaxExtent || R[3] > kCtaMaxExtent) return 0;
    const int32_t a0 = q0 < 0 ? q0 + p.nbx : (q0 >= p.nbx ? q0 - p.nbx : q0);
    const bool split = a0 + ncols > p.nbx;
    const int32_t nseg = split ? 2 * nrows : nrows;
    if (nseg > 32) return 0;
    int32_t beg = 0, cnt = 0;
    if (lane < nseg) {
        const int32_t row = split ? lane >> 1 : lane;
        int32_t ay = r0 + row;
        ay = ay < 0 ? ay + p.nby : (ay >= p.nby ? ay - p.nby : ay);
        int32_t c0, c1;
        if (!split) { c0 = a0; c1 = a0 + ncols; }
        else if ((lane & 1) == 0) { c0 = a0; c1 = p.nbx; }
        else { c0 = 0; c1 = a0 + ncols - p.nbx; }
        beg = __ldg(&p.bucket_start[ay * p.nbx + c0]);
        cnt = __ldg(&p.bucket_start[ay * p.nbx + c1]) - beg;
    }
    int32_t inc = cnt;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int32_t t = __shfl_up_sync(full, inc, o);
        if (lane >= o) inc += t;
    }
    const int32_t total = __shfl_sync(full, inc, 31);
    if (total > kCtaCapSites) return 0;
    const int32_t exc = inc - cnt;
    if (threadIdx.x == 0) sh.nkept = 0;
    __syncthreads();
    if (32 * wid < total) {                            // warp-uniform: this warp owns items [32 wid, 32 wid + 32)
        const int32_t i = 32 * wid + lane;             // this thread's item
        const int32_t seg = segment_of(inc, nseg, i);
        const int32_t sbeg = __shfl_sync(full, beg, seg & 31), sexc = __shfl_sync(full, exc, seg & 31);
        int32_t rx = 0, ry = 0, idx = 0;
        bool keep = false;
        if (i < total) {
            const int4 s = __ldg(&p.sorted[sbeg + (i - sexc)]);
            rx = s.x - cxm; ry = s.y - cym; idx = s.z;
            rx = rx >= halfx ? rx - Px : (rx < -halfx ? rx + Px : rx);
            ry = ry >= halfy ? ry - Py : (ry < -halfy ? ry + Py : ry);
            keep = abs(rx) <= HX + H && abs(ry) <= HY + H;
        }
        const unsigned ball = __ballot_sync(full, keep);
        int32_t base = 0;
        if (lane == 0 && ball) base = atomicAdd(&sh.nkept, __popc(ball));
        base = __shfl_sync(full, base, 0);
        if (keep) {
            const int32_t pos = base + __popc(ball & ((1u << lane) - 1u));
            sh.sxy[pos] = make_int2(rx, ry); sh.si[pos] = idx;
        }
    }
    return -1;                                         // the caller reads sh.nkept after its barrier
}

// 4 consecutive lanes (sub = 0..3) build the list of quadrant q; qcx, qcy: its centre relative to the
// CTA centre.  Lane sub == 0 publishes sh.count[q] = length | flags, or -1.
template <bool kFused, typename FS>
__device__ __forceinline__ void cta_build_list(const LabelParams& p, CtaShared& sh, FS& fs, int q, int sub,
                                               int32_t ns, const int32_t* R, int32_t qcx, int32_t qcy,
                                               bool active) {
    constexpr int kLanes = kCtaThreads / kCtaQ;         // lanes per quadrant (8)
    const unsigned full = 0xffffffffu;
    if (!active) ns = 0;
    // s*: the gathered site nearest to the quadrant centre (any one of them if several are)
    int32_t f = INT32_MAX, fi = 0;
    for (int32_t i = sub; i < ns; i += kLanes) {
        const int2 s2 = sh.sxy[i];
        const int32_t ox = s2.x - qcx, oy = s2.y - qcy;
        const int32_t d = ox * ox + oy * oy;
        if (d < f) { f = d; fi = i; }
    }
#pragma unroll
    for (int o = 1; o < kLanes; o <<= 1) {
        const int32_t g = __shfl_xor_sync(full, f, o), gi = __shfl_xor_sync(full, fi, o);
        if (g < f || (g == f && gi < fi)) { f = g; fi = gi; }
    }
    const int32_t U = isqrt_up(f) + p.r_quad;
    int32_t margin = min(qcx - kQHWX - R[0] + 1, R[1] - (qcx + kQHWX));
    margin = min(margin, min(qcy - kQHWY - R[2] + 1, R[3] - (qcy + kQHWY)));
    const bool ok = ns > 0 && U < margin && U <= kCtaMaxU;
    if (ok) {
        // Candidates: the sites that can be at least as near as s* to SOME cell of the quadrant.  For a site t,
        // g(c) = |c - t|^2 - |c - s*|^2 is linear in c, so over the box of cell centres [-hx, hx] x [-hy, hy] it is smallest
        // at a corner: min g = |o_t|^2 - |o_s|^2 - 2 (hx |dx| + hy |dy|), (dx, dy) = o_t - o_s.  min g > 0: s* is
        // strictly nearer than t on every cell and t never wins (nor ties).  Every site kept lies within U of the
        // box (it is at most as far from some corner as s*), so the bounds on the packed keys still hold.
        const int32_t osx = sh.sxy[fi].x - qcx, osy = sh.sxy[fi].y - qcy;
        for (int32_t i = sub; i < ns; i += kLanes) {
            const int2 s2 = sh.sxy[i];
            const int32_t ox = s2.x - qcx, oy = s2.y - qcy;
            const int32_t d = ox * ox + oy * oy;
            // |ox|, |oy| < 27000: d < 2^31; 2 (hx |dx| + hy |dy|) < 2 * 1920 * 108000 < 2^31
            if (d - f <= 2 * (kQHWX * abs(ox - osx) + kQHWY * abs(oy - osy))) {
                const int32_t slot = atomicAdd(&sh.count[q], 1);
                if (slot < kCtaListCap) {
                    if constexpr (kFused) {
                        sh.tmp[slot][q] = make_int4(-2 * ox, -2 * oy, d, sh.si[i]);
                        fs.tslot[slot][q] = (uint8_t)i;
                    } else {
                        sh.list[slot][q] = make_int4(-2 * ox, -2 * oy, d, sh.si[i]);
                        const uint32_t bit = 1u << (d & 31);
                        if (atomicOr(&sh.res[q][(d >> 5) & 7], bit) & bit) sh.coll[q] = 1;
                    }
                }
            }
        }
    }
    __syncwarp();
    const int32_t n = sh.count[q];
    __syncwarp();
    if constexpr (kFused) {
        if (ok && n <= kCtaListCap) {
            // order by original index: rank = number of survivors with a smaller index (indices distinct)
            for (int32_t k = sub; k < n; k += kLanes) {
                const int4 e = sh.tmp[k][q];
                int32_t r = 0;
                for (int32_t j = 0; j < n; ++j) r += (sh.tmp[j][q].w < e.w);
                sh.list[r][q] = e;
                fs.fin[r][q] = make_int2(e.w, (int32_t)fs.tslot[k][q]);
            }
        }
    } else {
        // two survivors share a residue (about 3 % of the quadrants): a tie is possible somewhere, so the list is
        // put in index order - the smallest-index rule then comes with the position in the packed key
        if (ok && n <= kCtaListCap && sh.coll[q]) {
            for (int32_t k = sub; k < n; k += kLanes) {
                const int4 e = sh.list[k][q];
                int32_t r = 0;
                for (int32_t j = 0; j < n; ++j) r += (sh.list[j][q].w < e.w);
                sh.tmp[r][q] = e;
            }
            __syncwarp(((1u << kLanes) - 1u) << ((threadIdx.x & 31) & ~(kLanes - 1)));   // the quadrant's lanes (they branch together)
            for (int32_t k = sub; k < n; k += kLanes) sh.list[k][q] = sh.tmp[k][q];
        }
    }
    if (sub == 0 && active)
        sh.count[q] = (ok && n <= kCtaListCap) ? (U <= kMaxUPacked ? n : n | kUnpackedFlag) : -1;
}

// ---- fused path: the adjacent pairs of a CTA's 32 x 32 cells, straight from the labelling registers.
// Every cell carries the SLOT (0..63) of its site in the CTA's gathered list, one byte per cell, four
// rows per register (lane = column); all comparisons below work on four rows at once.
// The compared pairs ("links": H = cell | right neighbour, V = cell | cell below) that join the same two
// slots form chains along the common border of the two regions.  Order the links of a warp's 32 x 16
// block by (row, H before V, column).  A link is reported only if none of the chain neighbours that
// PRECEDE it in that order joins the same two slots:
//   H link (a | b), u and v the cells above a and b:   u == b  (the V link u|a)   v == a  (the V link v|b)
//                                                      u == a and v == b  (the H link above)
//   V link (a over d), p and q the cells left of a and d, s the cell right of a:
//                                                      p == d  (the H link p|a)   s == d  (the H link a|s)
//                                                      p == a and q == d  (the V link to the left)
// The first link of every pair of slots in the block has no predecessor, so every adjacent pair is
// reported at least once - and a straight or staircase border exactly once, which is what keeps the work
// per cell small.  Reported links set one bit of the CTA's 64 x 64 bit matrix in shared memory (the
// de-duplication across the two warps), decoded into (label, label) keys at the end.
__device__ __forceinline__ void bm_set(uint32_t* bm, uint32_t a, uint32_t b) {
    const uint32_t idx = min(a, b) * kCtaCapSites + max(a, b);
    atomicOr(&bm[idx >> 5], 1u << (idx & 31));
}

// most significant bit of every byte: that byte of x (all bytes < 0x80) is not zero
__device__ __forceinline__ uint32_t nz7(uint32_t x) { return x + 0x7f7f7f7fu; }

// one bit-matrix entry per flagged byte (bit 7) of m: the pair (byte of aw, byte of bw) at that position
__device__ __forceinline__ void emit_flagged(uint32_t m, uint32_t aw, uint32_t bw, uint32_t* bm) {
    while (m) {
        const int s = (__ffs(m) - 1) & ~7;
        m &= m - 1;
        bm_set(bm, (aw >> s) & 255u, (bw >> s) & 255u);
    }
}

// W[i]: slots of rows 4i .. 4i+3 of this lane's column (a warp's 16 rows).  Links with the column to
// the right (lanes 0..30) and with the row below (rows 0..14); the row below row 15 is the other
// warp's or the next tile's business, the column right of lane 31 the seam kernel's.
__device__ __forceinline__ void cta_pairs(const uint32_t (&W)[4], int lane, uint32_t* bm) {
    const unsigned full = 0xffffffffu;
    constexpr uint32_t kNone = 0x7f7f7f7fu;                // a slot no cell carries
    uint32_t R[4], PL[4];
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        R[i] = __shfl_down_sync(full, W[i], 1);            // lane 31 reads itself: no H link, no cell to the right
        PL[i] = __shfl_up_sync(full, W[i], 1);
        if (lane == 0) PL[i] = kNone;                      // nothing to the left
    }
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const uint32_t a = W[i], b = R[i];
        const uint32_t u = i ? __funnelshift_l(W[i - 1], W[i], 8) : (W[0] << 8) | 0x7fu;   // the rows above
        const uint32_t v = i ? __funnelshift_l(R[i - 1], R[i], 8) : (R[0] << 8) | 0x7fu;
        const uint32_t mh = nz7(a ^ b) & nz7(u ^ b) & nz7(v ^ a) & nz7((u ^ a) | (v ^ b)) & 0x80808080u;
        emit_flagged(mh, a, b, bm);
        const uint32_t d = i < 3 ? __funnelshift_r(W[i], W[i + 1], 8) : (W[3] >> 8) | (W[3] & 0xff000000u);
        const uint32_t p = PL[i];
        const uint32_t q = i < 3 ? __funnelshift_r(PL[i], PL[i + 1], 8) : (PL[3] >> 8) | (PL[3] & 0xff000000u);
        const uint32_t mv = nz7(a ^ d) & nz7(p ^ d) & nz7(b ^ d) & nz7((p ^ a) | (q ^ d)) & 0x80808080u;
        emit_flagged(mv, a, d, bm);
    }
}

template <bool kFused>
__global__ void __launch_bounds__(kCtaThreads, kFused ? 20 : 24) label_cta_kernel(const __grid_constant__ LabelParams p,
                                                                int32_t* __restrict__ labels,
                                                                const __grid_constant__ RowSet rs) {
    constexpr int kLanes = kCtaThreads / kCtaQ;
    constexpr int HX = FP_HALF * (kQW * kCtaQX - 1), HY = FP_HALF * (kQH * kCtaQY - 1);
    __shared__ CtaShared sh;
    __shared__ typename std::conditional<kFused, CtaFusedShared, CtaNoFused>::type fs;
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int32_t X0 = p.wx0 + blockIdx.x * (kQW * kCtaQX), Y0 = p.wy0 + blockIdx.y * (kQH * kCtaQY);
    // ---- phases G + A; quadrants whose bound could not be proven get one retry with a wider halo
    if (threadIdx.x < kCtaQ) { sh.count[threadIdx.x] = 0; sh.coll[threadIdx.x] = 0; }
    (&sh.res[0][0])[threadIdx.x] = 0;
    static_assert(kCtaQ * 8 == kCtaThreads, "one residue word per thread");
    if constexpr (kFused) {
        for (int i = threadIdx.x; i < kCtaCapSites * kCtaCapSites / 32; i += kCtaThreads) fs.bm[i] = 0;
    }
    // first_fail: some quadrant was not proven with the first gather.  The retry gathers a different, larger site
    // list, so the slots (fin.y) of the quadrants proven first and of those proven on the retry index different
    // lists: the fused kernel never pairs them and hands such a tile to the label-image path (labels use fin.x
    // and are right either way).
    bool any_fail = false, first_fail = false;
    {
        const int q = threadIdx.x / kLanes, sub = threadIdx.x % kLanes;
        const int qx = q % kCtaQX, qy = q / kCtaQX;
        bool active = true;
        for (int attempt = 0; attempt < 2; ++attempt) {
            int32_t R[4] = {0, 0, 0, 0};
            const int32_t H = attempt == 0 ? p.halo_fast : 2 * p.halo_fast + p.w;
            const int32_t got = cta_gather(p, sh, lane, wid, FP_ONE * X0 + FP_HALF + HX,
                                           FP_ONE * Y0 + FP_HALF + HY, H, R);
            __syncthreads();
            const int32_t ns = got ? sh.nkept : 0;
            cta_build_list<kFused>(p, sh, fs, q, sub, ns, R, kQW * FP_ONE * qx + kQHWX - HX, kQH * FP_ONE * qy + kQHWY - HY, active);
            __syncthreads();
            active = sh.count[q] < 0;
            any_fail = __syncthreads_or(active);
            if (attempt == 0) first_fail = any_fail;
            if (!any_fail) break;
            if (attempt == 0 && active) {                                // reset the survivor counter and the residues
                sh.res[q][sub] = 0;
                if (sub == 0) { sh.count[q] = 0; sh.coll[q] = 0; }
            }
            __syncthreads();
        }
    }
    // fused: a tile with an unproven quadrant gets its pairs from the label image later (tile list)
    if constexpr (kFused) {
        if (first_fail && threadIdx.x == 0)
            p.dirty_tiles[atomicAdd(p.dirty_count, 1)] = blockIdx.y * gridDim.x + blockIdx.x;
    }
    // ---- phase B: warp = 32 x 16 cells, lane = column
    const int wx = 0, wy = wid;                          // a warp covers the tile's 32 columns and 16 of its rows
    static_assert(kQW * kCtaQX == 32 && kQH == 8 && kCtaQY == 4, "lane = column; two quadrant rows per warp");
    const int32_t x = X0 + 32 * wx + lane;
    const int qx = lane / kQW;
    const int32_t cxr = FP_ONE * (lane % kQW) - kQHWX;
    uint32_t W[4] = {0, 0, 0, 0};                        // fused: slots of the lane's 16 cells
#pragma unroll
    for (int h = 0; h < 2; ++h) {
        const int q = (2 * wy + h) * kCtaQX + qx;
        const int32_t y0 = Y0 + 16 * wy + 8 * h;
        if (x >= p.wx1 || y0 >= p.wy1) continue;
        const int32_t cnt = sh.count[q];
        int32_t* __restrict__ out = labels + (int64_t)(y0 - p.wy0) * p.pitch + (x - p.wx0);
        if (cnt < 0) {
            // not proven: the quadrant goes to label_fixup_kernel (one warp per quadrant, adaptive
            // halo).  The list holds every quadrant of the lattice, or is disabled (fail_cap == 0) and
            // the cells take the general search here; the quadrant's first lane is always in range.
            if (p.fail_cap > 0) {
                if ((lane & 7) == 0) p.fail_items[atomicAdd(p.fail_count, 1)] = make_int2(x, y0);
            } else {
                for (int j = 0; j < 8; ++j) {
                    if (y0 + j >= p.wy1) break;
                    const int32_t v = label_cell_general(p, x, y0 + j);
                    if constexpr (kFused) store_label(p, labels, x, y0 + j, v);
                    else out[(int64_t)j * p.pitch] = v;
                }
            }
            continue;
        }
        const int32_t n = cnt & (kUnpackedFlag - 1);
        int32_t sel[8];                                  // position of the winning candidate
        if (!(cnt & kUnpackedFlag)) {
            int32_t best[8];
#pragma unroll
            for (int j = 0; j < 8; ++j) best[j] = INT32_MAX;
            int32_t k = 0;
            for (; k + 2 <= n; k += 2) {                 // two candidates per step: 3-input min
                const int4 c0 = sh.list[k][q], c1 = sh.list[k + 1][q];
                const int32_t a0 = 16 * (c0.z + cxr * c0.x) + k, y0s = 16 * c0.y;
                const int32_t a1 = 16 * (c1.z + cxr * c1.x) + k + 1, y1s = 16 * c1.y;
#pragma unroll
                for (int j = 0; j < 8; ++j)
                    best[j] = min(best[j], min(a0 + (FP_ONE * j - kQHWY) * y0s, a1 + (FP_ONE * j - kQHWY) * y1s));
            }
            if (k < n) {
                const int4 c0 = sh.list[k][q];
                const int32_t a0 = 16 * (c0.z + cxr * c0.x) + k, y0s = 16 * c0.y;
#pragma unroll
                for (int j = 0; j < 8; ++j) best[j] = min(best[j], a0 + (FP_ONE * j - kQHWY) * y0s);
            }
#pragma unroll
            for (int j = 0; j < 8; ++j) sel[j] = best[j] & 15;                   // key = 16 t + position
        } else {
            // far sites (large U): same scan with an explicit (value, position) pair
            int32_t best[8];
#pragma unroll
            for (int j = 0; j < 8; ++j) { best[j] = INT32_MAX; sel[j] = 0; }
            for (int32_t k = 0; k < n; ++k) {
                const int4 c = sh.list[k][q];
                const int32_t a = c.z + cxr * c.x;
#pragma unroll
                for (int j = 0; j < 8; ++j) {
                    const int32_t t = a + (FP_ONE * j - kQHWY) * c.y;
                    if (t < best[j]) { best[j] = t; sel[j] = k; }
                }
            }
        }
        if constexpr (kFused) {                          // L % 32 == 0: no ragged rows
            int32_t lab[8];
#pragma unroll
            for (int j = 0; j < 8; ++j) {
                const int2 f = fs.fin[sel[j]][q];         // (label, slot)
                *out = f.x; out += p.pitch;
                lab[j] = f.x;
                W[2 * h + (j >> 2)] |= (uint32_t)f.y << (8 * (j & 3));
            }
            if (lane == 0 || lane == 31) {               // the tile's border columns, 8 labels = two 16-byte stores
                int4* __restrict__ c = reinterpret_cast<int4*>((lane ? p.col_right : p.col_left) + (int64_t)blockIdx.x * p.wy1 + y0);
                c[0] = make_int4(lab[0], lab[1], lab[2], lab[3]);
                c[1] = make_int4(lab[4], lab[5], lab[6], lab[7]);
            }
        } else if (y0 + 8 <= p.wy1) {
#pragma unroll
            for (int j = 0; j < 8; ++j) { *out = sh.list[sel[j]][q].w; out += p.pitch; }
        } else {
            for (int j = 0; j < 8; ++j)
                if (y0 + j < p.wy1) out[(int64_t)j * p.pitch] = sh.list[sel[j]][q].w;
        }
    }
    if constexpr (kFused) {
        if (first_fail) return;                          // CTA-uniform
        cta_pairs(W, lane, fs.bm);
        if (wid == 0) fs.seam[lane] = W[3] >> 24;        // row 15 of the tile
        __syncthreads();
        if (wid == 0) return;
        // the lower warp finishes alone (no further barrier): rows 15 | 16, then the bit matrix is decoded
        // and every distinct pair of the tile is appended to its adjacency row
        {
            const uint32_t a = fs.seam[lane], b = W[0] & 255u;
            const uint32_t pa = __shfl_up_sync(0xffffffffu, a, 1), pb = __shfl_up_sync(0xffffffffu, b, 1);
            if (a != b && (lane == 0 || pa != a || pb != b)) bm_set(fs.bm, a, b);
        }
        __syncwarp();
        constexpr int kWords = kCtaCapSites * kCtaCapSites / 32 / 32;      // bit-matrix words per lane (4)
#pragma unroll
        for (int k = 0; k < kWords; ++k) {
            uint32_t mk = fs.bm[kWords * lane + k];
            while (mk) {
                const uint32_t idx = 32u * (kWords * lane + k) + (__ffs(mk) - 1);
                mk &= mk - 1;
                const uint32_t la = (uint32_t)sh.si[idx / kCtaCapSites], lb = (uint32_t)sh.si[idx % kCtaCapSites];
                row_insert(rs, min(la, lb), max(la, lb));
            }
        }
    }
}

template <int TW, int TH>
__global__ void __launch_bounds__(kWarpsPerCta * 32) label_tile_kernel(LabelParams p,
                                                                       int32_t* __restrict__ labels,
                                                                       int use_fast) {
    constexpr int HX = FP_HALF * (TW - 1), HY = FP_HALF * (TH - 1);
    constexpr int GROUPS = 32 / TW;            // lane groups stacked in y
    constexpr int ROWS = TH / GROUPS;          // rows per lane
    static_assert(TW * GROUPS == 32 && ROWS * GROUPS == TH, "tile shape");
    __shared__ TileScratch scratch[kWarpsPerCta];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int64_t tile = (int64_t)blockIdx.x * kWarpsPerCta + wid;
    if (tile >= (int64_t)p.tiles_x * p.tiles_y) return;
    const int32_t tiy = (int32_t)(tile / p.tiles_x);
    const int32_t tx0 = p.wx0 + (int32_t)(tile - (int64_t)tiy * p.tiles_x) * TW, ty0 = p.wy0 + tiy * TH;
    const int32_t cxm = FP_ONE * tx0 + FP_HALF + HX, cym = FP_ONE * ty0 + FP_HALF + HY;

    if (use_fast && tile_fast<TW, TH>(p, scratch[wid].fast, lane, tx0, ty0, cxm, cym, labels)) return;
    __syncwarp();
    if (tile_generic<TW, TH>(p, scratch[wid].generic, lane, tx0, ty0, cxm, cym, labels)) return;
    const int32_t lx = lane % TW, ly0 = (lane / TW) * ROWS;
    const int32_t x = tx0 + lx;
#pragma unroll 1
    for (int j = 0; j < ROWS; ++j) {
        const int32_t y = ty0 + ly0 + j;
        if (x < p.wx1 && y < p.wy1) labels[(int64_t)(y - p.wy0) * p.pitch + (x - p.wx0)] = label_cell_general(p, x, y);
    }
}

// Second pass of the CTA path: the quadrants whose bound label_cta_kernel could not prove (sparse or
// clustered sites, voids wider than its halo).  One warp per 8 x 8 quadrant: the generic tile code
// with its adaptive halo, then the general search.
__global__ void __launch_bounds__(kWarpsPerCta * 32) label_fixup_kernel(LabelParams p, int32_t* __restrict__ labels) {
    constexpr int HX = FP_HALF * 7;
    __shared__ WarpScratch scratch[kWarpsPerCta];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int32_t n = min(*p.fail_count, p.fail_cap);
    if (blockIdx.x == 0 && threadIdx.x == 0) *p.fail_count_next = 0;
    for (int32_t i = blockIdx.x * kWarpsPerCta + wid; i < n; i += gridDim.x * kWarpsPerCta) {
        const int2 it = p.fail_items[i];
        const int32_t tx0 = it.x, ty0 = it.y;
        __syncwarp();
        if (tile_generic<8, 8>(p, scratch[wid], lane, tx0, ty0, FP_ONE * tx0 + FP_HALF + HX,
                               FP_ONE * ty0 + FP_HALF + HX, labels)) continue;
        const int32_t x = tx0 + (lane & 7), yb = ty0 + (lane >> 3) * 2;
#pragma unroll 1
        for (int j = 0; j < 2; ++j)
            if (x < p.wx1 && yb + j < p.wy1) store_label(p, labels, x, yb + j, label_cell_general(p, x, yb + j));
    }
}

}  // namespace

// which labelling kernel the current cell list gets: 1 general, 2 warp per tile, 3 CTA
static int label_path_for(const vor_ctx* ctx, double spacing) {
    int path = (int)ctx->label_path;
    if (path == 0) path = spacing >= 7.0 ? 3 : (spacing >= 4.0 ? 2 : 1);
    if (ctx->Lx < 16 || ctx->Ly < 16) path = 1;
    return path;
}

static double site_spacing(const vor_ctx* ctx) {               // mean distance between sites, in cells
    return sqrt((double)ctx->Lx * ctx->Ly / (double)ctx->n_hint);
}

// Labels the window [x0, x0 + ww) x [y0, y0 + wh) of the lattice into d_labels (row-major, ww columns).
// fused: rs != NULL -> the CTA kernel also extracts the adjacent pairs of every 32 x 32 tile (path 3 only,
// whole periodic lattice only)
static int label_launch(vor_ctx* ctx, int32_t* d_labels, int32_t x0, int32_t y0, int32_t ww, int32_t wh,
                        const RowSet* rs, cudaStream_t stream) {
    LabelParams p;
    p.Px = (int32_t)ctx->Px; p.Py = (int32_t)ctx->Py; p.nbx = ctx->nbx; p.nby = ctx->nby; p.w = ctx->w;
    p.wx0 = x0; p.wy0 = y0; p.wx1 = x0 + ww; p.wy1 = y0 + wh; p.pitch = ww;
    p.n = ctx->n_sites;
    p.n_dev = ctx->d_n_dev;
    p.bucket_start = ctx->d_bucket_start; p.sorted = ctx->d_sorted;
    p.fail_items = nullptr; p.fail_count = nullptr; p.fail_count_next = nullptr; p.fail_cap = 0;
    p.col_left = nullptr; p.col_right = nullptr; p.dirty_tiles = nullptr; p.dirty_count = nullptr;
    const double spacing = site_spacing(ctx);
    const int path = label_path_for(ctx, spacing);
    const int tw = path == 3 ? 16 : 8;
    if (path == 1) {
        const int64_t blocks = (int64_t)((ww + 15) / 16) * ((wh + 15) / 16);
        VOR_LAUNCH(label_general_kernel, (unsigned)blocks, 256, 0, stream, p, d_labels);
        return VOR_OK;
    }
    p.tiles_x = (ww + tw - 1) / tw;
    p.tiles_y = (wh + tw - 1) / tw;
    const double hx = 128.0 * (tw - 1);
    p.r_tile = (int32_t)ceil(sqrt(2.0 * hx * hx));
    p.halo0 = p.r_tile + (int32_t)(0.75 * spacing * FP_ONE);
    const double qh = 128.0 * (tw / 2 - 1);
    p.r_quad = (int32_t)ceil(sqrt(2.0 * qh * qh));
    if (path == 3) p.r_quad = (int32_t)ceil(sqrt((double)kQHWX * kQHWX + (double)kQHWY * kQHWY));   // 16 x 8 quadrants
    {   // limited to 2^24 units (65536 cells: far beyond any usable gather region), so that the retry's
        // 2 * halo_fast + w stays inside int32 for a handful of sites on a huge lattice
        const double hf = 0.01 * (double)ctx->label_halo_x100 * spacing * FP_ONE;
        p.halo_fast = p.r_quad + (int32_t)(hf < 16777216.0 ? hf : 16777216.0);
    }
    {   // magic numbers for floor(x / w), x < 2^32
        const uint32_t d = (uint32_t)ctx->w;
        uint32_t l = 0;
        while (((uint64_t)1 << l) < d) ++l;
        p.div_m = (uint32_t)((((uint64_t)1 << 32) * (((uint64_t)1 << l) - d)) / d + 1);
        p.div_s1 = l < 1 ? l : 1;
        p.div_s2 = l > 0 ? l - 1 : 0;
    }
    const int use_fast = ctx->label_fast_off ? 0 : 1;
    if (path == 3) {
        if (!ctx->d_lab_fail) {
            const int64_t q = (int64_t)((ctx->Lx + 7) / 8 + 1) * ((ctx->Ly + 7) / 8 + 1);   // any window's quadrants
            ctx->lab_fail_cap = q <= (1 << 24) ? (int32_t)q : 0;      // every quadrant fits, or no list at all
            VOR_CUDA(cudaMalloc((void**)&ctx->d_lab_fail, (size_t)(ctx->lab_fail_cap + 1) * sizeof(int2)));
            VOR_CUDA(cudaMalloc((void**)&ctx->d_lab_fail_n, 2 * sizeof(int32_t)));
            VOR_CUDA(cudaMemsetAsync(ctx->d_lab_fail_n, 0, 2 * sizeof(int32_t), stream));
        }
        p.fail_items = ctx->d_lab_fail; p.fail_cap = ctx->lab_fail_cap;
        p.fail_count = ctx->d_lab_fail_n + ctx->lab_fail_turn;
        p.fail_count_next = ctx->d_lab_fail_n + (1 - ctx->lab_fail_turn);
        ctx->lab_fail_turn = 1 - ctx->lab_fail_turn;
        dim3 grid((ww + kQW * kCtaQX - 1) / (kQW * kCtaQX), (wh + kQH * kCtaQY - 1) / (kQH * kCtaQY));
        if (rs) {
            p.col_left = ctx->d_fu_cols;
            p.col_right = ctx->d_fu_cols + (size_t)(ctx->Lx / 32) * ctx->Ly;
            p.dirty_tiles = ctx->d_fu_dirty;
            p.dirty_count = (int32_t*)&ctx->d_n_raw[4];
            VOR_LAUNCH(label_cta_kernel<true>, grid, kCtaThreads, 0, stream, p, d_labels, *rs);
        } else {
            VOR_LAUNCH(label_cta_kernel<false>, grid, kCtaThreads, 0, stream, p, d_labels, RowSet{});
        }
        // second pass over the unproven quadrants with the 8 x 8 tile geometry
        LabelParams p8 = p;
        const double h8 = 128.0 * 7;
        p8.r_tile = (int32_t)ceil(sqrt(2.0 * h8 * h8));
        p8.halo0 = p8.r_tile + (int32_t)(0.75 * spacing * FP_ONE);
        VOR_LAUNCH(label_fixup_kernel, 4 * ctx->num_sms, kWarpsPerCta * 32, 0, stream, p8, d_labels);
        return VOR_OK;
    }
    const int64_t tiles = (int64_t)p.tiles_x * p.tiles_y;
    const unsigned grid = (unsigned)((tiles + kWarpsPerCta - 1) / kWarpsPerCta);
    VOR_LAUNCH((label_tile_kernel<8, 8>), grid, kWarpsPerCta * 32, 0, stream, p, d_labels, use_fast);
    return VOR_OK;
}

extern "C" int vor_label(vor_ctx* ctx, int32_t* d_labels, void* stream_) {
    if (!ctx) return VOR_EINVAL;
    if (int drc_ = vor_check_device(ctx)) return drc_;
    if (!d_labels) return vor_fail(ctx, VOR_EINVAL, "vor_label: null labels");
    if (ctx->nbx <= 0) return vor_fail(ctx, VOR_ESTATE, "vor_label: call vor_build_cells first");
    return label_launch(ctx, d_labels, 0, 0, ctx->Lx, ctx->Ly, nullptr, (cudaStream_t)stream_);
}

extern "C" int vor_label_rows(vor_ctx* ctx, int32_t y0, int32_t n_rows, int32_t* d_labels, void* stream_) {
    if (!ctx) return VOR_EINVAL;
    if (int drc_ = vor_check_device(ctx)) return drc_;
    if (!d_labels) return vor_fail(ctx, VOR_EINVAL, "vor_label_rows: null labels");
    if (ctx->nbx <= 0) return vor_fail(ctx, VOR_ESTATE, "vor_label_rows: call vor_build_cells first");
    if (y0 < 0 || n_rows < 1 || (int64_t)y0 + n_rows > ctx->Ly)
        return vor_fail(ctx, VOR_EINVAL, "vor_label_rows: rows [y0, y0 + n_rows) must lie inside the lattice");
    return label_launch(ctx, d_labels, 0, y0, ctx->Lx, n_rows, nullptr, (cudaStream_t)stream_);
}

// Can the current cell list take the fused label -> edge path (vor_frame_*)?  It is written for the
// CTA kernel's 32 x 32 tiles on a periodic lattice they tile exactly.
bool vor_label_fusable(const vor_ctx* ctx) {
    if (ctx->nbx <= 0 || ctx->Lx % 32 != 0 || ctx->Ly % 32 != 0 || !ctx->per_x || !ctx->per_y || !ctx->fuse || ctx->d_fo_mask)
        return false;
    return label_path_for(ctx, site_spacing(ctx)) == 3;
}

// Labels + the adjacent pairs inside every 32 x 32 tile (inserted into the rows of rs); fills the compact
// border columns and the list of tiles left to vor_edges_fused_tail (edges.cu).
int vor_label_fused(vor_ctx* ctx, int32_t* d_labels, const RowSet& rs, cudaStream_t stream) {
    if (!ctx->d_fu_cols) {
        VOR_CUDA(cudaMalloc((void**)&ctx->d_fu_cols, 2 * (size_t)(ctx->Lx / 32) * ctx->Ly * sizeof(int32_t)));
        VOR_CUDA(cudaMalloc((void**)&ctx->d_fu_dirty, (size_t)(ctx->Lx / 32) * (ctx->Ly / 32) * sizeof(int32_t)));
    }
    return label_launch(ctx, d_labels, 0, 0, ctx->Lx, ctx->Ly, &rs, stream);
}
