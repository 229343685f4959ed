// CPU ORACLE — TEST INFRASTRUCTURE ONLY.
//
// Plain, slow, obviously-correct restatement of what the hot path of
// arXiv:1607.00908 ("GPU Based Detection of Topological Changes in Voronoi
// Diagrams") computes, in the reading fixed by BASELINE.json / SURVEY.md §8(c)
// and listed in DESIGN.md §3.  Only tests/, __graft_entry__.smoke() and
// bench.py's cpu_baseline / --impl reference legs may call it.  It shares no
// code with the CUDA path (paper_1607_00908_b200/csrc) and neither includes,
// links nor imports the other.
//
// Conventions:  L = lattice side, P = 256*L = period in
// fixed-point units; cell (x,y), 0<=x,y<L, has centre (256x+128, 256y+128);
// linear index = y*L + x.  Sites: int32 fixed point in [0,P).  Labels int32.
// Edge key = (uint64)i<<32 | j with i<j.
//
// Parity pins (tests/test_oracle_*.py): every function below is pinned — see
// DESIGN.md §4 for the table.  None is "parity unpinned".
//
// Build: g++ -O2 -ffp-contract=off -fopenmp -shared -fPIC (oracle/build.py).
// OpenMP is used only as "for each lattice row, independently"; threads<=0
// means "all cores the process may use".

#include <algorithm>
#include <cstdint>
#include <cstdlib>
#include <cstring>
#include <queue>
#include <set>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

typedef int64_t i64;
typedef uint64_t u64;

// Minimum-image squared distance between cell centre (cx,cy) and site (sx,sy),
// all in fixed point, period P.  PAPER.md:131 (§III.B.1: "calculating just the
// squared distance"), periodic metric per BASELINE.json config 1.
inline i64 min_image_d2(i64 cx, i64 cy, i64 sx, i64 sy, i64 P) {
    i64 ax = cx > sx ? cx - sx : sx - cx;
    i64 dx = ax < P - ax ? ax : P - ax;
    i64 ay = cy > sy ? cy - sy : sy - cy;
    i64 dy = ay < P - ay ? ay : P - ay;
    return dx * dx + dy * dy;
}

inline int resolve_threads(int threads) {
#ifdef _OPENMP
    return threads > 0 ? threads : omp_get_max_threads();
#else
    (void)threads;
    return 1;
#endif
}

// O1a for one cell: argmin over ALL sites of (d2, index), PAPER.md:35 (region
// definition) + PAPER.md:131 (each lattice site computes its distance from all
// the centres); ties to the smallest index (reading R1).
inline int32_t brute_one(int32_t L, int32_t n, const int32_t* sx, const int32_t* sy, i64 x, i64 y) {
    const i64 P = 256 * (i64)L;
    const i64 cx = 256 * x + 128, cy = 256 * y + 128;
    i64 best = INT64_MAX;
    int32_t besti = -1;
    for (int32_t i = 0; i < n; ++i) {
        i64 d2 = min_image_d2(cx, cy, sx[i], sy[i], P);
        if (d2 < best) { best = d2; besti = i; }   // strict '<' + ascending i  => smallest index wins ties
    }
    return besti;
}

// Cell list for O1b: buckets of `bs` x `bs` cells (w = 256*bs fixed-point units).
struct CellList {
    int32_t nb;                    // buckets per side
    i64 w;                         // bucket width in fixed point
    std::vector<int32_t> start;    // nb*nb+1
    std::vector<int32_t> items;    // site indices, bucket by bucket, ascending inside a bucket
};

CellList make_cell_list(int32_t L, int32_t bs, int32_t n, const int32_t* sx, const int32_t* sy) {
    CellList cl;
    cl.nb = L / bs;
    cl.w = 256 * (i64)bs;
    cl.start.assign((size_t)cl.nb * cl.nb + 1, 0);
    for (int32_t i = 0; i < n; ++i) {
        i64 b = (sy[i] / cl.w) * cl.nb + (sx[i] / cl.w);
        cl.start[b + 1]++;
    }
    for (size_t b = 0; b < (size_t)cl.nb * cl.nb; ++b) cl.start[b + 1] += cl.start[b];
    cl.items.resize(n);
    std::vector<int32_t> fill(cl.start.begin(), cl.start.end() - 1);
    for (int32_t i = 0; i < n; ++i) {
        i64 b = (sy[i] / cl.w) * cl.nb + (sx[i] / cl.w);
        cl.items[fill[b]++] = i;
    }
    return cl;
}

// O1b for one cell: ring search over cell-list buckets with the exactness stop
// rule of reading R3.  After all buckets at Chebyshev bucket
// distance <= r from the cell's own bucket have been scanned, every unscanned
// site has |dx| or |dy| strictly greater than r*w, hence d2 > (r*w)^2; stop when
// best_d2 <= (r*w)^2.  If the next ring would wrap onto itself (2r+1 >= nb) the
// cell is finished by the O1a loop over all sites.
inline int32_t ring_one(int32_t L, int32_t n, const int32_t* sx, const int32_t* sy,
                        const CellList& cl, i64 x, i64 y) {
    const i64 P = 256 * (i64)L;
    const i64 cx = 256 * x + 128, cy = 256 * y + 128;
    const int32_t nb = cl.nb;
    const int32_t bx = (int32_t)(cx / cl.w), by = (int32_t)(cy / cl.w);
    i64 best = INT64_MAX;
    int32_t besti = -1;
    for (int32_t r = 0;; ++r) {
        if (2 * r + 1 >= nb) return brute_one(L, n, sx, sy, x, y);
        for (int32_t oy = -r; oy <= r; ++oy) {
            for (int32_t ox = -r; ox <= r; ++ox) {
                if (std::max(std::abs(ox), std::abs(oy)) != r) continue;   // ring r only
                int32_t qx = ((bx + ox) % nb + nb) % nb, qy = ((by + oy) % nb + nb) % nb;
                size_t b = (size_t)qy * nb + qx;
                for (int32_t k = cl.start[b]; k < cl.start[b + 1]; ++k) {
                    int32_t i = cl.items[k];
                    i64 d2 = min_image_d2(cx, cy, sx[i], sy[i], P);
                    if (d2 < best || (d2 == best && i < besti)) { best = d2; besti = i; }
                }
            }
        }
        i64 rw = (i64)r * cl.w;
        if (besti >= 0 && r >= 1 && best <= rw * rw) return besti;
    }
}

}  // namespace

extern "C" {

// O1a — brute-force labels for the whole lattice.  labels[y*L+x].
void orc_label_brute(int32_t L, int32_t n, const int32_t* sx, const int32_t* sy,
                     int32_t* labels, int threads) {
    int nt = resolve_threads(threads);
    (void)nt;
#pragma omp parallel for schedule(static) num_threads(nt)
    for (int32_t y = 0; y < L; ++y)
        for (int32_t x = 0; x < L; ++x)
            labels[(size_t)y * L + x] = brute_one(L, n, sx, sy, x, y);
}

// O1a on m sampled cells (linear indices) — used at sizes where the full lattice
// is unaffordable (config 5).
void orc_label_brute_at(int32_t L, int32_t n, const int32_t* sx, const int32_t* sy,
                        int64_t m, const int64_t* cells, int32_t* out, int threads) {
    int nt = resolve_threads(threads);
    (void)nt;
#pragma omp parallel for schedule(static) num_threads(nt)
    for (int64_t k = 0; k < m; ++k)
        out[k] = brute_one(L, n, sx, sy, cells[k] % L, cells[k] / L);
}

// O1b — cell-list ring search for the whole lattice.  bucket_cells must divide L.
// Returns 0, or -1 on a bad bucket size.
int orc_label_cells(int32_t L, int32_t n, const int32_t* sx, const int32_t* sy,
                    int32_t bucket_cells, int32_t* labels, int threads) {
    if (bucket_cells < 1 || L % bucket_cells != 0) return -1;
    CellList cl = make_cell_list(L, bucket_cells, n, sx, sy);
    int nt = resolve_threads(threads);
    (void)nt;
#pragma omp parallel for schedule(static) num_threads(nt)
    for (int32_t y = 0; y < L; ++y)
        for (int32_t x = 0; x < L; ++x)
            labels[(size_t)y * L + x] = ring_one(L, n, sx, sy, cl, x, y);
    return 0;
}

// O1b on m sampled cells.
int orc_label_cells_at(int32_t L, int32_t n, const int32_t* sx, const int32_t* sy,
                       int32_t bucket_cells, int64_t m, const int64_t* cells, int32_t* out,
                       int threads) {
    if (bucket_cells < 1 || L % bucket_cells != 0) return -1;
    CellList cl = make_cell_list(L, bucket_cells, n, sx, sy);
    int nt = resolve_threads(threads);
    (void)nt;
#pragma omp parallel for schedule(static) num_threads(nt)
    for (int64_t k = 0; k < m; ++k)
        out[k] = ring_one(L, n, sx, sy, cl, cells[k] % L, cells[k] / L);
    return 0;
}

// O2 — site-adjacency (digital Delaunay) edge set from 4-connected label
// discontinuities including the periodic wrap (reading R6; the paper's analogue
// is the adjacency matrix of PAPER.md:121, 139-191, compressed by sort+unique,
// PAPER.md:207).  Output ascending packed keys (i<<32|j, i<j).  Returns the
// number of unique edges; writes at most `cap` of them.
int64_t orc_edges(int32_t L, const int32_t* labels, uint64_t* out, int64_t cap) {
    std::vector<u64> keys;
    for (int32_t y = 0; y < L; ++y) {
        for (int32_t x = 0; x < L; ++x) {
            int32_t a = labels[(size_t)y * L + x];
            int32_t b = labels[(size_t)y * L + (x + 1) % L];
            int32_t c = labels[(size_t)((y + 1) % L) * L + x];
            if (a != b) keys.push_back(((u64)(uint32_t)std::min(a, b) << 32) | (uint32_t)std::max(a, b));
            if (a != c) keys.push_back(((u64)(uint32_t)std::min(a, c) << 32) | (uint32_t)std::max(a, c));
        }
    }
    std::sort(keys.begin(), keys.end());
    keys.erase(std::unique(keys.begin(), keys.end()), keys.end());
    int64_t m = (int64_t)keys.size();
    for (int64_t k = 0; k < m && k < cap; ++k) out[k] = keys[k];
    return m;
}

// O3 — frame-to-frame diff (PAPER.md:213-221 translation + comparison; PAPER.md:223
// appearing/disappearing bubbles excluded; PAPER.md:266 breaking = in D_P only,
// arising = in D_N only).  p2n / n2p may be NULL (persistent identity).
// With maps: each prev edge (i,j) -> (p2n[i], p2n[j]), dropped if either is -1,
// re-packed (min,max), sorted, uniqued; each now edge with an endpoint whose
// n2p is -1 is dropped.  created = now \ prev, destroyed = prev \ now, both
// ascending, in NOW index space.  Counts returned through n_created/n_destroyed;
// at most cap entries written to each list.
void orc_diff(const uint64_t* prev, int64_t n_prev, const uint64_t* now, int64_t n_now,
              const int32_t* p2n, const int32_t* n2p,
              uint64_t* created, uint64_t* destroyed, int64_t cap,
              int64_t* n_created, int64_t* n_destroyed) {
    std::vector<u64> P, N;
    for (int64_t k = 0; k < n_prev; ++k) {
        int64_t i = (int64_t)(prev[k] >> 32), j = (int64_t)(prev[k] & 0xffffffffu);
        if (p2n) {
            i = p2n[i]; j = p2n[j];
            if (i < 0 || j < 0 || i == j) continue;
        }
        P.push_back(((u64)std::min(i, j) << 32) | (u64)std::max(i, j));
    }
    std::sort(P.begin(), P.end());
    P.erase(std::unique(P.begin(), P.end()), P.end());
    for (int64_t k = 0; k < n_now; ++k) {
        int64_t i = (int64_t)(now[k] >> 32), j = (int64_t)(now[k] & 0xffffffffu);
        if (n2p && (n2p[i] < 0 || n2p[j] < 0)) continue;
        N.push_back(now[k]);
    }
    std::sort(N.begin(), N.end());
    std::vector<u64> C, D;
    std::set_difference(N.begin(), N.end(), P.begin(), P.end(), std::back_inserter(C));
    std::set_difference(P.begin(), P.end(), N.begin(), N.end(), std::back_inserter(D));
    *n_created = (int64_t)C.size();
    *n_destroyed = (int64_t)D.size();
    for (int64_t k = 0; k < (int64_t)C.size() && k < cap; ++k) created[k] = C[k];
    for (int64_t k = 0; k < (int64_t)D.size() && k < cap; ++k) destroyed[k] = D[k];
}

// O4 — threshold + connected components (Ising-like variable from
// the threshold, then cluster labelling).  mask = above ? field>thr : field<thr
// (NaN -> false).  4-connected, periodic (readings R8, R9).  Scan linear indices
// ascending; an unvisited mask cell seeds a breadth-first search that writes the
// seed's linear index to every member — the seed is the component's minimum
// index by construction.  Background -1.
void orc_threshold_ccl(int32_t L, const float* field, float thr, int above, int32_t* ccl) {
    const size_t n = (size_t)L * L;
    std::vector<uint8_t> mask(n);
    for (size_t i = 0; i < n; ++i) mask[i] = above ? (field[i] > thr) : (field[i] < thr);
    for (size_t i = 0; i < n; ++i) ccl[i] = -1;
    std::vector<int32_t> queue;
    for (size_t seed = 0; seed < n; ++seed) {
        if (!mask[seed] || ccl[seed] != -1) continue;
        queue.clear();
        queue.push_back((int32_t)seed);
        ccl[seed] = (int32_t)seed;
        for (size_t head = 0; head < queue.size(); ++head) {
            int32_t c = queue[head];
            int32_t x = c % L, y = c / L;
            const int32_t nbr[4] = {
                y * L + (x + 1) % L, y * L + (x + L - 1) % L,
                ((y + 1) % L) * L + x, ((y + L - 1) % L) * L + x};
            for (int k = 0; k < 4; ++k)
                if (mask[nbr[k]] && ccl[nbr[k]] == -1) {
                    ccl[nbr[k]] = (int32_t)seed;
                    queue.push_back(nbr[k]);
                }
        }
    }
}

// O5 — per-component size and centre of mass (count the lattice
// points of each bubble, "sum, separately, the coordinates of the lattice points
// that form the bubble and divide by the size"; unweighted reading R10, periodic
// unwrap relative to the root cell R11, integer sums, floor to fixed point R12).
// Components with size < min_size are dropped; survivors are numbered 0..K-1 by
// ascending root index.  Returns K (writes at most cap entries).
int32_t orc_centroids(int32_t L, const int32_t* ccl, int32_t min_size,
                      double* cx, double* cy, int32_t* sx, int32_t* sy,
                      int32_t* size, int32_t* root, int32_t cap) {
    const size_t n = (size_t)L * L;
    const i64 P = 256 * (i64)L;
    std::vector<i64> cnt(n, 0), Sx(n, 0), Sy(n, 0);     // indexed by root cell
    for (size_t i = 0; i < n; ++i) {
        int32_t r = ccl[i];
        if (r < 0) continue;
        i64 x = (i64)(i % L), y = (i64)(i / L), xr = r % L, yr = r / L;
        i64 dx = x - xr;
        if (2 * dx >= L) dx -= L; else if (2 * dx < -(i64)L) dx += L;
        i64 dy = y - yr;
        if (2 * dy >= L) dy -= L; else if (2 * dy < -(i64)L) dy += L;
        cnt[r] += 1; Sx[r] += dx; Sy[r] += dy;
    }
    int32_t K = 0;
    for (size_t r = 0; r < n; ++r) {
        if (cnt[r] == 0 || cnt[r] < min_size) continue;
        if (K < cap) {
            i64 xr = (i64)(r % L), yr = (i64)(r / L), m = cnt[r];
            // floor division toward -inf, then non-negative mod P
            i64 qx = 256 * Sx[r], qy = 256 * Sy[r];
            i64 fx = qx >= 0 ? qx / m : -((-qx + m - 1) / m);
            i64 fy = qy >= 0 ? qy / m : -((-qy + m - 1) / m);
            sx[K] = (int32_t)((((256 * xr + 128 + fx) % P) + P) % P);
            sy[K] = (int32_t)((((256 * yr + 128 + fy) % P) + P) % P);
            double ux = (double)xr + 0.5 + (double)Sx[r] / (double)m;
            double uy = (double)yr + 0.5 + (double)Sy[r] / (double)m;
            if (ux < 0) ux += L; else if (ux >= L) ux -= L;
            if (uy < 0) uy += L; else if (uy >= L) uy -= L;
            cx[K] = ux; cy[K] = uy;
            size[K] = (int32_t)m;
            root[K] = (int32_t)r;
        }
        ++K;
    }
    return K;
}

// O6 — isomorphism Phi P->N by comparing the two sets of centres,
// unmatched = appeared / disappeared.  Rule (reading R13): mutual
// nearest neighbour under the minimum-image metric on fixed-point coordinates,
// within the inclusive radius, ties to the smallest index.  -1 = dead / born.
void orc_match(int32_t L, const int32_t* px, const int32_t* py, int32_t n_prev,
               const int32_t* nx, const int32_t* ny, int32_t n_now, int32_t radius_fp,
               int32_t* p2n, int32_t* n2p) {
    const i64 P = 256 * (i64)L, r2 = (i64)radius_fp * radius_fp;
    std::vector<int32_t> bp(n_now, -1), bn(n_prev, -1);
    for (int32_t j = 0; j < n_now; ++j) {
        i64 best = INT64_MAX;
        for (int32_t i = 0; i < n_prev; ++i) {
            i64 d2 = min_image_d2(nx[j], ny[j], px[i], py[i], P);
            if (d2 < best) { best = d2; bp[j] = i; }
        }
        if (best > r2) bp[j] = -1;
    }
    for (int32_t i = 0; i < n_prev; ++i) {
        i64 best = INT64_MAX;
        for (int32_t j = 0; j < n_now; ++j) {
            i64 d2 = min_image_d2(px[i], py[i], nx[j], ny[j], P);
            if (d2 < best) { best = d2; bn[i] = j; }
        }
        if (best > r2) bn[i] = -1;
    }
    for (int32_t i = 0; i < n_prev; ++i) p2n[i] = (bn[i] >= 0 && bp[bn[i]] == i) ? bn[i] : -1;
    for (int32_t j = 0; j < n_now; ++j) n2p[j] = (bp[j] >= 0 && bn[bp[j]] == j) ? bp[j] : -1;
}

// O7 — trigger and event counts (§III.B.3: every row of (E_P)_PN is compared with
// its isomorphic row of (E_N)_NN; a vertex whose rows differ gets local_trigger = 1, and
// global_trigger says whether any did; §III.B.4: the triggering indices are written to
// eventsIndices, their number to eventsNumber; for every active index, eventsCount =
// how many active sites are connected to it, "repeated for the active indices of the two
// triangulations").  Inputs: the two ascending unique edge lists in ONE index space (past list
// already translated) over n vertices.  Written out as the definition:
// row(i) = sorted neighbour list of i; trigger[i] = rows differ.
// Outputs: trigger[n] (0/1), events_indices (ascending, first *events_number entries),
// count_prev[n], count_now[n] (0 for inactive vertices).  Returns global_trigger.
int32_t orc_events(const u64* prev, i64 n_prev, const u64* now, i64 n_now, int32_t n,
                   int32_t* trigger, int32_t* events_indices, int32_t* events_number,
                   int32_t* count_prev, int32_t* count_now) {
    std::vector<std::vector<int32_t>> rp(n), rn(n);
    for (i64 k = 0; k < n_prev; ++k) {
        const int32_t i = (int32_t)(prev[k] >> 32), j = (int32_t)(prev[k] & 0xffffffffu);
        if (i < n && j < n) { rp[i].push_back(j); rp[j].push_back(i); }
    }
    for (i64 k = 0; k < n_now; ++k) {
        const int32_t i = (int32_t)(now[k] >> 32), j = (int32_t)(now[k] & 0xffffffffu);
        if (i < n && j < n) { rn[i].push_back(j); rn[j].push_back(i); }
    }
    int32_t m = 0, any = 0;
    for (int32_t i = 0; i < n; ++i) {
        std::sort(rp[i].begin(), rp[i].end());
        std::sort(rn[i].begin(), rn[i].end());
        trigger[i] = rp[i] != rn[i];
        if (trigger[i]) { events_indices[m++] = i; any = 1; }
    }
    *events_number = m;
    for (int32_t i = 0; i < n; ++i) {
        count_prev[i] = count_now[i] = 0;
        if (!trigger[i]) continue;
        for (int32_t j : rp[i]) count_prev[i] += trigger[j];
        for (int32_t j : rn[i]) count_now[i] += trigger[j];
    }
    return any;
}

// O8 — couples of active vertices and T1 pairing (§III.B.4: "we find which of the active
// points are connected and store them as couples ... discard those couples that are given by a simple
// permutation of another couple ... checks whether or not the couple is connected in both configurations.
// If the couple is connected in only one configuration, then this is dubbed either breaking or arising if
// it is found to be in D_P or in D_N"; an edge whose end points share two neighbours is
// in the bulk, one neighbour: on the boundary; PAPER.md:238 and Fig. 8: in a T1 event the breaking link
// is replaced by the arising link between its two common neighbours, the number of links is conserved).
// Inputs as O7.  A couple is a pair i < j of active vertices (trigger = 1, O7) connected in D_P or D_N.
// Outputs, one entry per couple in ascending (i, j) order:
//   couples      packed key (i << 32 | j)
//   cls          0 connected in both, 1 breaking (D_P only), 2 arising (D_N only)
//   common_prev  number of common neighbours of i and j in D_P, -1 if the couple is not connected there
//   common_now   the same in D_N
//   partner      breaking couple: if it has exactly two common neighbours c < d in D_P and (c, d) is an
//                arising couple, that couple's key (the T1 quadruple is {i, j, c, d}); arising couple: the
//                mirror statement in D_N with a breaking couple; otherwise ~0.
// Returns the number of couples (cap is only checked, never exceeded).
i64 orc_t1(const u64* prev, i64 n_prev, const u64* now, i64 n_now, int32_t n,
           u64* couples, int32_t* cls, int32_t* common_prev, int32_t* common_now, u64* partner, i64 cap) {
    std::vector<std::set<int32_t>> rp(n), rn(n);
    for (i64 k = 0; k < n_prev; ++k) {
        const int32_t i = (int32_t)(prev[k] >> 32), j = (int32_t)(prev[k] & 0xffffffffu);
        if (i < n && j < n) { rp[i].insert(j); rp[j].insert(i); }
    }
    for (i64 k = 0; k < n_now; ++k) {
        const int32_t i = (int32_t)(now[k] >> 32), j = (int32_t)(now[k] & 0xffffffffu);
        if (i < n && j < n) { rn[i].insert(j); rn[j].insert(i); }
    }
    std::vector<char> active(n);
    for (int32_t i = 0; i < n; ++i) active[i] = rp[i] != rn[i];
    auto shared = [](const std::set<int32_t>& a, const std::set<int32_t>& b) {
        std::vector<int32_t> c;
        for (int32_t v : a) if (b.count(v)) c.push_back(v);
        return c;                                        // ascending
    };
    const u64 none = ~(u64)0;
    i64 m = 0;
    for (int32_t i = 0; i < n; ++i) {
        if (!active[i]) continue;
        std::set<int32_t> nb = rp[i];
        nb.insert(rn[i].begin(), rn[i].end());
        for (int32_t j : nb) {
            if (j <= i || !active[j]) continue;          // a permutation of a couple is the same couple
            const bool in_p = rp[i].count(j) != 0, in_n = rn[i].count(j) != 0;
            const std::vector<int32_t> sp = shared(rp[i], rp[j]), sn = shared(rn[i], rn[j]);
            u64 pt = none;
            if (in_p && !in_n && sp.size() == 2) {       // breaking: do its two common neighbours arise?
                const int32_t c = sp[0], d = sp[1];
                if (rn[c].count(d) && !rp[c].count(d)) pt = ((u64)(uint32_t)c << 32) | (uint32_t)d;
            }
            if (in_n && !in_p && sn.size() == 2) {       // arising: do its two common neighbours break?
                const int32_t c = sn[0], d = sn[1];
                if (rp[c].count(d) && !rn[c].count(d)) pt = ((u64)(uint32_t)c << 32) | (uint32_t)d;
            }
            if (m < cap) {
                couples[m] = ((u64)(uint32_t)i << 32) | (uint32_t)j;
                cls[m] = in_p && in_n ? 0 : (in_p ? 1 : 2);
                common_prev[m] = in_p ? (int32_t)sp.size() : -1;
                common_now[m] = in_n ? (int32_t)sn.size() : -1;
                partner[m] = pt;
            }
            ++m;
        }
    }
    return m;
}

// ------------------------------------------------------------------------------------------------------
// O9 — the same definitions on the paper's own geometry: a rectangular
// Lx x Ly lattice (§IV: "Lx x Ly = 2048 x 1024"), each axis either periodic or closed by walls
// (§III.B.2: on the domain boundaries "the frame is given by all nearest neighbours that do
// not lie outside the domain"), obstacle sites carrying an excluded colour (§III.B.1: MAXLINK,
// "regions of the lattice with undefined colour which automatically will not be considered for the
// Delaunay triangulation"), 8-connected bubbles (reachable "along the directions of the
// Lattice Boltzmann model", D2Q9), density-weighted centres (§II eq. for z*), the bubble-size
// histogram ("characterize them according to their size"), bulk / boundary
// edges.  With Lx == Ly, both axes periodic, no exclusion, 4-connectivity and no weights
// these functions compute what O1..O6 compute (pinned by equality in tests/test_oracle_geometry.py).
// Conventions: cell (x, y), 0 <= x < Lx, 0 <= y < Ly, linear index y*Lx + x; Px = 256*Lx, Py = 256*Ly;
// on a walled axis the distance is the plain difference and nothing wraps.

namespace {

inline i64 axis_dist(i64 c, i64 s, i64 P, int periodic) {
    i64 a = c > s ? c - s : s - c;
    return periodic && P - a < a ? P - a : a;
}

inline int32_t brute_one_g(int32_t Lx, int32_t Ly, int px, int py, int32_t n, const int32_t* sx,
                           const int32_t* sy, i64 x, i64 y) {
    const i64 Px = 256 * (i64)Lx, Py = 256 * (i64)Ly;
    const i64 cx = 256 * x + 128, cy = 256 * y + 128;
    i64 best = INT64_MAX;
    int32_t besti = -1;
    for (int32_t i = 0; i < n; ++i) {
        const i64 dx = axis_dist(cx, sx[i], Px, px), dy = axis_dist(cy, sy[i], Py, py);
        const i64 d2 = dx * dx + dy * dy;
        if (d2 < best) { best = d2; besti = i; }
    }
    return besti;
}

}  // namespace

// O1a on the general geometry.  labels[y*Lx + x]; no site at all -> -1.
void orc_label_brute_g(int32_t Lx, int32_t Ly, int per_x, int per_y, int32_t n, const int32_t* sx,
                       const int32_t* sy, int32_t* labels, int threads) {
    int nt = resolve_threads(threads);
    (void)nt;
#pragma omp parallel for schedule(static) num_threads(nt)
    for (int32_t y = 0; y < Ly; ++y)
        for (int32_t x = 0; x < Lx; ++x)
            labels[(size_t)y * Lx + x] = brute_one_g(Lx, Ly, per_x, per_y, n, sx, sy, x, y);
}

void orc_label_brute_at_g(int32_t Lx, int32_t Ly, int per_x, int per_y, int32_t n, const int32_t* sx,
                          const int32_t* sy, int64_t m, const int64_t* cells, int32_t* out, int threads) {
    int nt = resolve_threads(threads);
    (void)nt;
#pragma omp parallel for schedule(static) num_threads(nt)
    for (int64_t k = 0; k < m; ++k)
        out[k] = brute_one_g(Lx, Ly, per_x, per_y, n, sx, sy, cells[k] % Lx, cells[k] / Lx);
}

// O1b on the general geometry: the ring search of reading R3 over nbx x nby buckets of bucket_cells cells.
// A ring position outside a walled axis holds no bucket; on a periodic axis it wraps.  The stop rule is
// unchanged (after ring r every unscanned site has |dx| or |dy| > r*w).  When a ring would wrap onto
// itself on a periodic axis, or has left the lattice on every side, the cell is finished by O1a.
int orc_label_cells_g(int32_t Lx, int32_t Ly, int per_x, int per_y, int32_t n, const int32_t* sx,
                      const int32_t* sy, int32_t bucket_cells, int32_t* labels, int threads) {
    if (bucket_cells < 1 || Lx % bucket_cells != 0 || Ly % bucket_cells != 0) return -1;
    const int32_t nbx = Lx / bucket_cells, nby = Ly / bucket_cells;
    const i64 w = 256 * (i64)bucket_cells, Px = 256 * (i64)Lx, Py = 256 * (i64)Ly;
    std::vector<int32_t> start((size_t)nbx * nby + 1, 0), items(n);
    for (int32_t i = 0; i < n; ++i) start[(size_t)(sy[i] / w) * nbx + sx[i] / w + 1]++;
    for (size_t b = 0; b < (size_t)nbx * nby; ++b) start[b + 1] += start[b];
    {
        std::vector<int32_t> fill(start.begin(), start.end() - 1);
        for (int32_t i = 0; i < n; ++i) items[fill[(size_t)(sy[i] / w) * nbx + sx[i] / w]++] = i;
    }
    int nt = resolve_threads(threads);
    (void)nt;
#pragma omp parallel for schedule(static) num_threads(nt)
    for (int32_t y = 0; y < Ly; ++y) {
        for (int32_t x = 0; x < Lx; ++x) {
            const i64 cx = 256 * (i64)x + 128, cy = 256 * (i64)y + 128;
            const int32_t bx = (int32_t)(cx / w), by = (int32_t)(cy / w);
            i64 best = INT64_MAX;
            int32_t besti = -1, result = -2;
            for (int32_t r = 0; result == -2; ++r) {
                const bool wraps = (per_x && 2 * r + 1 >= nbx) || (per_y && 2 * r + 1 >= nby);
                const bool outside = r > std::max(nbx, nby);
                if (wraps || outside) { result = brute_one_g(Lx, Ly, per_x, per_y, n, sx, sy, x, y); break; }
                for (int32_t oy = -r; oy <= r; ++oy) {
                    for (int32_t ox = -r; ox <= r; ++ox) {
                        if (std::max(std::abs(ox), std::abs(oy)) != r) continue;
                        int32_t qx = bx + ox, qy = by + oy;
                        if (per_x) qx = (qx % nbx + nbx) % nbx; else if (qx < 0 || qx >= nbx) continue;
                        if (per_y) qy = (qy % nby + nby) % nby; else if (qy < 0 || qy >= nby) continue;
                        const size_t b = (size_t)qy * nbx + qx;
                        for (int32_t k = start[b]; k < start[b + 1]; ++k) {
                            const int32_t i = items[k];
                            const i64 dx = axis_dist(cx, sx[i], Px, per_x), dy = axis_dist(cy, sy[i], Py, per_y);
                            const i64 d2 = dx * dx + dy * dy;
                            if (d2 < best || (d2 == best && i < besti)) { best = d2; besti = i; }
                        }
                    }
                }
                const i64 rw = (i64)r * w;
                if (besti >= 0 && r >= 1 && best <= rw * rw) result = besti;
            }
            labels[(size_t)y * Lx + x] = result;
        }
    }
    return 0;
}

// O2 on the general geometry: every cell against its right and its lower neighbour; a neighbour beyond a
// wall does not exist; a pair with the excluded colour on either side is not an edge.
// exclude < 0: nothing is excluded.
int64_t orc_edges_g(int32_t Lx, int32_t Ly, int per_x, int per_y, int32_t exclude, const int32_t* labels,
                    uint64_t* out, int64_t cap) {
    std::vector<u64> keys;
    auto add = [&](int32_t a, int32_t b) {
        if (a == b) return;
        if (exclude >= 0 && (a == exclude || b == exclude)) return;
        keys.push_back(((u64)(uint32_t)std::min(a, b) << 32) | (uint32_t)std::max(a, b));
    };
    for (int32_t y = 0; y < Ly; ++y) {
        for (int32_t x = 0; x < Lx; ++x) {
            const int32_t a = labels[(size_t)y * Lx + x];
            if (x + 1 < Lx) add(a, labels[(size_t)y * Lx + x + 1]);
            else if (per_x) add(a, labels[(size_t)y * Lx]);
            if (y + 1 < Ly) add(a, labels[(size_t)(y + 1) * Lx + x]);
            else if (per_y) add(a, labels[x]);
        }
    }
    std::sort(keys.begin(), keys.end());
    keys.erase(std::unique(keys.begin(), keys.end()), keys.end());
    const int64_t m = (int64_t)keys.size();
    for (int64_t k = 0; k < m && k < cap; ++k) out[k] = keys[k];
    return m;
}

// O4 on the general geometry; connectivity 4 (reading R9) or 8 (the D2Q9 directions of PAPER.md:95, 147).
int orc_threshold_ccl_g(int32_t Lx, int32_t Ly, int per_x, int per_y, const float* field, float thr, int above,
                        int connectivity, int32_t* ccl) {
    if (connectivity != 4 && connectivity != 8) return -1;
    const size_t n = (size_t)Lx * Ly;
    std::vector<uint8_t> mask(n);
    for (size_t i = 0; i < n; ++i) mask[i] = above ? (field[i] > thr) : (field[i] < thr);
    for (size_t i = 0; i < n; ++i) ccl[i] = -1;
    static const int DX[8] = {1, -1, 0, 0, 1, 1, -1, -1}, DY[8] = {0, 0, 1, -1, 1, -1, 1, -1};
    std::vector<int32_t> queue;
    for (size_t seed = 0; seed < n; ++seed) {
        if (!mask[seed] || ccl[seed] != -1) continue;
        queue.clear();
        queue.push_back((int32_t)seed);
        ccl[seed] = (int32_t)seed;
        for (size_t head = 0; head < queue.size(); ++head) {
            const int32_t c = queue[head], x = c % Lx, y = c / Lx;
            for (int k = 0; k < connectivity; ++k) {
                int32_t u = x + DX[k], v = y + DY[k];
                if (u < 0 || u >= Lx) { if (!per_x) continue; u = (u + Lx) % Lx; }
                if (v < 0 || v >= Ly) { if (!per_y) continue; v = (v + Ly) % Ly; }
                const size_t q = (size_t)v * Lx + u;
                if (mask[q] && ccl[q] == -1) { ccl[q] = (int32_t)seed; queue.push_back((int32_t)q); }
            }
        }
    }
    return 0;
}

// O5 on the general geometry, optionally weighted by the density (z* = sum(y rho) / sum(rho)).
// Weight of a cell: w = floor(rho * 65536) limited to [1, 2^24] (NaN -> 1): a fixed-point density, so that
// the sums are integers and do not depend on the order of accumulation (reading R10 carried over);
// field == NULL: w = 1, which is O5.  Offsets from the root cell are unwrapped on periodic axes only.
// sx = (256 xr + 128 + floor(256 Sx / W)) mod Px with Sx = sum(w dx), W = sum(w); cx = xr + 0.5 + Sx / W.
// size = number of cells (the weights do not enter min_size).
int32_t orc_centroids_g(int32_t Lx, int32_t Ly, int per_x, int per_y, const int32_t* ccl, const float* field,
                        int32_t min_size, double* cx, double* cy, int32_t* sx, int32_t* sy,
                        int32_t* size, int32_t* root, int32_t cap) {
    const size_t n = (size_t)Lx * Ly;
    const i64 Px = 256 * (i64)Lx, Py = 256 * (i64)Ly;
    std::vector<i64> cnt(n, 0), W(n, 0), Sx(n, 0), Sy(n, 0);
    for (size_t i = 0; i < n; ++i) {
        const int32_t r = ccl[i];
        if (r < 0) continue;
        i64 dx = (i64)(i % Lx) - r % Lx, dy = (i64)(i / Lx) - r / Lx;
        if (per_x) { if (2 * dx >= Lx) dx -= Lx; else if (2 * dx < -(i64)Lx) dx += Lx; }
        if (per_y) { if (2 * dy >= Ly) dy -= Ly; else if (2 * dy < -(i64)Ly) dy += Ly; }
        i64 w = 1;
        if (field) {
            const double s = (double)field[i] * 65536.0;      // exact: a power-of-two scale
            w = s >= 16777216.0 ? 16777216 : (s >= 1.0 ? (i64)s : 1);   // NaN fails both tests -> 1
        }
        cnt[r] += 1; W[r] += w; Sx[r] += w * dx; Sy[r] += w * dy;
    }
    auto floor_div = [](__int128 a, __int128 b) { return a >= 0 ? a / b : -((-a + b - 1) / b); };
    int32_t K = 0;
    for (size_t r = 0; r < n; ++r) {
        if (cnt[r] == 0 || cnt[r] < min_size) continue;
        if (K < cap) {
            const i64 xr = (i64)(r % Lx), yr = (i64)(r / Lx);
            const i64 fx = (i64)floor_div((__int128)256 * Sx[r], W[r]), fy = (i64)floor_div((__int128)256 * Sy[r], W[r]);
            sx[K] = (int32_t)((((256 * xr + 128 + fx) % Px) + Px) % Px);
            sy[K] = (int32_t)((((256 * yr + 128 + fy) % Py) + Py) % Py);
            double ux = (double)xr + 0.5 + (double)Sx[r] / (double)W[r];
            double uy = (double)yr + 0.5 + (double)Sy[r] / (double)W[r];
            if (ux < 0) ux += Lx; else if (ux >= Lx) ux -= Lx;
            if (uy < 0) uy += Ly; else if (uy >= Ly) uy -= Ly;
            cx[K] = ux; cy[K] = uy;
            size[K] = (int32_t)cnt[r];
            root[K] = (int32_t)r;
        }
        ++K;
    }
    return K;
}

// O6 on the general geometry.
void orc_match_g(int32_t Lx, int32_t Ly, int per_x, int per_y, const int32_t* px, const int32_t* py,
                 int32_t n_prev, const int32_t* nx, const int32_t* ny, int32_t n_now, int32_t radius_fp,
                 int32_t* p2n, int32_t* n2p) {
    const i64 Px = 256 * (i64)Lx, Py = 256 * (i64)Ly, r2 = (i64)radius_fp * radius_fp;
    auto d2 = [&](i64 ax, i64 ay, i64 bx, i64 by) {
        const i64 dx = axis_dist(ax, bx, Px, per_x), dy = axis_dist(ay, by, Py, per_y);
        return dx * dx + dy * dy;
    };
    std::vector<int32_t> bp(n_now, -1), bn(n_prev, -1);
    for (int32_t j = 0; j < n_now; ++j) {
        i64 best = INT64_MAX;
        for (int32_t i = 0; i < n_prev; ++i) {
            const i64 d = d2(nx[j], ny[j], px[i], py[i]);
            if (d < best) { best = d; bp[j] = i; }
        }
        if (best > r2) bp[j] = -1;
    }
    for (int32_t i = 0; i < n_prev; ++i) {
        i64 best = INT64_MAX;
        for (int32_t j = 0; j < n_now; ++j) {
            const i64 d = d2(px[i], py[i], nx[j], ny[j]);
            if (d < best) { best = d; bn[i] = j; }
        }
        if (best > r2) bn[i] = -1;
    }
    for (int32_t i = 0; i < n_prev; ++i) p2n[i] = (bn[i] >= 0 && bp[bn[i]] == i) ? bn[i] : -1;
    for (int32_t j = 0; j < n_now; ++j) n2p[j] = (bp[j] >= 0 && bn[bp[j]] == j) ? bp[j] : -1;
}

// Bubble-size histogram: hist[b] = number of bubbles with size in
// [b*bin_width, (b+1)*bin_width); the last bin also takes every larger bubble.
void orc_size_histogram(const int32_t* size, int32_t K, int32_t bin_width, int32_t n_bins, int64_t* hist) {
    for (int32_t b = 0; b < n_bins; ++b) hist[b] = 0;
    for (int32_t k = 0; k < K; ++k) {
        i64 b = size[k] / bin_width;
        if (b >= n_bins) b = n_bins - 1;
        if (b >= 0) hist[b] += 1;
    }
}

// Bulk / boundary edges: for every edge (i, j) of an ascending unique list over n
// vertices, the number of neighbours i and j share - "two: the edge is in the bulk; only one: on the
// boundary".  Keys with a label >= n take no part and get -1.
void orc_edge_commons(const u64* edges, i64 n_edges, int32_t n, int32_t* commons) {
    std::vector<std::set<int32_t>> row(n);
    for (i64 k = 0; k < n_edges; ++k) {
        const int32_t i = (int32_t)(edges[k] >> 32), j = (int32_t)(edges[k] & 0xffffffffu);
        if (i < n && j < n) { row[i].insert(j); row[j].insert(i); }
    }
    for (i64 k = 0; k < n_edges; ++k) {
        const int32_t i = (int32_t)(edges[k] >> 32), j = (int32_t)(edges[k] & 0xffffffffu);
        if (i >= n || j >= n) { commons[k] = -1; continue; }
        int32_t c = 0;
        for (int32_t v : row[i]) c += (int32_t)row[j].count(v);
        commons[k] = c;
    }
}

// O10 — bulk and boundary vertices of an event (§III.B.4): "two points connected by a boundary
// edge belong to the boundary" (a boundary edge: its end points share only one neighbour); a point is involved
// in a BULK event if it is "connected to, at least, three other active points", in a BOUNDARY event if it is
// "connected to, at least, one other active boundary point" - for each of the two triangulations.
// Inputs as O7 (two ascending unique lists in one index space, n vertices); active = O7's trigger.
// Outputs: boundary_prev[n], boundary_now[n] (0/1, for every vertex), vclass[n] = bit 0 bulk event in D_P,
// bit 1 boundary event in D_P, bit 2 bulk event in D_N, bit 3 boundary event in D_N; 0 for inactive vertices.
void orc_event_vertices(const u64* prev, i64 n_prev, const u64* now, i64 n_now, int32_t n,
                        int32_t* boundary_prev, int32_t* boundary_now, int32_t* vclass) {
    std::vector<std::set<int32_t>> row[2];
    row[0].resize(n); row[1].resize(n);
    const u64* lists[2] = {prev, now};
    const i64 counts[2] = {n_prev, n_now};
    for (int t = 0; t < 2; ++t)
        for (i64 k = 0; k < counts[t]; ++k) {
            const int32_t i = (int32_t)(lists[t][k] >> 32), j = (int32_t)(lists[t][k] & 0xffffffffu);
            if (i < n && j < n) { row[t][i].insert(j); row[t][j].insert(i); }
        }
    std::vector<char> active(n);
    for (int32_t v = 0; v < n; ++v) active[v] = row[0][v] != row[1][v];
    int32_t* boundary[2] = {boundary_prev, boundary_now};
    for (int t = 0; t < 2; ++t)
        for (int32_t v = 0; v < n; ++v) {
            boundary[t][v] = 0;
            for (int32_t u : row[t][v]) {
                int32_t shared = 0;
                for (int32_t w : row[t][v]) shared += (int32_t)row[t][u].count(w);
                if (shared == 1) boundary[t][v] = 1;
            }
        }
    for (int32_t v = 0; v < n; ++v) {
        vclass[v] = 0;
        if (!active[v]) continue;
        for (int t = 0; t < 2; ++t) {
            int32_t act = 0, bnd = 0;
            for (int32_t u : row[t][v]) { act += active[u]; bnd += active[u] && boundary[t][u]; }
            if (act >= 3) vclass[v] |= 1 << (2 * t);
            if (bnd >= 1) vclass[v] |= 2 << (2 * t);
        }
    }
}

int orc_num_threads(int threads) { return resolve_threads(threads); }

}  // extern "C"
