/* vor.h — C ABI of libvor: the data-parallel hot path of arXiv:1607.00908
 * ("GPU Based Detection of Topological Changes in Voronoi Diagrams"), re-designed for one
 * NVIDIA B200 (sm_100a).  "PAPER.md:n" cites a line of the paper text plus its section.
 *
 * Conventions
 *   L            lattice side: vor_create makes an L x L torus; vor_create_geom an Lx x Ly lattice whose axes
 *                are periodic or walled (then read Lx / Ly for L below).  P = 256*L is the period in
 *                fixed-point units (1 cell = 256 units).
 *   cell (x,y)   0 <= x,y < L, centre (256x+128, 256y+128), linear index y*L + x.
 *   sites        SoA int32 arrays sx[n], sy[n], each coordinate in [0, P).  Coordinates outside
 *                that range are undefined behaviour.
 *   labels       int32[L*L], row-major.
 *   edge key     (uint64)i << 32 | j with i < j (site indices); lists are ascending and unique.
 *   -1           background cell / unmatched component.
 *
 * Pointers named d_* are DEVICE memory owned by the caller (e.g. torch tensors); h_* are HOST
 * memory owned by the caller.  The library neither frees nor keeps them beyond the stream work it
 * enqueues, except where stated.  `stream` is a cudaStream_t passed as void* (NULL = default
 * stream).  All d_* entry points are asynchronous: they enqueue work and return; counts are
 * written to device scalars so that no call forces a host synchronisation.
 *
 * Every function returns a vor_status.  Nothing throws or aborts across this boundary.
 * Capacity overflows never write out of bounds: the kernels store the REQUIRED count in the
 * device scalar, write nothing beyond `cap`, and latch a sticky device-side flag that the next
 * vor_sync_status() reports as VOR_ECAPACITY.
 */
#ifndef VOR_H_
#define VOR_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct vor_ctx vor_ctx; /* opaque; owns all scratch memory (cell list, key buffers, sort and
                                   union-find temporaries, the e2e pipeline's device buffers) */

typedef enum {
    VOR_OK = 0,
    VOR_EINVAL = -1,    /* bad argument (null pointer, size out of range) */
    VOR_ECAPACITY = -2, /* an output or scratch buffer was too small (sticky, see above) */
    VOR_ECUDA = -3,     /* a CUDA runtime call failed; vor_last_error() has the text */
    VOR_ESTATE = -4,    /* call order violation (e.g. vor_label before vor_build_cells) */
    VOR_ELIMIT = -5     /* a size exceeds a fixed, compiled-in maximum (vor_diff_rows_static only) */
} vor_status;

/* Create a context for an L x L lattice (2 <= L <= 2^22) and at most max_sites sites
 * (1 <= max_sites < 2^31).  max_raw_keys sizes the scratch that receives the (partly
 * de-duplicated) edge keys before sorting; 0 selects a default (max(2^20, 16*max_sites), never
 * more than the hard worst case 2*L*L).  Allocates device memory on the CURRENT device;
 * every later call on the context must be made with that device current (VOR_ESTATE otherwise). */
int vor_create(vor_ctx** out, int32_t L, int32_t max_sites, int64_t max_raw_keys);
/* The paper's own geometry: an Lx x Ly lattice (§IV: 2048 x 1024),
 * each axis periodic (1) or closed by walls (0; beyond the domain boundary there are no
 * neighbours).  Cell (x, y) has linear index y*Lx + x; label and field images are Ly rows of Lx entries; site
 * coordinates lie in [0, 256 Lx) x [0, 256 Ly).  On a walled axis distances are plain differences and nothing
 * wraps, in every call on this context (labels, edges, bubbles, centres, matching).  vor_create(L) is
 * vor_create_geom(L, L, 1, 1).  2 <= Lx, Ly <= 2^22 (2^21 on a walled axis).  The labelling kernels treat a
 * walled axis as a window of a periodic lattice twice as long, where the minimum image is the plain distance. */
int vor_create_geom(vor_ctx** out, int32_t Lx, int32_t Ly, int32_t periodic_x, int32_t periodic_y,
                    int32_t max_sites, int64_t max_raw_keys);
int vor_destroy(vor_ctx* ctx);

/* Text of the last failure on this context (ctx-owned storage; never free it). */
const char* vor_last_error(const vor_ctx* ctx);

/* Synchronise `stream`, then return and clear the sticky device-side status. */
int vor_sync_status(vor_ctx* ctx, void* stream);

/* Number of CUDA kernels this context has launched so far (bench.py's gpu_launches). */
int64_t vor_launch_count(const vor_ctx* ctx);

/* Copy `bytes` bytes from device memory (e.g. a pointer returned by vor_frame_results /
 * field_frame_results) to the host buffer h_dst on `stream` and wait for the copy.  For callers
 * that hold only raw pointers; a torch caller copies its own tensors. */
int vor_download(vor_ctx* ctx, const void* d_src, void* h_dst, int64_t bytes, void* stream);

/* Diagnostics of the last call (synchronises the device; for tuning notes, never on the hot path):
 *   "label_unproven_quadrants"  8x8-cell quadrants the CTA labelling kernel handed to its second pass
 *   "edges_raw_keys"            CTA-distinct keys the emit kernel produced (before the rows de-duplicate)
 *   "edges_overflow_keys"       keys that did not fit their adjacency row
 * Unknown names -> VOR_EINVAL (negative). */
int64_t vor_stat(vor_ctx* ctx, const char* name);

/* Per-kernel timing for bench.py's roofline figures.  vor_profile_begin() arms the context: every
 * kernel the library launches afterwards (at most 256) is bracketed by CUDA events on its own stream.
 * vor_profile_end() disarms it, synchronises `stream`, and returns the number n of launches timed
 * (or a negative vor_status): ms[i] = duration of launch i, names = their kernel names separated by
 * '\n' (truncated to names_len bytes; n is reduced accordingly).  Launch order is preserved. */
int vor_profile_begin(vor_ctx* ctx);
int vor_profile_end(vor_ctx* ctx, void* stream, char* names, int32_t names_len, float* ms, int32_t cap);

/* Tuning knobs (integers).  Unknown names -> VOR_EINVAL.
 *   "bucket_occupancy_x100"  target sites per cell-list bucket * 100 (default 100)
 *   "row_slots"              adjacency-matrix slots used per site in vor_edges: 4, 8, 12 or 16
 *                            (default 16); pairs that do not fit take the sorted overflow path,
 *                            so the result never depends on it
 *   "sites_hint"             expected number of bubbles for field_frame_device (0 = max_sites)
 *   "label_path" (0 auto, 1 general ring search, 2 warp-per-tile, 3 CTA), "label_halo_x100",
 *   "label_fast_off", "edges_generic"   kernel selection for the parity tests; results never depend
 *                            on them */
int vor_set_option(vor_ctx* ctx, const char* name, int64_t value);

/* ---- a1: counting-sort cell list of the sites (not in the paper, which loops over all centres,
 * PAPER.md:131 §III.B.1; named by BASELINE.json north_star).  Reads d_sx/d_sy[n_sites]; the
 * context keeps its own bucket-ordered copy, so the caller may overwrite the inputs once the
 * stream work has run. */
int vor_build_cells(vor_ctx* ctx, const int32_t* d_sx, const int32_t* d_sy, int32_t n_sites,
                    void* stream);

/* Same with the number of sites in a DEVICE scalar (e.g. the bubble count field_centroids just wrote),
 * so that a field-driven frame needs no host synchronisation.  Reads min(*d_n_sites, cap) sites;
 * 1 <= cap <= max_sites.  n_hint (1..cap, else cap) is the expected number: it only sizes the buckets
 * and selects kernels, results never depend on it.  Labels produced afterwards are < cap; zero sites
 * give the label -1 everywhere.  *d_n_sites must stay valid until vor_label has run. */
int vor_build_cells_dev(vor_ctx* ctx, const int32_t* d_sx, const int32_t* d_sy, const int32_t* d_n_sites,
                        int32_t cap, int32_t n_hint, void* stream);

/* ---- a2: digital Voronoi colouring (§II region definition; PAPER.md:129-131
 * §III.B.1 "coloring itself with the label of the nearest center of mass", squared distance).
 * labels[y*L+x] = argmin_i (minimum-image squared distance from the cell centre to site i, i),
 * exact integer arithmetic, ties to the smallest index.  Uses the cell list of the last
 * vor_build_cells on this context (none -> VOR_ESTATE).  Writes d_labels[L*L]. */
int vor_label(vor_ctx* ctx, int32_t* d_labels, void* stream);
/* The same for the strip of rows [y0, y0 + n_rows) of the lattice only (y0 + n_rows <= Ly): writes n_rows * Lx
 * labels.  One rank of a row-strip decomposition labels its rows plus the first row of the next strip
 * (PAPER.md:304 multi-GPU as future work) - no halo exchange. */
int vor_label_rows(vor_ctx* ctx, int32_t y0, int32_t n_rows, int32_t* d_labels, void* stream);
/* Obstacles (§III.B.1): sites where d_mask[i] != 0 take the fixed colour `colour` (the paper's
 * MAXLINK, any value >= the number of sites) instead of a label; d_mask and d_labels hold n_rows * Lx entries.
 * Pass the same colour as `exclude` to vor_edges_image: such sites take part in no edge. */
int vor_paint_obstacles(vor_ctx* ctx, const uint8_t* d_mask, int32_t colour, int32_t* d_labels, int32_t n_rows,
                        void* stream);

/* ---- a3+a4: site adjacency (digital Delaunay edge set; PAPER.md:121 adjacency matrix,
 * PAPER.md:207 compress by sort+unique).  Rule (R6): every 4-connected label
 * discontinuity, including across the periodic wrap, contributes the pair (min,max).
 * Reads d_labels[L*L] (any int32 >= 0; values below the n_sites of the last vor_build_cells - or
 * below max_sites if there was none - take the fast adjacency-row path, larger ones the sorted
 * overflow path); writes the ascending unique keys to d_edges[0..min(E,cap)) and E to *d_n_edges. */
int vor_edges(vor_ctx* ctx, const int32_t* d_labels, uint64_t* d_edges, int64_t cap,
              int64_t* d_n_edges, void* stream);
/* Same, and also the offset of every site's row in the list: the keys (a, b), b > a, of site a are
 * d_edges[d_row_ptr[a] .. d_row_ptr[a+1]) - the paper's adjacency matrix in compressed form
 * (PAPER.md:207, 215).  d_row_ptr has n_rows + 1 entries, n_rows = n_sites of the last vor_build_cells
 * (max_sites if there was none); keys whose smaller label is >= n_rows follow after d_row_ptr[n_rows].
 * Offsets are clamped to cap; cap must be < 2^32.  d_row_ptr may be NULL (= vor_edges). */
int vor_edges_rows(vor_ctx* ctx, const int32_t* d_labels, uint64_t* d_edges, int64_t cap,
                   int64_t* d_n_edges, uint32_t* d_row_ptr, void* stream);

/* General form of vor_edges_rows.  The image has n_rows rows of Lx labels: the whole domain (n_rows = Ly,
 * wrap_y = the context's periodicity in y) or a strip of consecutive rows (wrap_y = 0: nothing is adjacent
 * across its first and last row; the last row of a strip is the first row of the next one, so that the union
 * of the strips' lists is the lattice's list).  The x axis wraps as the context says.  exclude >= 0: pairs
 * with that label on either side are not edges (obstacle colour); -1: none.  d_row_ptr may be NULL. */
int vor_edges_image(vor_ctx* ctx, const int32_t* d_labels, int32_t n_rows, int32_t wrap_y, int32_t exclude,
                    uint64_t* d_edges, int64_t cap, int64_t* d_n_edges, uint32_t* d_row_ptr, void* stream);

/* Union of n_lists ASCENDING key lists (row strips of one lattice, one per rank, brought together by an
 * all-gather): list l occupies d_lists[l * stride .. l * stride + min(d_counts[l], stride)); the ascending
 * unique union goes to d_out[0..min(E, cap)), E to *d_n_out.  Labels are < n_labels.  stride * n_lists must not
 * exceed the context's max_raw_keys. */
int vor_merge_lists(vor_ctx* ctx, const uint64_t* d_lists, int64_t stride, const int64_t* d_counts,
                    int32_t n_lists, int32_t n_labels, uint64_t* d_out, int64_t cap, int64_t* d_n_out, void* stream);

/* ---- a5: frame-to-frame comparison (§III.B.3 translation + comparison;
 * PAPER.md:223 appearing/disappearing bubbles excluded; §III.B.4 "breaking" = in
 * D_P only, "arising" = in D_N only).  d_prev/d_now are ascending unique key lists with device
 * counts; cap_prev / cap_now are the capacities of the two buffers and a count above its capacity
 * (an upstream overflow, already latched in the sticky status) is clamped to it, so a chained call
 * never reads out of bounds.  d_p2n[i] (prev label -> now label or -1) and d_n2p (now -> prev or -1) may both be
 * NULL: persistent identity.  With maps: prev edges are translated, dropped if an endpoint is -1
 * or both endpoints collapse, re-sorted and uniqued; now edges with an unmatched endpoint are
 * dropped.  created = now \ prev, destroyed = prev \ now, ascending, in NOW index space.
 * n_prev_labels / n_now_labels bound the label values (needed only with maps; pass 0 otherwise). */
int vor_diff(vor_ctx* ctx, const uint64_t* d_prev, const int64_t* d_n_prev,
             const uint64_t* d_now, const int64_t* d_n_now, int64_t cap_prev, int64_t cap_now,
             const int32_t* d_p2n, const int32_t* d_n2p, int32_t n_prev_labels, int32_t n_now_labels,
             uint64_t* d_created, uint64_t* d_destroyed, int64_t cap,
             int64_t* d_n_created, int64_t* d_n_destroyed, void* stream);
/* The same comparison the way the paper does it ("each thread accesses a given row of
 * (E_P)_PN and its isomorphic one in (E_N)_NN"): persistent identity, both lists with the row offsets
 * vor_edges_rows returned for the SAME n_rows; keys beyond d_*_row_ptr[n_rows] are not compared.
 * No searching and no count arguments: the offsets delimit everything that is read. */
int vor_diff_rows(vor_ctx* ctx, const uint64_t* d_prev, const uint32_t* d_prev_row_ptr,
                  const uint64_t* d_now, const uint32_t* d_now_row_ptr, int32_t n_rows,
                  uint64_t* d_created, uint64_t* d_destroyed, int64_t cap,
                  int64_t* d_n_created, int64_t* d_n_destroyed, void* stream);

/* ---- a5 for callers that must not allocate.
 * Who needs this: code that runs where a device allocation is forbidden or impossible - inside a host framework
 * whose memory pool owns the whole GPU and hands out only the buffers it was asked for up front, in a
 * process that fixed its memory budget at start-up, or on a latency path where cudaMalloc's implicit device-wide
 * synchronisation is not acceptable.  Every other call of this library needs a vor_ctx, and vor_create (plus
 * a few lazily sized buffers, vor_diff_rows' among them) calls cudaMalloc.  This call takes NO context and
 * never calls cudaMalloc, cudaFree or any routine that allocates: the comparison's working memory (one mask
 * word per row and two counters per block of 512 rows) is a fixed array that is part of the library image.
 *
 * The result is exactly vor_diff_rows': created = now \ prev, destroyed = prev \ now, ascending; the counts
 * hold the REQUIRED numbers and nothing is written past `cap`.  There is no context to latch an overflow in:
 * compare *d_n_created / *d_n_destroyed with cap yourself.  All pointers are device memory owned by the
 * caller; the call enqueues two kernels on `stream` and returns.
 *
 * Limit: n_rows <= VOR_DIFF_ROWS_STATIC_MAX_ROWS (2^20 rows; the array costs 4.02 MiB of device memory on
 * every GPU that loads libvor, from load until the process exits).  A larger n_rows returns VOR_ELIMIT and
 * does nothing; a null pointer, cap < 0 or n_rows < 1 returns VOR_EINVAL.
 *
 * First call on each device: the library looks up the array's device address (cudaGetSymbolAddress, with the
 * caller's current device - keep the device whose memory you pass current).  Make that first call during
 * set-up, before you start any stream capture on that device.  Later calls only launch.
 *
 * The array is shared by every call in the process on that device and keeps whatever the last call left in
 * it.  Nothing in it has to start at zero: each call overwrites every word it later reads.  For the same
 * reason two calls whose kernels can run at the same time on one GPU (different streams, different threads)
 * corrupt each other: issue them on one stream, or order them with events. */
#define VOR_DIFF_ROWS_STATIC_MAX_ROWS (1 << 20)
int vor_diff_rows_static(const uint64_t* d_prev, const uint32_t* d_prev_row_ptr,
                         const uint64_t* d_now, const uint32_t* d_now_row_ptr, int32_t n_rows,
                         uint64_t* d_created, uint64_t* d_destroyed, int64_t cap,
                         int64_t* d_n_created, int64_t* d_n_destroyed, void* stream);

/* ---- trigger and event counts: the paper's own outputs on top of the diff (PAPER.md:215-221
 * §III.B.3 local_trigger / global_trigger; §III.B.4 eventsIndices / eventsNumber;
 * PAPER.md:236 eventsCount for both triangulations).  All four lists are ascending unique key lists
 * in ONE index space with labels < n_labels (site path: as given to / returned by vor_diff; keys
 * with a label >= n_labels are ignored).  d_created / d_destroyed must be the diff of d_prev / d_now.
 * cap_*: capacities of the four list buffers; device counts above them are clamped (see vor_diff).
 * Outputs, device memory owned by the caller:
 *   d_trigger[n_labels]         1 if the vertex's adjacency row changed (endpoint of a created or
 *                               destroyed edge), else 0
 *   d_events_indices[n_labels]  the active vertices in ascending order (first *d_events_number entries)
 *   d_events_number, d_global_trigger   device scalars (global_trigger = events_number > 0)
 *   d_count_prev / d_count_now[n_labels]  for an active vertex: number of active vertices adjacent to
 *                               it in the past / present edge list; 0 for inactive vertices. */
int vor_events(vor_ctx* ctx, const uint64_t* d_prev, const int64_t* d_n_prev,
               const uint64_t* d_now, const int64_t* d_n_now, int64_t cap_prev, int64_t cap_now,
               const uint64_t* d_created, const int64_t* d_n_created,
               const uint64_t* d_destroyed, const int64_t* d_n_destroyed, int64_t cap_created,
               int64_t cap_destroyed, int32_t n_labels,
               int32_t* d_trigger, int32_t* d_events_indices, int32_t* d_events_number,
               int32_t* d_global_trigger, int32_t* d_count_prev, int32_t* d_count_now, void* stream);

/* ---- couples of active vertices and T1 pairing: the paper's final output (§III.B.4: the
 * active points that are connected are stored as couples, a permutation of a couple is the same couple, a
 * couple connected in only one configuration is "breaking" (D_P only) or "arising" (D_N only);
 * an edge whose end points share two neighbours lies in the bulk, one: on the boundary;
 * PAPER.md:238 and Fig. 8: a T1 event replaces the breaking link by the arising link between its two common
 * neighbours).  Lists, counts and capacities as for vor_events; d_trigger[n_labels] as vor_events wrote it.
 * A couple is a pair i < j of active vertices connected in the past or the present list.  Outputs (device,
 * caller-owned, capacity `cap` each), one entry per couple in ascending key order, *d_n_couples of them
 * (the REQUIRED number; more than cap latches VOR_ECAPACITY and nothing is written past cap):
 *   d_couples      packed key
 *   d_class        0 connected in both, 1 breaking, 2 arising
 *   d_common_prev  number of common neighbours of i and j in the past list, -1 if not connected there
 *   d_common_now   the same in the present list
 *   d_partner      breaking couple with exactly two common neighbours c < d in the past list whose pair
 *                  (c, d) is arising: that key - {i, j, c, d} is the T1 quadruple; arising couple: the mirror
 *                  statement in the present list with a breaking pair; otherwise ~0.
 * The context builds both adjacency matrices in compressed symmetric form (sorted rows) in
 * its own scratch, sized on the first call from the capacities; cap_prev + cap_now must be < 2^31. */
int vor_t1_events(vor_ctx* ctx, const uint64_t* d_prev, const int64_t* d_n_prev,
                  const uint64_t* d_now, const int64_t* d_n_now, int64_t cap_prev, int64_t cap_now,
                  const uint64_t* d_created, const int64_t* d_n_created,
                  const uint64_t* d_destroyed, const int64_t* d_n_destroyed, int64_t cap_created,
                  int64_t cap_destroyed, const int32_t* d_trigger, int32_t n_labels,
                  uint64_t* d_couples, int32_t* d_class, int32_t* d_common_prev, int32_t* d_common_now,
                  uint64_t* d_partner, int64_t cap, int64_t* d_n_couples, void* stream);

/* ---- bulk and boundary edges (§III.B.4: "if two connected points share two neighbours,
 * then the edge is in the bulk; if two connected points share only one neighbour, then the edge is on the
 * boundary").  d_commons[k] = number of neighbours the two end points of edge k share in the ascending unique
 * list d_edges (device count clamped to cap_edges < 2^31; labels < n_labels, keys with a larger label get -1).
 * On a torus every edge of a triangulation is a bulk edge; walls and obstacles create boundary edges. */
int vor_edge_commons(vor_ctx* ctx, const uint64_t* d_edges, const int64_t* d_n_edges, int64_t cap_edges,
                     int32_t n_labels, int32_t* d_commons, void* stream);

/* Bulk and boundary vertices of an event (§III.B.4): "two points connected by a boundary edge
 * belong to the boundary"; an active point takes part in a BULK event if it is "connected to, at least, three
 * other active points", in a BOUNDARY event if it is "connected to, at least, one other active boundary point" -
 * evaluated in each of the two triangulations.  Lists, counts, capacities and d_trigger as for vor_t1_events.
 * Outputs (device, n_labels entries each): d_boundary_prev / d_boundary_now 1 for a boundary vertex of the past /
 * present triangulation, else 0; d_vclass bit 0 bulk event in D_P, bit 1 boundary event in D_P, bit 2 bulk
 * event in D_N, bit 3 boundary event in D_N, 0 for inactive vertices. */
int vor_event_vertices(vor_ctx* ctx, const uint64_t* d_prev, const int64_t* d_n_prev,
                       const uint64_t* d_now, const int64_t* d_n_now, int64_t cap_prev, int64_t cap_now,
                       const int32_t* d_trigger, int32_t n_labels, int32_t* d_boundary_prev,
                       int32_t* d_boundary_now, int32_t* d_vclass, void* stream);

/* ---- a6: bubble identification (§III.A: threshold -> two-valued variable ->
 * cluster labelling).  mask = above ? field > thr : field < thr (strict; NaN -> background).
 * 4-connected periodic components; d_ccl[c] = smallest linear index in c's component, or -1. */
int field_threshold_ccl(vor_ctx* ctx, const float* d_field, float thr, int above,
                        int32_t* d_ccl, void* stream);
/* The same with connectivity 4 (above) or 8: cells touching at a corner belong to one bubble - "moving along
 * the directions of the Lattice Boltzmann model" (D2Q9). */
int field_threshold_ccl_conn(vor_ctx* ctx, const float* d_field, float thr, int above, int32_t connectivity,
                             int32_t* d_ccl, void* stream);

/* ---- a7: bubble sizes and centres of mass (§III.A: count the lattice points
 * of each bubble; sum the coordinates and divide by the size).  Unweighted, periodic unwrap
 * relative to the root cell, integer sums; components smaller than min_size are dropped; the K
 * survivors are ordered by ascending root.  Outputs (each capacity `cap`): centroid in lattice
 * units (float64, in [0,L)), fixed-point site coordinates (floor), size, root; K to *d_n_comp. */
int field_centroids(vor_ctx* ctx, const int32_t* d_ccl, int32_t min_size,
                    double* d_cx, double* d_cy, int32_t* d_sx, int32_t* d_sy,
                    int32_t* d_size, int32_t* d_root, int32_t cap, int32_t* d_n_comp, void* stream);

/* Density-weighted centres of mass (§II: z* = sum(y rho) / sum(rho)).  d_field[Lx*Ly] is the
 * density; the weight of a cell is the fixed-point value floor(rho * 65536) limited to [1, 2^24] (NaN -> 1), so
 * that the sums stay integers and the result does not depend on the order of the atomic additions.  size is
 * still the number of cells (min_size applies to it); d_field == NULL is field_centroids. */
int field_centroids_weighted(vor_ctx* ctx, const int32_t* d_ccl, const float* d_field, int32_t min_size,
                             double* d_cx, double* d_cy, int32_t* d_sx, int32_t* d_sy,
                             int32_t* d_size, int32_t* d_root, int32_t cap, int32_t* d_n_comp, void* stream);
/* Bubble-size histogram ("characterize them according to their size"):
 * d_hist[b] = number of bubbles among the first min(*d_n_comp, cap) entries of d_size whose size lies in
 * [b * bin_width, (b + 1) * bin_width); the last of the n_bins bins also takes every larger bubble. */
int field_size_histogram(vor_ctx* ctx, const int32_t* d_size, const int32_t* d_n_comp, int32_t cap,
                         int32_t bin_width, int32_t n_bins, int64_t* d_hist, void* stream);

/* ---- a8: isomorphism Phi P->N "by simply comparing the two sets of centers of mass"
 * (§III.B.3); unmatched = appeared / disappeared.  Mutual nearest
 * neighbour under the minimum-image metric on fixed-point coordinates, squared distance
 * <= radius_fp^2, ties to the smallest index.  Counts are device scalars (int32) so the call
 * chains after field_centroids without a host sync; cap_* bound the array lengths. */
int match_sites(vor_ctx* ctx, const int32_t* d_px, const int32_t* d_py, const int32_t* d_n_prev,
                const int32_t* d_nx, const int32_t* d_ny, const int32_t* d_n_now,
                int32_t cap_prev, int32_t cap_now, int32_t radius_fp,
                int32_t* d_p2n, int32_t* d_n2p, void* stream);

/* ---- end-to-end, HOST buffers (bench.py's e2e leg): one site-driven frame.
 * Copies h_sx/h_sy[n_sites] to the device, runs a1..a5 against the edge list kept from the
 * previous call on this context (the first call diffs against an empty list), copies the
 * created/destroyed lists (at most cap each) and h_counts[3] = {n_edges, n_created, n_destroyed}
 * back, and synchronises.  The label image stays on the device (not copying it is
 * the point of the method); vor_frame_results() exposes it. */
int vor_frame_host(vor_ctx* ctx, const int32_t* h_sx, const int32_t* h_sy, int32_t n_sites,
                   uint64_t* h_created, uint64_t* h_destroyed, int64_t cap, int64_t* h_counts,
                   void* stream);
/* Pipelined form of vor_frame_host for a stream of frames: vor_frame_submit() enqueues the upload
 * (on a copy stream of the context), a1..a5 (on `stream`) and the download of the counts, and
 * returns without waiting; vor_frame_collect() waits for the OLDEST frame in flight, downloads its
 * created / destroyed lists (on a second copy stream) and returns them like vor_frame_host.  At most
 * two frames may be in flight (a third submit -> VOR_ESTATE), so submit(k+1) before collect(k)
 * overlaps frame k's downloads and frame k+1's upload with the kernels.  Page-locked caller buffers
 * are used directly; the input arrays of a submitted frame must stay unchanged until it is
 * collected.  Frames are diffed in submission order; vor_frame_reset() drops frames in flight. */
int vor_frame_submit(vor_ctx* ctx, const int32_t* h_sx, const int32_t* h_sy, int32_t n_sites, void* stream);
int vor_frame_collect(vor_ctx* ctx, uint64_t* h_created, uint64_t* h_destroyed, int64_t cap,
                      int64_t* h_counts);
/* Same pipeline with DEVICE site arrays and no host copies or synchronisation: results stay in
 * context-owned device buffers (vor_frame_results).  bench.py's device-resident leg. */
int vor_frame_device(vor_ctx* ctx, const int32_t* d_sx, const int32_t* d_sy, int32_t n_sites,
                     void* stream);
/* Variants of the frame calls (vor_frame_* and field_frame_*), kept until changed: bubbles 4- or 8-connected
 * (field_threshold_ccl_conn), density-weighted centres (field_centroids_weighted with the frame's field), and an
 * obstacle mask d_obstacles[Lx*Ly] (device memory that must stay valid; NULL = none) whose sites take
 * obstacle_colour after labelling and take part in no edge (vor_paint_obstacles, vor_edges_image) - together with
 * walled axes (vor_create_geom) the paper's own set-up: a confined channel with posts. */
int vor_frame_options(vor_ctx* ctx, int32_t connectivity, int32_t weighted, const uint8_t* d_obstacles,
                      int32_t obstacle_colour);
/* Forget the previous frame's edge list (start a new sequence). */
int vor_frame_reset(vor_ctx* ctx);
/* Device pointers to the context-owned results of the last vor_frame_* call:
 * labels int32[L*L]; edges / created / destroyed uint64 lists; counts int64[3] (device). */
int vor_frame_results(vor_ctx* ctx, const int32_t** d_labels, const uint64_t** d_edges,
                      const uint64_t** d_created, const uint64_t** d_destroyed,
                      const int64_t** d_counts);

/* ---- end-to-end, field-driven frames (PAPER.md:93-101 bubbles and centres of mass; PAPER.md:211-223
 * the trigger: isomorphism, translation, comparison): a6 -> a7 -> a8 -> a1 -> a2 -> a3/a4 -> a5 with the
 * maps, all enqueued on `stream` without a host synchronisation.  Bubbles are the sites (at most the
 * context's max_sites; more latch VOR_ECAPACITY); matching radius in fixed-point units.  The first frame
 * of a sequence has nothing to compare with: created = destroyed = empty.  Same pipeline rules as
 * vor_frame_submit / vor_frame_collect (two frames in flight, results in submission order); do not mix
 * site and field frames on one context.  h_counts[4] = {n_bubbles, n_edges, n_created, n_destroyed};
 * lists in NOW index space.  vor_frame_reset() starts a new sequence. */
int field_frame_device(vor_ctx* ctx, const float* d_field, float thr, int above, int32_t min_size,
                       int32_t radius_fp, void* stream);
int field_frame_submit(vor_ctx* ctx, const float* h_field, float thr, int above, int32_t min_size,
                       int32_t radius_fp, void* stream);
int field_frame_collect(vor_ctx* ctx, uint64_t* h_created, uint64_t* h_destroyed, int64_t cap,
                        int64_t* h_counts);
/* Device pointers to the context-owned results of the last field_frame_device / field_frame_submit:
 * bubble image, Voronoi labels, per-bubble arrays (first counts[0] entries), the maps P->N and N->P
 * (max_sites entries each), edges, created, destroyed, counts int64[4] (device; field_frame_device only).
 * Any out-pointer may be NULL. */
int field_frame_results(vor_ctx* ctx, const int32_t** d_ccl, const int32_t** d_labels,
                        const double** d_cx, const double** d_cy, const int32_t** d_sx,
                        const int32_t** d_sy, const int32_t** d_size, const int32_t** d_root,
                        const int32_t** d_p2n, const int32_t** d_n2p, const uint64_t** d_edges,
                        const uint64_t** d_created, const uint64_t** d_destroyed,
                        const int64_t** d_counts);

#ifdef __cplusplus
}
#endif
#endif /* VOR_H_ */
