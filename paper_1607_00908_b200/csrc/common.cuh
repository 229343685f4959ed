// Shared declarations of libvor's translation units (context layout, launch helpers).
// Product code: never includes or links anything from oracle/.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>
#include <string.h>

#include "../../include/vor.h"

#define FP_ONE 256
#define FP_HALF 128

constexpr int kNumSMs = 148;               // B200: 2 dies x 74 SMs (grid sizing of the streaming kernels)
constexpr int kSortThreads = 1024;         // block size of the persistent cooperative kernels
constexpr int kMaxCoopBlocks = 1024;       // allocation bound for per-block scratch of those kernels
constexpr int kRowStride = 16;             // adjacency-row slots per site (64-byte rows)
constexpr uint32_t kEmptySlot = 0xffffffffu;
constexpr int kMatchGrid = 512;            // match_sites: buckets per side (at most), kMatchSlots sites per bucket
constexpr int kMatchSlots = 4;
constexpr int kMaxProfLaunches = 256;      // launches timed per vor_profile_begin/end bracket

// error flag bits latched on the device (ctx->d_flags[0])
enum : int {
    FLAG_RAWKEY_OVERFLOW = 1,
    FLAG_EDGE_CAP = 2,
    FLAG_DIFF_CAP = 4,
    FLAG_COMP_CAP = 8,
    FLAG_MATCH_CAP = 16,
};

struct vor_ctx {
    int32_t Lx, Ly;            // the domain: label / field images are Ly rows of Lx cells
    int32_t per_x, per_y;      // 1 = periodic axis, 0 = closed by walls
    // the LABELLING lattice: the domain itself on a periodic axis, twice the domain on a walled axis (inside
    // the domain the minimum image on the doubled period is the plain distance, so the periodic kernels label
    // a walled domain as a window of it); the cell list covers this lattice
    int32_t FLx, FLy;
    int64_t Px, Py;            // 256 * FLx, 256 * FLy
    int32_t max_sites;
    int64_t max_raw_keys;
    int device;

    // options
    int64_t bucket_occ_x100;
    int64_t label_path;            // 0 auto, 1 general, 2 tile 8x8, 3 CTA
    int64_t label_halo_x100;       // fast-path halo = r_quad + this/100 * mean site spacing
    int64_t label_fast_off;        // 1 = skip the quadrant fast path (testing)

    // ---- cell list (a1)
    int64_t nbuckets_max;      // allocation bound for nbx * nby
    int64_t w_min, w_gcd;      // smallest admissible bucket width; gcd(Px, Py) (every width divides it)
    int32_t nbx, nby;          // buckets per axis of the last build (0 = none)
    int32_t w;                 // bucket width in fixed-point units, w * nbx == Px, w * nby == Py
    int32_t n_sites;           // of the last build (vor_build_cells_dev: the upper bound `cap`)
    int32_t n_hint;            // expected number of sites (kernel selection, bucket and halo sizes only)
    const int32_t* d_n_dev;    // vor_build_cells_dev: the exact number lives on the device; else NULL
    int32_t* d_bucket_start;   // [nbuckets_max + 1]
    int32_t* d_bucket_fill;    // [nbuckets_max]  (scatter cursors)
    int4* d_sorted;            // [max_sites]  (x, y, original index, bucket)
    int32_t* d_scan_part;      // scratch for device scans

    int2* d_lab_fail;          // CTA label path: quadrants whose bound was not proven (x0, y0), lazily sized
    int32_t* d_lab_fail_n;     // their number: two device scalars used alternately (the fix-up kernel of one
                               //   call zeroes the other call's counter, so no memset is needed)
    int32_t lab_fail_cap;
    int lab_fail_turn;

    // ---- edges (a3/a4)
    uint32_t* d_rows;          // [max_sites * kRowStride] per-site lists of larger-index neighbours
    uint32_t* d_row_cnt;       // [max_sites] entries appended to each row; all 0 between calls (the
                               //   finish kernel restores that), so stale row contents are never read
    int64_t row_slots;         // slots used per row (option; 4..kRowStride, multiple of 4)
    int64_t edges_generic;     // 1 = force the generic emit kernel (testing)
    uint64_t* d_keys_a;        // [max_raw_keys]  overflow keys / sort ping
    uint64_t* d_keys_b;        // [max_raw_keys]  sort pong
    int64_t* d_n_raw;          // device control block [8]: 0 = raw/overflow key count, 1 = filtered
                               //   overflow count, 2 = OR of the overflow keys, 3 = raw key count, 4 = dirty tiles (fused path)
    uint32_t* d_hist;          // [kMaxCoopBlocks * 256] per-block digit histograms
    int64_t* d_blk_count;      // [2 * kMaxCoopBlocks] per-block counts for compactions

    // ---- fused label -> edge path (vor_frame_*): compact border columns of the 32-cell tile columns
    int32_t* d_fu_cols;        // [2][Lx / 32][Ly]: left, then right border column of every tile column
    int32_t* d_fu_dirty;       // [(Lx / 32) * (Ly / 32)] tiles whose pairs the labelling kernel could not extract itself
    int64_t fuse;              // option: 1 = vor_frame_* labels and extracts the pairs in one kernel

    // ---- row-by-row diff: membership mask per row [dr_rows], then the per-block counts
    uint32_t* d_dr_scratch;
    int64_t dr_rows;

    // ---- vor_t1_events: degrees, offsets, unsorted and sorted adjacency lists, union list (lazily sized)
    void* d_t1[5];
    size_t t1_bytes[5];

    // ---- diff with maps: translated / filtered lists
    uint64_t* d_tr_prev;       // lazily sized to max_raw_keys
    uint64_t* d_tr_now;
    uint32_t* d_tr_rowptr[2];  // [max_sites + 1] row offsets of the two lists (rows path)
    int64_t* d_tr_counts;      // [4]

    // ---- field path (a6..a8)
    int32_t* d_rank;           // [Lx*Ly] root -> component rank
    int64_t* d_acc;            // [3 * max_comp] n, Sx, Sy
    int32_t* d_comp_root;      // [max_comp]
    int32_t* d_comp_wcount;    // per-warp counts of the compactions
    int32_t max_comp;
    int32_t* d_comp_count;     // device scalars [4]
    int32_t* d_best;           // [best_cap] best partner per prev / now (lazily sized)
    int64_t best_cap;
    int32_t* d_mgrid;          // match grid: [2][kMatchGrid^2] counts, then [2][kMatchGrid^2 * kMatchSlots] site ids

    // ---- frame pipeline (e2e)
    int32_t* d_fr_sx;
    int32_t* d_fr_sy;
    int32_t* d_fr_labels;      // [Lx*Ly]
    uint64_t* d_fr_edges[2];   // ping-pong prev / now
    int64_t* d_fr_nedges[2];
    uint32_t* d_fr_rowptr[2];  // [max_sites + 1] row offsets of the two lists (vor_edges_rows)
    int32_t fr_prev_sites;     // number of sites of the previous frame
    uint64_t* d_fr_created;
    uint64_t* d_fr_destroyed;
    int64_t* d_fr_counts;      // [3]
    int64_t* h_fr_counts;      // pinned [3]
    int32_t* h_fr_sites;       // pinned [2 * max_sites]
    uint64_t* h_fr_lists;      // pinned [2 * fr_cap]
    int64_t fr_cap;
    int fr_cur;                // index of the "now" buffer of the last frame; -1 = none
    int fr_have_prev;
    // field-driven frames (field_frame_*): bubble image, two generations of bubble arrays, the isomorphism
    int32_t* d_ff_ccl;         // [Lx*Ly]
    double* d_ff_cxy[2];       // [2 * max_sites] cx, cy
    int32_t* d_ff_comp[2];     // [4 * max_sites + 4] sx, sy, size, root, then the device count
    int32_t* d_ff_maps;        // [2 * max_sites] p2n, n2p
    int64_t* d_ff_tmpcount;    // [2] created / destroyed counts before they are gathered
    float* d_ff_field[2];      // device copies of submitted host fields (lazily)
    int ff_cur;                // generation of the last field frame; -1 = none
    // vor_frame_options: variants of the frame calls
    int32_t fo_connectivity;   // bubbles: 4 (default, also when 0) or 8
    int32_t fo_weighted;       // density-weighted centres
    const uint8_t* d_fo_mask;  // obstacle sites (caller-owned, may be NULL)
    int32_t fo_colour;
    int32_t ff_hint;           // bubbles in an earlier frame (sizes the next cell list)
    int32_t* h_ff_count;       // pinned [1]: bubble count of the latest frame whose kernels have finished
    // pipelined variant (vor_frame_submit / vor_frame_collect): two frames in flight, copies on own streams
    int32_t* d_pp_sx[2];
    int32_t* d_pp_sy[2];
    uint64_t* d_pp_created[2];
    uint64_t* d_pp_destroyed[2];
    int64_t* d_pp_counts[2];   // [4]: n_edges, n_created, n_destroyed, sticky flags
    int64_t* h_pp_counts[2];   // pinned [4]
    int32_t* h_pp_sites[2];    // pinned staging [2 * max_sites] for pageable inputs
    cudaStream_t pp_h2d, pp_d2h, pp_lst;   // uploads; counts (waits for the kernels); list downloads
    cudaEvent_t pp_ev_in[2], pp_ev_done[2], pp_ev_cnt[2];
    int64_t pp_head, pp_tail;  // frames submitted / collected

    int32_t* d_flags;          // [1] sticky error bits
    int num_sms;               // of the device the context lives on
    int coop_blocks[8];        // cached grid sizes of the cooperative kernels (0 = not yet queried)
    int64_t launches;
    // per-launch timing (vor_profile_begin / vor_profile_end): events around every kernel launch
    int prof_on;
    int prof_n;
    cudaEvent_t prof_ev[kMaxProfLaunches][2];
    const char* prof_name[kMaxProfLaunches];
    char err[512];
};

inline void vor_prof_mark(vor_ctx* ctx, int which, const char* name, cudaStream_t stream) {
    if (!ctx->prof_on || ctx->prof_n >= kMaxProfLaunches) return;
    cudaEventRecord(ctx->prof_ev[ctx->prof_n][which], stream);
    if (which == 1) ctx->prof_name[ctx->prof_n++] = name;
}

inline int vor_fail(vor_ctx* ctx, int code, const char* what) {
    if (ctx) snprintf(ctx->err, sizeof(ctx->err), "%s", what);
    return code;
}

inline int vor_cuda_fail(vor_ctx* ctx, cudaError_t e, const char* where) {
    if (ctx) snprintf(ctx->err, sizeof(ctx->err), "%s: %s", where, cudaGetErrorString(e));
    return VOR_ECUDA;
}

// Every entry point that enqueues work or allocates lazily runs on the device the context was created on.
inline int vor_check_device(vor_ctx* ctx) {
    int d = -1;
    if (cudaGetDevice(&d) != cudaSuccess || d != ctx->device)
        return vor_fail(ctx, VOR_ESTATE, "the current CUDA device is not the one this context was created on");
    return VOR_OK;
}

#define VOR_CUDA(call)                                                          \
    do {                                                                        \
        cudaError_t e_ = (call);                                                \
        if (e_ != cudaSuccess) return vor_cuda_fail(ctx, e_, #call);            \
    } while (0)

// Grid size for a cooperative (grid-synchronising) kernel: every block must be co-resident.
inline int vor_coop_grid(vor_ctx* ctx, int slot, const void* func, int threads, int max_per_sm) {
    if (ctx->coop_blocks[slot] == 0) {
        int per_sm = 0;
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, func, threads, 0) != cudaSuccess || per_sm < 1)
            per_sm = 1;
        if (per_sm > max_per_sm) per_sm = max_per_sm;
        int g = per_sm * ctx->num_sms;
        if (g > kMaxCoopBlocks) g = kMaxCoopBlocks;
        ctx->coop_blocks[slot] = g;
    }
    return ctx->coop_blocks[slot];
}

#define VOR_LAUNCH_COOP(kernel, grid, block, stream, ...)                                         \
    do {                                                                                           \
        void* args_[] = {__VA_ARGS__};                                                             \
        vor_prof_mark(ctx, 0, #kernel, (stream));                                                  \
        cudaError_t e_ = cudaLaunchCooperativeKernel((const void*)kernel, dim3(grid), dim3(block), \
                                                     args_, 0, (stream));                          \
        vor_prof_mark(ctx, 1, #kernel, (stream));                                                  \
        ctx->launches++;                                                                           \
        if (e_ != cudaSuccess) return vor_cuda_fail(ctx, e_, #kernel);                             \
    } while (0)

// launch + count + check
#define VOR_LAUNCH(kernel, grid, block, smem, stream, ...)                      \
    do {                                                                        \
        vor_prof_mark(ctx, 0, #kernel, (stream));                               \
        kernel<<<(grid), (block), (smem), (stream)>>>(__VA_ARGS__);             \
        vor_prof_mark(ctx, 1, #kernel, (stream));                               \
        ctx->launches++;                                                        \
        cudaError_t e_ = cudaGetLastError();                                    \
        if (e_ != cudaSuccess) return vor_cuda_fail(ctx, e_, #kernel);          \
    } while (0)

// internal entry points shared between translation units
int vor_sort_unique_keys(vor_ctx* ctx, uint64_t* d_keys_in_a, const int64_t* d_n_in, int key_bits,
                         uint64_t* d_out, int64_t cap, int64_t* d_n_out, int flag_bit,
                         int64_t n_hint /* expected number of keys, 0 = unknown */, cudaStream_t stream);
int vor_reset_rows(vor_ctx* ctx);
