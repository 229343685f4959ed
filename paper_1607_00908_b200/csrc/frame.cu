// One site-driven frame of the hot path (a1..a5) on context-owned buffers: the call a user makes
// once per simulation snapshot (the paper's "trigger").  The previous frame's
// edge list is the only state carried between calls.
#include "common.cuh"
#include "rows.cuh"

namespace {

__global__ void gather_counts_kernel(const int64_t* __restrict__ n_edges, const int64_t* __restrict__ n_created,
                                     const int64_t* __restrict__ n_destroyed, const int32_t* __restrict__ flags,
                                     int64_t* __restrict__ out) {
    out[0] = *n_edges; out[1] = *n_created; out[2] = *n_destroyed; out[3] = *flags;
}

// a1..a5 for one frame on the context's label image and ping-pong edge lists; the flip lists and
// the 4 counts go to the given buffers.  The edge lists carry their row offsets (vor_edges_rows), so
// consecutive frames with the same number of sites are compared row by row (vor_diff_rows).
int frame_compute(vor_ctx* ctx, const int32_t* d_sx, const int32_t* d_sy, int32_t n_sites,
                  uint64_t* d_created, uint64_t* d_destroyed, int64_t* d_counts, cudaStream_t stream) {
    int rc;
    const int now = ctx->fr_cur < 0 ? 0 : 1 - ctx->fr_cur, prev = 1 - now;
    if (ctx->fr_cur < 0) {                               // no previous frame: an empty list with empty rows
        VOR_CUDA(cudaMemsetAsync(ctx->d_fr_nedges[prev], 0, sizeof(int64_t), stream));
        VOR_CUDA(cudaMemsetAsync(ctx->d_fr_rowptr[prev], 0, ((size_t)ctx->max_sites + 1) * sizeof(uint32_t), stream));
        ctx->fr_prev_sites = n_sites;
    }
    if ((rc = vor_build_cells(ctx, d_sx, d_sy, n_sites, stream)) != VOR_OK) return rc;
    if (vor_label_fusable(ctx)) {
        // labelling and pair extraction in one kernel: the label image is written (vor_frame_results) but
        // never read back, except for the rows along the tile seams (do not move the lattice)
        VOR_CUDA(cudaMemsetAsync(ctx->d_n_raw, 0, 8 * sizeof(int64_t), stream));
        const RowSet rs = vor_row_set(ctx);
        if ((rc = vor_label_fused(ctx, ctx->d_fr_labels, rs, stream)) != VOR_OK) return rc;
        if ((rc = vor_edges_fused_tail(ctx, ctx->d_fr_labels, rs, stream)) != VOR_OK) return rc;
        if ((rc = vor_edges_finish(ctx, rs, ctx->d_fr_edges[now], ctx->fr_cap, ctx->d_fr_nedges[now],
                                   ctx->d_fr_rowptr[now], false, stream)) != VOR_OK) return rc;
    } else {
        if ((rc = vor_label(ctx, ctx->d_fr_labels, stream)) != VOR_OK) return rc;
        if (ctx->d_fo_mask &&
            (rc = vor_paint_obstacles(ctx, ctx->d_fo_mask, ctx->fo_colour, ctx->d_fr_labels, ctx->Ly, stream)) != VOR_OK) return rc;
        if ((rc = vor_edges_image(ctx, ctx->d_fr_labels, ctx->Ly, ctx->per_y, ctx->d_fo_mask ? ctx->fo_colour : -1,
                                  ctx->d_fr_edges[now], ctx->fr_cap, ctx->d_fr_nedges[now], ctx->d_fr_rowptr[now],
                                  stream)) != VOR_OK) return rc;
    }
    if (n_sites == ctx->fr_prev_sites)
        rc = vor_diff_rows(ctx, ctx->d_fr_edges[prev], ctx->d_fr_rowptr[prev], ctx->d_fr_edges[now],
                           ctx->d_fr_rowptr[now], n_sites, d_created, d_destroyed, ctx->fr_cap,
                           &d_counts[1], &d_counts[2], stream);
    else                                                 // the number of sites changed: plain list comparison
        rc = vor_diff(ctx, ctx->d_fr_edges[prev], ctx->d_fr_nedges[prev], ctx->d_fr_edges[now],
                      ctx->d_fr_nedges[now], ctx->fr_cap, ctx->fr_cap, nullptr, nullptr, 0, 0, d_created, d_destroyed,
                      ctx->fr_cap, &d_counts[1], &d_counts[2], stream);
    if (rc != VOR_OK) return rc;
    VOR_LAUNCH(gather_counts_kernel, 1, 1, 0, stream, ctx->d_fr_nedges[now], &d_counts[1], &d_counts[2],
               ctx->d_flags, d_counts);
    ctx->fr_cur = now;
    ctx->fr_prev_sites = n_sites;
    return VOR_OK;
}

int ensure_pipe_buffers(vor_ctx* ctx) {
    if (ctx->pp_h2d) return VOR_OK;
    for (int k = 0; k < 2; ++k) {
        VOR_CUDA(cudaMalloc((void**)&ctx->d_pp_sx[k], (size_t)ctx->max_sites * sizeof(int32_t)));
        VOR_CUDA(cudaMalloc((void**)&ctx->d_pp_sy[k], (size_t)ctx->max_sites * sizeof(int32_t)));
        VOR_CUDA(cudaMalloc((void**)&ctx->d_pp_created[k], (size_t)ctx->fr_cap * sizeof(uint64_t)));
        VOR_CUDA(cudaMalloc((void**)&ctx->d_pp_destroyed[k], (size_t)ctx->fr_cap * sizeof(uint64_t)));
        VOR_CUDA(cudaMalloc((void**)&ctx->d_pp_counts[k], 8 * sizeof(int64_t)));
        VOR_CUDA(cudaMallocHost((void**)&ctx->h_pp_counts[k], 8 * sizeof(int64_t)));
        VOR_CUDA(cudaMallocHost((void**)&ctx->h_pp_sites[k], 2 * (size_t)ctx->max_sites * sizeof(int32_t)));
        VOR_CUDA(cudaEventCreateWithFlags(&ctx->pp_ev_in[k], cudaEventDisableTiming));
        VOR_CUDA(cudaEventCreateWithFlags(&ctx->pp_ev_done[k], cudaEventDisableTiming));
        VOR_CUDA(cudaEventCreateWithFlags(&ctx->pp_ev_cnt[k], cudaEventDisableTiming));
    }
    VOR_CUDA(cudaStreamCreateWithFlags(&ctx->pp_d2h, cudaStreamNonBlocking));
    VOR_CUDA(cudaStreamCreateWithFlags(&ctx->pp_lst, cudaStreamNonBlocking));
    VOR_CUDA(cudaStreamCreateWithFlags(&ctx->pp_h2d, cudaStreamNonBlocking));
    return VOR_OK;
}

// Page-locked host memory (cudaMallocHost / cudaHostRegister / torch pin_memory) can be the source or
// target of a true asynchronous DMA; anything else is staged through the context's pinned buffers.
bool is_pinned(const void* p) {
    cudaPointerAttributes a;
    if (cudaPointerGetAttributes(&a, p) != cudaSuccess) { cudaGetLastError(); return false; }
    return a.type == cudaMemoryTypeHost;
}

int ensure_frame_buffers(vor_ctx* ctx) {
    if (ctx->d_fr_labels) return VOR_OK;
    const size_t cells = (size_t)ctx->Lx * ctx->Ly;
    int64_t cap = 4 * (int64_t)ctx->max_sites + 1024;
    if (cap > ctx->max_raw_keys) cap = ctx->max_raw_keys;
    if (cap > 0xffffffffll) cap = 0xffffffffll;            // 32-bit row offsets
    ctx->fr_cap = cap;
    VOR_CUDA(cudaMalloc((void**)&ctx->d_fr_sx, (size_t)ctx->max_sites * sizeof(int32_t)));
    VOR_CUDA(cudaMalloc((void**)&ctx->d_fr_sy, (size_t)ctx->max_sites * sizeof(int32_t)));
    VOR_CUDA(cudaMalloc((void**)&ctx->d_fr_labels, cells * sizeof(int32_t)));
    for (int k = 0; k < 2; ++k) {
        VOR_CUDA(cudaMalloc((void**)&ctx->d_fr_edges[k], (size_t)cap * sizeof(uint64_t)));
        VOR_CUDA(cudaMalloc((void**)&ctx->d_fr_nedges[k], sizeof(int64_t)));
        VOR_CUDA(cudaMemset(ctx->d_fr_nedges[k], 0, sizeof(int64_t)));
        VOR_CUDA(cudaMalloc((void**)&ctx->d_fr_rowptr[k], ((size_t)ctx->max_sites + 1) * sizeof(uint32_t)));
    }
    VOR_CUDA(cudaMalloc((void**)&ctx->d_fr_created, (size_t)cap * sizeof(uint64_t)));
    VOR_CUDA(cudaMalloc((void**)&ctx->d_fr_destroyed, (size_t)cap * sizeof(uint64_t)));
    VOR_CUDA(cudaMalloc((void**)&ctx->d_fr_counts, 8 * sizeof(int64_t)));
    VOR_CUDA(cudaMallocHost((void**)&ctx->h_fr_counts, 8 * sizeof(int64_t)));
    VOR_CUDA(cudaMallocHost((void**)&ctx->h_fr_sites, 2 * (size_t)ctx->max_sites * sizeof(int32_t)));
    VOR_CUDA(cudaMallocHost((void**)&ctx->h_fr_lists, 2 * (size_t)cap * sizeof(uint64_t)));
    ctx->fr_cur = -1;
    return VOR_OK;
}


// ---- field-driven frame (a6..a8, then a1..a5 with the isomorphism): PAPER.md:93-101 (bubbles and their
// centres of mass), 213-223 (translation, comparison, appearing / disappearing bubbles).  Nothing on
// this chain needs a host synchronisation: the number of bubbles stays in a device scalar
// (vor_build_cells_dev), the maps are sized by the context's max_sites.
__global__ void gather_field_counts_kernel(const int32_t* __restrict__ n_comp, const int64_t* __restrict__ n_edges,
                                           const int64_t* __restrict__ n_created, const int64_t* __restrict__ n_destroyed,
                                           int have_prev, const int32_t* __restrict__ flags, int64_t* __restrict__ out) {
    out[0] = *n_comp; out[1] = *n_edges;
    out[2] = have_prev ? *n_created : 0; out[3] = have_prev ? *n_destroyed : 0;
    out[4] = *flags;
}

int ensure_field_buffers(vor_ctx* ctx) {
    if (ctx->d_ff_ccl) return VOR_OK;
    const size_t cells = (size_t)ctx->Lx * ctx->Ly, K = (size_t)ctx->max_sites;
    VOR_CUDA(cudaMalloc((void**)&ctx->d_ff_ccl, cells * sizeof(int32_t)));
    for (int k = 0; k < 2; ++k) {
        VOR_CUDA(cudaMalloc((void**)&ctx->d_ff_cxy[k], 2 * K * sizeof(double)));
        VOR_CUDA(cudaMalloc((void**)&ctx->d_ff_comp[k], (4 * K + 4) * sizeof(int32_t)));   // sx, sy, size, root, n
    }
    VOR_CUDA(cudaMalloc((void**)&ctx->d_ff_maps, 2 * K * sizeof(int32_t)));
    VOR_CUDA(cudaMalloc((void**)&ctx->d_ff_tmpcount, 2 * sizeof(int64_t)));
    VOR_CUDA(cudaMallocHost((void**)&ctx->h_ff_count, sizeof(int32_t)));
    *ctx->h_ff_count = 0;
    ctx->ff_cur = -1;
    return VOR_OK;
}

struct FieldArgs { float thr; int above; int32_t min_size; int32_t radius_fp; };

int field_frame_compute(vor_ctx* ctx, const float* d_field, const FieldArgs& fa, uint64_t* d_created,
                        uint64_t* d_destroyed, int64_t* d_counts, cudaStream_t stream) {
    int rc;
    const int32_t K = ctx->max_sites;
    const bool have_prev = ctx->ff_cur >= 0;
    const int now = have_prev ? 1 - ctx->ff_cur : 0, prev = 1 - now;
    double* cx = ctx->d_ff_cxy[now]; double* cy = cx + K;
    int32_t* c = ctx->d_ff_comp[now]; const int32_t* pc = ctx->d_ff_comp[prev];
    int32_t* p2n = ctx->d_ff_maps; int32_t* n2p = p2n + K;
    // the bubble count of an earlier frame, copied to page-locked memory behind that frame's kernels: whatever
    // has arrived by now sizes this frame's buckets and halo (a hint: results never depend on it), no waiting
    const int32_t seen = *(volatile int32_t*)ctx->h_ff_count;
    if (seen > 0) ctx->ff_hint = seen < K ? seen : K;
    if ((rc = field_threshold_ccl_conn(ctx, d_field, fa.thr, fa.above, ctx->fo_connectivity == 8 ? 8 : 4, ctx->d_ff_ccl,
                                       stream)) != VOR_OK) return rc;
    if ((rc = field_centroids_weighted(ctx, ctx->d_ff_ccl, ctx->fo_weighted ? d_field : nullptr, fa.min_size, cx, cy, c,
                                       c + K, c + 2 * K, c + 3 * K, K, c + 4 * K, stream)) != VOR_OK) return rc;
    VOR_CUDA(cudaMemcpyAsync(ctx->h_ff_count, c + 4 * K, sizeof(int32_t), cudaMemcpyDeviceToHost, stream));
    if (have_prev && (rc = match_sites(ctx, pc, pc + K, pc + 4 * K, c, c + K, c + 4 * K, K, K, fa.radius_fp,
                                       p2n, n2p, stream)) != VOR_OK) return rc;
    if ((rc = vor_build_cells_dev(ctx, c, c + K, c + 4 * K, K, ctx->ff_hint > 0 ? ctx->ff_hint : K, stream)) != VOR_OK)
        return rc;
    if ((rc = vor_label(ctx, ctx->d_fr_labels, stream)) != VOR_OK) return rc;
    if (ctx->d_fo_mask &&
        (rc = vor_paint_obstacles(ctx, ctx->d_fo_mask, ctx->fo_colour, ctx->d_fr_labels, ctx->Ly, stream)) != VOR_OK) return rc;
    if ((rc = vor_edges_image(ctx, ctx->d_fr_labels, ctx->Ly, ctx->per_y, ctx->d_fo_mask ? ctx->fo_colour : -1,
                              ctx->d_fr_edges[now], ctx->fr_cap, ctx->d_fr_nedges[now], nullptr, stream)) != VOR_OK) return rc;
    if (have_prev && (rc = vor_diff(ctx, ctx->d_fr_edges[prev], ctx->d_fr_nedges[prev], ctx->d_fr_edges[now],
                                    ctx->d_fr_nedges[now], ctx->fr_cap, ctx->fr_cap, p2n, n2p, K, K,
                                    d_created, d_destroyed, ctx->fr_cap, &ctx->d_ff_tmpcount[0],
                                    &ctx->d_ff_tmpcount[1], stream)) != VOR_OK) return rc;
    VOR_LAUNCH(gather_field_counts_kernel, 1, 1, 0, stream, c + 4 * K, ctx->d_fr_nedges[now], &ctx->d_ff_tmpcount[0],
               &ctx->d_ff_tmpcount[1], have_prev ? 1 : 0, ctx->d_flags, d_counts);
    ctx->ff_cur = now;
    ctx->fr_cur = -1;                                    // the site-path state shares the edge buffers
    return VOR_OK;
}
}  // namespace

extern "C" int vor_frame_options(vor_ctx* ctx, int32_t connectivity, int32_t weighted, const uint8_t* d_obstacles,
                                 int32_t obstacle_colour) {
    if (!ctx) return VOR_EINVAL;
    if (connectivity != 4 && connectivity != 8)
        return vor_fail(ctx, VOR_EINVAL, "vor_frame_options: connectivity must be 4 or 8");
    if (d_obstacles && obstacle_colour < 0)
        return vor_fail(ctx, VOR_EINVAL, "vor_frame_options: the obstacle colour must be >= 0");
    ctx->fo_connectivity = connectivity;
    ctx->fo_weighted = weighted != 0;
    ctx->d_fo_mask = d_obstacles;
    ctx->fo_colour = obstacle_colour;
    return VOR_OK;
}

extern "C" int vor_frame_reset(vor_ctx* ctx) {
    if (!ctx) return VOR_EINVAL;
    if (int drc_ = vor_check_device(ctx)) return drc_;
    ctx->fr_cur = -1;
    ctx->ff_cur = -1;
    if (ctx->pp_h2d) {                                   // drop frames still in flight
        cudaStreamSynchronize(ctx->pp_h2d);
        cudaStreamSynchronize(ctx->pp_d2h);
        cudaStreamSynchronize(ctx->pp_lst);
    }
    ctx->pp_tail = ctx->pp_head;
    return VOR_OK;
}

extern "C" int vor_frame_device(vor_ctx* ctx, const int32_t* d_sx, const int32_t* d_sy,
                                int32_t n_sites, void* stream_) {
    if (!ctx) return VOR_EINVAL;
    if (int drc_ = vor_check_device(ctx)) return drc_;
    int rc = ensure_frame_buffers(ctx);
    if (rc != VOR_OK) return rc;
    return frame_compute(ctx, d_sx, d_sy, n_sites, ctx->d_fr_created, ctx->d_fr_destroyed, ctx->d_fr_counts,
                         (cudaStream_t)stream_);
}

extern "C" int vor_frame_host(vor_ctx* ctx, const int32_t* h_sx, const int32_t* h_sy, int32_t n_sites,
                              uint64_t* h_created, uint64_t* h_destroyed, int64_t cap,
                              int64_t* h_counts, void* stream_) {
    if (!ctx) return VOR_EINVAL;
    if (int drc_ = vor_check_device(ctx)) return drc_;
    if (!h_sx || !h_sy || !h_counts || cap < 0 || (cap > 0 && (!h_created || !h_destroyed)))
        return vor_fail(ctx, VOR_EINVAL, "vor_frame_host: null pointer or negative capacity");
    if (n_sites < 1 || n_sites > ctx->max_sites)
        return vor_fail(ctx, VOR_EINVAL, "vor_frame_host: n_sites out of range");
    int rc = ensure_frame_buffers(ctx);
    if (rc != VOR_OK) return rc;
    cudaStream_t stream = (cudaStream_t)stream_;
    // pageable caller buffers are staged through pinned memory so that the copies are true async DMA
    const int32_t* src_x = h_sx;
    const int32_t* src_y = h_sy;
    if (!is_pinned(h_sx) || !is_pinned(h_sy)) {
        memcpy(ctx->h_fr_sites, h_sx, (size_t)n_sites * sizeof(int32_t));
        memcpy(ctx->h_fr_sites + ctx->max_sites, h_sy, (size_t)n_sites * sizeof(int32_t));
        src_x = ctx->h_fr_sites; src_y = ctx->h_fr_sites + ctx->max_sites;
    }
    VOR_CUDA(cudaMemcpyAsync(ctx->d_fr_sx, src_x, (size_t)n_sites * sizeof(int32_t),
                             cudaMemcpyHostToDevice, stream));
    VOR_CUDA(cudaMemcpyAsync(ctx->d_fr_sy, src_y, (size_t)n_sites * sizeof(int32_t),
                             cudaMemcpyHostToDevice, stream));
    if ((rc = vor_frame_device(ctx, ctx->d_fr_sx, ctx->d_fr_sy, n_sites, stream)) != VOR_OK) return rc;
    VOR_CUDA(cudaMemcpyAsync(ctx->h_fr_counts, ctx->d_fr_counts, 3 * sizeof(int64_t),
                             cudaMemcpyDeviceToHost, stream));
    VOR_CUDA(cudaStreamSynchronize(stream));
    h_counts[0] = ctx->h_fr_counts[0]; h_counts[1] = ctx->h_fr_counts[1]; h_counts[2] = ctx->h_fr_counts[2];
    int64_t nc = h_counts[1] < ctx->fr_cap ? h_counts[1] : ctx->fr_cap;
    int64_t nd = h_counts[2] < ctx->fr_cap ? h_counts[2] : ctx->fr_cap;
    if (nc > cap) nc = cap;
    if (nd > cap) nd = cap;
    const bool direct = (nc == 0 || is_pinned(h_created)) && (nd == 0 || is_pinned(h_destroyed));
    uint64_t* dst_c = direct ? h_created : ctx->h_fr_lists;
    uint64_t* dst_d = direct ? h_destroyed : ctx->h_fr_lists + ctx->fr_cap;
    if (nc > 0)
        VOR_CUDA(cudaMemcpyAsync(dst_c, ctx->d_fr_created, (size_t)nc * sizeof(uint64_t),
                                 cudaMemcpyDeviceToHost, stream));
    if (nd > 0)
        VOR_CUDA(cudaMemcpyAsync(dst_d, ctx->d_fr_destroyed, (size_t)nd * sizeof(uint64_t),
                                 cudaMemcpyDeviceToHost, stream));
    rc = vor_sync_status(ctx, stream);
    if (!direct) {
        if (nc > 0) memcpy(h_created, dst_c, (size_t)nc * sizeof(uint64_t));
        if (nd > 0) memcpy(h_destroyed, dst_d, (size_t)nd * sizeof(uint64_t));
    }
    if (rc == VOR_OK && (h_counts[1] > cap || h_counts[2] > cap))
        return vor_fail(ctx, VOR_ECAPACITY, "vor_frame_host: created/destroyed list larger than cap");
    return rc;
}

extern "C" int vor_frame_results(vor_ctx* ctx, const int32_t** d_labels, const uint64_t** d_edges,
                                 const uint64_t** d_created, const uint64_t** d_destroyed,
                                 const int64_t** d_counts) {
    if (!ctx) return VOR_EINVAL;
    if (int drc_ = vor_check_device(ctx)) return drc_;
    if (ctx->fr_cur < 0 || !ctx->d_fr_labels) return vor_fail(ctx, VOR_ESTATE, "no frame processed yet");
    if (d_labels) *d_labels = ctx->d_fr_labels;
    if (d_edges) *d_edges = ctx->d_fr_edges[ctx->fr_cur];
    if (d_created) *d_created = ctx->d_fr_created;
    if (d_destroyed) *d_destroyed = ctx->d_fr_destroyed;
    if (d_counts) *d_counts = ctx->d_fr_counts;
    return VOR_OK;
}

extern "C" int vor_frame_submit(vor_ctx* ctx, const int32_t* h_sx, const int32_t* h_sy, int32_t n_sites,
                                void* stream_) {
    if (!ctx) return VOR_EINVAL;
    if (int drc_ = vor_check_device(ctx)) return drc_;
    if (!h_sx || !h_sy) return vor_fail(ctx, VOR_EINVAL, "vor_frame_submit: null pointer");
    if (n_sites < 1 || n_sites > ctx->max_sites)
        return vor_fail(ctx, VOR_EINVAL, "vor_frame_submit: n_sites out of range");
    int rc = ensure_frame_buffers(ctx);
    if (rc != VOR_OK) return rc;
    if ((rc = ensure_pipe_buffers(ctx)) != VOR_OK) return rc;
    if (ctx->pp_head - ctx->pp_tail >= 2)
        return vor_fail(ctx, VOR_ESTATE, "vor_frame_submit: two frames in flight, collect one first");
    cudaStream_t stream = (cudaStream_t)stream_;
    const int s = (int)(ctx->pp_head & 1);
    // inputs: own stream, so that the upload overlaps the previous frame's kernels; the slot's device
    // buffers were last read by frame head-2, which has been collected, hence finished
    const int32_t* src_x = h_sx;
    const int32_t* src_y = h_sy;
    if (!is_pinned(h_sx) || !is_pinned(h_sy)) {
        memcpy(ctx->h_pp_sites[s], h_sx, (size_t)n_sites * sizeof(int32_t));
        memcpy(ctx->h_pp_sites[s] + ctx->max_sites, h_sy, (size_t)n_sites * sizeof(int32_t));
        src_x = ctx->h_pp_sites[s]; src_y = ctx->h_pp_sites[s] + ctx->max_sites;
    }
    VOR_CUDA(cudaMemcpyAsync(ctx->d_pp_sx[s], src_x, (size_t)n_sites * sizeof(int32_t), cudaMemcpyHostToDevice, ctx->pp_h2d));
    VOR_CUDA(cudaMemcpyAsync(ctx->d_pp_sy[s], src_y, (size_t)n_sites * sizeof(int32_t), cudaMemcpyHostToDevice, ctx->pp_h2d));
    VOR_CUDA(cudaEventRecord(ctx->pp_ev_in[s], ctx->pp_h2d));
    VOR_CUDA(cudaStreamWaitEvent(stream, ctx->pp_ev_in[s], 0));
    if ((rc = frame_compute(ctx, ctx->d_pp_sx[s], ctx->d_pp_sy[s], n_sites, ctx->d_pp_created[s],
                            ctx->d_pp_destroyed[s], ctx->d_pp_counts[s], stream)) != VOR_OK) return rc;
    VOR_CUDA(cudaEventRecord(ctx->pp_ev_done[s], stream));
    VOR_CUDA(cudaStreamWaitEvent(ctx->pp_d2h, ctx->pp_ev_done[s], 0));
    VOR_CUDA(cudaMemcpyAsync(ctx->h_pp_counts[s], ctx->d_pp_counts[s], 4 * sizeof(int64_t), cudaMemcpyDeviceToHost, ctx->pp_d2h));
    VOR_CUDA(cudaEventRecord(ctx->pp_ev_cnt[s], ctx->pp_d2h));
    ctx->pp_head++;
    return VOR_OK;
}

extern "C" int vor_frame_collect(vor_ctx* ctx, uint64_t* h_created, uint64_t* h_destroyed, int64_t cap,
                                 int64_t* h_counts) {
    if (!ctx) return VOR_EINVAL;
    if (int drc_ = vor_check_device(ctx)) return drc_;
    if (!h_counts || cap < 0 || (cap > 0 && (!h_created || !h_destroyed)))
        return vor_fail(ctx, VOR_EINVAL, "vor_frame_collect: null pointer or negative capacity");
    if (!ctx->pp_h2d || ctx->pp_tail == ctx->pp_head)
        return vor_fail(ctx, VOR_ESTATE, "vor_frame_collect: no frame in flight");
    const int s = (int)(ctx->pp_tail & 1);
    VOR_CUDA(cudaEventSynchronize(ctx->pp_ev_cnt[s]));
    const int64_t* c = ctx->h_pp_counts[s];
    h_counts[0] = c[0]; h_counts[1] = c[1]; h_counts[2] = c[2];
    int64_t nc = c[1] < ctx->fr_cap ? c[1] : ctx->fr_cap, nd = c[2] < ctx->fr_cap ? c[2] : ctx->fr_cap;
    if (nc > cap) nc = cap;
    if (nd > cap) nd = cap;
    const bool direct = (nc == 0 || is_pinned(h_created)) && (nd == 0 || is_pinned(h_destroyed));
    uint64_t* dst_c = direct ? h_created : ctx->h_fr_lists;
    uint64_t* dst_d = direct ? h_destroyed : ctx->h_fr_lists + ctx->fr_cap;
    // own stream: pp_d2h already holds the wait for the NEXT frame's kernels
    if (nc > 0) VOR_CUDA(cudaMemcpyAsync(dst_c, ctx->d_pp_created[s], (size_t)nc * sizeof(uint64_t), cudaMemcpyDeviceToHost, ctx->pp_lst));
    if (nd > 0) VOR_CUDA(cudaMemcpyAsync(dst_d, ctx->d_pp_destroyed[s], (size_t)nd * sizeof(uint64_t), cudaMemcpyDeviceToHost, ctx->pp_lst));
    VOR_CUDA(cudaStreamSynchronize(ctx->pp_lst));
    if (!direct) {
        if (nc > 0) memcpy(h_created, dst_c, (size_t)nc * sizeof(uint64_t));
        if (nd > 0) memcpy(h_destroyed, dst_d, (size_t)nd * sizeof(uint64_t));
    }
    ctx->pp_tail++;
    if (c[3] != 0) {                                     // a kernel of this (or an earlier) frame latched an overflow
        VOR_CUDA(cudaDeviceSynchronize());
        return vor_sync_status(ctx, nullptr);
    }
    if (c[1] > cap || c[2] > cap)
        return vor_fail(ctx, VOR_ECAPACITY, "vor_frame_collect: created/destroyed list larger than cap");
    return VOR_OK;
}

// ------------------------------------------------------------------------------------ field frames
extern "C" int field_frame_device(vor_ctx* ctx, const float* d_field, float thr, int above, int32_t min_size,
                                  int32_t radius_fp, void* stream_) {
    if (!ctx) return VOR_EINVAL;
    if (int drc_ = vor_check_device(ctx)) return drc_;
    if (!d_field || radius_fp < 0) return vor_fail(ctx, VOR_EINVAL, "field_frame_device: null field or negative radius");
    int rc = ensure_frame_buffers(ctx);
    if (rc != VOR_OK || (rc = ensure_field_buffers(ctx)) != VOR_OK) return rc;
    const FieldArgs fa{thr, above, min_size, radius_fp};
    return field_frame_compute(ctx, d_field, fa, ctx->d_fr_created, ctx->d_fr_destroyed, ctx->d_fr_counts,
                               (cudaStream_t)stream_);
}

extern "C" int field_frame_submit(vor_ctx* ctx, const float* h_field, float thr, int above, int32_t min_size,
                                  int32_t radius_fp, void* stream_) {
    if (!ctx) return VOR_EINVAL;
    if (int drc_ = vor_check_device(ctx)) return drc_;
    if (!h_field || radius_fp < 0) return vor_fail(ctx, VOR_EINVAL, "field_frame_submit: null field or negative radius");
    int rc = ensure_frame_buffers(ctx);
    if (rc != VOR_OK || (rc = ensure_field_buffers(ctx)) != VOR_OK || (rc = ensure_pipe_buffers(ctx)) != VOR_OK) return rc;
    if (ctx->pp_head - ctx->pp_tail >= 2)
        return vor_fail(ctx, VOR_ESTATE, "field_frame_submit: two frames in flight, collect one first");
    cudaStream_t stream = (cudaStream_t)stream_;
    const int s = (int)(ctx->pp_head & 1);
    const size_t bytes = (size_t)ctx->Lx * ctx->Ly * sizeof(float);
    if (!ctx->d_ff_field[s]) VOR_CUDA(cudaMalloc((void**)&ctx->d_ff_field[s], bytes));
    // pinned caller memory is DMA'd directly; pageable memory goes through the driver's staging copy
    VOR_CUDA(cudaMemcpyAsync(ctx->d_ff_field[s], h_field, bytes, cudaMemcpyHostToDevice, ctx->pp_h2d));
    VOR_CUDA(cudaEventRecord(ctx->pp_ev_in[s], ctx->pp_h2d));
    VOR_CUDA(cudaStreamWaitEvent(stream, ctx->pp_ev_in[s], 0));
    const FieldArgs fa{thr, above, min_size, radius_fp};
    if ((rc = field_frame_compute(ctx, ctx->d_ff_field[s], fa, ctx->d_pp_created[s], ctx->d_pp_destroyed[s],
                                  ctx->d_pp_counts[s], stream)) != VOR_OK) return rc;
    VOR_CUDA(cudaEventRecord(ctx->pp_ev_done[s], stream));
    VOR_CUDA(cudaStreamWaitEvent(ctx->pp_d2h, ctx->pp_ev_done[s], 0));
    VOR_CUDA(cudaMemcpyAsync(ctx->h_pp_counts[s], ctx->d_pp_counts[s], 5 * sizeof(int64_t), cudaMemcpyDeviceToHost, ctx->pp_d2h));
    VOR_CUDA(cudaEventRecord(ctx->pp_ev_cnt[s], ctx->pp_d2h));
    ctx->pp_head++;
    return VOR_OK;
}

extern "C" int field_frame_collect(vor_ctx* ctx, uint64_t* h_created, uint64_t* h_destroyed, int64_t cap,
                                   int64_t* h_counts) {
    if (!ctx) return VOR_EINVAL;
    if (int drc_ = vor_check_device(ctx)) return drc_;
    if (!h_counts || cap < 0 || (cap > 0 && (!h_created || !h_destroyed)))
        return vor_fail(ctx, VOR_EINVAL, "field_frame_collect: null pointer or negative capacity");
    if (!ctx->pp_h2d || !ctx->d_ff_ccl || ctx->pp_tail == ctx->pp_head)
        return vor_fail(ctx, VOR_ESTATE, "field_frame_collect: no frame in flight");
    const int s = (int)(ctx->pp_tail & 1);
    VOR_CUDA(cudaEventSynchronize(ctx->pp_ev_cnt[s]));
    const int64_t* c = ctx->h_pp_counts[s];
    for (int k = 0; k < 4; ++k) h_counts[k] = c[k];
    if (c[0] > 0) ctx->ff_hint = (int32_t)(c[0] < ctx->max_sites ? c[0] : ctx->max_sites);   // sizes the next cell lists
    int64_t nc = c[2] < ctx->fr_cap ? c[2] : ctx->fr_cap, nd = c[3] < ctx->fr_cap ? c[3] : ctx->fr_cap;
    if (nc > cap) nc = cap;
    if (nd > cap) nd = cap;
    const bool direct = (nc == 0 || is_pinned(h_created)) && (nd == 0 || is_pinned(h_destroyed));
    uint64_t* dst_c = direct ? h_created : ctx->h_fr_lists;
    uint64_t* dst_d = direct ? h_destroyed : ctx->h_fr_lists + ctx->fr_cap;
    if (nc > 0) VOR_CUDA(cudaMemcpyAsync(dst_c, ctx->d_pp_created[s], (size_t)nc * sizeof(uint64_t), cudaMemcpyDeviceToHost, ctx->pp_lst));
    if (nd > 0) VOR_CUDA(cudaMemcpyAsync(dst_d, ctx->d_pp_destroyed[s], (size_t)nd * sizeof(uint64_t), cudaMemcpyDeviceToHost, ctx->pp_lst));
    VOR_CUDA(cudaStreamSynchronize(ctx->pp_lst));
    if (!direct) {
        if (nc > 0) memcpy(h_created, dst_c, (size_t)nc * sizeof(uint64_t));
        if (nd > 0) memcpy(h_destroyed, dst_d, (size_t)nd * sizeof(uint64_t));
    }
    ctx->pp_tail++;
    if (c[4] != 0) {
        VOR_CUDA(cudaDeviceSynchronize());
        return vor_sync_status(ctx, nullptr);
    }
    if (c[2] > cap || c[3] > cap)
        return vor_fail(ctx, VOR_ECAPACITY, "field_frame_collect: created/destroyed list larger than cap");
    return VOR_OK;
}

extern "C" int field_frame_results(vor_ctx* ctx, const int32_t** d_ccl, const int32_t** d_labels,
                                   const double** d_cx, const double** d_cy, const int32_t** d_sx,
                                   const int32_t** d_sy, const int32_t** d_size, const int32_t** d_root,
                                   const int32_t** d_p2n, const int32_t** d_n2p, const uint64_t** d_edges,
                                   const uint64_t** d_created, const uint64_t** d_destroyed,
                                   const int64_t** d_counts) {
    if (!ctx) return VOR_EINVAL;
    if (int drc_ = vor_check_device(ctx)) return drc_;
    if (!ctx->d_ff_ccl || ctx->ff_cur < 0) return vor_fail(ctx, VOR_ESTATE, "no field frame processed yet");
    const int32_t K = ctx->max_sites;
    const int32_t* c = ctx->d_ff_comp[ctx->ff_cur];
    if (d_ccl) *d_ccl = ctx->d_ff_ccl;
    if (d_labels) *d_labels = ctx->d_fr_labels;
    if (d_cx) *d_cx = ctx->d_ff_cxy[ctx->ff_cur];
    if (d_cy) *d_cy = ctx->d_ff_cxy[ctx->ff_cur] + K;
    if (d_sx) *d_sx = c;
    if (d_sy) *d_sy = c + K;
    if (d_size) *d_size = c + 2 * K;
    if (d_root) *d_root = c + 3 * K;
    if (d_p2n) *d_p2n = ctx->d_ff_maps;
    if (d_n2p) *d_n2p = ctx->d_ff_maps + K;
    if (d_edges) *d_edges = ctx->d_fr_edges[ctx->ff_cur];
    if (d_created) *d_created = ctx->d_fr_created;
    if (d_destroyed) *d_destroyed = ctx->d_fr_destroyed;
    if (d_counts) *d_counts = ctx->d_fr_counts;
    return VOR_OK;
}
