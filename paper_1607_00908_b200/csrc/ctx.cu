// Context life cycle, options, sticky status.  See include/vor.h.
#include <stdlib.h>

#include "common.cuh"

namespace {

template <typename T>
cudaError_t dmalloc(T** p, size_t n) {
    return cudaMalloc((void**)p, (n ? n : 1) * sizeof(T));
}

}  // namespace

extern "C" {

int vor_create(vor_ctx** out, int32_t L, int32_t max_sites, int64_t max_raw_keys) {
    return vor_create_geom(out, L, L, 1, 1, max_sites, max_raw_keys);
}

int vor_create_geom(vor_ctx** out, int32_t Lx, int32_t Ly, int32_t periodic_x, int32_t periodic_y,
                    int32_t max_sites, int64_t max_raw_keys) {
    if (!out) return VOR_EINVAL;
    *out = nullptr;
    const int32_t lim_x = periodic_x ? (1 << 22) : (1 << 21), lim_y = periodic_y ? (1 << 22) : (1 << 21);
    if (Lx < 2 || Ly < 2 || Lx > lim_x || Ly > lim_y || max_sites < 1) return VOR_EINVAL;
    vor_ctx* ctx = (vor_ctx*)calloc(1, sizeof(vor_ctx));
    if (!ctx) return VOR_ECUDA;
    ctx->Lx = Lx; ctx->Ly = Ly;
    ctx->per_x = periodic_x != 0; ctx->per_y = periodic_y != 0;
    ctx->FLx = ctx->per_x ? Lx : 2 * Lx;
    ctx->FLy = ctx->per_y ? Ly : 2 * Ly;
    ctx->Px = (int64_t)FP_ONE * ctx->FLx;
    ctx->Py = (int64_t)FP_ONE * ctx->FLy;
    ctx->max_sites = max_sites;
    const int64_t worst = 2 * (int64_t)Lx * Ly;
    if (max_raw_keys <= 0) {
        max_raw_keys = 16 * (int64_t)max_sites;
        if (max_raw_keys < (1 << 20)) max_raw_keys = 1 << 20;
    }
    if (max_raw_keys > worst) max_raw_keys = worst;
    ctx->max_raw_keys = max_raw_keys;
    ctx->bucket_occ_x100 = 100;
    ctx->label_halo_x100 = 130;
    ctx->row_slots = kRowStride;
    ctx->fr_cur = -1;
    ctx->ff_cur = -1;
    cudaError_t e = cudaGetDevice(&ctx->device);
    if (e != cudaSuccess) { free(ctx); return VOR_ECUDA; }
    int coop = 0;
    if (cudaDeviceGetAttribute(&ctx->num_sms, cudaDevAttrMultiProcessorCount, ctx->device) != cudaSuccess ||
        cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, ctx->device) != cudaSuccess ||
        ctx->num_sms < 1 || !coop) {
        free(ctx);
        return VOR_ECUDA;
    }

    // bucket widths are common divisors of Px and Py; the smallest one vor_build_cells may pick is at least
    // 2 cells wide and gives at most 4096 buckets per axis - or, when no divisor does, the largest divisor
    {
        int64_t g = ctx->Px, t = ctx->Py;
        while (t) { const int64_t r = g % t; g = t; t = r; }
        int64_t wmin = g;
        for (int64_t d = 1; d * d <= g; ++d) {
            if (g % d) continue;
            const int64_t c[2] = {d, g / d};
            for (int k = 0; k < 2; ++k)
                if (c[k] >= 2 * FP_ONE && ctx->Px / c[k] <= 4096 && ctx->Py / c[k] <= 4096 && c[k] < wmin) wmin = c[k];
        }
        ctx->w_min = wmin;
        ctx->w_gcd = g;
        ctx->nbuckets_max = (ctx->Px / wmin) * (ctx->Py / wmin);
    }
    const size_t nbuckets = (size_t)ctx->nbuckets_max;
    bool ok = true;
    ok = ok && dmalloc(&ctx->d_bucket_start, nbuckets + 1) == cudaSuccess;
    ok = ok && dmalloc(&ctx->d_bucket_fill, nbuckets) == cudaSuccess;
    ok = ok && dmalloc(&ctx->d_sorted, (size_t)max_sites) == cudaSuccess;
    ok = ok && dmalloc(&ctx->d_scan_part, 8192) == cudaSuccess;
    ok = ok && dmalloc(&ctx->d_keys_a, (size_t)max_raw_keys) == cudaSuccess;
    ok = ok && dmalloc(&ctx->d_keys_b, (size_t)max_raw_keys) == cudaSuccess;
    ok = ok && dmalloc(&ctx->d_rows, (size_t)max_sites * kRowStride) == cudaSuccess;
    ok = ok && dmalloc(&ctx->d_row_cnt, (size_t)max_sites) == cudaSuccess;
    ok = ok && dmalloc(&ctx->d_n_raw, 8) == cudaSuccess;
    ok = ok && dmalloc(&ctx->d_hist, (size_t)kMaxCoopBlocks * 256) == cudaSuccess;
    ok = ok && dmalloc(&ctx->d_blk_count, (size_t)2 * kMaxCoopBlocks) == cudaSuccess;
    ok = ok && dmalloc(&ctx->d_tr_counts, 4) == cudaSuccess;
    ok = ok && dmalloc(&ctx->d_comp_count, 4) == cudaSuccess;
    ok = ok && dmalloc(&ctx->d_flags, 4) == cudaSuccess;
    if (ok) ok = cudaMemset(ctx->d_flags, 0, 4 * sizeof(int32_t)) == cudaSuccess;
    if (ok) ok = vor_reset_rows(ctx) == VOR_OK;
    if (!ok) {
        vor_destroy(ctx);
        return VOR_ECUDA;
    }
    *out = ctx;
    return VOR_OK;
}

int vor_destroy(vor_ctx* ctx) {
    if (!ctx) return VOR_EINVAL;
    cudaFree(ctx->d_bucket_start); cudaFree(ctx->d_bucket_fill); cudaFree(ctx->d_sorted);
    cudaFree(ctx->d_scan_part); cudaFree(ctx->d_keys_a); cudaFree(ctx->d_keys_b);
    cudaFree(ctx->d_lab_fail); cudaFree(ctx->d_lab_fail_n);
    cudaFree(ctx->d_fu_cols); cudaFree(ctx->d_fu_dirty);
    cudaFree(ctx->d_rows); cudaFree(ctx->d_row_cnt); cudaFree(ctx->d_n_raw); cudaFree(ctx->d_hist); cudaFree(ctx->d_blk_count);
    cudaFree(ctx->d_tr_prev); cudaFree(ctx->d_tr_now); cudaFree(ctx->d_tr_rowptr[0]); cudaFree(ctx->d_tr_rowptr[1]); cudaFree(ctx->d_tr_counts); cudaFree(ctx->d_dr_scratch);
    for (int k = 0; k < 5; ++k) cudaFree(ctx->d_t1[k]);
    cudaFree(ctx->d_rank); cudaFree(ctx->d_acc); cudaFree(ctx->d_comp_root); cudaFree(ctx->d_comp_wcount);
    cudaFree(ctx->d_comp_count); cudaFree(ctx->d_best); cudaFree(ctx->d_mgrid);
    cudaFree(ctx->d_fr_sx); cudaFree(ctx->d_fr_sy); cudaFree(ctx->d_fr_labels);
    cudaFree(ctx->d_fr_edges[0]); cudaFree(ctx->d_fr_edges[1]);
    cudaFree(ctx->d_fr_nedges[0]); cudaFree(ctx->d_fr_nedges[1]);
    cudaFree(ctx->d_fr_rowptr[0]); cudaFree(ctx->d_fr_rowptr[1]);
    cudaFree(ctx->d_ff_ccl); cudaFree(ctx->d_ff_maps); cudaFree(ctx->d_ff_tmpcount); cudaFreeHost(ctx->h_ff_count);
    for (int k = 0; k < 2; ++k) { cudaFree(ctx->d_ff_cxy[k]); cudaFree(ctx->d_ff_comp[k]); cudaFree(ctx->d_ff_field[k]); }
    cudaFree(ctx->d_fr_created); cudaFree(ctx->d_fr_destroyed); cudaFree(ctx->d_fr_counts);
    cudaFreeHost(ctx->h_fr_counts); cudaFreeHost(ctx->h_fr_sites); cudaFreeHost(ctx->h_fr_lists);
    for (int k = 0; k < 2; ++k) {
        cudaFree(ctx->d_pp_sx[k]); cudaFree(ctx->d_pp_sy[k]); cudaFree(ctx->d_pp_created[k]);
        cudaFree(ctx->d_pp_destroyed[k]); cudaFree(ctx->d_pp_counts[k]);
        cudaFreeHost(ctx->h_pp_counts[k]); cudaFreeHost(ctx->h_pp_sites[k]);
        if (ctx->pp_ev_in[k]) { cudaEventDestroy(ctx->pp_ev_in[k]); cudaEventDestroy(ctx->pp_ev_done[k]); cudaEventDestroy(ctx->pp_ev_cnt[k]); }
    }
    if (ctx->pp_h2d) { cudaStreamDestroy(ctx->pp_h2d); cudaStreamDestroy(ctx->pp_d2h); cudaStreamDestroy(ctx->pp_lst); }
    cudaFree(ctx->d_flags);
    if (ctx->prof_ev[0][0])
        for (int i = 0; i < kMaxProfLaunches; ++i)
            for (int k = 0; k < 2; ++k) cudaEventDestroy(ctx->prof_ev[i][k]);
    free(ctx);
    return VOR_OK;
}

const char* vor_last_error(const vor_ctx* ctx) { return ctx ? ctx->err : "null context"; }

int vor_download(vor_ctx* ctx, const void* d_src, void* h_dst, int64_t bytes, void* stream_) {
    if (!ctx) return VOR_EINVAL;
    if (!d_src || !h_dst || bytes < 0) return vor_fail(ctx, VOR_EINVAL, "vor_download: null pointer or negative size");
    cudaStream_t stream = (cudaStream_t)stream_;
    VOR_CUDA(cudaMemcpyAsync(h_dst, d_src, (size_t)bytes, cudaMemcpyDeviceToHost, stream));
    VOR_CUDA(cudaStreamSynchronize(stream));
    return VOR_OK;
}

int64_t vor_launch_count(const vor_ctx* ctx) { return ctx ? ctx->launches : 0; }

int64_t vor_stat(vor_ctx* ctx, const char* name) {
    if (!ctx || !name) return VOR_EINVAL;
    if (cudaDeviceSynchronize() != cudaSuccess) return VOR_ECUDA;
    if (!strcmp(name, "label_unproven_quadrants")) {
        if (!ctx->d_lab_fail_n) return 0;
        int32_t v = 0;                                      // the counter the last vor_label call used
        if (cudaMemcpy(&v, ctx->d_lab_fail_n + (1 - ctx->lab_fail_turn), sizeof(v), cudaMemcpyDeviceToHost) != cudaSuccess)
            return VOR_ECUDA;
        return v;
    }
    if (!strcmp(name, "edges_raw_keys") || !strcmp(name, "edges_overflow_keys")) {
        int64_t v[4] = {0, 0, 0, 0};
        if (cudaMemcpy(v, ctx->d_n_raw, sizeof(v), cudaMemcpyDeviceToHost) != cudaSuccess) return VOR_ECUDA;
        return name[6] == 'r' ? v[3] : v[0];
    }
    return vor_fail(ctx, VOR_EINVAL, "unknown statistic");
}

int vor_profile_begin(vor_ctx* ctx) {
    if (!ctx) return VOR_EINVAL;
    if (!ctx->prof_ev[0][0])
        for (int i = 0; i < kMaxProfLaunches; ++i)
            for (int k = 0; k < 2; ++k) VOR_CUDA(cudaEventCreate(&ctx->prof_ev[i][k]));
    ctx->prof_n = 0;
    ctx->prof_on = 1;
    return VOR_OK;
}

int vor_profile_end(vor_ctx* ctx, void* stream, char* names, int32_t names_len, float* ms, int32_t cap) {
    if (!ctx || !names || !ms || names_len < 1 || cap < 0) return VOR_EINVAL;
    ctx->prof_on = 0;
    VOR_CUDA(cudaStreamSynchronize((cudaStream_t)stream));
    int n = ctx->prof_n < cap ? ctx->prof_n : cap;
    int used = 0;
    names[0] = 0;
    for (int i = 0; i < n; ++i) {
        VOR_CUDA(cudaEventElapsedTime(&ms[i], ctx->prof_ev[i][0], ctx->prof_ev[i][1]));
        const int len = (int)strlen(ctx->prof_name[i]);
        if (used + len + 2 > names_len) { n = i; break; }
        memcpy(names + used, ctx->prof_name[i], len);
        names[used + len] = '\n';
        used += len + 1;
        names[used] = 0;
    }
    return n;
}

int vor_set_option(vor_ctx* ctx, const char* name, int64_t value) {
    if (!ctx || !name) return VOR_EINVAL;
    if (!strcmp(name, "bucket_occupancy_x100")) {
        if (value < 1) return vor_fail(ctx, VOR_EINVAL, "bucket_occupancy_x100 must be >= 1");
        ctx->bucket_occ_x100 = value;
        return VOR_OK;
    }
    if (!strcmp(name, "label_halo_x100")) {
        if (value < 0 || value > 1000) return vor_fail(ctx, VOR_EINVAL, "label_halo_x100 must be in [0,1000]");
        ctx->label_halo_x100 = value;
        return VOR_OK;
    }
    if (!strcmp(name, "sites_hint")) {
        if (value < 0 || value > ctx->max_sites) return vor_fail(ctx, VOR_EINVAL, "sites_hint must be in [0, max_sites]");
        ctx->ff_hint = (int32_t)value;
        return VOR_OK;
    }
    if (!strcmp(name, "row_slots")) {
        if (value < 4 || value > kRowStride || value % 4)
            return vor_fail(ctx, VOR_EINVAL, "row_slots must be 4, 8, 12 or 16");
        ctx->row_slots = value;
        return VOR_OK;
    }
    if (!strcmp(name, "fuse")) {
        ctx->fuse = value != 0;
        return VOR_OK;
    }
    if (!strcmp(name, "edges_generic")) {
        ctx->edges_generic = value != 0;
        return VOR_OK;
    }
    if (!strcmp(name, "label_fast_off")) {
        ctx->label_fast_off = value != 0;
        return VOR_OK;
    }
    if (!strcmp(name, "label_path")) {
        if (value < 0 || value > 3) return vor_fail(ctx, VOR_EINVAL, "label_path must be in [0,3]");
        ctx->label_path = value;
        return VOR_OK;
    }
    return vor_fail(ctx, VOR_EINVAL, "unknown option");
}

int vor_sync_status(vor_ctx* ctx, void* stream) {
    if (!ctx) return VOR_EINVAL;
    VOR_CUDA(cudaStreamSynchronize((cudaStream_t)stream));
    int32_t flags = 0;
    VOR_CUDA(cudaMemcpy(&flags, ctx->d_flags, sizeof(flags), cudaMemcpyDeviceToHost));
    if (flags) {
        VOR_CUDA(cudaMemset(ctx->d_flags, 0, sizeof(int32_t)));
        snprintf(ctx->err, sizeof(ctx->err), "capacity exceeded:%s%s%s%s%s",
                 (flags & FLAG_RAWKEY_OVERFLOW) ? " raw-key scratch (max_raw_keys)" : "",
                 (flags & FLAG_EDGE_CAP) ? " edge list" : "",
                 (flags & FLAG_DIFF_CAP) ? " created/destroyed list" : "",
                 (flags & FLAG_COMP_CAP) ? " component arrays" : "",
                 (flags & FLAG_MATCH_CAP) ? " match arrays" : "");
        return VOR_ECAPACITY;
    }
    return VOR_OK;
}

}  // extern "C"

// All adjacency rows empty (the invariant vor_edges relies on between calls).
int vor_reset_rows(vor_ctx* ctx) {
    VOR_CUDA(cudaMemset(ctx->d_row_cnt, 0, (size_t)ctx->max_sites * sizeof(uint32_t)));
    return VOR_OK;
}
