// Adjacency rows shared by the kernels that find label discontinuities (edges.cu: from a label image;
// label.cu, fused variant: straight from the labelling kernel's registers): row a of the matrix collects the
// larger-index neighbours b of site a (§III.B: one row per label, pre-filled with a
// sentinel).  See edges.cu for how the rows become the sorted edge list.
#pragma once

#include "common.cuh"

constexpr uint64_t kEmptyKey = ~0ull;

struct RowSet {
    uint32_t* rows;            // [n_rows * kRowStride]
    uint32_t* cnt;             // [n_rows] entries appended to each row (may exceed S: the excess overflowed)
    int32_t n_rows;
    int32_t S;                 // slots used per row
    uint64_t* ovf;             // overflow keys (unordered, may repeat)
    int64_t ovf_cap;
    unsigned long long* n_ovf;
    uint64_t* raw;             // per-CTA distinct keys, appended by the emit kernels
    int64_t raw_cap;
    unsigned long long* n_raw;
    int32_t* flags;
    uint32_t exclude;          // label that takes part in no edge (obstacle colour), 0xffffffff = none
};

__device__ __forceinline__ void ovf_push(const RowSet& rs, uint32_t a, uint32_t b) {
    const unsigned long long pos = atomicAdd(rs.n_ovf, 1ull);
    if ((int64_t)pos < rs.ovf_cap) rs.ovf[pos] = ((uint64_t)a << 32) | b;
    else atomicOr(rs.flags, FLAG_RAWKEY_OVERFLOW);
}

// Append b to row a (a < b).  The row may receive the same b more than once (from different CTAs):
// the finish kernel drops the repeats when it sorts the row.
__device__ __forceinline__ void row_insert(const RowSet& rs, uint32_t a, uint32_t b) {
    if (a == rs.exclude || b == rs.exclude) return;
    if (a < (uint32_t)rs.n_rows) {
        const uint32_t slot = atomicAdd(rs.cnt + a, 1u);
        if (slot < (uint32_t)rs.S) {
            rs.rows[(size_t)a * kRowStride + slot] = b;
            return;
        }
    }
    ovf_push(rs, a, b);
}

// host side (edges.cu)
RowSet vor_row_set(vor_ctx* ctx);
int vor_edges_finish(vor_ctx* ctx, const RowSet& rs, uint64_t* d_edges, int64_t cap, int64_t* d_n_edges,
                     uint32_t* d_row_ptr, bool have_raw, cudaStream_t stream);
// fused label -> edge path: label.cu labels and extracts the pairs inside the 32 x 32 tiles, edges.cu
// adds the tile seams and the tiles the labelling kernel could not finish
bool vor_label_fusable(const vor_ctx* ctx);
int vor_label_fused(vor_ctx* ctx, int32_t* d_labels, const RowSet& rs, cudaStream_t stream);
int vor_edges_fused_tail(vor_ctx* ctx, const int32_t* d_labels, const RowSet& rs, cudaStream_t stream);
