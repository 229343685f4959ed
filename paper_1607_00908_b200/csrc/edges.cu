// a3 + a4 — site-adjacency (digital Delaunay) edge set.
// Paper: the Delaunay graph as an adjacency matrix with one row per label, pre-filled with a
// sentinel (§III.B), filled from the coloured lattice and
// "compressed" by sort + unique per row.  This build's rule (R6,
// BASELINE.json): every 4-connected label discontinuity (right, down, periodic wrap) contributes the
// pair (min,max), packed as (min << 32 | max); the result is the ascending unique list.
//
//   emit    stream the label image once (128-bit loads); every warp compacts the lane-rows that hold a
//           discontinuity into a shared-memory queue and inserts their pairs, 32 records at a time,
//           into a per-CTA hash set; the CTA's distinct pairs go to a global raw-key list.
//   insert  every raw key (a < b) is appended to row a of a global adjacency matrix (kRowStride
//           slots per site): slot = atomicAdd(row counter), plain store.  A pair seen by several
//           CTAs is appended several times; pairs that do not fit (row full, or label >= number of
//           rows) go to an overflow list.
//   finish  ONE cooperative kernel: [only if the overflow list is not empty: radix-sort it, drop
//           duplicates and keys already present in their row] -> every row is sorted in registers,
//           its duplicates dropped, written back and counted -> grid sync -> every row is copied to
//           its final position (merged with its overflow keys, if any); the row counters are reset
//           to 0 on the way.
// The matrix rows are in ascending site order and each row is sorted, so the concatenation IS the
// globally sorted list: no global sort on the common path.
#include <cooperative_groups.h>

#include "common.cuh"
#include "rows.cuh"

namespace cg = cooperative_groups;

namespace {

// ------------------------------------------------------------------------------------ emit
constexpr int kHashSlots = 512;
constexpr int kMaxProbe = 32;
constexpr int kQueueCap = 32 + 256;     // < 32 pending + at most 8 pairs per lane per row

__device__ __forceinline__ uint32_t hash_key(uint32_t a, uint32_t b) {
    uint32_t h = a * 0x9E3779B1u ^ (b * 0x85EBCA77u);
    return h ^ (h >> 15);
}

template <int kSlots = kHashSlots>
__device__ __forceinline__ void hash_insert(uint32_t a, uint32_t b, unsigned long long* table,
                                            const RowSet& rs) {
    const uint32_t lo = min(a, b), hi = max(a, b);
    if (lo == rs.exclude || hi == rs.exclude) return;       // obstacle colour: no edge
    const unsigned long long key = ((unsigned long long)lo << 32) | hi;
    uint32_t h = hash_key(lo, hi) & (kSlots - 1);
    for (int probe = 0; probe < kMaxProbe; ++probe) {
        const unsigned long long cur = table[h];
        if (cur == key) return;
        if (cur == kEmptyKey) {
            const unsigned long long old = atomicCAS(&table[h], kEmptyKey, key);
            if (old == kEmptyKey || old == key) return;
        }
        h = (h + 1) & (kSlots - 1);
    }
    row_insert(rs, lo, hi);    // table crowded (very dense sites): straight to the matrix
}

// ---- streaming kernel (L % 4 == 0, 16-byte aligned image).
// A warp owns a strip of 128 columns x kStripRows rows and walks down it, 4 columns per lane, kPf
// rows in flight per lane (register prefetch; pointers advance by L, no per-row address arithmetic).
// Work is done in three stages of decreasing volume, each one dense over the 32 lanes:
//   A  per row and lane: is any of the lane's 8 compared pairs (cell | right neighbour, row above |
//      cell) a discontinuity?  A few ORs of XORs.  A lane-row that repeats the row above exactly over
//      its 5 columns is skipped: it has no vertical pair and its horizontal pairs are those of the row
//      above, which its owner (this warp, or the warp / CTA above) reports.  The chain ends at
//      row 0 at the latest, which is never skipped, so every distinct pair is reported at least once;
//      the set insertion downstream makes "at least once" enough.  "Dirty" lane-rows are compacted
//      (ballot) into a queue of 9-label records {row, row above, right neighbour}.
//   B  32 records at a time: if the 9 labels take only two values {a, b} - the usual case, one
//      boundary crossing the window - the record contributes exactly the key (a, b): one hash
//      insertion.  Otherwise (a Voronoi vertex nearby) the record moves on to a second queue.
//   C  32 such records at a time: each of the 8 compared pairs that differ is inserted.
// The CTA's hash set ends up holding every distinct key of its tile; it is appended to a global
// raw-key list (one atomic per CTA) that the finish kernel inserts into the adjacency matrix.
constexpr int kStrWarpsX = 2, kStrWarpsY = 2;
constexpr int kStrWarps = kStrWarpsX * kStrWarpsY;
constexpr int kStrThreads = 32 * kStrWarps;                     // 128
constexpr int kStripCols = 128;
constexpr int kStripRows = 32;                                  // rows per warp
constexpr int kPf = 4;                                          // rows in flight per lane
constexpr int kRecCap = 96;                                     // < 32 pending + 2 rows x 32
constexpr int kMultiCap = 64;                                   // < 32 pending + 32 per batch

struct RecQueue {                                               // SoA: conflict-free 128-bit accesses
    int4 c[kRecCap];       // the lane-row's 4 labels
    int4 pc[kRecCap];      // the 4 labels above them
    int32_t rr3[kRecCap];  // right neighbour of c.w
};

struct StreamShared {
    unsigned long long table[kHashSlots];
    RecQueue rec[kStrWarps];
    int32_t multi[kStrWarps][kMultiCap * 9];   // 9 labels per record (c0..c3, rr3, pc0..pc3); odd stride
    int32_t scan[kStrWarps + 1];
};

// Append the CTA's distinct keys to the global raw list (falls back to direct insertion if full).
template <int kSlots = kHashSlots>
__device__ __forceinline__ void hash_flush(const unsigned long long* table, const RowSet& rs,
                                           int32_t* scan /* [warps + 1] */) {
    constexpr int kPer = kSlots / kStrThreads;
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    unsigned long long mine[kPer];
    int cnt = 0;
#pragma unroll
    for (int k = 0; k < kPer; ++k) {
        mine[k] = table[k * kStrThreads + threadIdx.x];
        cnt += mine[k] != kEmptyKey;
    }
    int inc = cnt;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int t = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += t;
    }
    if (lane == 31) scan[wid] = inc;
    __syncthreads();
    int wbase = 0, total = 0;
#pragma unroll
    for (int w = 0; w < kStrWarps; ++w) {
        if (w < wid) wbase += scan[w];
        total += scan[w];
    }
    __shared__ long long base_sh;
    if (threadIdx.x == 0) base_sh = total ? (long long)atomicAdd(rs.n_raw, (unsigned long long)total) : 0;
    __syncthreads();
    // a key whose reserved slot lies beyond the list's capacity goes straight to the matrix, so every
    // slot below min(n_raw, raw_cap) is written and rows_insert_kernel never reads a stale one
    int64_t pos = base_sh + wbase + inc - cnt;
#pragma unroll
    for (int k = 0; k < kPer; ++k) {
        if (mine[k] == kEmptyKey) continue;
        if (pos < rs.raw_cap) rs.raw[pos] = mine[k];
        else row_insert(rs, (uint32_t)(mine[k] >> 32), (uint32_t)mine[k]);
        ++pos;
    }
}

// The image has H rows of W labels (W % 4 == 0); wrap_x / wrap_y: the last column / row is adjacent to the
// first one (periodic axis); otherwise the image ends there (a wall, or the end of a strip of rows).
__global__ void __launch_bounds__(kStrThreads, 8) edges_stream_kernel(const int32_t* __restrict__ labels,
                                                                      int32_t W, int32_t H, int wrap_x, int wrap_y,
                                                                      const RowSet rs) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    StreamShared& sh = *reinterpret_cast<StreamShared*>(smem_raw);
    for (int i = threadIdx.x; i < kHashSlots; i += kStrThreads) sh.table[i] = kEmptyKey;
    __syncthreads();
    const unsigned full = 0xffffffffu;
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const unsigned lt = (1u << lane) - 1u;
    const int32_t xbase = (blockIdx.x * kStrWarpsX + (wid % kStrWarpsX)) * kStripCols;
    const int32_t x0 = xbase + 4 * lane;
    const int32_t ybeg = (blockIdx.y * kStrWarpsY + (wid / kStrWarpsX)) * kStripRows;
    const int32_t yend = min(ybeg + kStripRows, H);
    RecQueue& rq = sh.rec[wid];
    int32_t* __restrict__ mq = sh.multi[wid];
    int rn = 0, mn = 0;                            // warp-uniform queue fills

    // stage C: every differing pair of `take` queued multi-label records.  Pair k < 4 is
    // (label k, label k + 1) of {c0..c3, rr3}; pair k >= 4 is (pc[k-4], c[k-4]) = (label k + 1, label k - 4).
    auto process_multi = [&](int take) {
        mn -= take;
        const int32_t* __restrict__ r = mq + (mn + lane) * 9;
        unsigned bits = 0;                             // bit k: pair k differs
        if (lane < take) {
#pragma unroll
            for (int k = 0; k < 8; ++k) bits |= (unsigned)(r[k < 4 ? k : k + 1] != r[k < 4 ? k + 1 : k - 4]) << k;
        }
        while (__any_sync(full, bits != 0)) {          // every trip is dense over the lanes that still have pairs
            if (bits) {
                const int k = __ffs(bits) - 1;
                bits &= bits - 1;
                hash_insert(r[k < 4 ? k : k + 1], r[k < 4 ? k + 1 : k - 4], sh.table, rs);
            }
        }
        __syncwarp();
    };
    // stage B: one dense pass over `take` queued records
    auto process_recs = [&](int take) {
        rn -= take;
        int4 c = make_int4(0, 0, 0, 0), pc = c;
        int32_t rr3 = 0;
        if (lane < take) { c = rq.c[rn + lane]; pc = rq.pc[rn + lane]; rr3 = rq.rr3[rn + lane]; }
        __syncwarp();
        const uint32_t a = (uint32_t)c.x;
        const uint32_t t1 = c.y ^ a, t2 = c.z ^ a, t3 = c.w ^ a, t4 = rr3 ^ a;
        const uint32_t t5 = pc.x ^ a, t6 = pc.y ^ a, t7 = pc.z ^ a, t8 = pc.w ^ a;
        // two labels {a, b}  <=>  every non-zero t equals the largest one (b = a ^ max t)
        const uint32_t mx = max(max(max(t1, t2), max(t3, t4)), max(max(t5, t6), max(t7, t8)));
        const uint32_t lo = min(min(min(t1 - 1u, t2 - 1u), min(t3 - 1u, t4 - 1u)),
                                min(min(t5 - 1u, t6 - 1u), min(t7 - 1u, t8 - 1u)));   // 0 -> 2^32 - 1
        const bool any = mx != 0, two = lo == mx - 1u;
        if (any && two) hash_insert(a, a ^ mx, sh.table, rs);
        const bool multi = any && !two;
        const unsigned mm = __ballot_sync(full, multi);
        if (mm) {
            if (multi) {
                int32_t* __restrict__ r = mq + (mn + __popc(mm & lt)) * 9;
                r[0] = c.x; r[1] = c.y; r[2] = c.z; r[3] = c.w; r[4] = rr3;
                r[5] = pc.x; r[6] = pc.y; r[7] = pc.z; r[8] = pc.w;
            }
            mn += __popc(mm);
            __syncwarp();
            if (mn >= 32) process_multi(32);
        }
    };

    if (xbase < W && ybeg < H) {                   // warp-uniform
        const bool active = x0 < W;                // W % 4 == 0: a lane's 4 columns are all in or all out
        const bool halo = active && (lane == 31 || x0 + 4 >= W);   // right neighbour not in the next lane
        const uint32_t amask = active ? 0xffffffffu : 0u;
        // inactive lanes (ragged last strip) read a valid address and never report anything
        const uint32_t col = active ? x0 : xbase;
        // beyond the last column: column 0 (periodic) or the last column itself (wall: no pair)
        const uint32_t colh = halo ? (x0 + 4 >= W ? (wrap_x ? 0 : x0 + 3) : x0 + 4) : xbase;
        const int32_t* __restrict__ p = labels + (int64_t)ybeg * W + col;      // load cursors: main, halo
        const int32_t* __restrict__ ph = labels + (int64_t)ybeg * W + colh;
        int4 pc;
        int32_t prr3;
        {
            // above row 0: the last row (periodic) or row 0 itself (no pair)
            const int32_t* __restrict__ up = labels + (int64_t)(ybeg == 0 ? (wrap_y ? H - 1 : 0) : ybeg - 1) * W;
            pc = __ldg(reinterpret_cast<const int4*>(up + col));
            int32_t hup = 0;
            if (halo) hup = __ldg(up + colh);
            const int32_t nb = __shfl_down_sync(full, pc.x, 1);
            prr3 = halo ? hup : nb;
        }
        uint32_t force = ybeg == 0 ? 1u : 0u;      // row 0 ends every chain: nothing is skipped there
        // The load cursor stops on the strip's last row: a ragged strip re-reads it, and a repeated
        // row equals the row above it, so it is never dirty.  Every strip runs kStripRows rows.
        int32_t ahead = yend - ybeg - 1;           // rows below the cursor
        int4 buf[kPf];
        int32_t hb[kPf] = {0, 0, 0, 0};
#pragma unroll
        for (int j = 0; j < kPf; ++j) {
            buf[j] = __ldcs(reinterpret_cast<const int4*>(p));
            if (halo) hb[j] = __ldg(ph);        // only the lane next to the strip border uses it
            const int32_t step = ahead > 0 ? W : 0;
            p += step; ph += step;
            --ahead;
        }
#pragma unroll 1
        for (int it = 0; it < kStripRows / kPf; ++it) {
#pragma unroll
            for (int j = 0; j < kPf; ++j) {
                const int4 c = buf[j];
                const int32_t hc = hb[j];
                buf[j] = __ldcs(reinterpret_cast<const int4*>(p));
                if (halo) hb[j] = __ldg(ph);        // only the lane next to the strip border uses it
                const int32_t step = ahead > 0 ? W : 0;
                p += step; ph += step;
                --ahead;
                const int32_t nb = __shfl_down_sync(full, c.x, 1);
                const int32_t rr3 = halo ? hc : nb;
                const uint32_t dh = (c.x ^ c.y) | (c.y ^ c.z) | (c.z ^ c.w) | (c.w ^ rr3);
                const uint32_t dv = (pc.x ^ c.x) | (pc.y ^ c.y) | (pc.z ^ c.z) | (pc.w ^ c.w);
                uint32_t any = (dv | dh) & amask;
                // dv5 == 0: identical to the row above over the 5 columns -> skipped (see above)
                uint32_t dv5 = dv | (uint32_t)(rr3 ^ prr3) | force;
                asm volatile("" : "+r"(any), "+r"(dv5));     // keep the OR-of-XOR form (LOP3)
                const bool dirty = (any != 0) & (dv5 != 0);
                const unsigned m = __ballot_sync(full, dirty);
                if (m) {
                    if (dirty) {
                        const int pos = rn + __popc(m & lt);
                        rq.c[pos] = c; rq.pc[pos] = pc; rq.rr3[pos] = rr3;
                    }
                    rn += __popc(m);
                }
                pc = c; prr3 = rr3; force = 0;
                if (j & 1) {                       // every second row: at most 31 + 64 records queued
                    __syncwarp();
                    while (rn >= 32) process_recs(32);
                }
            }
        }
        if (rn > 0) process_recs(rn);
        if (mn > 0) process_multi(mn);
    }
    __syncthreads();
    hash_flush(sh.table, rs, sh.scan);
}

// ---- generic kernel (any L, any alignment): scalar loads, every discontinuity goes to the hash set.
constexpr int kEmitThreads = 128;
constexpr int kEmitCols = 128;          // per CTA tile: 32 lanes x 4 labels
constexpr int kEmitRowsPerWarp = 16;
constexpr int kEmitRows = (kEmitThreads / 32) * kEmitRowsPerWarp;   // 128

__global__ void __launch_bounds__(kEmitThreads) edges_emit_kernel(const int32_t* __restrict__ labels,
                                                                  int32_t W, int32_t H, int wrap_x, int wrap_y,
                                                                  const RowSet rs) {
    __shared__ unsigned long long table[kHashSlots];
    __shared__ uint2 queue[kEmitThreads / 32][kQueueCap];
    __shared__ int32_t scan[kEmitThreads / 32 + 1];
    static_assert(kEmitThreads == kStrThreads, "hash_flush is written for one block size");
    for (int i = threadIdx.x; i < kHashSlots; i += kEmitThreads) table[i] = kEmptyKey;
    __syncthreads();
    const unsigned full = 0xffffffffu;
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int32_t x0 = blockIdx.x * kEmitCols + lane * 4;
    const int32_t ybeg = blockIdx.y * kEmitRows + wid * kEmitRowsPerWarp;
    uint2* __restrict__ q = queue[wid];
    int qn = 0;                                    // warp-uniform queue fill
    if (ybeg < H) {
        auto load_row = [&](const int32_t* __restrict__ row, int32_t* v) {
#pragma unroll
            for (int k = 0; k < 4; ++k) v[k] = x0 + k < W ? __ldg(row + x0 + k) : 0;
        };
        int32_t c[4], nx[4];
        load_row(labels + (int64_t)ybeg * W, c);
        const int32_t yend = min(ybeg + kEmitRowsPerWarp, H);
        for (int32_t y = ybeg; y < yend; ++y) {
            const int32_t* __restrict__ row = labels + (int64_t)y * W;
            // below the last row: row 0 (periodic) or the row itself (no pair)
            load_row(labels + (int64_t)(y + 1 == H ? (wrap_y ? 0 : y) : y + 1) * W, nx);
            // right neighbours: next column, next lane's first column, or column 0 through the wrap
            int32_t rr[4] = {c[1], c[2], c[3], __shfl_down_sync(full, c[0], 1)};
            if (lane == 31 && x0 + 4 < W) rr[3] = __ldg(row + x0 + 4);
            if (x0 + 4 >= W && x0 < W) {
                const int32_t first = __ldg(row);
#pragma unroll
                for (int k = 0; k < 4; ++k)
                    if (x0 + k + 1 >= W) rr[k] = wrap_x ? first : c[k];
            }
            unsigned bits = 0;
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                const bool valid = x0 + k < W;
                bits |= (unsigned)(valid && c[k] != rr[k]) << k;
                bits |= (unsigned)(valid && c[k] != nx[k]) << (4 + k);
            }
            const int cnt = __popc(bits);
            int inc = cnt;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int t = __shfl_up_sync(full, inc, o);
                if (lane >= o) inc += t;
            }
            const int total = __shfl_sync(full, inc, 31);
            if (total) {
                int pos = qn + inc - cnt;
#pragma unroll
                for (int k = 0; k < 4; ++k)
                    if (bits & (1u << k)) q[pos++] = make_uint2((uint32_t)c[k], (uint32_t)rr[k]);
#pragma unroll
                for (int k = 0; k < 4; ++k)
                    if (bits & (16u << k)) q[pos++] = make_uint2((uint32_t)c[k], (uint32_t)nx[k]);
                qn += total;
                __syncwarp();
                while (qn >= 32) {
                    qn -= 32;
                    const uint2 it = q[qn + lane];
                    hash_insert(it.x, it.y, table, rs);
                }
                __syncwarp();
            }
#pragma unroll
            for (int k = 0; k < 4; ++k) c[k] = nx[k];
        }
        if (lane < qn) {
            const uint2 it = q[lane];
            hash_insert(it.x, it.y, table, rs);
        }
    }
    __syncthreads();
    hash_flush(table, rs, scan);
}

// ------------------------------------------------------------------------------------ block helpers
constexpr int kSortWarps = kSortThreads / 32;
constexpr int kKeysPerThread = 4;
constexpr int kSubTile = kSortThreads * kKeysPerThread;       // 4096 keys

struct CoopShared {
    uint32_t cnt[kSortWarps][256];     // radix: per-warp digit counts, then per-warp bases
    uint32_t running[256];
    uint32_t wsum[8];
    int64_t red[32];
    int32_t wtot[kSortWarps];
};

// chunk of block b: [b*C, min((b+1)*C, n)), C = ceil(n / gridDim) rounded up to a multiple of `unit`
__device__ __forceinline__ void block_chunk(int64_t n, int64_t unit, int64_t* beg, int64_t* end) {
    int64_t C = (n + gridDim.x - 1) / gridDim.x;
    C = (C + unit - 1) / unit * unit;
    const int64_t b = (int64_t)blockIdx.x * C;
    *beg = b < n ? b : n;
    *end = b + C < n ? b + C : n;
}

// sum over the block, returned to every thread (two barriers)
__device__ __forceinline__ int64_t block_sum_i64(int64_t v, int64_t* sh /* [32] */) {
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    if (lane == 0) sh[wid] = v;
    __syncthreads();
    int64_t t = lane < (int)(blockDim.x >> 5) ? sh[lane] : 0;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
    __syncthreads();
    return t;
}

// (sum of partial[b] for b < me, sum of all) over `count` per-block values
__device__ __forceinline__ void partial_prefix(const int64_t* __restrict__ partial, int count, int me,
                                               int64_t* sh, int64_t* before, int64_t* all) {
    int64_t bf = 0, al = 0;
    for (int b = threadIdx.x; b < count; b += blockDim.x) {
        const int64_t v = __ldcg(partial + b);
        al += v;
        if (b < me) bf += v;
    }
    *before = block_sum_i64(bf, sh);
    *all = block_sum_i64(al, sh);
}

// Order-preserving compaction step for one batch of blockDim.x items: returns this thread's output
// position (valid if keep) and advances *run by the batch total.
__device__ __forceinline__ int64_t compact_pos(bool keep, int64_t* run, int32_t* wtot) {
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const unsigned ball = __ballot_sync(0xffffffffu, keep);
    if (lane == 0) wtot[wid] = __popc(ball);
    __syncthreads();
    int32_t wbase = 0, total = 0;
    for (int w = 0; w < (int)(blockDim.x >> 5); ++w) {
        const int32_t t = wtot[w];
        if (w < wid) wbase += t;
        total += t;
    }
    const int64_t pos = *run + wbase + __popc(ball & ((1u << lane) - 1u));
    *run += total;
    __syncthreads();
    return pos;
}

// ------------------------------------------------------------------------------------ radix sort
struct DigitSpec {
    int label_bits;    // significant bits of each 32-bit half (32 = sort the key as it is)
    int shift;         // 8 * pass
};

__device__ __forceinline__ uint64_t compact_key(uint64_t key, int label_bits) {
    return ((key >> 32) << label_bits) | (key & 0xffffffffull);
}
__device__ __forceinline__ uint32_t digit_of(uint64_t key, DigitSpec ds) {
    return (uint32_t)(compact_key(key, ds.label_bits) >> ds.shift) & 255u;
}

__device__ void radix_hist(const uint64_t* __restrict__ in, int64_t n, DigitSpec ds,
                           uint32_t* __restrict__ hist, CoopShared& sh) {
    if (threadIdx.x < 256) sh.running[threadIdx.x] = 0;
    __syncthreads();
    int64_t beg, end;
    block_chunk(n, kSubTile, &beg, &end);
    for (int64_t i = beg + threadIdx.x; i < end; i += kSortThreads)
        atomicAdd(&sh.running[digit_of(in[i], ds)], 1u);
    __syncthreads();
    if (threadIdx.x < 256) hist[blockIdx.x * 256 + threadIdx.x] = sh.running[threadIdx.x];
    __syncthreads();
}

// stable: every block owns a contiguous chunk, processed front to back
__device__ void radix_scatter(const uint64_t* __restrict__ in, uint64_t* __restrict__ out, int64_t n,
                              DigitSpec ds, const uint32_t* __restrict__ hist, CoopShared& sh) {
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    int64_t beg, end;
    block_chunk(n, kSubTile, &beg, &end);
    // global base of (digit d, this block) = sum over digits < d of all blocks + blocks < me of d
    if (threadIdx.x < 256) {
        const int d = threadIdx.x;
        uint32_t total = 0, before = 0;
        for (int b = 0; b < (int)gridDim.x; ++b) {
            const uint32_t v = __ldcg(hist + b * 256 + d);
            total += v;
            if (b < (int)blockIdx.x) before += v;
        }
        uint32_t inc = total;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t t = __shfl_up_sync(0xffffffffu, inc, o);
            if (lane >= o) inc += t;
        }
        if (lane == 31) sh.wsum[wid] = inc;
        sh.running[d] = inc - total + before;          // completed below with the warp offsets
    }
    __syncthreads();
    if (threadIdx.x < 256) {
        uint32_t off = 0;
        for (int k = 0; k < wid; ++k) off += sh.wsum[k];
        sh.running[threadIdx.x] += off;
    }
    __syncthreads();
    for (int64_t sub = beg; sub < end; sub += kSubTile) {
        for (int i = threadIdx.x; i < kSortWarps * 256; i += kSortThreads) (&sh.cnt[0][0])[i] = 0;
        __syncthreads();
        uint64_t key[kKeysPerThread];
        uint32_t dg[kKeysPerThread], rk[kKeysPerThread];
        const int64_t wbase = sub + (int64_t)wid * (32 * kKeysPerThread);
#pragma unroll
        for (int it = 0; it < kKeysPerThread; ++it) {
            const int64_t i = wbase + it * 32 + lane;
            const bool valid = i < end;
            key[it] = valid ? in[i] : 0;
            dg[it] = valid ? digit_of(key[it], ds) : 256u;
            const unsigned peers = __match_any_sync(0xffffffffu, dg[it]);
            const int leader = __ffs(peers) - 1;
            uint32_t old = 0;
            if (valid && lane == leader) {
                old = sh.cnt[wid][dg[it]];
                sh.cnt[wid][dg[it]] = old + __popc(peers);
            }
            old = __shfl_sync(0xffffffffu, old, leader);
            rk[it] = old + __popc(peers & ((1u << lane) - 1u));
            __syncwarp();
        }
        __syncthreads();
        if (threadIdx.x < 256) {
            const int d = threadIdx.x;
            uint32_t run = sh.running[d];
#pragma unroll 4
            for (int w = 0; w < kSortWarps; ++w) {
                const uint32_t t = sh.cnt[w][d];
                sh.cnt[w][d] = run;
                run += t;
            }
            sh.running[d] = run;
        }
        __syncthreads();
#pragma unroll
        for (int it = 0; it < kKeysPerThread; ++it)
            if (dg[it] < 256u) out[sh.cnt[wid][dg[it]] + rk[it]] = key[it];
        __syncthreads();
    }
}

// LSD radix sort of a[0..n) with b as the pong buffer; passes whose digit is 0 in every key
// (per `mask`, an OR of the compacted keys or any superset) are skipped.  Returns the sorted buffer.
__device__ uint64_t* coop_sort(cg::grid_group& grid, uint64_t* a, uint64_t* b, int64_t n,
                               int label_bits, uint64_t mask, uint32_t* hist, CoopShared& sh) {
    uint64_t* src = a;
    uint64_t* dst = b;
    for (int pass = 0; pass < 8; ++pass) {
        if (((mask >> (8 * pass)) & 255ull) == 0) continue;
        const DigitSpec ds{label_bits, 8 * pass};
        radix_hist(src, n, ds, hist, sh);
        grid.sync();
        radix_scatter(src, dst, n, ds, hist, sh);
        grid.sync();
        uint64_t* t = src; src = dst; dst = t;
    }
    return src;
}

// Ascending unique keys of the sorted list `keys` that satisfy `keep`, written to out[0..cap).
// Returns the number of survivors (to every thread).  Two grid syncs.
template <typename Keep>
__device__ int64_t coop_unique(cg::grid_group& grid, const uint64_t* __restrict__ keys, int64_t n,
                               uint64_t* __restrict__ out, int64_t cap, Keep keep,
                               int64_t* __restrict__ partial, CoopShared& sh) {
    int64_t beg, end;
    block_chunk(n, kSortThreads, &beg, &end);
    int64_t c = 0;
    for (int64_t i = beg + threadIdx.x; i < end; i += kSortThreads) {
        const uint64_t k = keys[i];
        c += (i == 0 || k != keys[i - 1]) && keep(k);
    }
    c = block_sum_i64(c, sh.red);
    if (threadIdx.x == 0) partial[blockIdx.x] = c;
    grid.sync();
    int64_t before, all;
    partial_prefix(partial, gridDim.x, blockIdx.x, sh.red, &before, &all);
    int64_t run = before;
    for (int64_t sub = beg; sub < end; sub += kSortThreads) {
        const int64_t i = sub + threadIdx.x;
        uint64_t k = 0;
        bool head = false;
        if (i < end) {
            k = keys[i];
            head = (i == 0 || k != keys[i - 1]) && keep(k);
        }
        const int64_t pos = compact_pos(head, &run, sh.wtot);
        if (head && pos < cap) out[pos] = k;
    }
    grid.sync();
    return all;
}

struct KeepAll {
    __device__ bool operator()(uint64_t) const { return true; }
};
// overflow key (a, b) is redundant if row a already holds b
struct KeepNotInRow {
    const uint32_t* rows;
    const uint32_t* cnt;
    int32_t n_rows, S;
    __device__ bool operator()(uint64_t key) const {
        const uint32_t a = (uint32_t)(key >> 32), b = (uint32_t)key;
        if (a >= (uint32_t)n_rows) return true;
        const uint32_t* row = rows + (size_t)a * kRowStride;
        const int n = (int)min(__ldcg(cnt + a), (uint32_t)S);
        for (int k = 0; k < n; ++k)
            if (__ldcg(row + k) == b) return false;
        return true;
    }
};

__device__ __forceinline__ int64_t lower_bound_u64(const uint64_t* __restrict__ a, int64_t n, uint64_t key) {
    int64_t lo = 0, hi = n;
    while (lo < hi) {
        const int64_t mid = (lo + hi) >> 1;
        if (a[mid] < key) lo = mid + 1; else hi = mid;
    }
    return lo;
}

// ------------------------------------------------------------------------------------ insert
// The CTAs' distinct keys (raw list) -> adjacency matrix: exact set insertion, full rows overflow.
// One atomic on a 4-byte counter (the counters stay in L2) and one fire-and-forget store per key.
constexpr int kInsertThreads = 256;

__global__ void __launch_bounds__(kInsertThreads) rows_insert_kernel(const RowSet rs) {
    const unsigned long long have = *rs.n_raw;
    const int64_t n_raw = (int64_t)have < rs.raw_cap ? (int64_t)have : rs.raw_cap;
    for (int64_t i = (int64_t)blockIdx.x * kInsertThreads + threadIdx.x; i < n_raw;
         i += (int64_t)gridDim.x * kInsertThreads) {
        const uint64_t key = __ldcs(rs.raw + i);
        row_insert(rs, (uint32_t)(key >> 32), (uint32_t)key);
    }
}

// ------------------------------------------------------------------------------------ finish
template <int N>
__device__ __forceinline__ void bitonic_sort(uint32_t* e) {
#pragma unroll
    for (int k = 2; k <= N; k <<= 1) {
#pragma unroll
        for (int j = k >> 1; j > 0; j >>= 1) {
#pragma unroll
            for (int i = 0; i < N; ++i) {
                const int l = i ^ j;
                if (l > i) {
                    const uint32_t lo = min(e[i], e[l]), hi = max(e[i], e[l]);
                    const bool up = (i & k) == 0;
                    e[i] = up ? lo : hi;
                    e[l] = up ? hi : lo;
                }
            }
        }
    }
}

struct FinishParams {
    RowSet rs;                 // matrix, raw list (keys_b) and overflow list (keys_a)
    uint32_t* rows;
    int32_t n_rows;
    int32_t S;
    uint64_t* keys_a;          // overflow keys (unordered)
    uint64_t* keys_b;          // raw keys of the emit kernel; later the sort's pong buffer
    int64_t keys_cap;
    int64_t* ctl;              // [0] overflow count, [2] OR of the overflow keys, [3] raw key count
    uint32_t* hist;
    int64_t* partial;          // [2 * gridDim]
    uint64_t* out;
    int64_t cap;
    int64_t* n_out;
    int32_t* flags;
    uint32_t* row_ptr;         // optional [n_rows + 1]: offset of each site's first key in `out`
};

__global__ void __launch_bounds__(kSortThreads) edges_finish_kernel(const FinishParams p) {
    __shared__ CoopShared sh;
    cg::grid_group grid = cg::this_grid();
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;

    // (the CTAs' distinct keys were inserted into the adjacency matrix by rows_insert_kernel)
    // ---- overflow keys (normally none): sorted, unique, not already in their row
    const uint64_t* ovf = nullptr;
    int64_t n_ovf = __ldcg(p.ctl) < p.keys_cap ? __ldcg(p.ctl) : p.keys_cap;
    if (n_ovf > 0) {                                   // grid-uniform
        int64_t beg, end;
        block_chunk(n_ovf, kSortThreads, &beg, &end);
        unsigned long long m = 0;
        for (int64_t i = beg + threadIdx.x; i < end; i += kSortThreads) m |= p.keys_a[i];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) m |= __shfl_xor_sync(0xffffffffu, m, o);
        if (lane == 0 && m) atomicOr((unsigned long long*)&p.ctl[2], m);
        grid.sync();
        const uint64_t mask = (uint64_t)__ldcg(&p.ctl[2]);
        uint64_t* sorted = coop_sort(grid, p.keys_a, p.keys_b, n_ovf, 32, mask, p.hist, sh);
        uint64_t* dst = sorted == p.keys_a ? p.keys_b : p.keys_a;
        n_ovf = coop_unique(grid, sorted, n_ovf, dst, p.keys_cap, KeepNotInRow{p.rows, p.rs.cnt, p.n_rows, p.S},
                            p.partial, sh);
        ovf = dst;
    }

    // ---- rows, pass 1: sort every row in registers, drop repeats, write it back, count
    int64_t rbeg, rend;
    block_chunk(p.n_rows, kSortThreads, &rbeg, &rend);
    {
        int64_t c = 0;
        for (int64_t a = rbeg + threadIdx.x; a < rend; a += kSortThreads) {
            const int n = (int)min(__ldcg(p.rs.cnt + a), (uint32_t)p.S);
            if (n == 0) continue;
            uint32_t* row = p.rows + (size_t)a * kRowStride;
            if (n == 1) { c += 1; continue; }              // nothing to sort; the counter is already right
            uint32_t e[kRowStride];
#pragma unroll
            for (int q = 0; q < kRowStride; q += 4) {
                uint4 v = make_uint4(kEmptySlot, kEmptySlot, kEmptySlot, kEmptySlot);
                if (q < n) v = __ldcg(reinterpret_cast<const uint4*>(row + q));
                e[q] = q < n ? v.x : kEmptySlot; e[q + 1] = q + 1 < n ? v.y : kEmptySlot;
                e[q + 2] = q + 2 < n ? v.z : kEmptySlot; e[q + 3] = q + 3 < n ? v.w : kEmptySlot;
            }
            if (n > 8) bitonic_sort<16>(e);
            else if (n > 4) bitonic_sort<8>(e);
            else bitonic_sort<4>(e);
            int m = 0;                                      // ascending, repeats adjacent, padding last
#pragma unroll
            for (int k = 0; k < kRowStride; ++k) {
                if (k < n && (k == 0 || e[k] != e[k - 1])) { row[m] = e[k]; ++m; }
            }
            p.rs.cnt[a] = (uint32_t)m;
            c += m;
        }
        c = block_sum_i64(c, sh.red);
        if (threadIdx.x == 0) p.partial[gridDim.x + blockIdx.x] = c;
    }
    grid.sync();

    // ---- rows, pass 2: copy every row to its final position; reset the counters
    int64_t before, all;
    partial_prefix(p.partial + gridDim.x, gridDim.x, blockIdx.x, sh.red, &before, &all);
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        *p.n_out = all + n_ovf;
        if (all + n_ovf > p.cap) atomicOr(p.flags, FLAG_EDGE_CAP);
    }
    int64_t run = before;
    for (int64_t base = rbeg; base < rend; base += kSortThreads) {
        const int64_t a = base + threadIdx.x;
        int n = 0;
        if (a < rend) {
            n = (int)min(__ldcg(p.rs.cnt + a), (uint32_t)p.S);
            if (n) p.rs.cnt[a] = 0;                        // leave the row empty for the next call
        }
        // exclusive scan of n over the block
        int inc = n;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int t = __shfl_up_sync(0xffffffffu, inc, o);
            if (lane >= o) inc += t;
        }
        if (lane == 31) sh.wtot[wid] = inc;
        __syncthreads();
        int wbase = 0, total = 0;
        for (int w = 0; w < kSortWarps; ++w) {
            const int t = sh.wtot[w];
            if (w < wid) wbase += t;
            total += t;
        }
        int64_t pos = run + wbase + inc - n;
        run += total;
        __syncthreads();
        const uint64_t hi = (uint64_t)a << 32;
        int64_t o0 = 0, o1 = 0;
        if (a < rend && n_ovf > 0) {
            o0 = lower_bound_u64(ovf, n_ovf, hi);
            o1 = lower_bound_u64(ovf, n_ovf, hi + (1ull << 32));
            pos += o0;
        }
        if (a < rend && p.row_ptr) p.row_ptr[a] = (uint32_t)(pos < p.cap ? pos : p.cap);
        if (a < rend && n > 0) {
            const uint32_t* row = p.rows + (size_t)a * kRowStride;
            if (o1 == o0) {
#pragma unroll
                for (int q = 0; q < kRowStride; q += 4) {
                    if (q < n) {
                        const uint4 v = __ldcg(reinterpret_cast<const uint4*>(row + q));
                        const uint32_t e[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
                        for (int k = 0; k < 4; ++k)
                            if (q + k < n && pos + q + k < p.cap) p.out[pos + q + k] = hi | e[k];
                    }
                }
            } else {
                // rare: merge the row with its overflow keys (disjoint by construction)
                int i = 0;
                int64_t j = o0;
                while (i < n || j < o1) {
                    uint64_t key;
                    if (j >= o1 || (i < n && (hi | __ldcg(row + i)) < ovf[j])) key = hi | __ldcg(row + i++);
                    else key = ovf[j++];
                    if (pos < p.cap) p.out[pos] = key;
                    ++pos;
                }
            }
        } else if (a < rend && n_ovf > 0) {
            // an empty row can still own overflow keys only if S == 0, which set_option forbids
        }
    }
    // ---- overflow keys whose smaller label has no row come last
    int64_t t0 = 0;
    if (n_ovf > 0) t0 = lower_bound_u64(ovf, n_ovf, (uint64_t)p.n_rows << 32);
    if (p.row_ptr && blockIdx.x == 0 && threadIdx.x == 0)
        p.row_ptr[p.n_rows] = (uint32_t)(all + t0 < p.cap ? all + t0 : p.cap);
    if (n_ovf > 0) {
        for (int64_t j = t0 + (int64_t)blockIdx.x * kSortThreads + threadIdx.x; j < n_ovf;
             j += (int64_t)gridDim.x * kSortThreads)
            if (all + j < p.cap) p.out[all + j] = ovf[j];
    }
}

// ------------------------------------------------------------------------------------ fused path: seams and left-over tiles
// The labelling kernel (label.cu, fused variant) appends the distinct adjacent pairs found INSIDE every
// 32 x 32 tile to the adjacency rows itself.  What is left:
//   fused_seam_kernel   the pairs across the tile borders.  Line c < L/32: the vertical seam right of tile
//                       column c, from the compact border columns the labelling kernel wrote; the other
//                       L/32 lines: the horizontal seam below tile row c - L/32, rows 32k+31 | 32k+32 of the
//                       label image.  Both are coalesced reads of 1/16 of the image.  A run of the same pair
//                       along a line is reported once per warp; a CTA de-duplicates its 2048 positions
//                       through a small hash set before it touches the rows.
//   fused_dirty_kernel  the tiles the labelling kernel could not finish (an unproven quadrant: their labels
//                       came from the second labelling pass): the pairs inside them, from the label image.
constexpr int kSeamThreads = 256;
constexpr int kSeamPer = 8;                     // positions per thread
constexpr int kSeamSlots = 512;                 // about 200 distinct pairs cross 2048 positions at config 5
constexpr int kTailThreads = 256;
constexpr int kTailSlots = 2048;

__global__ void __launch_bounds__(kSeamThreads) fused_seam_kernel(const int32_t* __restrict__ labels,
                                                                  const int32_t* __restrict__ col_left,
                                                                  const int32_t* __restrict__ col_right,
                                                                  int32_t Lx, int32_t Ly, const RowSet rs) {
    __shared__ unsigned long long table[kSeamSlots];
    const unsigned full = 0xffffffffu;
    const int lane = threadIdx.x & 31;
    const int32_t nt = Lx >> 5, c = blockIdx.y;
    for (int i = threadIdx.x; i < kSeamSlots; i += kSeamThreads) table[i] = kEmptyKey;
    __syncthreads();
    const int32_t* __restrict__ pa;
    const int32_t* __restrict__ pb;
    const int32_t len = c < nt ? Ly : Lx;              // positions along this seam line
    if (c < nt) {
        pa = col_right + (int64_t)c * Ly;
        pb = col_left + (int64_t)(c + 1 == nt ? 0 : c + 1) * Ly;
    } else {
        const int32_t y = 32 * (c - nt) + 31;
        pa = labels + (int64_t)y * Lx;
        pb = labels + (int64_t)(y + 1 == Ly ? 0 : y + 1) * Lx;
    }
    const int32_t i0 = blockIdx.x * (kSeamThreads * kSeamPer) + threadIdx.x;
    int32_t a[kSeamPer], b[kSeamPer];
#pragma unroll
    for (int k = 0; k < kSeamPer; ++k) {           // Lx, Ly % 32 == 0: whole warps are in or out of range
        const int32_t i = i0 + k * kSeamThreads;
        a[k] = i < len ? __ldcs(pa + i) : 0;
        b[k] = i < len ? __ldcs(pb + i) : 0;
    }
#pragma unroll
    for (int k = 0; k < kSeamPer; ++k) {
        const int32_t qa = __shfl_up_sync(full, a[k], 1), qb = __shfl_up_sync(full, b[k], 1);
        if (a[k] != b[k] && (lane == 0 || qa != a[k] || qb != b[k]))
            hash_insert<kSeamSlots>((uint32_t)a[k], (uint32_t)b[k], table, rs);
    }
    __syncthreads();
    for (int i = threadIdx.x; i < kSeamSlots; i += kSeamThreads) {
        const unsigned long long key = table[i];
        if (key != kEmptyKey) row_insert(rs, (uint32_t)(key >> 32), (uint32_t)key);
    }
}

// The pairs inside one 32 x 32 tile from the label image, lane = column, all 32 rows in flight at once.
__device__ __noinline__ void tail_dirty_tile(const int32_t* __restrict__ p, int32_t L, int lane,
                                             unsigned long long* table, const RowSet& rs) {
    const unsigned full = 0xffffffffu;
    int32_t v[32];
#pragma unroll
    for (int r = 0; r < 32; ++r) v[r] = __ldg(p + (int64_t)r * L);
    int32_t upr = 0;                                  // right neighbour of the row above
#pragma unroll
    for (int r = 0; r < 32; ++r) {
        // every shuffle is executed by the whole warp, outside the conditions
        const int32_t cur = v[r], right = __shfl_down_sync(full, cur, 1);
        const int32_t below = v[r < 31 ? r + 1 : 31];
        const int32_t lc = __shfl_up_sync(full, cur, 1), lb = __shfl_up_sync(full, below, 1);
        if (lane < 31 && cur != right && (r == 0 || cur != v[r > 0 ? r - 1 : 0] || right != upr))
            hash_insert<kTailSlots>((uint32_t)cur, (uint32_t)right, table, rs);
        if (r < 31 && cur != below && (lane == 0 || lc != cur || lb != below))
            hash_insert<kTailSlots>((uint32_t)cur, (uint32_t)below, table, rs);
        upr = right;
    }
}

__global__ void __launch_bounds__(kTailThreads) fused_dirty_kernel(const int32_t* __restrict__ labels,
                                                                   const int32_t* __restrict__ dirty_tiles,
                                                                   const int32_t* __restrict__ dirty_count,
                                                                   int32_t L, const RowSet rs) {
    __shared__ unsigned long long table[kTailSlots];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int32_t nt = L >> 5, n = *dirty_count;           // L = Lx: tiles per tile row, label pitch
    if ((int32_t)(blockIdx.x * (kTailThreads / 32)) >= n) return;
    for (int i = threadIdx.x; i < kTailSlots; i += kTailThreads) table[i] = kEmptyKey;
    __syncthreads();
    for (int32_t t = blockIdx.x * (kTailThreads / 32) + wid; t < n; t += gridDim.x * (kTailThreads / 32)) {
        const int32_t tile = dirty_tiles[t];
        tail_dirty_tile(labels + (int64_t)(tile / nt) * 32 * L + (tile % nt) * 32 + lane, L, lane, table, rs);
    }
    __syncthreads();
    for (int i = threadIdx.x; i < kTailSlots; i += kTailThreads) {
        const unsigned long long key = table[i];
        if (key != kEmptyKey) row_insert(rs, (uint32_t)(key >> 32), (uint32_t)key);
    }
}

// ------------------------------------------------------------------------------------ plain sort + unique
struct SortUniqueParams {
    uint64_t* keys_a;
    uint64_t* keys_b;
    const int64_t* n_in;
    int64_t keys_cap;
    int label_bits;
    uint32_t* hist;
    int64_t* partial;
    uint64_t* out;
    int64_t cap;
    int64_t* n_out;
    int32_t* flags;
    int flag_bit;
};

__global__ void __launch_bounds__(kSortThreads) sort_unique_kernel(const SortUniqueParams p) {
    __shared__ CoopShared sh;
    cg::grid_group grid = cg::this_grid();
    const int64_t n = __ldcg(p.n_in) < p.keys_cap ? __ldcg(p.n_in) : p.keys_cap;
    const int bits = 2 * p.label_bits;
    const uint64_t mask = bits >= 64 ? ~0ull : ((1ull << bits) - 1ull);
    uint64_t* sorted = coop_sort(grid, p.keys_a, p.keys_b, n, p.label_bits, mask, p.hist, sh);
    const int64_t all = coop_unique(grid, sorted, n, p.out, p.cap, KeepAll{}, p.partial, sh);
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        *p.n_out = all;
        if (all > p.cap) atomicOr(p.flags, p.flag_bit);
    }
}

}  // namespace

// Sort the *d_n_in keys held in ctx->d_keys_a (d_keys_in_a must be that buffer) and write the
// ascending unique list to d_out[0..cap), its length to *d_n_out.  key_bits = significant bits of
// each 32-bit half.  Uses ctx->d_keys_b as the pong buffer.  One cooperative launch.
int vor_sort_unique_keys(vor_ctx* ctx, uint64_t* d_keys_in_a, const int64_t* d_n_in, int key_bits,
                         uint64_t* d_out, int64_t cap, int64_t* d_n_out, int flag_bit,
                         int64_t n_hint, cudaStream_t stream) {
    SortUniqueParams p{d_keys_in_a, ctx->d_keys_b, d_n_in, ctx->max_raw_keys, key_bits, ctx->d_hist,
                       ctx->d_blk_count, d_out, cap, d_n_out, ctx->d_flags, flag_bit};
    int grid = vor_coop_grid(ctx, 1, (const void*)sort_unique_kernel, kSortThreads, 1);
    // short lists: fewer blocks make the grid synchronisations cheaper (any grid size is correct)
    if (n_hint > 0) {
        const int64_t want = (n_hint + kSubTile - 1) / kSubTile;
        if (want < grid) grid = want < 1 ? 1 : (int)want;
    }
    VOR_LAUNCH_COOP(sort_unique_kernel, grid, kSortThreads, stream, (void*)&p);
    return VOR_OK;
}

// The RowSet of this context: adjacency matrix, raw-key list (keys_b) and overflow list (keys_a).
RowSet vor_row_set(vor_ctx* ctx) {
    RowSet rs;
    rs.rows = ctx->d_rows;
    rs.cnt = ctx->d_row_cnt;
    rs.n_rows = ctx->n_sites > 0 ? ctx->n_sites : ctx->max_sites;
    rs.S = (int32_t)ctx->row_slots;
    rs.ovf = ctx->d_keys_a;
    rs.ovf_cap = ctx->max_raw_keys;
    rs.n_ovf = (unsigned long long*)ctx->d_n_raw;
    rs.raw = ctx->d_keys_b;
    rs.raw_cap = ctx->max_raw_keys;
    rs.n_raw = (unsigned long long*)&ctx->d_n_raw[3];
    rs.flags = ctx->d_flags;
    rs.exclude = 0xffffffffu;
    return rs;
}

int vor_edges_fused_tail(vor_ctx* ctx, const int32_t* d_labels, const RowSet& rs, cudaStream_t stream) {
    const int32_t Lx = ctx->Lx, Ly = ctx->Ly, ntx = Lx / 32, nty = Ly / 32;
    const int32_t* col_left = ctx->d_fu_cols;
    const int32_t* col_right = ctx->d_fu_cols + (size_t)ntx * Ly;
    const int32_t longest = Lx > Ly ? Lx : Ly;
    const dim3 grid((longest + kSeamThreads * kSeamPer - 1) / (kSeamThreads * kSeamPer), ntx + nty);
    VOR_LAUNCH(fused_seam_kernel, grid, kSeamThreads, 0, stream, d_labels, col_left, col_right, Lx, Ly, rs);
    VOR_LAUNCH(fused_dirty_kernel, 4 * ctx->num_sms, kTailThreads, 0, stream, d_labels, ctx->d_fu_dirty,
               (const int32_t*)&ctx->d_n_raw[4], Lx, rs);
    return VOR_OK;
}

// [insert the raw keys into the matrix, then] sort / merge / concatenate the rows (see the file header)
int vor_edges_finish(vor_ctx* ctx, const RowSet& rs, uint64_t* d_edges, int64_t cap, int64_t* d_n_edges,
                     uint32_t* d_row_ptr, bool have_raw, cudaStream_t stream) {
    FinishParams fp{rs, ctx->d_rows, rs.n_rows, rs.S, ctx->d_keys_a, ctx->d_keys_b, ctx->max_raw_keys,
                    ctx->d_n_raw, ctx->d_hist, ctx->d_blk_count, d_edges, cap, d_n_edges, ctx->d_flags, d_row_ptr};
    if (have_raw) VOR_LAUNCH(rows_insert_kernel, 8 * ctx->num_sms, kInsertThreads, 0, stream, rs);
    const int fgrid = vor_coop_grid(ctx, 0, (const void*)edges_finish_kernel, kSortThreads, 1);
    VOR_LAUNCH_COOP(edges_finish_kernel, fgrid, kSortThreads, stream, (void*)&fp);
    return VOR_OK;
}

// labels: n_rows rows of Lx labels; wrap_y: the last row is adjacent to the first one
static int edges_image(vor_ctx* ctx, const int32_t* d_labels, int32_t n_rows, int wrap_y, int32_t exclude,
                       uint64_t* d_edges, int64_t cap, int64_t* d_n_edges, uint32_t* d_row_ptr,
                       cudaStream_t stream) {
    VOR_CUDA(cudaMemsetAsync(ctx->d_n_raw, 0, 8 * sizeof(int64_t), stream));
    const int32_t W = ctx->Lx, H = n_rows;
    RowSet rs = vor_row_set(ctx);
    if (exclude >= 0) rs.exclude = (uint32_t)exclude;
    const bool vec = (W % 4 == 0) && (((uintptr_t)d_labels & 15) == 0) && !ctx->edges_generic;
    if (vec) {
        static_assert(sizeof(StreamShared) <= 27 * 1024, "eight CTAs per SM");
        VOR_CUDA(cudaFuncSetAttribute(edges_stream_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                      (int)sizeof(StreamShared)));
        dim3 grid((W + kStrWarpsX * kStripCols - 1) / (kStrWarpsX * kStripCols),
                  (H + kStrWarpsY * kStripRows - 1) / (kStrWarpsY * kStripRows));
        VOR_LAUNCH(edges_stream_kernel, grid, kStrThreads, sizeof(StreamShared), stream, d_labels, W, H,
                   ctx->per_x, wrap_y, rs);
    } else {
        dim3 grid((W + kEmitCols - 1) / kEmitCols, (H + kEmitRows - 1) / kEmitRows);
        VOR_LAUNCH(edges_emit_kernel, grid, kEmitThreads, 0, stream, d_labels, W, H, ctx->per_x, wrap_y, rs);
    }
    return vor_edges_finish(ctx, rs, d_edges, cap, d_n_edges, d_row_ptr, true, stream);
}

extern "C" int vor_edges(vor_ctx* ctx, const int32_t* d_labels, uint64_t* d_edges, int64_t cap,
                         int64_t* d_n_edges, void* stream_) {
    return vor_edges_rows(ctx, d_labels, d_edges, cap, d_n_edges, nullptr, stream_);
}

extern "C" int vor_edges_rows(vor_ctx* ctx, const int32_t* d_labels, uint64_t* d_edges, int64_t cap,
                              int64_t* d_n_edges, uint32_t* d_row_ptr, void* stream_) {
    if (!ctx) return VOR_EINVAL;
    if (int drc_ = vor_check_device(ctx)) return drc_;
    return vor_edges_image(ctx, d_labels, ctx->Ly, ctx->per_y, -1, d_edges, cap, d_n_edges, d_row_ptr, stream_);
}

extern "C" int vor_edges_image(vor_ctx* ctx, const int32_t* d_labels, int32_t n_rows, int32_t wrap_y,
                               int32_t exclude, uint64_t* d_edges, int64_t cap, int64_t* d_n_edges,
                               uint32_t* d_row_ptr, void* stream_) {
    if (!ctx) return VOR_EINVAL;
    if (int drc_ = vor_check_device(ctx)) return drc_;
    if (!d_labels || !d_edges || !d_n_edges || cap < 0)
        return vor_fail(ctx, VOR_EINVAL, "vor_edges: null pointer or negative capacity");
    if (n_rows < 1) return vor_fail(ctx, VOR_EINVAL, "vor_edges_image: n_rows must be >= 1");
    if (d_row_ptr && cap > 0xffffffffll)
        return vor_fail(ctx, VOR_EINVAL, "vor_edges_rows: row offsets are 32-bit, cap must be < 2^32");
    return edges_image(ctx, d_labels, n_rows, wrap_y != 0, exclude, d_edges, cap, d_n_edges, d_row_ptr,
                       (cudaStream_t)stream_);
}

// Obstacle sites take a fixed large colour instead of a bubble's label (§III.B.1: "a
// supplementary binary field which takes the value 1 on those sites which are considered obstacles ... we can
// set their colour to be a fixed large number, MAXLINK").  Pass the same colour as `exclude` to vor_edges_image.
namespace {
__global__ void paint_obstacles_kernel(const uint8_t* __restrict__ mask, int32_t colour, int64_t n,
                                       int32_t* __restrict__ labels) {
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x)
        if (mask[i]) labels[i] = colour;
}
}  // namespace

extern "C" int vor_paint_obstacles(vor_ctx* ctx, const uint8_t* d_mask, int32_t colour, int32_t* d_labels,
                                   int32_t n_rows, void* stream_) {
    if (!ctx) return VOR_EINVAL;
    if (int drc_ = vor_check_device(ctx)) return drc_;
    if (!d_mask || !d_labels) return vor_fail(ctx, VOR_EINVAL, "vor_paint_obstacles: null pointer");
    if (colour < 0 || n_rows < 1) return vor_fail(ctx, VOR_EINVAL, "vor_paint_obstacles: colour >= 0, n_rows >= 1");
    const int64_t n = (int64_t)ctx->Lx * n_rows;
    const int grid = (int)((n + 255) / 256 < 8 * kNumSMs ? (n + 255) / 256 : 8 * kNumSMs);
    VOR_LAUNCH(paint_obstacles_kernel, grid, 256, 0, (cudaStream_t)stream_, d_mask, colour, n, d_labels);
    return VOR_OK;
}
