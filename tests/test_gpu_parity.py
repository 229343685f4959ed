"""-m gpu: element-by-element parity of the CUDA path (through the C ABI) with the CPU oracle.

Integer / index work: bit-exact.  Centroids (float64): |diff| <= 1e-9 lattice units (north_star).
"""
import zlib

import numpy as np
import pytest

import oracle
from helpers import FP, hex_sites, pack, pairs, read_golden, rhombus_sites
from paper_1607_00908_b200 import workloads as W

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def G():
    import gpu_util
    return gpu_util


def make(L, max_sites, **kw):
    from paper_1607_00908_b200.binding import Vor
    return Vor(L, max_sites, **kw)


def rnd(seed, L, n):
    rng = np.random.default_rng(seed)
    return rng.integers(0, FP * L, n).astype(np.int32), rng.integers(0, FP * L, n).astype(np.int32)


# ------------------------------------------------------------------ labels (a1 + a2)
def check_labels(G, L, sx, sy, paths=(0, 1, 2, 3), ref=None, occ=None):
    ref = oracle.label_brute(L, sx, sy) if ref is None else ref
    v = make(L, max(len(sx), 1))
    if occ:
        v.vor_set_option("bucket_occupancy_x100", occ)
    for path in paths:
        for fast_off in ((0, 1) if path in (0, 2) else (0,)):
            v.vor_set_option("label_path", path)
            v.vor_set_option("label_fast_off", fast_off)
            got = G.gpu_labels(v, sx, sy)
            bad = np.argwhere(got != ref)
            assert len(bad) == 0, f"path {path} fast_off {fast_off}: {len(bad)} cells differ, first {bad[:5].tolist()}"
    v.close()


def test_labels_config1_both_frames(G):
    w = W.config(1)
    for sx, sy in w.frames():
        check_labels(G, w.L, sx, sy)


def test_labels_config2_two_frames(G):
    w = W.config(2)
    for sx, sy in w.frames(2):
        check_labels(G, w.L, sx, sy)


@pytest.mark.parametrize("L,n,halo", [(16, 4, 130), (16, 2, 1000), (32, 9, 130), (48, 20, 400), (75, 30, 130),
                                        (75, 3, 1000), (96, 12, 700), (128, 5, 1000)])
def test_labels_small_lattices_where_the_halo_exceeds_the_period(G, L, n, halo):
    """on small lattices the gather halo of the CTA path (above all the retry's 2 * halo + bucket width) is
    larger than half a period or than the period itself; the kernel must refuse such a region up front (no negative
    argument to its bucket division, no int32 overflow in the span test) and fall back - same labels on every path,
    for the default and for very wide halos."""
    rng = np.random.default_rng(1000 * L + n)
    sx, sy = rng.integers(0, FP * L, n).astype(np.int32), rng.integers(0, FP * L, n).astype(np.int32)
    ref = oracle.label_brute(L, sx, sy)
    v = make(L, n)
    v.vor_set_option("label_halo_x100", halo)
    for path in (3, 2, 0):
        v.vor_set_option("label_path", path)
        got = G.gpu_labels(v, sx, sy)
        assert np.array_equal(got, ref), (path, int((got != ref).sum()))
    v.close()


@pytest.mark.parametrize("L", [512, 1024])
def test_labels_scaled_config5(G, L):
    w = W.scaled(5, L)
    fr = list(w.frames(6))
    for sx, sy in (fr[0], fr[5]):
        check_labels(G, L, sx, sy, ref=oracle.label_cells(L, sx, sy, 16))


ADVERSARIAL = [
    ("single", 64, lambda rng, P: (np.array([5], np.int32), np.array([P - 1], np.int32))),
    ("one_bucket", 64, lambda rng, P: (rng.integers(0, 8 * FP, 30).astype(np.int32),
                                       rng.integers(0, 8 * FP, 30).astype(np.int32))),
    ("empty_quadrants", 256, lambda rng, P: (rng.integers(0, P // 4, 200).astype(np.int32),
                                             rng.integers(P // 2, 3 * P // 4, 200).astype(np.int32))),
    ("corners", 64, lambda rng, P: (np.array([0, P - 1, 0, P - 1], np.int32),
                                    np.array([0, 0, P - 1, P - 1], np.int32))),
    ("lattice_aligned_ties", 256, lambda rng, P: ((rng.integers(0, 16, 150) * 16 * FP + 128).astype(np.int32),
                                                  (rng.integers(0, 16, 150) * 16 * FP + 128).astype(np.int32))),
    ("regular_grid_all_ties", 256, lambda rng, P: (np.tile(np.arange(16) * 16 * FP, 16).astype(np.int32),
                                                   np.repeat(np.arange(16) * 16 * FP, 16).astype(np.int32))),
    ("regular_grid_reversed_indices", 256, lambda rng, P: (np.tile(np.arange(16) * 16 * FP, 16)[::-1].astype(np.int32).copy(),
                                                            np.repeat(np.arange(16) * 16 * FP, 16)[::-1].astype(np.int32).copy())),
    ("half_cell_grid_shuffled", 512, lambda rng, P: tuple(a.astype(np.int32) for a in (lambda o: (
        (np.tile(np.arange(32) * 16 * FP + 128, 32))[o], (np.repeat(np.arange(32) * 16 * FP + 128, 32))[o]))(rng.permutation(1024)))),
    ("dense", 48, lambda rng, P: (rng.integers(0, P, 3000).astype(np.int32),
                                  rng.integers(0, P, 3000).astype(np.int32))),
    ("duplicates", 128, lambda rng, P: (np.repeat(rng.integers(0, P, 40), 3).astype(np.int32),
                                        np.repeat(rng.integers(0, P, 40), 3).astype(np.int32))),
    ("cluster_plus_void", 512, lambda rng, P: (np.concatenate([rng.integers(0, P // 16, 300), rng.integers(0, P, 30)]).astype(np.int32),
                                               np.concatenate([rng.integers(0, P // 16, 300), rng.integers(0, P, 30)]).astype(np.int32))),
]


@pytest.mark.parametrize("name,L,gen", ADVERSARIAL, ids=[a[0] for a in ADVERSARIAL])
def test_labels_adversarial(G, name, L, gen):
    import zlib
    rng = np.random.default_rng(zlib.crc32(name.encode()))          # the same inputs in every process
    sx, sy = gen(rng, FP * L)
    check_labels(G, L, sx, sy)


@pytest.mark.parametrize("L,n", [(100, 40), (250, 434), (17, 5), (2, 1), (2, 3), (333, 3000), (1000, 3000)])
def test_labels_ragged_lattices(G, L, n):
    sx, sy = rnd(L * 7 + n, L, n)
    check_labels(G, L, sx, sy)


@pytest.mark.parametrize("occ", [25, 400])
def test_labels_bucket_size_independent(G, occ):
    w = W.scaled(5, 512)
    sx, sy = next(iter(w.frames(1)))
    check_labels(G, 512, sx, sy, occ=occ)


@pytest.mark.parametrize("halo", [0, 30, 60, 150, 400])
def test_labels_halo_independent(G, halo):
    """The fast path's halo is a performance knob: too small a halo must fall back, never mislabel."""
    w = W.scaled(5, 512)
    sx, sy = list(w.frames(4))[3]
    ref = oracle.label_cells(512, sx, sy, 16)
    v = make(512, len(sx))
    v.vor_set_option("label_halo_x100", halo)
    for path in (2, 3):
        v.vor_set_option("label_path", path)
        assert np.array_equal(G.gpu_labels(v, sx, sy), ref)
    v.close()


def test_labels_hex_and_rhombus_constructions(G):
    g = read_golden("hex_lattice.txt")
    sx, sy = hex_sites(g["L"][0], g["cols"][0], g["rows"][0], g["jitter"][0], seed=3)
    check_labels(G, g["L"][0], sx, sy)
    sx, sy = rhombus_sites(256, 24)        # exactly cocircular rhombus: ties along Voronoi edges
    check_labels(G, 256, sx, sy)


# ------------------------------------------------------------------ edges (a3 + a4)
def check_edges(G, labels, max_sites, row_slots=(16,)):
    L = labels.shape[0]
    v = make(L, max_sites)
    ref = oracle.edges(labels)
    for s in row_slots:
        v.vor_set_option("row_slots", s)
        for generic in (0, 1, 0):                      # repeated: the rows must be left empty
            v.vor_set_option("edges_generic", generic)
            got = G.gpu_edges(v, labels, cap=max(1024, 2 * L * L))
            assert got.dtype == np.uint64 and np.array_equal(got, ref), (s, generic, len(got), len(ref))
    v.close()


def test_edges_hand_images(G):
    lab = np.array([[3, 3, 7, 7], [3, 3, 7, 7], [3, 5, 7, 7], [3, 3, 7, 7]], dtype=np.int32)
    check_edges(G, lab, 8)
    check_edges(G, np.full((6, 6), 9, np.int32), 16)           # no edges at all
    lab = np.zeros((6, 6), np.int32); lab[:, 5] = 2; lab[5, :] = 4   # wrap-only adjacency
    check_edges(G, lab, 8)
    rng = np.random.default_rng(0)
    check_edges(G, rng.integers(0, 1000, (37, 37)).astype(np.int32), 1000)      # ragged, noise labels
    check_edges(G, rng.integers(0, 2 ** 31 - 1, (64, 64)).astype(np.int32), 1)  # 31-bit labels
    check_edges(G, rng.integers(0, 50000, (256, 256)).astype(np.int32), 50000)  # hash-set overflow path
    check_edges(G, rng.integers(0, 3, (4, 4)).astype(np.int32), 3)              # one lane, halo = column 0
    check_edges(G, rng.integers(0, 9, (132, 132)).astype(np.int32), 9)          # ragged strips, noisy rows
    lab = np.zeros((520, 520), np.int32); lab[:, 130:391] = 1; lab[259:262, :] = 2   # long straight boundaries
    lab[300:, 128] = 3; lab[77, 3:9] = 4
    check_edges(G, lab, 5)


@pytest.mark.parametrize("cfg,L", [(1, None), (2, None), (5, 512), (5, 1000), (5, 2048)])
def test_edges_on_oracle_labels(G, cfg, L):
    w = W.config(cfg) if L is None else W.scaled(cfg, L)
    sx, sy = next(iter(w.frames(1)))
    lab = oracle.label_cells(w.L, sx, sy, 8)
    check_edges(G, lab, w.n_sites, row_slots=(16, 4))   # 4 slots: many rows spill to the overflow path


def test_edges_overflow_paths(G):
    """Rows that overflow, labels beyond the row range, and both at once."""
    rng = np.random.default_rng(11)
    # a hub: label 0 touches 300 other labels (row 0 overflows for any slot count)
    lab = np.zeros((64, 64), np.int32)
    ys, xs = np.nonzero((np.arange(64)[:, None] % 3 == 1) & (np.arange(64)[None, :] % 3 == 1))
    lab[ys[:300], xs[:300]] = 1 + np.arange(300)
    check_edges(G, lab, 400, row_slots=(16, 8, 4))
    # max_sites smaller than the largest label: pairs whose smaller label has no row
    check_edges(G, rng.integers(0, 500, (96, 96)).astype(np.int32), 100, row_slots=(16, 4))
    check_edges(G, rng.integers(0, 40, (200, 200)).astype(np.int32), 40, row_slots=(16, 12, 4))
    # stripes: every label has exactly two neighbours, one of them through the wrap
    check_edges(G, np.repeat(np.arange(50, dtype=np.int32), 4)[None, :].repeat(200, 0), 50)


def test_edges_capacity_overflow_is_reported(G):
    from paper_1607_00908_b200.binding import VorError, VOR_ECAPACITY
    w = W.scaled(5, 512)
    sx, sy = next(iter(w.frames(1)))
    lab = oracle.label_cells(w.L, sx, sy, 16)
    ref = oracle.edges(lab)
    v = make(w.L, w.n_sites)
    d = G.dev(lab.ravel())
    out = torch.full((100,), -1, dtype=torch.int64, device="cuda")
    guard = out[90:]                                   # cap = 90: entries beyond must stay untouched
    n = torch.zeros(1, dtype=torch.int64, device="cuda")
    v.lib.vor_edges(v.h, d.data_ptr(), out.data_ptr(), 90, n.data_ptr(), None)
    with pytest.raises(VorError) as e:
        v.vor_sync_status()
    assert e.value.status == VOR_ECAPACITY
    assert int(n.item()) == len(ref)                   # required count is reported
    assert np.array_equal(G.u64(out, 90), ref[:90]) and bool((guard == -1).all())
    v.vor_sync_status()                                # sticky flag was cleared
    v.close()


def test_edges_tiny_raw_key_scratch_is_still_exact(G):
    """max_raw_keys far below the number of CTA-distinct keys: the emit kernels' raw list fills up and the
    remaining keys go straight to the adjacency rows; the result must not change."""
    w = W.scaled(5, 1024)
    sx, sy = next(iter(w.frames(1)))
    lab = oracle.label_cells(w.L, sx, sy, 16)
    ref = oracle.edges(lab)
    for generic in (0, 1):
        v = make(w.L, w.n_sites, max_raw_keys=1000)
        v.vor_set_option("edges_generic", generic)
        for _ in range(2):                              # twice: stale keys of the first call must not leak
            assert np.array_equal(G.gpu_edges(v, lab, cap=len(ref) + 10), ref)
        v.close()


def row_offsets(keys, n_rows):
    """row_ptr by definition: offset of the first key whose smaller label is >= a."""
    return np.searchsorted(keys >> np.uint64(32), np.arange(n_rows + 1, dtype=np.uint64), side="left")


@pytest.mark.parametrize("slots", [16, 4])
def test_edges_rows_offsets_and_row_diff(G, slots):
    """vor_edges_rows returns the compressed adjacency matrix; vor_diff_rows compares
    two of them row by row.  Also with rows that spilled to the sorted overflow path (4 slots)."""
    w = W.scaled(5, 1024)
    v = make(w.L, w.n_sites)
    v.vor_set_option("row_slots", slots)
    lists = []
    for sx, sy in w.frames(3):
        lab = oracle.label_cells(w.L, sx, sy, 16)
        e, ptr = G.gpu_edges_rows(v, lab, w.n_sites)
        ref = oracle.edges(lab)
        assert np.array_equal(e, ref)
        assert np.array_equal(ptr, row_offsets(ref, w.n_sites))
        lists.append((e, ptr))
    empty = (np.empty(0, np.uint64), np.zeros(w.n_sites + 1, np.int64))
    for (a, pa), (b, pb) in ((empty, lists[0]), (lists[0], lists[1]), (lists[1], lists[2]), (lists[2], lists[2]),
                             (lists[2], empty)):
        c, d = G.gpu_diff_rows(v, a, pa, b, pb, w.n_sites)
        rc, rd = oracle.diff(a, b)
        assert np.array_equal(c, rc) and np.array_equal(d, rd)
    v.close()


def test_diff_rows_long_rows_and_random_graphs(G):
    """Rows longer than the in-register path (hubs), empty rows, several batches per block."""
    rng = np.random.default_rng(23)
    v = make(64, 64)
    for n, m in ((1, 0), (5, 6), (300, 2000), (3000, 9000), (700000, 2000000)):
        def graph(hub):
            i = rng.integers(0, n, m); j = rng.integers(0, n, m)
            if hub and n > 100:                            # vertex 3 touches ~half of the others: a long row
                i = np.concatenate([i, np.full(n // 2, 3)]); j = np.concatenate([j, rng.integers(0, n, n // 2)])
            keep = i != j
            lo, hi = np.minimum(i, j)[keep].astype(np.uint64), np.maximum(i, j)[keep].astype(np.uint64)
            return np.unique((lo << np.uint64(32)) | hi)
        a = graph(True)
        b = np.unique(np.concatenate([a[rng.random(len(a)) < 0.9], graph(False)[: max(1, m // 10)]])) if m else a
        c, d = G.gpu_diff_rows(v, a, row_offsets(a, n), b, row_offsets(b, n), n)
        rc, rd = oracle.diff(a, b)
        assert np.array_equal(c, rc) and np.array_equal(d, rd), (n, m)
    v.close()


def test_overflowed_lists_chain_safely(G):
    """a vor_edges call whose output overflowed reports the REQUIRED count; vor_diff and
    vor_events chained behind it clamp to the buffer capacities instead of reading past them."""
    from paper_1607_00908_b200.binding import VorError, VOR_ECAPACITY
    w = W.scaled(5, 512)
    fr = list(w.frames(2))
    labs = [oracle.label_cells(w.L, sx, sy, 16) for sx, sy in fr]
    refs = [oracle.edges(l) for l in labs]
    v = make(w.L, w.n_sites)
    cap = 500                                            # far below the ~2900 edges
    i64 = dict(dtype=torch.int64, device="cuda"); i32 = dict(dtype=torch.int32, device="cuda")
    e = [torch.full((cap + 64,), -1, **i64) for _ in range(2)]
    n = [torch.zeros(1, **i64) for _ in range(2)]
    for k in range(2):
        v.lib.vor_edges(v.h, G.dev(labs[k].ravel()).data_ptr(), e[k].data_ptr(), cap, n[k].data_ptr(), None)
    c, d = torch.full((cap + 64,), -1, **i64), torch.full((cap + 64,), -1, **i64)
    nc, nd = torch.zeros(1, **i64), torch.zeros(1, **i64)
    v.lib.vor_diff(v.h, e[0].data_ptr(), n[0].data_ptr(), e[1].data_ptr(), n[1].data_ptr(), cap, cap, None, None, 0, 0,
                   c.data_ptr(), d.data_ptr(), cap, nc.data_ptr(), nd.data_ptr(), None)
    nl = w.n_sites
    trig, idx, cp, cn = (torch.empty(nl, **i32) for _ in range(4))
    m, g = torch.zeros(1, **i32), torch.zeros(1, **i32)
    v.lib.vor_events(v.h, e[0].data_ptr(), n[0].data_ptr(), e[1].data_ptr(), n[1].data_ptr(), cap, cap,
                     c.data_ptr(), nc.data_ptr(), d.data_ptr(), nd.data_ptr(), cap, cap, nl,
                     trig.data_ptr(), idx.data_ptr(), m.data_ptr(), g.data_ptr(), cp.data_ptr(), cn.data_ptr(), None)
    with pytest.raises(VorError) as ex:
        v.vor_sync_status()
    assert ex.value.status == VOR_ECAPACITY
    assert [int(t.item()) for t in n] == [len(r) for r in refs]          # required counts
    for k in range(2):                                                   # guards untouched, prefix correct
        assert bool((e[k][cap:] == -1).all()) and np.array_equal(G.u64(e[k], cap), refs[k][:cap])
    # the chained calls saw exactly the clamped lists
    rc, rd = oracle.diff(refs[0][:cap], refs[1][:cap])
    assert int(nc.item()) == len(rc) and int(nd.item()) == len(rd)
    assert np.array_equal(G.u64(c, min(cap, len(rc))), rc[:cap]) and bool((c[cap:] == -1).all())
    ev = oracle.events(refs[0][:cap], refs[1][:cap], nl)
    assert np.array_equal(trig.cpu().numpy(), ev["trigger"])
    v.close()


# ------------------------------------------------------------------ diff (a5)
def test_diff_hand_and_random(G):
    v = make(64, 64)
    prev = pack([(0, 1), (0, 2), (1, 2), (2, 5), (7, 9)])
    now = pack([(0, 1), (1, 2), (1, 5), (2, 5), (3, 4), (7, 9)])
    for a, b in ((prev, now), (now, prev), (prev, prev), (np.empty(0, np.uint64), now), (now, np.empty(0, np.uint64))):
        c, d = G.gpu_diff(v, a, b)
        rc, rd = oracle.diff(a, b)
        assert np.array_equal(c, rc) and np.array_equal(d, rd)
    rng = np.random.default_rng(5)
    for n in (10, 5000, 200000, 3000000):
        mk = lambda: np.unique((rng.integers(0, 3000, n).astype(np.uint64) << np.uint64(32))
                               | rng.integers(3000, 6000, n).astype(np.uint64))
        a, b = mk(), mk()
        c, d = G.gpu_diff(v, a, b)
        rc, rd = oracle.diff(a, b)
        assert np.array_equal(c, rc) and np.array_equal(d, rd)
    # very different densities: the window of the dense list does not fit in shared memory
    dense = np.unique(rng.integers(0, 1 << 40, 2000000).astype(np.uint64))
    sparse = np.unique(np.concatenate([dense[::1000], rng.integers(0, 1 << 40, 1500).astype(np.uint64)]))
    for a, b in ((dense, sparse), (sparse, dense)):
        c, d = G.gpu_diff(v, a, b)
        rc, rd = oracle.diff(a, b)
        assert np.array_equal(c, rc) and np.array_equal(d, rd)
    v.close()


def test_diff_with_maps(G):
    v = make(64, 64)
    p2n = np.array([2, 0, -1, 1], np.int32); n2p = np.array([1, 3, 0, -1], np.int32)
    prev = pack([(0, 1), (0, 2), (1, 3), (2, 3)]); now = pack([(0, 1), (1, 2), (0, 3), (2, 3)])
    c, d = G.gpu_diff(v, prev, now, p2n, n2p)
    rc, rd = oracle.diff(prev, now, p2n, n2p)
    assert np.array_equal(c, rc) and np.array_equal(d, rd) and pairs(c) == {(1, 2)} and pairs(d) == {(0, 2)}
    rng = np.random.default_rng(8)
    for _ in range(3):
        K = 500
        perm = rng.permutation(K).astype(np.int32)
        p2n = perm.copy(); p2n[rng.random(K) < 0.1] = -1
        n2p = np.full(K, -1, np.int32); ok = p2n >= 0; n2p[p2n[ok]] = np.nonzero(ok)[0]
        mk = lambda: np.unique((rng.integers(0, K // 2, 3000).astype(np.uint64) << np.uint64(32))
                               | rng.integers(K // 2, K, 3000).astype(np.uint64))
        a, b = mk(), mk()
        c, d = G.gpu_diff(v, a, b, p2n, n2p)
        rc, rd = oracle.diff(a, b, p2n, n2p)
        assert np.array_equal(c, rc) and np.array_equal(d, rd)
    v.close()


def test_rhombus_flip_end_to_end_golden(G):
    g = read_golden("rhombus_flip.txt")
    L = g["L"][0]
    v = make(L, 14)
    e = []
    for h in (g["h_prev"][0], g["h_now"][0]):
        sx, sy = rhombus_sites(L, h)
        e.append(G.gpu_edges(v, G.gpu_labels(v, sx, sy)))
    c, d = G.gpu_diff(v, e[0], e[1])
    assert pairs(c) == {tuple(g["created"])} and pairs(d) == {tuple(g["destroyed"])}
    assert len(e[0]) == len(e[1]) == g["n_edges_each"][0]
    v.close()


# ------------------------------------------------------------------ frame pipeline (a1..a5 chained)
@pytest.mark.parametrize("cfg,L,nfr", [(1, None, 2), (2, None, 100), (5, 1024, 10)])
def test_frame_host_sequence_matches_oracle(G, cfg, L, nfr):
    w = W.config(cfg) if L is None else W.scaled(cfg, L)
    v = make(w.L, w.n_sites)
    cap = 8 * w.n_sites + 64
    hc = np.empty(cap, np.uint64); hd = np.empty(cap, np.uint64); cnt = np.zeros(3, np.int64)
    prev = np.empty(0, np.uint64)
    for sx, sy in w.frames(nfr):
        v.vor_frame_host(sx, sy, hc, hd, cnt)
        lab = oracle.label_cells(w.L, sx, sy, w.bucket_cells)
        e = oracle.edges(lab)
        rc, rd = oracle.diff(prev, e)
        assert cnt.tolist() == [len(e), len(rc), len(rd)]
        assert np.array_equal(hc[:cnt[1]], rc) and np.array_equal(hd[:cnt[2]], rd)
        pl, pe, _, _, _ = v.vor_frame_results()
        assert np.array_equal(G.from_device_ptr(pl, w.L * w.L, torch.int32).cpu().numpy().reshape(w.L, w.L), lab)
        assert np.array_equal(G.u64(G.from_device_ptr(pe, len(e), torch.int64)), e)
        prev = e
    v.close()


FUSED_CASES = [a for a in ADVERSARIAL if a[1] % 32 == 0] + [
    ("uniform_sparse", 512, lambda rng, P: (rng.integers(0, P, 400).astype(np.int32), rng.integers(0, P, 400).astype(np.int32))),
    ("two_sites", 32, lambda rng, P: (np.array([100, 5000], np.int32), np.array([200, 7000], np.int32))),
    ("stripes", 256, lambda rng, P: ((np.arange(12) * (P // 12) + 77).astype(np.int32), np.full(12, P // 2, np.int32))),
]


@pytest.mark.parametrize("name,L,gen", FUSED_CASES, ids=[a[0] for a in FUSED_CASES])
def test_frame_fused_label_edges_adversarial(G, name, L, gen):
    """vor_frame_* labels and extracts the pairs in ONE kernel where the lattice allows it (L % 32 == 0,
    CTA labelling path); tiles with an unproven quadrant, the tile seams and the periodic wrap take the
    side paths.  Labels, edge list and flips must equal the oracle's, and the unfused calls' results."""
    rng = np.random.default_rng(zlib.crc32(name.encode()))   # fixed per case: str hashes change per process
    P = FP * L
    sx, sy = gen(rng, P)
    frames = [(sx, sy), (((sx.astype(np.int64) + rng.integers(-600, 600, len(sx))) % P).astype(np.int32),
                         ((sy.astype(np.int64) + rng.integers(-600, 600, len(sy))) % P).astype(np.int32))]
    cap = max(64, 16 * len(sx))
    for fuse_off in (0, 1):
        v = make(L, len(sx))
        v.vor_set_option("fuse", 1 - fuse_off)
        v.vor_set_option("label_path", 3)            # the fused path belongs to the CTA kernel
        hc = np.empty(cap, np.uint64); hd = np.empty(cap, np.uint64); cnt = np.zeros(3, np.int64)
        prev = np.empty(0, np.uint64)
        for fx, fy in frames:
            v.vor_frame_host(fx, fy, hc, hd, cnt)
            lab = oracle.label_brute(L, fx, fy)
            e = oracle.edges(lab)
            rc, rd = oracle.diff(prev, e)
            pl, pe, _, _, _ = v.vor_frame_results()
            got = G.from_device_ptr(pl, L * L, torch.int32).cpu().numpy().reshape(L, L)
            assert np.array_equal(got, lab), (fuse_off, int((got != lab).sum()))
            assert cnt.tolist() == [len(e), len(rc), len(rd)], (fuse_off, cnt.tolist(), len(e), len(rc), len(rd))
            assert np.array_equal(G.u64(G.from_device_ptr(pe, len(e), torch.int64)), e)
            assert np.array_equal(hc[:cnt[1]], rc) and np.array_equal(hd[:cnt[2]], rd)
            prev = e
        v.close()


@pytest.mark.parametrize("seed", [11, 12])
def test_frame_fused_retry_with_wider_halo(G, seed):
    """a dense half and a sparse half on one lattice.  The halo follows the MEAN spacing (~9.5 cells), so
    in the sparse half (spacing ~24 cells) most quadrants fail the first attempt of the CTA kernel and succeed on
    its retry with the wider halo (<= 64 sites gathered).  The fused kernel must not pair slots of the two
    attempts' site lists: such a tile takes its pairs from the label image."""
    L = 1024
    P = FP * L
    rng = np.random.default_rng(seed)
    nd, ns = (L // 2) * L // 49, (L // 2) * L // 576
    sx = np.concatenate([rng.integers(0, P // 2, nd), rng.integers(P // 2, P, ns)]).astype(np.int32)
    sy = rng.integers(0, P, nd + ns).astype(np.int32)
    perm = rng.permutation(nd + ns)
    sx, sy = sx[perm], sy[perm]
    lab = oracle.label_cells(L, sx, sy, 16)
    e = oracle.edges(lab)
    cap = 16 * len(sx)
    res = []
    for fuse in (1, 0):
        v = make(L, len(sx))
        v.vor_set_option("fuse", fuse)
        v.vor_set_option("label_path", 3)
        hc = np.empty(cap, np.uint64); hd = np.empty(cap, np.uint64); cnt = np.zeros(3, np.int64)
        v.vor_frame_host(sx, sy, hc, hd, cnt)
        pl, pe, _, _, _ = v.vor_frame_results()
        got = G.from_device_ptr(pl, L * L, torch.int32).cpu().numpy().reshape(L, L)
        assert np.array_equal(got, lab), (fuse, int((got != lab).sum()))
        ge = G.u64(G.from_device_ptr(pe, min(int(cnt[0]), cap), torch.int64))
        res.append((int(cnt[0]), len(np.setdiff1d(ge, e)), len(np.setdiff1d(e, ge))))
        v.close()
    assert res == [(len(e), 0, 0)] * 2, f"(count, spurious, missing) fused / unfused: {res}, expected {len(e)}"


@pytest.mark.parametrize("pin", [False, True])
def test_frame_pipeline_submit_collect(G, pin):
    """Two frames in flight (submit k+1 before collect k): same results, in order, as the oracle;
    a third submit and a collect with nothing in flight are refused."""
    from paper_1607_00908_b200.binding import VorError, VOR_ESTATE
    w = W.scaled(5, 1024)
    v = make(w.L, w.n_sites)
    cap = 8 * w.n_sites + 64
    def buf(n, dt):
        return torch.empty(n, dtype=dt, pin_memory=True).numpy() if pin else np.empty(n, torch.empty(0, dtype=dt).numpy().dtype)
    hc, hd = buf(cap, torch.int64).view(np.uint64), buf(cap, torch.int64).view(np.uint64)
    cnt = np.zeros(3, np.int64)
    frames = []
    for sx, sy in w.frames(5):
        px, py = buf(w.n_sites, torch.int32), buf(w.n_sites, torch.int32)
        px[:] = sx; py[:] = sy
        frames.append((px, py))
    refs, prev = [], np.empty(0, np.uint64)
    for sx, sy in frames:
        e = oracle.edges(oracle.label_cells(w.L, sx, sy, w.bucket_cells))
        refs.append((e,) + oracle.diff(prev, e))
        prev = e
    with pytest.raises(VorError) as ex:
        v.vor_frame_collect(hc, hd, cnt)
    assert ex.value.status == VOR_ESTATE
    def collect(k):
        v.vor_frame_collect(hc, hd, cnt)
        e, rc, rd = refs[k]
        assert cnt.tolist() == [len(e), len(rc), len(rd)], k
        assert np.array_equal(hc[:cnt[1]], rc) and np.array_equal(hd[:cnt[2]], rd), k
    v.vor_frame_submit(*frames[0])
    for k in range(1, len(frames)):
        v.vor_frame_submit(*frames[k])
        if k == 1:
            with pytest.raises(VorError) as ex:
                v.vor_frame_submit(*frames[2])
            assert ex.value.status == VOR_ESTATE
        collect(k - 1)
    collect(len(frames) - 1)
    # the synchronous call continues the same sequence (same previous edge list)
    sx, sy = frames[-1]
    v.vor_frame_host(sx, sy, hc, hd, cnt)
    assert cnt.tolist() == [len(refs[-1][0]), 0, 0]
    v.close()


# ------------------------------------------------------------------ field path (a6..a8)
def check_field_frame(G, v, field, thr, min_size, above=True):
    ref_ccl = oracle.threshold_ccl(field, thr, above)
    ccl = G.gpu_ccl(v, field, thr, above)
    got = ccl.cpu().numpy().reshape(v.L, v.L)
    assert np.array_equal(got, ref_ccl), f"{(got != ref_ccl).sum()} ccl cells differ"
    rc = oracle.centroids(ref_ccl, min_size)
    gc = G.gpu_centroids(v, ccl, min_size)
    for k in ("sx", "sy", "size", "root"):
        assert np.array_equal(gc[k], rc[k]), k
    assert len(gc["cx"]) == len(rc["cx"])
    if len(rc["cx"]):
        assert np.abs(gc["cx"] - rc["cx"]).max() <= 1e-9 and np.abs(gc["cy"] - rc["cy"]).max() <= 1e-9
    return rc


def test_ccl_and_centroids_hand_cases(G):
    L = 8
    v = make(L, 64)
    f = np.zeros((L, L), np.float32)
    f[0, 0] = f[0, 7] = f[7, 0] = 2; f[4, :] = 2; f[2, 3] = 2
    check_field_frame(G, v, f, 1.0, 1)
    check_field_frame(G, v, np.full((L, L), 5, np.float32), 1.0, 1)
    check_field_frame(G, v, np.zeros((L, L), np.float32), 1.0, 1)
    check_field_frame(G, v, np.zeros((L, L), np.float32), 1.0, 1, above=False)
    check_field_frame(G, v, np.full((L, L), np.nan, np.float32), 1.0, 1)
    check_field_frame(G, v, np.full((L, L), 1.0, np.float32), 1.0, 1)
    check_field_frame(G, v, np.full((L, L), 1e-40, np.float32), 0.0, 1)      # denormal > 0
    v.close()


@pytest.mark.parametrize("L,p,seed", [(64, 0.4, 0), (100, 0.59, 1), (257, 0.62, 2), (512, 0.5, 3)])
def test_ccl_and_centroids_random_masks(G, L, p, seed):
    rng = np.random.default_rng(seed)
    v = make(L, 1024)
    check_field_frame(G, v, rng.random((L, L)).astype(np.float32), 1.0 - p, 1)
    check_field_frame(G, v, rng.random((L, L)).astype(np.float32), 1.0 - p, 20)
    v.close()


def test_ccl_serpentine_long_chains(G):
    L = 256
    f = np.zeros((L, L), np.float32)
    f[::2, :] = 1                                  # rows, joined alternately at the ends: one snake
    f[1::4, L - 1] = 1
    f[3::4, 0] = 1
    v = make(L, 16)
    check_field_frame(G, v, f, 0.5, 1)
    v.close()


@pytest.mark.parametrize("cfg,L,nfr", [(3, 256, 3), (3, 1024, 2), (4, 512, 3), (3, None, 2), (4, None, 2)])
def test_field_pipeline_scaled_configs(G, cfg, L, nfr):
    """threshold -> CCL -> centroids -> match -> label -> edges -> diff(maps), frame by frame.
    L = None: the configuration at its full BASELINE.json size (2048^2 / 4096^2)."""
    w = W.config(cfg) if L is None else W.scaled(cfg, L)
    L = w.L
    v = make(L, 65536)
    R = int(w.match_radius_cells * FP)
    prev_c, prev_e = None, None
    for field in w.frames(nfr):
        rc = check_field_frame(G, v, field, w.threshold, w.min_size)
        K = len(rc["sx"])
        assert K > 3
        lab = oracle.label_cells(L, rc["sx"], rc["sy"], 16 if L % 16 == 0 else 1)
        assert np.array_equal(G.gpu_labels(v, rc["sx"], rc["sy"]), lab)
        e = oracle.edges(lab)
        assert np.array_equal(G.gpu_edges(v, lab), e)
        if prev_c is not None:
            p2n, n2p = oracle.match(L, prev_c["sx"], prev_c["sy"], rc["sx"], rc["sy"], R)
            gp, gn = G.gpu_match(v, prev_c["sx"], prev_c["sy"], rc["sx"], rc["sy"], R)
            assert np.array_equal(gp, p2n) and np.array_equal(gn, n2p)
            assert (p2n >= 0).mean() > 0.5
            c, d = G.gpu_diff(v, prev_e, e, p2n, n2p)
            oc, od = oracle.diff(prev_e, e, p2n, n2p)
            assert np.array_equal(c, oc) and np.array_equal(d, od)
        prev_c, prev_e = rc, e
    v.close()


def oracle_field_chain(w, fields):
    """The oracle's chain a6 -> a7 -> a8 -> a1..a5 (maps) frame by frame: (K, edges, created, destroyed, parts)."""
    L, R = w.L, int(w.match_radius_cells * FP)
    prev_c, prev_e = None, None
    for field in fields:
        ccl = oracle.threshold_ccl(field, w.threshold, True)
        c = oracle.centroids(ccl, w.min_size)
        lab = oracle.label_cells(L, c["sx"], c["sy"], 16 if L % 16 == 0 else 1)
        e = oracle.edges(lab)
        if prev_c is None:
            rc = rd = np.empty(0, np.uint64)
            maps = None
        else:
            maps = oracle.match(L, prev_c["sx"], prev_c["sy"], c["sx"], c["sy"], R)
            rc, rd = oracle.diff(prev_e, e, *maps)
        yield len(c["sx"]), e, rc, rd, dict(ccl=ccl, comp=c, labels=lab, maps=maps)
        prev_c, prev_e = c, e


@pytest.mark.parametrize("cfg,L,nfr", [(3, 512, 4), (4, 512, 3), (3, None, None), (4, None, None)])
def test_field_frames_chained_on_the_device(G, cfg, L, nfr):
    """field_frame_submit / field_frame_collect: the whole field-driven frame chained on the device (GPU
    bubbles -> GPU centroids -> GPU maps -> GPU labels -> GPU edges -> GPU diff with the GPU maps, no host
    sync in between), compared with the oracle chain.  L = None: every frame of the configuration at its
    full BASELINE.json size (config 3: 50 frames of 2048^2, config 4: 20 frames of 4096^2)."""
    w = W.config(cfg) if L is None else W.scaled(cfg, L)
    L = w.L
    v = make(L, 65536)
    R = int(w.match_radius_cells * FP)
    cap = 8 * 65536
    hc, hd, cnt = np.empty(cap, np.uint64), np.empty(cap, np.uint64), np.zeros(4, np.int64)
    fields = list(w.frames(nfr))
    refs = oracle_field_chain(w, fields)

    def collect(k):
        v.field_frame_collect(hc, hd, cnt)
        K, e, rc, rd, _ = next(refs)
        assert cnt.tolist() == [K, len(e), len(rc), len(rd)], (k, cnt.tolist(), K, len(e), len(rc), len(rd))
        assert np.array_equal(hc[:cnt[2]], rc) and np.array_equal(hd[:cnt[3]], rd), k
        assert K > 3

    v.field_frame_submit(fields[0].ravel(), w.threshold, True, w.min_size, R)
    for k in range(1, len(fields)):
        v.field_frame_submit(fields[k].ravel(), w.threshold, True, w.min_size, R)
        collect(k - 1)
    collect(len(fields) - 1)
    v.close()


def test_field_frame_device_results(G):
    """field_frame_device on device-resident fields: every intermediate the context exposes (bubble image,
    centroids, maps, labels, edges) equals the oracle's, and a new sequence starts after vor_frame_reset."""
    w = W.scaled(3, 512)
    L = w.L
    v = make(L, 4096)
    R = int(w.match_radius_cells * FP)
    fields = list(w.frames(3))
    for rep in range(2):
        for k, (K, e, rc, rd, parts) in enumerate(oracle_field_chain(w, fields)):
            v.field_frame_device(G.dev(fields[k].ravel()), w.threshold, True, w.min_size, R)
            v.vor_sync_status()
            r = v.field_frame_results()
            get = lambda name, n, dt: G.from_device_ptr(r[name], n, dt).cpu().numpy()
            assert get("counts", 4, torch.int64).tolist() == [K, len(e), len(rc), len(rd)]
            assert np.array_equal(get("ccl", L * L, torch.int32).reshape(L, L), parts["ccl"])
            assert np.array_equal(get("labels", L * L, torch.int32).reshape(L, L), parts["labels"])
            for name in ("sx", "sy", "size", "root"):
                assert np.array_equal(get(name, K, torch.int32), parts["comp"][name]), name
            assert np.abs(get("cx", K, torch.float64) - parts["comp"]["cx"]).max() <= 1e-9
            assert np.abs(get("cy", K, torch.float64) - parts["comp"]["cy"]).max() <= 1e-9
            assert np.array_equal(get("edges", len(e), torch.int64).view(np.uint64), e)
            assert np.array_equal(get("created", len(rc), torch.int64).view(np.uint64), rc)
            assert np.array_equal(get("destroyed", len(rd), torch.int64).view(np.uint64), rd)
            if parts["maps"] is not None:
                assert np.array_equal(get("p2n", len(parts["maps"][0]), torch.int32), parts["maps"][0])
                assert np.array_equal(get("n2p", K, torch.int32), parts["maps"][1])
        v.vor_frame_reset()
    v.close()


def test_build_cells_dev_count_on_the_device(G):
    """vor_build_cells_dev: the number of sites is a device scalar below the capacity; labels equal the
    oracle's on the first n sites whatever the hint; zero sites give -1 everywhere."""
    L = 256
    sx, sy = rnd(3, L, 500)
    v = make(L, 500)
    lab = torch.empty(L * L, dtype=torch.int32, device="cuda")
    for n, hint in ((500, 0), (137, 500), (137, 10), (1, 0), (0, 0)):
        v.vor_build_cells_dev(G.dev(sx), G.dev(sy), torch.tensor([n], dtype=torch.int32, device="cuda"), hint)
        v.vor_label(lab)
        v.vor_sync_status()
        ref = oracle.label_brute(L, sx[:n], sy[:n]) if n else np.full((L, L), -1, np.int32)
        assert np.array_equal(lab.cpu().numpy().reshape(L, L), ref), (n, hint)
    v.close()


def test_match_invariants_and_random(G):
    v = make(64, 256)
    rng = np.random.default_rng(13)
    P = FP * 64
    for _ in range(4):
        px, py = rng.integers(0, P, 80).astype(np.int32), rng.integers(0, P, 80).astype(np.int32)
        nx, ny = rng.integers(0, P, 70).astype(np.int32), rng.integers(0, P, 70).astype(np.int32)
        for R in (0, 3 * FP, 6 * FP, 40 * FP):
            a, b = G.gpu_match(v, px, py, nx, ny, R)
            ra, rb = oracle.match(64, px, py, nx, ny, R)
            assert np.array_equal(a, ra) and np.array_equal(b, rb)
    a, b = G.gpu_match(v, np.array([1000, 1000]), np.array([1000, 1000]), np.array([1100]), np.array([1000]), 4 * FP)
    assert a.tolist() == [0, -1] and b.tolist() == [0]
    # a crowded bucket (grid path overflows -> brute-force redo) next to the seam, plus scattered points
    cx = np.concatenate([rng.integers(P - 300, P + 300, 150) % P, rng.integers(0, P, 60)]).astype(np.int32)
    cy = np.concatenate([rng.integers(-200, 400, 150) % P, rng.integers(0, P, 60)]).astype(np.int32)
    mx = ((cx.astype(np.int64) + rng.integers(-150, 150, len(cx))) % P).astype(np.int32)
    my = ((cy.astype(np.int64) + rng.integers(-150, 150, len(cy))) % P).astype(np.int32)
    for R in (1 * FP, 3 * FP):
        a, b = G.gpu_match(v, cx, cy, mx[::-1].copy(), my[::-1].copy(), R)
        ra, rb = oracle.match(64, cx, cy, mx[::-1].copy(), my[::-1].copy(), R)
        assert np.array_equal(a, ra) and np.array_equal(b, rb)
    v.close()
    # grid path proper: many well-separated points on a large lattice, seam included
    L = 2048
    v = make(L, 8192)
    P = FP * L
    g = np.arange(64) * (P // 64)
    px, py = (np.repeat(g, 64) + rng.integers(0, 2000, 4096)) % P, (np.tile(g, 64) + rng.integers(0, 2000, 4096)) % P
    keep = rng.random(4096) > 0.05
    nx = ((px + rng.integers(-700, 700, 4096)) % P)[keep][::-1].copy()
    ny = ((py + rng.integers(-700, 700, 4096)) % P)[keep][::-1].copy()
    a, b = G.gpu_match(v, px.astype(np.int32), py.astype(np.int32), nx.astype(np.int32), ny.astype(np.int32), 4 * FP)
    ra, rb = oracle.match(L, px.astype(np.int32), py.astype(np.int32), nx.astype(np.int32), ny.astype(np.int32), 4 * FP)
    assert np.array_equal(a, ra) and np.array_equal(b, rb) and (ra >= 0).sum() > 3000
    v.close()


# ------------------------------------------------------------------ event layer (trigger, eventsIndices, eventsCount)
def check_events(G, v, prev, now, n):
    got, ref = G.gpu_events(v, prev, now, n), oracle.events(prev, now, n)
    for k in ("trigger", "events_indices", "count_prev", "count_now"):
        assert np.array_equal(got[k], ref[k]), k
    assert got["global_trigger"] == ref["global_trigger"]
    return got


def test_events_hand_random_and_golden(G):
    v = make(64, 64)
    common = [(0, 1), (1, 2), (2, 3), (0, 3), (0, 4), (1, 4), (2, 5), (3, 5), (4, 5)]
    ev = check_events(G, v, pack(common + [(1, 3)]), pack(common + [(0, 2)]), 6)
    assert ev["count_prev"].tolist() == [2, 3, 2, 3, 0, 0] and ev["count_now"].tolist() == [3, 2, 3, 2, 0, 0]
    check_events(G, v, pack(common), pack(common), 6)                  # nothing happened
    check_events(G, v, np.empty(0, np.uint64), pack([(0, 2)]), 3)      # empty past list
    check_events(G, v, pack([(0, 1), (1, 2), (0, 2)]), pack([(0, 1), (1, 2)]), 3)
    check_events(G, v, pack([(0, 1)]), pack([(0, 1)]), 1)              # n_labels below the labels: keys ignored
    rng = np.random.default_rng(17)
    for n in (2, 33, 1000, 5000):                                      # several batches and a ragged tail
        i = rng.integers(0, n, 6 * n); j = rng.integers(0, n, 6 * n)
        keep = i != j
        a = np.unique((np.minimum(i, j)[keep].astype(np.uint64) << np.uint64(32)) | np.maximum(i, j)[keep].astype(np.uint64))
        b = np.unique(np.concatenate([a[rng.random(len(a)) < 0.97], a[:5] + np.uint64(1) if len(a) > 5 else a]))
        b = b[(b & np.uint64(0xffffffff)) < np.uint64(n)]
        b = b[(b >> np.uint64(32)) < (b & np.uint64(0xffffffff))]
        check_events(G, v, a, b, n)
    v.close()
    g = read_golden("rhombus_flip.txt")
    L = g["L"][0]
    v = make(L, 16)
    lists = []
    for h in (g["h_prev"][0], g["h_now"][0]):
        sx, sy = rhombus_sites(L, h)
        lists.append(G.gpu_edges(v, G.gpu_labels(v, sx, sy)))
    ev = check_events(G, v, lists[0], lists[1], g["n_sites"][0])
    assert ev["events_indices"].tolist() == g["events_indices"]
    assert ev["count_prev"][:4].tolist() == g["count_prev"] and ev["count_now"][:4].tolist() == g["count_now"]
    v.close()


# ------------------------------------------------------------------ couples of active vertices, T1 pairing
T1_KEYS = ("couples", "cls", "common_prev", "common_now", "partner")


def check_t1(G, v, prev, now, n):
    got, ref = G.gpu_t1(v, prev, now, n), oracle.t1(prev, now, n)
    assert got["n_couples"] == len(ref["couples"]) and not got["overflow"]
    for k in T1_KEYS:
        assert np.array_equal(got[k], ref[k]), k
    return got


def random_graph_pair(rng, n, deg, keep=0.9, fresh=0.1):
    """Two ascending unique key lists over n vertices sharing most of their edges."""
    def draw(m):
        i = rng.integers(0, n, m); j = rng.integers(0, n, m)
        ok = i != j
        return (np.minimum(i, j)[ok].astype(np.uint64) << np.uint64(32)) | np.maximum(i, j)[ok].astype(np.uint64)
    a = np.unique(draw(deg * n // 2))
    b = np.unique(np.concatenate([a[rng.random(len(a)) < keep], draw(max(1, int(fresh * deg * n / 2)))]))
    return a, b


def test_t1_events_hand_graphs_random_graphs_and_golden(G):
    v = make(64, 64)
    key = lambda i, j: (min(i, j) << 32) | max(i, j)
    common = [(0, 1), (1, 2), (2, 3), (0, 3), (0, 4), (1, 4), (2, 5), (3, 5), (4, 5)]
    r = check_t1(G, v, pack(common + [(1, 3)]), pack(common + [(0, 2)]), 6)              # one T1
    k = r["couples"].tolist()
    assert int(r["partner"][k.index(key(1, 3))]) == key(0, 2) and int(r["partner"][k.index(key(0, 2))]) == key(1, 3)
    rh = lambda o: [(o, o + 1), (o + 1, o + 2), (o + 2, o + 3), (o, o + 3)]
    glue = [(3, 4), (2, 4), (2, 5)]
    check_t1(G, v, pack(rh(0) + rh(4) + glue + [(1, 3), (4, 6)]), pack(rh(0) + rh(4) + glue + [(0, 2), (5, 7)]), 8)
    check_t1(G, v, pack([(0, 1), (1, 2), (0, 2)]), pack([(0, 1), (1, 2)]), 3)            # Fig. 8 boundary event
    full = [(0, 1), (0, 2), (0, 3), (1, 2), (1, 3), (2, 3)]
    check_t1(G, v, pack(full), pack(full[1:]), 4)                                        # tetrahedron: no partner
    check_t1(G, v, pack(common), pack(common), 6)                                        # nothing happened
    check_t1(G, v, np.empty(0, np.uint64), np.empty(0, np.uint64), 3)
    check_t1(G, v, np.empty(0, np.uint64), pack([(0, 2)]), 3)
    check_t1(G, v, pack([(0, 1), (1, 2), (0, 2), (1, 5)]), pack([(0, 1), (1, 2), (2, 6)]), 3)   # labels >= n ignored
    check_events(G, v, pack([(0, 1)]), pack([(0, 1), (0, 7)]), 3)                        # ... by the trigger as well
    rng = np.random.default_rng(23)
    for n, deg in ((2, 1), (7, 3), (33, 6), (1000, 6), (5000, 6), (300, 40)):
        for _ in range(3):
            a, b = random_graph_pair(rng, n, deg)
            check_t1(G, v, a, b, n)
    # hubs: two adjacent vertices joined to (almost) everybody, long rows through the merge intersection
    n = 3000
    a, b = random_graph_pair(rng, n, 4)
    hub = lambda h, skip: np.array([key(h, t) for t in range(n) if t != h and t % 7 != skip], np.uint64)
    a = np.unique(np.concatenate([a, hub(5, 0), hub(1700, 1), np.array([key(5, 1700)], np.uint64)]))
    b = np.unique(np.concatenate([b, hub(5, 2), hub(1700, 1)]))
    check_t1(G, v, a, b, n)
    # capacity: the required number is reported, nothing is written past cap, the status says so
    ref = oracle.t1(a, b, n)
    got = G.gpu_t1(v, a, b, n, cap=100)
    assert got["overflow"] and got["n_couples"] == len(ref["couples"]) > 100
    assert np.array_equal(got["couples"], ref["couples"][:100]) and np.array_equal(got["partner"], ref["partner"][:100])
    v.close()
    g = read_golden("rhombus_flip.txt")
    L = g["L"][0]
    v = make(L, 16)
    lists = []
    for h in (g["h_prev"][0], g["h_now"][0]):
        sx, sy = rhombus_sites(L, h)
        lists.append(G.gpu_edges(v, G.gpu_labels(v, sx, sy)))
    r = check_t1(G, v, lists[0], lists[1], g["n_sites"][0])
    k = r["couples"].tolist()
    assert int(r["partner"][k.index(key(*g["destroyed"]))]) == key(*g["created"])
    assert int(r["partner"][k.index(key(*g["created"]))]) == key(*g["destroyed"])
    v.close()


def test_event_vertices_bulk_and_boundary(G):
    def check(prev, now, n):
        got, ref = G.gpu_event_vertices(v, prev, now, n), oracle.event_vertices(prev, now, n)
        for k in ("boundary_prev", "boundary_now", "vclass"):
            assert np.array_equal(got[k], ref[k]), k
        return got
    v = make(64, 64)
    common = [(0, 1), (1, 2), (2, 3), (0, 3), (0, 4), (1, 4), (2, 5), (3, 5), (4, 5)]
    r = check(pack(common + [(1, 3)]), pack(common + [(0, 2)]), 6)
    assert [c & 5 for c in r["vclass"][:4].tolist()] == [4, 1, 4, 1]
    r = check(pack([(0, 1), (1, 2), (0, 2)]), pack([(0, 1), (1, 2)]), 3)               # Fig. 8 bottom
    assert r["vclass"].tolist() == [2, 0, 2] and r["boundary_prev"].tolist() == [1, 1, 1]
    check(pack(common), pack(common), 6)
    check(np.empty(0, np.uint64), pack([(0, 2)]), 3)
    check(pack([(0, 1), (1, 2), (0, 2), (1, 5)]), pack([(0, 1), (1, 2), (2, 6)]), 3)
    rng = np.random.default_rng(41)
    for n, deg in ((7, 3), (33, 6), (1000, 6), (5000, 6), (300, 40)):
        a, b = random_graph_pair(rng, n, deg)
        check(a, b, n)
    v.close()
    # walled lattice: the triangulation has a boundary; two frames of moving sites
    import importlib
    geo = importlib.import_module("test_gpu_geometry")
    Lx, Ly = 256, 192
    sx, sy = geo.jitter_sites(rng, Lx, Ly, 14.0)
    vg = geo.make(Lx, Ly, (0, 0), len(sx))
    lists = []
    for t in range(2):
        lists.append(G.gpu_edges_image(vg, G.gpu_labels(vg, sx, sy), False))
        sx = np.clip(sx + rng.integers(-500, 500, len(sx)), 0, FP * Lx - 1).astype(np.int32)
        sy = np.clip(sy + rng.integers(-500, 500, len(sy)), 0, FP * Ly - 1).astype(np.int32)
    got = G.gpu_event_vertices(vg, lists[0], lists[1], len(sx))
    ref = oracle.event_vertices(lists[0], lists[1], len(sx))
    for k in ("boundary_prev", "boundary_now", "vclass"):
        assert np.array_equal(got[k], ref[k]), k
    assert ref["boundary_prev"].sum() > 20 and (ref["vclass"] & 1).sum() > 5 and (ref["vclass"] & 2).sum() > 0
    vg.close()


# ------------------------------------------------------------------ full size, bench.py's launch configuration
def test_config5_full_size_all_frames(G):
    """BASELINE config 5 at its full size (16384^2 cells, 10^6 sites), ALL 10 frames of the random walk,
    through the same calls, buffers and capacities bench.py times.  Every label, edge key, row offset and
    flip of every frame is compared with the oracle (O1b finishes a full frame in seconds), and O1b itself
    is cross-checked here against brute force over all 10^6 sites on sampled cells.  The later frames are
    the disordered regime (candidate lists overflow, quadrants go to the fix-up pass)."""
    w = W.config(5)
    L, n = w.L, w.n_sites
    v = make(L, n, max_raw_keys=max(1 << 20, 16 * n))
    cap_e = 4 * n + 1024
    i64 = dict(dtype=torch.int64, device="cuda"); i32 = dict(dtype=torch.int32, device="cuda")
    labels = torch.empty(L * L, **i32)
    edges = [torch.empty(cap_e, **i64) for _ in range(2)]
    n_edges = [torch.zeros(1, **i64) for _ in range(2)]
    row_ptr = [torch.zeros(n + 1, **i32) for _ in range(2)]
    created, destroyed = torch.empty(cap_e, **i64), torch.empty(cap_e, **i64)
    created2, destroyed2 = torch.empty(cap_e, **i64), torch.empty(cap_e, **i64)
    n_c, n_d, n_c2, n_d2 = (torch.zeros(1, **i64) for _ in range(4))
    rng = np.random.default_rng(5)
    prev = np.empty(0, np.uint64)
    assert w.n_frames == 10
    vf = make(L, n, max_raw_keys=max(1 << 20, 16 * n))   # the frame call, with the fused label -> edge kernel
    vf.vor_set_option("fuse", 1)
    for i, (sx, sy) in enumerate(w.frames()):
        now, prv = i & 1, 1 - (i & 1)
        vf.vor_frame_device(G.dev(sx), G.dev(sy))
        v.vor_build_cells(G.dev(sx), G.dev(sy))
        v.vor_label(labels)
        v.vor_edges_rows(labels, edges[now], n_edges[now], row_ptr[now])
        v.vor_diff_rows(edges[prv], row_ptr[prv], edges[now], row_ptr[now], n, created, destroyed, n_c, n_d)
        v.vor_diff(edges[prv], n_edges[prv], edges[now], n_edges[now], created2, destroyed2, n_c2, n_d2)
        v.vor_sync_status()
        ref = oracle.label_cells(L, sx, sy, w.bucket_cells)
        got = labels.cpu().numpy().reshape(L, L)
        assert np.array_equal(got, ref), f"frame {i}: {int((got != ref).sum())} labels differ"
        cells = rng.integers(0, L * L, 1500)
        assert np.array_equal(ref.ravel()[cells], oracle.label_brute_at(L, sx, sy, cells))
        e = oracle.edges(ref)
        assert np.array_equal(G.u64(edges[now], int(n_edges[now].item())), e), i
        assert np.array_equal(row_ptr[now].cpu().numpy().view(np.uint32), row_offsets(e, n)), i
        rc, rd = oracle.diff(prev, e)
        for c_, d_, nc_, nd_ in ((created, destroyed, n_c, n_d), (created2, destroyed2, n_c2, n_d2)):
            assert np.array_equal(G.u64(c_, int(nc_.item())), rc), i
            assert np.array_equal(G.u64(d_, int(nd_.item())), rd), i
        vf.vor_sync_status()
        pl, pe, pc, pd, pn = vf.vor_frame_results()
        assert G.from_device_ptr(pn, 3, torch.int64).cpu().tolist() == [len(e), len(rc), len(rd)], i
        assert bool((G.from_device_ptr(pl, L * L, torch.int32) == labels).all()), i
        assert np.array_equal(G.u64(G.from_device_ptr(pe, len(e), torch.int64)), e), i
        assert np.array_equal(G.u64(G.from_device_ptr(pc, len(rc), torch.int64)), rc), i
        assert np.array_equal(G.u64(G.from_device_ptr(pd, len(rd), torch.int64)), rd), i
        if i in (1, 9):                             # event layer at full size, on the device-resident lists
            trig, idx, cp, cn = (torch.empty(n, **i32) for _ in range(4))
            m, g = torch.zeros(1, **i32), torch.zeros(1, **i32)
            v.vor_events(edges[prv], n_edges[prv], edges[now], n_edges[now], created, n_c, destroyed, n_d,
                         trig, idx, m, g, cp, cn)
            v.vor_sync_status()
            ev = oracle.events(prev, e, n)
            assert np.array_equal(trig.cpu().numpy(), ev["trigger"]) and int(g.item()) == 1
            assert np.array_equal(idx[:int(m.item())].cpu().numpy(), ev["events_indices"])
            assert np.array_equal(cp.cpu().numpy(), ev["count_prev"]) and np.array_equal(cn.cpu().numpy(), ev["count_now"])
            couples, partner = torch.empty(cap_e, **i64), torch.empty(cap_e, **i64)   # couples and T1 quadruples
            cls, kp, kn = (torch.empty(cap_e, **i32) for _ in range(3))
            nk = torch.zeros(1, **i64)
            v.vor_t1_events(edges[prv], n_edges[prv], edges[now], n_edges[now], created, n_c, destroyed, n_d, trig,
                            couples, cls, kp, kn, partner, nk)
            v.vor_sync_status()
            t1 = oracle.t1(prev, e, n)
            k = int(nk.item())
            assert k == len(t1["couples"]) and np.array_equal(G.u64(couples, k), t1["couples"]), i
            assert np.array_equal(G.u64(partner, k), t1["partner"]) and np.array_equal(cls[:k].cpu().numpy(), t1["cls"]), i
            assert np.array_equal(kp[:k].cpu().numpy(), t1["common_prev"]), i
            assert np.array_equal(kn[:k].cpu().numpy(), t1["common_now"]), i
            n_t1 = int(((t1["cls"] == 1) & (t1["partner"] != np.uint64(0xFFFFFFFFFFFFFFFF))).sum())
            assert n_t1 > 0.3 * len(rd)               # about half the breaking links of such a frame are isolated T1 events
            del couples, partner, cls, kp, kn, t1
        prev = e
        del ref, got
    assert 2.9 * n < len(prev) < 3.0 * n            # E slightly below 3N (R6), as the survey's probe found
    v.close(); vf.close()
