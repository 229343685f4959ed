"""Pins for the oracle's labelling (O1a brute force, O1b cell-list ring search).

What fixes the expected values (none of it is the oracle's own formula retyped):
 - the region definition PAPER.md:35 / colouring PAPER.md:131 evaluated by a LIBRARY nearest-
   neighbour routine (scipy cKDTree with periodic boxsize) on float64 coordinates;
 - exact equivariances of the definition (translation by whole cells, transpose, mirror);
 - hand-constructed tie cases (reading R1: smallest index) that also pin the +0.5 cell-centre
   convention (R2) and the minimum-image wrap;
 - O1b == O1a on adversarial inputs (proves the R3 stop rule).
"""
import zlib

import numpy as np
import pytest
from scipy.spatial import cKDTree

import oracle
from paper_1607_00908_b200 import workloads as W

FP = 256


def rand_sites(rng, L, n):
    P = FP * L
    return (rng.integers(0, P, n).astype(np.int32), rng.integers(0, P, n).astype(np.int32))


@pytest.mark.parametrize("L,n,seed", [(64, 32, 1), (96, 7, 2), (128, 300, 3)])
def test_brute_matches_periodic_kdtree(L, n, seed):
    rng = np.random.default_rng(seed)
    sx, sy = rand_sites(rng, L, n)
    lab = oracle.label_brute(L, sx, sy)
    pts = np.stack([sx / FP, sy / FP], axis=1)
    tree = cKDTree(pts, boxsize=float(L))
    yy, xx = np.mgrid[0:L, 0:L]
    q = np.stack([xx.ravel() + 0.5, yy.ravel() + 0.5], axis=1)
    d, idx = tree.query(q, k=2)
    clear = (d[:, 1] - d[:, 0]) > 1e-9          # leave exact ties to the tie tests
    assert clear.mean() > 0.95
    assert np.array_equal(lab.ravel()[clear], idx[clear, 0])


def test_coverage_and_conditional_own_cell():
    w = W.config(1)
    sx, sy = next(iter(w.frames(1)))
    L, P = w.L, FP * w.L
    lab = oracle.label_brute(L, sx, sy)
    assert lab.shape == (L, L) and lab.min() >= 0 and lab.max() < w.n_sites
    # R5: a site's own cell carries its label whenever no other site is within sqrt(2) cells
    for i in range(w.n_sites):
        dx = np.abs(sx.astype(np.int64) - sx[i]); dx = np.minimum(dx, P - dx)
        dy = np.abs(sy.astype(np.int64) - sy[i]); dy = np.minimum(dy, P - dy)
        d2 = dx * dx + dy * dy
        d2[i] = np.iinfo(np.int64).max
        if d2.min() > 2 * FP * FP:
            assert lab[sy[i] // FP, sx[i] // FP] == i


def test_translation_equivariance_across_seam():
    rng = np.random.default_rng(5)
    L, n = 64, 40
    P = FP * L
    sx, sy = rand_sites(rng, L, n)
    lab = oracle.label_brute(L, sx, sy)
    for kx, ky in [(1, 0), (0, 1), (37, 0), (13, 59)]:
        sx2 = ((sx.astype(np.int64) + kx * FP) % P).astype(np.int32)
        sy2 = ((sy.astype(np.int64) + ky * FP) % P).astype(np.int32)
        lab2 = oracle.label_brute(L, sx2, sy2)
        assert np.array_equal(lab2, np.roll(lab, (ky, kx), axis=(0, 1)))


def test_transpose_and_mirror_equivariance():
    rng = np.random.default_rng(6)
    L, n = 48, 25
    P = FP * L
    sx, sy = rand_sites(rng, L, n)
    lab = oracle.label_brute(L, sx, sy)
    assert np.array_equal(oracle.label_brute(L, sy, sx), lab.T)
    # mirror x -> P - x maps cell x to cell L-1-x (centres 256x+128 -> P - 256x - 128)
    mx = ((P - sx.astype(np.int64)) % P).astype(np.int32)
    # sites with sx == 0 map to themselves; mirror is exact for all others, ties keep index order
    assert np.array_equal(oracle.label_brute(L, mx, sy), lab[:, ::-1])


def test_tie_goes_to_smallest_index_and_centre_offset():
    L = 32
    c = lambda x: FP * x + 128          # fixed-point centre of cell x
    # two sites at the centres of cells 10 and 12 of row 5: cell 11 is exactly equidistant
    for order in ((10, 12), (12, 10)):
        sx = np.array([c(order[0]), c(order[1])], dtype=np.int32)
        sy = np.array([c(5), c(5)], dtype=np.int32)
        lab = oracle.label_brute(L, sx, sy)
        assert lab[5, order[0]] == 0 and lab[5, order[1]] == 1
        assert lab[5, 11] == 0                       # tie -> smaller index (R1)
        assert np.all(lab[:, 11] == 0)               # the whole equidistant column
    # a missing +128 centre offset would break the tie in favour of the left site: caught by (12,10)


def test_tie_column_mirror_symmetric_sites_with_wrap():
    L = 16
    P = FP * L
    # sites mirror-symmetric about the column of cell centres x=3 AND (through the wrap) x=11
    sx = np.array([FP * 3 + 128 - 700, FP * 3 + 128 + 700], dtype=np.int32)
    sy = np.array([1000, 1000], dtype=np.int32)
    lab = oracle.label_brute(L, sx, sy)
    assert np.all(lab[:, 3] == 0) and np.all(lab[:, 11] == 0)
    assert np.all(lab[:, 1] == 0) and np.all(lab[:, 5] == 1)
    assert np.all(lab[:, 12] == 0) and np.all(lab[:, 10] == 1)   # wrap side: site 0 is nearer via -x


def test_duplicate_sites_and_crowded_out_site():
    L = 16
    sx = np.array([2000, 2000, 100], dtype=np.int32)
    sy = np.array([2000, 2000, 100], dtype=np.int32)
    lab = oracle.label_brute(L, sx, sy)
    assert set(np.unique(lab)) == {0, 2}            # R4: the duplicate (larger index) owns nothing


ADVERSARIAL = [
    ("single", 64, 8, lambda rng, P: (np.array([5], np.int32), np.array([P - 1], np.int32))),
    ("one_bucket", 64, 8, lambda rng, P: (rng.integers(0, 8 * FP, 30).astype(np.int32),
                                          rng.integers(0, 8 * FP, 30).astype(np.int32))),
    ("empty_quadrants", 64, 8, lambda rng, P: (rng.integers(0, P // 4, 20).astype(np.int32),
                                               rng.integers(P // 2, 3 * P // 4, 20).astype(np.int32))),
    ("bucket_borders", 64, 8, lambda rng, P: ((rng.integers(0, 8, 50) * 8 * FP).astype(np.int32),
                                              (rng.integers(0, 8, 50) * 8 * FP - 1).clip(0).astype(np.int32))),
    ("corners", 64, 16, lambda rng, P: (np.array([0, P - 1, 0, P - 1], np.int32),
                                        np.array([0, 0, P - 1, P - 1], np.int32))),
    ("lattice_aligned_ties", 64, 8, lambda rng, P: ((rng.integers(0, 64, 100) * FP + 128).astype(np.int32),
                                                    (rng.integers(0, 64, 100) * FP + 128).astype(np.int32))),
    ("two_buckets_per_side", 64, 32, lambda rng, P: (rng.integers(0, P, 10).astype(np.int32),
                                                     rng.integers(0, P, 10).astype(np.int32))),
    ("one_bucket_per_side", 64, 64, lambda rng, P: (rng.integers(0, P, 10).astype(np.int32),
                                                    rng.integers(0, P, 10).astype(np.int32))),
    ("dense", 48, 4, lambda rng, P: (rng.integers(0, P, 3000).astype(np.int32),
                                     rng.integers(0, P, 3000).astype(np.int32))),
]


@pytest.mark.parametrize("name,L,bs,gen", ADVERSARIAL, ids=[a[0] for a in ADVERSARIAL])
def test_cell_list_equals_brute_adversarial(name, L, bs, gen):
    rng = np.random.default_rng(zlib.crc32(name.encode()))   # fixed per case: str hashes change per process
    sx, sy = gen(rng, FP * L)
    assert np.array_equal(oracle.label_cells(L, sx, sy, bs), oracle.label_brute(L, sx, sy))


def test_cell_list_equals_brute_configs_1_2_and_scaled_5():
    for w, bs, nfr in [(W.config(1), 8, 2), (W.config(2), 16, 1), (W.scaled(5, 512), 16, 3)]:
        for sx, sy in w.frames(nfr):
            assert np.array_equal(oracle.label_cells(w.L, sx, sy, bs), oracle.label_brute(w.L, sx, sy))


def test_sampled_api_matches_full():
    w = W.scaled(5, 256)
    sx, sy = next(iter(w.frames(1)))
    full = oracle.label_brute(w.L, sx, sy).ravel()
    cells = np.random.default_rng(0).integers(0, w.L * w.L, 500)
    assert np.array_equal(oracle.label_brute_at(w.L, sx, sy, cells), full[cells])
    assert np.array_equal(oracle.label_cells_at(w.L, sx, sy, 16, cells), full[cells])
