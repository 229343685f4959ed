"""Pins for the oracle's field path: threshold+CCL (O4), centroids (O5), matching (O6).

Expected values: scipy.ndimage.label (library) with the periodic seams unioned by hand; hand-drawn
masks; the closed-form centroid of a symmetric disc; exact shift equivariance; matching invariants.
"""
import numpy as np
import pytest
from scipy import ndimage

import oracle
from helpers import FP


def periodic_partition_scipy(mask):
    """4-connected periodic components via scipy + union of labels across the two seams."""
    lab, k = ndimage.label(mask, structure=[[0, 1, 0], [1, 1, 1], [0, 1, 0]])
    parent = list(range(k + 1))

    def find(a):
        while parent[a] != a:
            parent[a] = parent[parent[a]]
            a = parent[a]
        return a

    L = mask.shape[0]
    for i in range(L):
        for a, b in ((lab[i, 0], lab[i, L - 1]), (lab[0, i], lab[L - 1, i])):
            if a and b:
                ra, rb = find(a), find(b)
                if ra != rb:
                    parent[max(ra, rb)] = min(ra, rb)
    out = np.array([find(a) for a in range(k + 1)])[lab]
    return out          # 0 = background


def assert_same_partition_with_min_index_labels(ccl, ref):
    L = ccl.shape[0]
    assert np.array_equal(ccl >= 0, ref > 0)
    idx = np.arange(L * L).reshape(L, L)
    for r in np.unique(ref[ref > 0]):
        members = ref == r
        labs = np.unique(ccl[members])
        assert len(labs) == 1                               # one oracle label per scipy component
        assert labs[0] == idx[members].min()                # and it is the minimum linear index
    assert len(np.unique(ccl[ccl >= 0])) == len(np.unique(ref[ref > 0]))


@pytest.mark.parametrize("seed,L,p", [(0, 32, 0.4), (1, 64, 0.55), (2, 50, 0.62), (3, 17, 0.5)])
def test_ccl_equals_scipy_periodic(seed, L, p):
    rng = np.random.default_rng(seed)
    field = rng.random((L, L)).astype(np.float32)
    ccl = oracle.threshold_ccl(field, 1.0 - p, above=True)
    assert_same_partition_with_min_index_labels(ccl, periodic_partition_scipy(field > np.float32(1.0 - p)))


def test_ccl_hand_cases():
    L = 8
    f = np.zeros((L, L), np.float32)
    # component crossing the corner: cells (0,0), (0,7), (7,0) [row, col]
    f[0, 0] = f[0, 7] = f[7, 0] = 2
    # ring around the torus along row 4
    f[4, :] = 2
    # single cell
    f[2, 3] = 2
    ccl = oracle.threshold_ccl(f, 1.0, above=True)
    assert ccl[0, 0] == ccl[0, 7] == ccl[7, 0] == 0
    assert np.all(ccl[4, :] == 4 * L)
    assert ccl[2, 3] == 2 * L + 3
    assert (ccl >= 0).sum() == 3 + L + 1 and ccl[1, 1] == -1
    # full lattice / empty mask / polarity / NaN
    assert np.all(oracle.threshold_ccl(np.full((L, L), 5, np.float32), 1.0) == 0)
    assert np.all(oracle.threshold_ccl(np.zeros((L, L), np.float32), 1.0) == -1)
    assert np.all(oracle.threshold_ccl(np.zeros((L, L), np.float32), 1.0, above=False) == 0)
    g = np.full((L, L), np.nan, np.float32)
    assert np.all(oracle.threshold_ccl(g, 1.0, True) == -1) and np.all(oracle.threshold_ccl(g, 1.0, False) == -1)
    # strict comparison: field == thr is background
    assert np.all(oracle.threshold_ccl(np.full((L, L), 1.0, np.float32), 1.0) == -1)
    # diagonal neighbours are NOT connected (4-connectivity, R9)
    d = np.zeros((L, L), np.float32); d[1, 1] = d[2, 2] = 2
    c = oracle.threshold_ccl(d, 1.0)
    assert c[1, 1] != c[2, 2]


def disc_mask(L, cx, cy, r):
    yy, xx = np.mgrid[0:L, 0:L]
    dx = np.abs(xx + 0.5 - cx); dx = np.minimum(dx, L - dx)
    dy = np.abs(yy + 0.5 - cy); dy = np.minimum(dy, L - dy)
    return dx * dx + dy * dy <= r * r


@pytest.mark.parametrize("cx,cy", [(20.5, 30.5), (20.0, 30.0), (0.5, 0.5), (0.0, 63.5), (63.5, 0.0)])
def test_centroid_of_symmetric_disc_is_its_centre(cx, cy):
    """A disc rasterised about a cell centre or a cell corner is point-symmetric about it, so the
    mean of its cell centres is exactly that point — also across the periodic seams."""
    L = 64
    m = disc_mask(L, cx, cy, 6.3)
    ccl = oracle.threshold_ccl(m.astype(np.float32), 0.5)
    c = oracle.centroids(ccl, 1)
    assert len(c["cx"]) == 1 and c["size"][0] == m.sum()
    assert abs(c["cx"][0] - cx % L) < 1e-12 and abs(c["cy"][0] - cy % L) < 1e-12
    assert c["sx"][0] == int(round(cx * FP)) % (FP * L) and c["sy"][0] == int(round(cy * FP)) % (FP * L)
    assert c["root"][0] == ccl[ccl >= 0].min()


def test_centroid_hand_case_floor_rounding():
    L = 16
    f = np.zeros((L, L), np.float32)
    f[3, 5] = f[3, 6] = f[4, 5] = 2            # L-shaped triple: mean x = 5.5+1/3, mean y = 3.5+1/3
    c = oracle.centroids(oracle.threshold_ccl(f, 1.0), 1)
    assert c["size"][0] == 3 and c["root"][0] == 3 * L + 5
    assert abs(c["cx"][0] - (5.5 + 1 / 3)) < 1e-12 and abs(c["cy"][0] - (3.5 + 1 / 3)) < 1e-12
    assert c["sx"][0] == 5 * FP + 128 + (FP * 1) // 3 and c["sy"][0] == 3 * FP + 128 + (FP * 1) // 3
    # negative offset: root is the min index (top-left-most in row order), members to its LEFT below
    f = np.zeros((L, L), np.float32)
    f[3, 5] = f[4, 5] = f[4, 4] = 2            # mean x = 5.5 - 1/3 -> floor(-256/3) = -86
    c = oracle.centroids(oracle.threshold_ccl(f, 1.0), 1)
    assert c["sx"][0] == 5 * FP + 128 - 86 and abs(c["cx"][0] - (5.5 - 1 / 3)) < 1e-12


def test_centroid_upper_wrap_branch_hand_case():
    """Root (minimum index) at x = L-2 with the lower rows wrapping to x = 0..3: the unwrapped mean lies
    beyond L and must come back by -L (the `>= L` branch).  Expected value by hand: unwrapped cell
    centres x = 14.5, 15.5 | 15.5, 16.5, 17.5, 18.5, 19.5 | 16.5, 17.5, 18.5, 19.5 -> sum 189.5, n 11."""
    L = 16
    f = np.zeros((L, L), np.float32)
    f[3, 14] = f[3, 15] = 2
    f[4, 15] = f[4, 0] = f[4, 1] = f[4, 2] = f[4, 3] = 2
    f[5, 0] = f[5, 1] = f[5, 2] = f[5, 3] = 2
    for g, (kx, ky, ks, kt) in ((f, ("cx", "cy", "sx", "sy")), (np.ascontiguousarray(f.T), ("cy", "cx", "sy", "sx"))):
        c = oracle.centroids(oracle.threshold_ccl(g, 1.0), 1)
        assert len(c["cx"]) == 1 and c["size"][0] == 11
        assert abs(c[kx][0] - (189.5 / 11 - L)) < 1e-12          # 1.2272...: wrapped back into [0, L)
        assert abs(c[ky][0] - (3.5 * 2 + 4.5 * 5 + 5.5 * 4) / 11) < 1e-12
        # fixed point: floor(256 * 30 / 11) = 698 past the root's centre 14.5, mod P
        assert c[ks][0] == (14 * FP + 128 + (FP * 30) // 11) % (FP * L)
        assert c[kt][0] == 3 * FP + 128 + (FP * (5 + 8)) // 11
    # the root itself: row-major minimum (3,14) for f; for the transpose the minimum index is (0,4)
    assert oracle.centroids(oracle.threshold_ccl(f, 1.0), 1)["root"][0] == 3 * L + 14


def test_centroids_shift_equivariance_and_min_size():
    rng = np.random.default_rng(9)
    L = 96
    base = ndimage.gaussian_filter(rng.standard_normal((L, L)), 3.0, mode="wrap").astype(np.float32)
    thr = float(np.quantile(base, 0.8))
    ccl = oracle.threshold_ccl(base, thr)
    c0 = oracle.centroids(ccl, 5)
    sizes = np.bincount(ccl[ccl >= 0])
    kept = sizes[sizes >= 5]
    assert c0["size"].sum() == kept.sum() and len(c0["size"]) == len(kept)
    assert np.all(np.diff(c0["root"]) > 0)
    for kx, ky in [(1, 0), (40, 77), (95, 95)]:
        c1 = oracle.centroids(oracle.threshold_ccl(np.roll(base, (ky, kx), axis=(0, 1)), thr), 5)
        # components are renumbered by their new roots: compare as multisets of (size, shifted position)
        a = sorted(zip(c0["size"].tolist(), ((c0["sx"].astype(np.int64) + kx * FP) % (FP * L)).tolist(),
                       ((c0["sy"].astype(np.int64) + ky * FP) % (FP * L)).tolist()))
        b = sorted(zip(c1["size"].tolist(), c1["sx"].tolist(), c1["sy"].tolist()))
        # unwrap reference (root cell) changes with the shift; for components narrower than L/2 the
        # integer mean is reference-independent up to the floor of an exact rational: identical
        assert a == b


def test_match_invariants():
    rng = np.random.default_rng(12)
    L = 128
    P = FP * L
    n = 60
    # well separated points (jittered grid 8x8 minus a few)
    g = 8
    ix, iy = np.meshgrid(np.arange(g), np.arange(g), indexing="xy")
    x = ((ix.ravel() + 0.5) * (L / g) + rng.uniform(-2, 2, g * g))[:n]
    y = ((iy.ravel() + 0.5) * (L / g) + rng.uniform(-2, 2, g * g))[:n]
    px = (np.floor(x * FP).astype(np.int64) % P).astype(np.int32)
    py = (np.floor(y * FP).astype(np.int64) % P).astype(np.int32)
    R = 4 * FP
    p2n, n2p = oracle.match(L, px, py, px, py, R)
    assert np.array_equal(p2n, np.arange(n)) and np.array_equal(n2p, np.arange(n))      # identical frames
    nx = ((px.astype(np.int64) + 3 * FP) % P).astype(np.int32)                           # rigid shift < radius
    ny = ((py.astype(np.int64) - 2 * FP) % P).astype(np.int32)
    p2n, n2p = oracle.match(L, px, py, nx, ny, R)
    assert np.array_equal(p2n, np.arange(n)) and np.array_equal(n2p, np.arange(n))
    p2n, n2p = oracle.match(L, np.delete(px, 7), np.delete(py, 7), nx, ny, R)            # one born
    assert (n2p == -1).sum() == 1 and n2p[7] == -1 and (p2n >= 0).all()
    assert np.array_equal(p2n, np.delete(np.arange(n), 7))
    perm = rng.permutation(n)                                                            # relabelled
    p2n, n2p = oracle.match(L, px, py, nx[perm], ny[perm], R)
    assert np.array_equal(perm[p2n], np.arange(n)) and np.array_equal(n2p, perm)
    # shift beyond the radius -> nothing matches; radius is inclusive
    fx = ((px.astype(np.int64) + 5 * FP) % P).astype(np.int32)
    p2n, n2p = oracle.match(L, px, py, fx, py, R)
    assert (p2n == -1).all() and (n2p == -1).all()
    ex = ((px.astype(np.int64) + 4 * FP) % P).astype(np.int32)
    p2n, n2p = oracle.match(L, px, py, ex, py, R)
    assert np.array_equal(p2n, np.arange(n))


def test_match_is_injective_and_mutual_on_random_clouds():
    rng = np.random.default_rng(13)
    L, P = 64, FP * 64
    for _ in range(5):
        px, py = rng.integers(0, P, 80).astype(np.int32), rng.integers(0, P, 80).astype(np.int32)
        nx, ny = rng.integers(0, P, 70).astype(np.int32), rng.integers(0, P, 70).astype(np.int32)
        p2n, n2p = oracle.match(L, px, py, nx, ny, 6 * FP)
        m = p2n[p2n >= 0]
        assert len(np.unique(m)) == len(m)
        for i, j in enumerate(p2n):
            if j >= 0:
                assert n2p[j] == i
        for j, i in enumerate(n2p):
            if i >= 0:
                assert p2n[i] == j
        # two coincident prev points compete for one now point: smallest index wins (R13)
    px = np.array([1000, 1000], np.int32); py = np.array([1000, 1000], np.int32)
    p2n, n2p = oracle.match(L, px, py, np.array([1100], np.int32), np.array([1000], np.int32), 4 * FP)
    assert p2n.tolist() == [0, -1] and n2p.tolist() == [0]
