"""Pins for oracle O9: the definitions on a rectangular lattice with periodic or walled axes, obstacle
colour, 8-connected bubbles, density-weighted centres, size histogram, bulk / boundary edges
(PAPER.md:29-31, 95-99, 135, 147, 205, 248-252, 278).

What fixes the expected values: equality with the pinned square / periodic functions O1..O6 where the
geometries coincide; library routines (scipy cKDTree with and without a periodic box, scipy.ndimage.label
with the 4- and 8-neighbour structure plus hand seam unions, numpy bincount); exact equivariances
(transpose swaps the two axes, a walled lattice equals a window of a periodic lattice twice its size);
hand-painted images and graphs; closed-form centres of mass.
"""
import numpy as np
import pytest
from scipy import ndimage
from scipy.spatial import cKDTree

import oracle
from helpers import FP, pack, pairs


def rand_sites(rng, Lx, Ly, n):
    return rng.integers(0, FP * Lx, n).astype(np.int32), rng.integers(0, FP * Ly, n).astype(np.int32)


# ------------------------------------------------------------------ where the geometries coincide: O1..O6
def test_square_periodic_geometry_is_o1_to_o6():
    rng = np.random.default_rng(1)
    L, n = 48, 30
    sx, sy = rand_sites(rng, L, L, n)
    lab = oracle.label_brute(L, sx, sy)
    assert np.array_equal(oracle.label_brute_g(L, L, 1, 1, sx, sy), lab)
    assert np.array_equal(oracle.label_cells_g(L, L, 1, 1, sx, sy, 8), lab)
    cells = rng.integers(0, L * L, 100)
    assert np.array_equal(oracle.label_brute_at_g(L, L, 1, 1, sx, sy, cells), lab.ravel()[cells])
    assert np.array_equal(oracle.edges_g(lab), oracle.edges(lab))
    f = rng.random((L, L)).astype(np.float32)
    ccl = oracle.threshold_ccl(f, 0.5)
    assert np.array_equal(oracle.threshold_ccl_g(f, 0.5), ccl)
    a, b = oracle.centroids(ccl, 3), oracle.centroids_g(ccl, 3)
    for k in a:
        assert np.array_equal(a[k], b[k]), k
    px, py = rand_sites(rng, L, L, 40)
    nx = ((px.astype(np.int64) + rng.integers(-300, 300, 40)) % (FP * L)).astype(np.int32)
    ny = ((py.astype(np.int64) + rng.integers(-300, 300, 40)) % (FP * L)).astype(np.int32)
    for x, y in zip(oracle.match(L, px, py, nx, ny, 400), oracle.match_g(L, L, 1, 1, px, py, nx, ny, 400)):
        assert np.array_equal(x, y)


# ------------------------------------------------------------------ labels
@pytest.mark.parametrize("Lx,Ly,per,n,seed", [(96, 48, (1, 1), 40, 2), (40, 72, (1, 1), 9, 3), (64, 32, (0, 1), 25, 4),
                                              (48, 48, (0, 0), 30, 5), (32, 80, (1, 0), 12, 6)])
def test_labels_match_kdtree_periodic_box_or_plain(Lx, Ly, per, n, seed):
    """scipy's nearest neighbour: boxsize per axis; a walled axis gets a box so wide that nothing wraps."""
    rng = np.random.default_rng(seed)
    sx, sy = rand_sites(rng, Lx, Ly, n)
    lab = oracle.label_brute_g(Lx, Ly, per[0], per[1], sx, sy)
    box = [float(Lx) if per[0] else 4.0 * Lx, float(Ly) if per[1] else 4.0 * Ly]
    tree = cKDTree(np.stack([sx / FP, sy / FP], axis=1), boxsize=box)
    yy, xx = np.mgrid[0:Ly, 0:Lx]
    d, idx = tree.query(np.stack([xx.ravel() + 0.5, yy.ravel() + 0.5], axis=1), k=2)
    clear = (d[:, 1] - d[:, 0]) > 1e-9
    assert clear.mean() > 0.95
    assert np.array_equal(lab.ravel()[clear], idx[clear, 0])
    assert np.array_equal(oracle.label_cells_g(Lx, Ly, per[0], per[1], sx, sy, 8), lab)      # R3 ring search
    assert np.array_equal(oracle.label_cells_g(Lx, Ly, per[0], per[1], sx, sy, 4), lab)


def test_transpose_swaps_the_axes():
    rng = np.random.default_rng(7)
    Lx, Ly = 56, 24
    sx, sy = rand_sites(rng, Lx, Ly, 20)
    for per in ((1, 1), (0, 1), (1, 0), (0, 0)):
        a = oracle.label_brute_g(Lx, Ly, per[0], per[1], sx, sy)
        assert np.array_equal(oracle.label_brute_g(Ly, Lx, per[1], per[0], sy, sx), a.T)


def test_walled_lattice_is_a_window_of_a_periodic_lattice_twice_its_size():
    """Inside the domain a plain difference never exceeds the domain, i.e. half the doubled period: the
    minimum image on the doubled lattice is the plain distance (this is how the CUDA path labels walled
    domains; here it pins the walled branch of O9 against the periodic branch)."""
    rng = np.random.default_rng(8)
    Lx, Ly = 40, 24
    sx, sy = rand_sites(rng, Lx, Ly, 15)
    assert np.array_equal(oracle.label_brute_g(Lx, Ly, 0, 0, sx, sy),
                          oracle.label_brute_g(2 * Lx, 2 * Ly, 1, 1, sx, sy)[:Ly, :Lx])
    assert np.array_equal(oracle.label_brute_g(Lx, Ly, 0, 1, sx, sy),
                          oracle.label_brute_g(2 * Lx, Ly, 1, 1, sx, sy)[:, :Lx])


def test_wall_hand_case_and_ties():
    # two sites at the two ends of a 16 x 4 channel: with walls the split is in the middle, on a periodic
    # axis the seam is a second border; ties on the middle column go to the smaller index
    Lx, Ly = 16, 4
    sx, sy = np.array([FP * 2, FP * 14], np.int32), np.array([FP * 2, FP * 2], np.int32)
    wall = oracle.label_brute_g(Lx, Ly, 0, 1, sx, sy)
    assert np.all(wall[:, :8] == 0) and np.all(wall[:, 8:] == 1)           # centres 0.5 .. 7.5 | 8.5 .. 15.5
    sx2 = np.array([FP * 2 + 128, FP * 12 + 128], np.int32)                 # mirror images about the centre 7.5 of column 7
    tie = oracle.label_brute_g(Lx, Ly, 0, 1, sx2, sy)
    assert np.all(tie[:, 7] == 0) and np.all(tie[:, 6] == 0) and np.all(tie[:, 8] == 1) and np.all(tie[:, 0] == 0)
    assert np.all(oracle.label_brute_g(Lx, Ly, 0, 1, sx2[::-1].copy(), sy)[:, 7] == 0)   # ... whichever side it is on
    per = oracle.label_brute_g(Lx, Ly, 1, 1, np.array([FP * 1, FP * 9], np.int32), sy)
    # centre 12.5 is 3.5 from the site at 9 and 4.5 from the image of the site at 1 (17); centre 13.5 the reverse
    assert per[0, 15] == 0 and per[0, 13] == 0 and per[0, 12] == 1 and per[0, 5] == 1 and per[0, 4] == 0
    assert np.all(oracle.label_brute_g(Lx, Ly, 0, 1, np.array([FP * 1, FP * 9], np.int32), sy)[:, 13:] == 1)


# ------------------------------------------------------------------ edges: walls, obstacles, rectangles
def test_edges_hand_image_walls_and_obstacles():
    lab = np.array([[0, 0, 1, 1, 1, 2],
                    [0, 0, 1, 1, 2, 2],
                    [3, 3, 3, 9, 2, 2],
                    [3, 3, 3, 9, 9, 2]], np.int32)
    inner = {(0, 1), (1, 2), (0, 3), (1, 3), (1, 9), (2, 9), (3, 9)}
    assert pairs(oracle.edges_g(lab, 0, 0)) == inner
    # periodic in x adds column 5 | column 0: (2,0), (2,0), (2,3), (2,3); in y row 3 | row 0: (3,0), (3,1), (9,1), (2,2)
    assert pairs(oracle.edges_g(lab, 1, 0)) == inner | {(0, 2), (2, 3)}
    assert pairs(oracle.edges_g(lab, 0, 1)) == inner | {(0, 3), (1, 3), (1, 9)}
    assert pairs(oracle.edges_g(lab, 1, 1)) == inner | {(0, 2), (2, 3)}
    # colour 9 is an obstacle: every pair with it disappears, nothing else changes
    assert pairs(oracle.edges_g(lab, 0, 0, exclude=9)) == {(0, 1), (1, 2), (0, 3), (1, 3)}
    assert pairs(oracle.edges_g(lab, 1, 1, exclude=9)) == {(0, 1), (1, 2), (0, 3), (1, 3), (0, 2), (2, 3)}
    # the obstacle separates 2 from 3 inside the domain: they meet only through the periodic seam
    assert (2, 3) not in pairs(oracle.edges_g(lab, 0, 0, exclude=9))


def test_apply_obstacles_and_exclusion():
    rng = np.random.default_rng(9)
    Lx, Ly, n = 64, 32, 12
    sx, sy = rand_sites(rng, Lx, Ly, n)
    lab = oracle.label_brute_g(Lx, Ly, 0, 1, sx, sy)
    mask = np.zeros((Ly, Lx), np.uint8)
    mask[:, :3] = 1                                             # a wall of posts on the left
    mask[8:12, 3:20] = 1
    MAXLINK = 0x77777777
    col = oracle.apply_obstacles(lab, mask, MAXLINK)
    assert np.all(col[mask == 1] == MAXLINK) and np.array_equal(col[mask == 0], lab[mask == 0])
    e = pairs(oracle.edges_g(col, 0, 1, exclude=MAXLINK))
    assert all(max(p) < n for p in e)
    # brute force over the cell pairs that survive
    ref = set()
    for y in range(Ly):
        for x in range(Lx):
            for (u, v) in ((x + 1, y), (x, (y + 1) % Ly)):
                if u < Lx and not mask[y, x] and not mask[v, u] and lab[y, x] != lab[v, u]:
                    ref.add((min(lab[y, x], lab[v, u]), max(lab[y, x], lab[v, u])))
    assert e == ref


# ------------------------------------------------------------------ bubbles: 8-connectivity, walls, rectangles
def partition_scipy(mask, per_x, per_y, conn):
    st = np.ones((3, 3), int) if conn == 8 else [[0, 1, 0], [1, 1, 1], [0, 1, 0]]
    lab, k = ndimage.label(mask, structure=st)
    parent = list(range(k + 1))

    def find(a):
        while parent[a] != a:
            parent[a] = parent[parent[a]]
            a = parent[a]
        return a

    def union(a, b):
        if a and b:
            ra, rb = find(a), find(b)
            if ra != rb:
                parent[max(ra, rb)] = min(ra, rb)

    Ly, Lx = mask.shape
    steps = (-1, 0, 1) if conn == 8 else (0,)
    if per_x:
        for y in range(Ly):
            for d in steps:
                v = y + d
                if 0 <= v < Ly or per_y:
                    union(lab[y, Lx - 1], lab[v % Ly, 0])
    if per_y:
        for x in range(Lx):
            for d in steps:
                u = x + d
                if 0 <= u < Lx or per_x:
                    union(lab[Ly - 1, x], lab[0, u % Lx])
    return np.array([find(a) for a in range(k + 1)])[lab]


def assert_partition(ccl, ref):
    Ly, Lx = ccl.shape
    assert np.array_equal(ccl >= 0, ref > 0)
    idx = np.arange(Lx * Ly).reshape(Ly, Lx)
    for r in np.unique(ref[ref > 0]):
        labs = np.unique(ccl[ref == r])
        assert len(labs) == 1 and labs[0] == idx[ref == r].min()
    assert len(np.unique(ccl[ccl >= 0])) == len(np.unique(ref[ref > 0]))


@pytest.mark.parametrize("Lx,Ly,per,conn,p,seed", [(32, 32, (1, 1), 8, 0.35, 0), (48, 20, (1, 1), 8, 0.4, 1),
                                                   (48, 20, (1, 1), 4, 0.55, 2), (40, 40, (0, 0), 4, 0.55, 3),
                                                   (40, 24, (0, 1), 8, 0.38, 4), (24, 40, (1, 0), 4, 0.6, 5),
                                                   (17, 9, (1, 1), 8, 0.45, 6)])
def test_ccl_equals_scipy(Lx, Ly, per, conn, p, seed):
    rng = np.random.default_rng(seed)
    f = rng.random((Ly, Lx)).astype(np.float32)
    ccl = oracle.threshold_ccl_g(f, 1.0 - p, True, per[0], per[1], conn)
    assert_partition(ccl, partition_scipy(f > np.float32(1.0 - p), per[0], per[1], conn))


def test_ccl_diagonal_hand_cases():
    f = np.zeros((6, 8), np.float32)
    f[1, 1] = f[2, 2] = 2                                  # a diagonal pair
    f[0, 7] = f[5, 0] = 2                                  # diagonal across the corner of the torus
    f[2, 7] = f[3, 0] = 2                                  # diagonal across the x seam only
    c4 = oracle.threshold_ccl_g(f, 1.0, True, 1, 1, 4)
    assert len(np.unique(c4[c4 >= 0])) == 6
    c8 = oracle.threshold_ccl_g(f, 1.0, True, 1, 1, 8)
    assert c8[1, 1] == c8[2, 2] == 1 * 8 + 1
    assert c8[0, 7] == c8[5, 0] == 7
    assert c8[2, 7] == c8[3, 0] == 2 * 8 + 7
    c8w = oracle.threshold_ccl_g(f, 1.0, True, 0, 0, 8)    # walls: only the inner diagonal remains joined
    assert c8w[1, 1] == c8w[2, 2] and len(np.unique(c8w[c8w >= 0])) == 5
    c8x = oracle.threshold_ccl_g(f, 1.0, True, 1, 0, 8)    # periodic in x only: the x-seam diagonal joins
    assert c8x[2, 7] == c8x[3, 0] and c8x[0, 7] != c8x[5, 0]
    with pytest.raises(ValueError):
        oracle.threshold_ccl_g(f, 1.0, True, 1, 1, 6)


# ------------------------------------------------------------------ centres of mass: weights, walls, rectangles
def test_weighted_centre_closed_forms():
    Lx, Ly = 16, 8
    ccl = -np.ones((Ly, Lx), np.int32)
    ccl[2, 3] = ccl[2, 4] = 2 * Lx + 3                      # two cells, weights 1 : 3 -> 3/4 of the way
    f = np.zeros((Ly, Lx), np.float32)
    f[2, 3], f[2, 4] = 1.0, 3.0
    c = oracle.centroids_g(ccl, 1, 1, 1, f)
    assert c["size"].tolist() == [2] and c["cx"][0] == 3.5 + 0.75 and c["cy"][0] == 2.5
    assert c["sx"][0] == FP * 3 + 128 + 192 and c["sy"][0] == FP * 2 + 128
    # equal weights: exactly the unweighted centre, whatever the common value
    for v in (0.25, 1.0, 7.5):
        g = np.full((Ly, Lx), v, np.float32)
        a, b = oracle.centroids_g(ccl, 1, 1, 1, g), oracle.centroids_g(ccl, 1)
        assert all(np.array_equal(a[k], b[k]) for k in a)
    # the weight is floor(rho * 65536) limited to [1, 2^24]: zero, negative and NaN densities weigh one unit
    f2 = np.zeros((Ly, Lx), np.float32)
    f2[2, 3], f2[2, 4] = np.nan, 3.0 / 65536.0              # weights 1 and 3
    assert oracle.centroids_g(ccl, 1, 1, 1, f2)["cx"][0] == 3.5 + 0.75
    f2[2, 3], f2[2, 4] = -5.0, 1e9                          # weights 1 and 2^24
    assert oracle.centroids_g(ccl, 1, 1, 1, f2)["cx"][0] == 3.5 + 16777216.0 / 16777217.0


def test_weighted_disc_with_symmetric_density():
    """A disc with a radially symmetric density about a cell centre has its centre of mass there, also
    across the seam; a linear density gradient moves it by the closed-form amount on a 1-d bar."""
    Lx, Ly = 64, 40
    yy, xx = np.mgrid[0:Ly, 0:Lx]
    for cxr, cyr in ((20, 17), (0, 0), (63, 39)):
        dx = (xx - cxr + Lx // 2) % Lx - Lx // 2
        dy = (yy - cyr + Ly // 2) % Ly - Ly // 2
        r2 = dx * dx + dy * dy
        mask = r2 <= 36
        rho = np.where(mask, 1.0 + r2 / 8.0, 0.0).astype(np.float32)      # multiples of 1/8: exact weights
        ccl = oracle.threshold_ccl_g(mask.astype(np.float32), 0.5, True, 1, 1, 4)
        c = oracle.centroids_g(ccl, 1, 1, 1, rho)
        assert len(c["cx"]) == 1 and abs(c["cx"][0] - (cxr + 0.5)) < 1e-12 and abs(c["cy"][0] - (cyr + 0.5)) < 1e-12
        assert c["sx"][0] == FP * cxr + 128 and c["sy"][0] == FP * cyr + 128
    # bar of 4 cells, weights 1, 2, 3, 4 (x 65536): centre = x0 + 0.5 + (0*1 + 1*2 + 2*3 + 3*4) / 10
    ccl = -np.ones((4, 8), np.int32)
    ccl[1, 2:6] = 8 + 2
    f = np.zeros((4, 8), np.float32)
    f[1, 2:6] = [1, 2, 3, 4]
    c = oracle.centroids_g(ccl, 1, 0, 0, f)
    assert c["cx"][0] == 2.5 + 2.0 and c["sx"][0] == FP * 2 + 128 + 512


def test_centres_do_not_unwrap_across_a_wall():
    Lx, Ly = 16, 8
    ccl = -np.ones((Ly, Lx), np.int32)
    ccl[3, 0] = ccl[3, 15] = 3 * Lx                          # two cells at the two ends of row 3, one label
    per = oracle.centroids_g(ccl, 1, 1, 1)
    assert per["cx"][0] == 0.0                               # neighbours through the seam: centre on the seam
    wall = oracle.centroids_g(ccl, 1, 0, 1)
    assert wall["cx"][0] == 8.0                              # plain mean of 0.5 and 15.5
    assert wall["sx"][0] == FP * 8


def test_match_across_seam_only_when_periodic():
    Lx, Ly = 32, 16
    px, py = np.array([FP * 31 + 200], np.int32), np.array([FP * 4], np.int32)
    nx, ny = np.array([40], np.int32), np.array([FP * 4], np.int32)         # 96 units away through the seam
    assert oracle.match_g(Lx, Ly, 1, 1, px, py, nx, ny, 100)[0].tolist() == [0]
    assert oracle.match_g(Lx, Ly, 0, 1, px, py, nx, ny, 100)[0].tolist() == [-1]
    assert oracle.match_g(Lx, Ly, 1, 1, px, py, nx, ny, 95)[0].tolist() == [-1]
    # y axis likewise, on a rectangle whose periods differ
    py2, ny2 = np.array([FP * 15 + 250], np.int32), np.array([2], np.int32)
    assert oracle.match_g(Lx, Ly, 1, 1, nx, py2, nx, ny2, 10)[0].tolist() == [0]
    assert oracle.match_g(Lx, Ly, 1, 0, nx, py2, nx, ny2, 10)[0].tolist() == [-1]


# ------------------------------------------------------------------ size histogram, bulk / boundary edges
def test_size_histogram_is_bincount():
    rng = np.random.default_rng(10)
    size = rng.integers(1, 500, 1000).astype(np.int32)
    for width, bins in ((1, 600), (16, 32), (50, 4)):
        ref = np.bincount(np.minimum(size // width, bins - 1), minlength=bins)
        assert np.array_equal(oracle.size_histogram(size, width, bins), ref)
    assert oracle.size_histogram(np.array([], np.int32), 4, 3).tolist() == [0, 0, 0]


def test_edge_commons_hand_strip_and_sets():
    # a strip of triangles 0-1-2-3-4-5 (zig-zag): outer edges share one neighbour, inner diagonals two
    #   0---2---4
    #    \ / \ / \
    #     1---3---5
    e = [(0, 1), (0, 2), (1, 2), (1, 3), (2, 3), (2, 4), (3, 4), (3, 5), (4, 5)]
    c = oracle.edge_commons(pack(e), 6)
    want = {(0, 1): 1, (0, 2): 1, (1, 2): 2, (1, 3): 1, (2, 3): 2, (2, 4): 1, (3, 4): 2, (3, 5): 1, (4, 5): 1}
    assert c.tolist() == [want[p] for p in sorted(e)]
    rng = np.random.default_rng(12)
    n = 40
    allp = [(i, j) for i in range(n) for j in range(i + 1, n) if rng.random() < 0.2]
    rows = [set() for _ in range(n)]
    for i, j in allp:
        rows[i].add(j); rows[j].add(i)
    got = oracle.edge_commons(pack(allp), n)
    assert got.tolist() == [len(rows[i] & rows[j]) for i, j in sorted(allp)]
    assert oracle.edge_commons(pack([(0, 1), (1, 7)]), 3).tolist() == [0, -1]       # labels >= n take no part


def test_triangulated_torus_has_only_bulk_edges_and_walls_make_a_boundary():
    """On the torus every edge of a well-resolved triangulation is shared by two triangles;
    with walls the edges of the outer hull are shared by one."""
    from helpers import hex_sites
    L = 256
    sx, sy = hex_sites(L, 16, 18, 0.8, seed=3)
    per = oracle.edges(oracle.label_brute(L, sx, sy))
    assert set(oracle.edge_commons(per, len(sx)).tolist()) == {2}
    wall = oracle.edges_g(oracle.label_brute_g(L, L, 0, 0, sx, sy), 0, 0)
    c = oracle.edge_commons(wall, len(sx))
    assert (c == 1).sum() > 40 and (c == 2).sum() > 500 and set(c.tolist()) <= {1, 2}
