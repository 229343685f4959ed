"""Pins for the oracle's edge extraction (O2) and diff (O3).

Expected values come from geometry, not from the oracle: an exact brute-force periodic Delaunay
referee (tests/referee_delaunay.py), scipy's Delaunay on 3x3 replicated points (library), the torus
Euler relation E = 3N, the hexagonal degree-6 fact and the closed-form rhombus flip
(tests/golden/*.txt).
"""
import numpy as np
import pytest
from scipy.spatial import Delaunay

import oracle
from helpers import FP, fixed, hex_sites, pack, pairs, read_golden, rhombus_sites
from referee_delaunay import periodic_delaunay


def digital_edges(L, sx, sy):
    return oracle.edges(oracle.label_brute(L, sx, sy))


def test_edges_hand_case_2x2_blocks():
    # 4x4 lattice painted by hand: left half 3, right half 7, except one cell of 5
    lab = np.array([[3, 3, 7, 7],
                    [3, 3, 7, 7],
                    [3, 5, 7, 7],
                    [3, 3, 7, 7]], dtype=np.int32)
    # 3|7 across x=1|2 and across the wrap x=3|0; 5 touches 3 (left, up, down) and 7 (right)
    assert pairs(oracle.edges(lab)) == {(3, 7), (3, 5), (5, 7)}
    e = oracle.edges(lab)
    assert e.dtype == np.uint64 and np.all(np.diff(e.astype(np.int64)) > 0)      # ascending, unique (R16)


def test_edges_wrap_only_adjacency():
    # labels differ only across the periodic seams: row 0 vs last row, col 0 vs last col
    L = 6
    lab = np.zeros((L, L), dtype=np.int32)
    lab[0, :] = 1                       # row 0 differs from row 1 (down) and from row L-1 (wrap)
    assert pairs(oracle.edges(lab)) == {(0, 1)}
    lab = np.zeros((L, L), dtype=np.int32)
    lab[:, L - 1] = 2
    lab[L - 1, :] = 4
    assert pairs(oracle.edges(lab)) == {(0, 2), (0, 4), (2, 4)}
    assert len(oracle.edges(np.full((L, L), 9, np.int32))) == 0        # R7: own image -> no key


def test_edge_set_is_symmetric_under_label_transpose():
    rng = np.random.default_rng(11)
    L = 64
    sx = rng.integers(0, FP * L, 50).astype(np.int32)
    sy = rng.integers(0, FP * L, 50).astype(np.int32)
    lab = oracle.label_brute(L, sx, sy)
    e = pairs(oracle.edges(lab))
    # adjacency is a symmetric relation: computing it on the transposed / flipped image (which
    # swaps the roles of "right" and "down", and of a and b in every comparison) gives the same set
    assert pairs(oracle.edges(np.ascontiguousarray(lab.T))) == e
    assert pairs(oracle.edges(np.ascontiguousarray(lab[::-1, ::-1]))) == e
    assert all(i < j for i, j in e)


def test_hexagonal_lattice_degree_six():
    g = read_golden("hex_lattice.txt")
    L, cols, rows = g["L"][0], g["cols"][0], g["rows"][0]
    sx, sy = hex_sites(L, cols, rows, g["jitter"][0], seed=3)
    n = cols * rows
    assert n == g["n_sites"][0]
    e = oracle.edges(oracle.label_brute(L, sx, sy))
    assert len(e) == g["n_edges"][0] == 3 * n
    i, j = oracle.unpack(e)
    deg = np.bincount(np.concatenate([i, j]), minlength=n)
    assert np.all(deg == g["degree"][0])


def _jittered(rng, L, g, jitter):
    sp = L / g
    ix, iy = np.meshgrid(np.arange(g), np.arange(g), indexing="xy")
    x = (ix.ravel() + 0.5 + rng.uniform(-jitter, jitter, g * g)) * sp
    y = (iy.ravel() + 0.5 + rng.uniform(-jitter, jitter, g * g)) * sp
    return fixed(np.mod(x, L), L), fixed(np.mod(y, L), L)


def test_digital_edges_equal_exact_periodic_delaunay_tiny():
    """Well-separated sites at fine resolution: digital edge set == Delaunay graph, E = 3N, F = 2N."""
    rng = np.random.default_rng(21)
    L, P = 256, FP * 256
    accepted = 0
    for _ in range(12):
        sx, sy = _jittered(rng, L, 4, 0.3)
        E, T, min_ve = periodic_delaunay(sx.tolist(), sy.tolist(), P)
        if min_ve < 3 * FP:                 # rejection: shortest Voronoi edge >= 3 cells
            continue
        accepted += 1
        n = len(sx)
        assert len(E) == 3 * n and len(T) == 2 * n          # torus Euler relation (referee sanity)
        assert pairs(digital_edges(L, sx, sy)) == E
        if accepted == 2:
            break
    assert accepted >= 2


def test_rhombus_configuration_against_referee_and_golden():
    g = read_golden("rhombus_flip.txt")
    L = g["L"][0]
    for h in (g["h_prev"][0], g["h_now"][0]):
        sx, sy = rhombus_sites(L, h)
        E, T, min_ve = periodic_delaunay(sx.tolist(), sy.tolist(), FP * L)
        assert min_ve > 3 * FP
        d = pairs(digital_edges(L, sx, sy))
        assert d == E and len(d) == g["n_edges_each"][0] == 3 * g["n_sites"][0]


def _scipy_periodic_delaunay(sx, sy, L):
    n = len(sx)
    x, y = sx / FP, sy / FP
    px = np.concatenate([x + ox * L for oy in (-1, 0, 1) for ox in (-1, 0, 1)])
    py = np.concatenate([y + oy * L for oy in (-1, 0, 1) for ox in (-1, 0, 1)])
    tri = Delaunay(np.stack([px, py], axis=1))
    E = set()
    for s in tri.simplices:
        # keep simplices with a vertex in the base image (block 4 of the 9)
        if not np.any((s >= 4 * n) & (s < 5 * n)):
            continue
        for a, b in ((s[0], s[1]), (s[1], s[2]), (s[2], s[0])):
            i, j = int(a % n), int(b % n)
            if i != j:
                E.add((min(i, j), max(i, j)))
    return E, tri, np.stack([px, py], axis=1)


def test_digital_edges_vs_scipy_delaunay_medium():
    """N=400 jittered sites on 512^2 (spacing 25.6).  The digital edge set may differ from the
    Delaunay graph only next to a Voronoi edge shorter than ~1.5 cells (reading R6; PAPER.md:111,
    "the lattice acts as a natural cutoff"): it may MISS the Delaunay edge A-C dual to such a short
    Voronoi edge, and it may ADD the flipped diagonal B-D of the quadrilateral A,B,C,D around it.
    Everything else must agree exactly."""
    rng = np.random.default_rng(33)
    L = 512
    sx, sy = _jittered(rng, L, 20, 0.35)
    E, tri, pts = _scipy_periodic_delaunay(sx, sy, L)
    n = len(sx)
    assert len(E) == 3 * n
    D = pairs(digital_edges(L, sx, sy))
    cc = {}
    for s in tri.simplices:
        a, b, c = pts[s]
        d = 2 * ((b[0] - a[0]) * (c[1] - a[1]) - (b[1] - a[1]) * (c[0] - a[0]))
        a2, b2, c2 = a @ a, b @ b, c @ c
        u = np.array([(a2 * (b[1] - c[1]) + b2 * (c[1] - a[1]) + c2 * (a[1] - b[1])) / d,
                      (a2 * (c[0] - b[0]) + b2 * (a[0] - c[0]) + c2 * (b[0] - a[0])) / d])
        for k in range(3):
            p, q, opp = s[k], s[(k + 1) % 3], s[(k + 2) % 3]
            cc.setdefault((min(p, q), max(p, q)), []).append((u, opp))
    may_miss, may_add = set(), set()
    for (p, q), us in cc.items():
        if len(us) == 2 and np.hypot(*(us[0][0] - us[1][0])) < 1.5:
            i, j = int(p % n), int(q % n)
            may_miss.add((min(i, j), max(i, j)))
            i, j = int(us[0][1] % n), int(us[1][1] % n)
            may_add.add((min(i, j), max(i, j)))
    assert (E - D) <= may_miss
    assert (D - E) <= may_add
    assert len(E - D) + len(D - E) <= 0.03 * len(E)
    assert len(D & E) >= 0.97 * len(E)


# ---------------------------------------------------------------- diff (O3)

def test_flip_matches_golden():
    g = read_golden("rhombus_flip.txt")
    L = g["L"][0]
    e_prev = digital_edges(L, *rhombus_sites(L, g["h_prev"][0]))
    e_now = digital_edges(L, *rhombus_sites(L, g["h_now"][0]))
    created, destroyed = oracle.diff(e_prev, e_now)
    assert pairs(created) == {tuple(g["created"])}
    assert pairs(destroyed) == {tuple(g["destroyed"])}
    # and back again
    created, destroyed = oracle.diff(e_now, e_prev)
    assert pairs(created) == {tuple(g["destroyed"])} and pairs(destroyed) == {tuple(g["created"])}


def test_diff_hand_case_and_invariants():
    prev = pack([(0, 1), (0, 2), (1, 2), (2, 5), (7, 9)])
    now = pack([(0, 1), (1, 2), (1, 5), (2, 5), (3, 4), (7, 9)])
    c, d = oracle.diff(prev, now)
    assert pairs(c) == {(1, 5), (3, 4)} and pairs(d) == {(0, 2)}
    assert np.all(np.diff(c.astype(np.int64)) > 0)
    c, d = oracle.diff(prev, prev)
    assert len(c) == 0 and len(d) == 0
    c, d = oracle.diff(np.empty(0, np.uint64), now)
    assert np.array_equal(c, now) and len(d) == 0

    rng = np.random.default_rng(4)
    for _ in range(5):
        a = np.unique(rng.integers(0, 40, 60)); b = np.unique(rng.integers(0, 40, 60))
        mk = lambda v: pack([(int(t) // 7, 7 + int(t)) for t in v])
        pa, pb = mk(a), mk(b)
        c, d = oracle.diff(pa, pb)
        sa, sb, sc, sd = pairs(pa), pairs(pb), pairs(c), pairs(d)
        assert len(sb) == len(sa) + len(sc) - len(sd)
        assert not (sc & sa) and sd <= sa and (sa - sd) | sc == sb


def test_diff_with_translation_maps():
    # prev labels 0..3, now labels 0..3 ; prev 0->2, 1->0, 2->dead, 3->1 ; now 3 is born
    p2n = np.array([2, 0, -1, 1], np.int32)
    n2p = np.array([1, 3, 0, -1], np.int32)
    prev = pack([(0, 1), (0, 2), (1, 3), (2, 3)])
    #   translated: (0,1)->(2,0)=(0,2) ; (0,2) dropped ; (1,3)->(0,1) ; (2,3) dropped
    now = pack([(0, 1), (1, 2), (0, 3), (2, 3)])
    #   filtered:   (0,1) ; (1,2) ; (0,3) dropped (3 born) ; (2,3) dropped
    c, d = oracle.diff(prev, now, p2n, n2p)
    assert pairs(c) == {(1, 2)} and pairs(d) == {(0, 2)}
    # identity maps behave like no maps
    ident = np.arange(10, dtype=np.int32)
    c2, d2 = oracle.diff(prev, now, ident, ident)
    c3, d3 = oracle.diff(prev, now)
    assert np.array_equal(c2, c3) and np.array_equal(d2, d3)


def test_well_resolved_flips_conserve_links():
    """a bulk T1 conserves the number of links; on a torus every event is bulk."""
    from paper_1607_00908_b200 import workloads as W
    w = W.config(2)
    fr = list(w.frames(4))
    e = [oracle.edges(oracle.label_cells(w.L, sx, sy, 16)) for sx, sy in fr]
    for a, b in zip(e[:-1], e[1:]):
        c, d = oracle.diff(a, b)
        assert len(b) == len(a) + len(c) - len(d)
