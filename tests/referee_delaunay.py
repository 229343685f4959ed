"""Independent referee: brute-force periodic Delaunay graph on tiny inputs.

Closed form, exact integer arithmetic (Python ints): replicate the N sites over
the 3x3 periodic images; a non-degenerate triangle of image points with at least
one vertex in the base image is Delaunay iff no image point lies STRICTLY inside
its circumcircle (§I: "connects two sites by an edge whenever there
exists a circle that contains those two sites and no other site").  Edges are
mapped back mod N.  Shares nothing with oracle/ or the CUDA path.
"""
from __future__ import annotations

import itertools
import math


def _orient(a, b, c):
    return (b[0] - a[0]) * (c[1] - a[1]) - (b[1] - a[1]) * (c[0] - a[0])


def _incircle(a, b, c, d):
    """> 0 iff d strictly inside the circumcircle of CCW triangle abc (exact)."""
    ax, ay = a[0] - d[0], a[1] - d[1]
    bx, by = b[0] - d[0], b[1] - d[1]
    cx, cy = c[0] - d[0], c[1] - d[1]
    return ((ax * ax + ay * ay) * (bx * cy - by * cx)
            - (bx * bx + by * by) * (ax * cy - ay * cx)
            + (cx * cx + cy * cy) * (ax * by - ay * bx))


def _circumcentre(a, b, c):
    d = 2.0 * _orient(a, b, c)
    a2, b2, c2 = a[0] ** 2 + a[1] ** 2, b[0] ** 2 + b[1] ** 2, c[0] ** 2 + c[1] ** 2
    ux = (a2 * (b[1] - c[1]) + b2 * (c[1] - a[1]) + c2 * (a[1] - b[1])) / d
    uy = (a2 * (c[0] - b[0]) + b2 * (a[0] - c[0]) + c2 * (b[0] - a[0])) / d
    return ux, uy


def _canon(t):
    """Rotate (keeping orientation) so the smallest (index, ox, oy) vertex comes first, then
    translate that vertex into the base image: one representative per periodic triangle."""
    k = min(range(3), key=lambda m: t[m])
    t = (t[k], t[(k + 1) % 3], t[(k + 2) % 3])
    ox, oy = t[0][1], t[0][2]
    return tuple((v[0], v[1] - ox, v[2] - oy) for v in t)


def periodic_delaunay(sx, sy, P):
    """sites: python ints in [0,P).  Returns (edges:set[(i,j)] i<j, triangles, min_voronoi_edge).

    triangles: list of ((i,ox,oy),(j,..),(k,..)) image triples with a base-image vertex first.
    min_voronoi_edge: shortest distance between circumcentres of two Delaunay triangles sharing
    an edge, in the same units as the inputs (float; only used to reject near-degenerate inputs).
    """
    n = len(sx)
    pts = []   # (x, y, index, ox, oy)
    for oy in (-1, 0, 1):
        for ox in (-1, 0, 1):
            for i in range(n):
                pts.append((int(sx[i]) + ox * P, int(sy[i]) + oy * P, i, ox, oy))
    base = [p for p in pts if p[3] == 0 and p[4] == 0]
    # Validity domain: every accepted triangle must have circumradius R < P/2 (asserted below).
    # Then its circumcircle, which touches a base-image vertex, lies inside [-P, 2P)^2, so testing
    # emptiness against the 3x3 images is complete, and its vertices are within 2R < P of each
    # other, so partners may be restricted to |dx|,|dy| <= P.  Inputs too sparse for this (N < ~10)
    # trip the assertion instead of returning a wrong graph.
    tris = set()
    for a in base:
        near = [p for p in pts if p is not a and abs(p[0] - a[0]) <= P and abs(p[1] - a[1]) <= P]
        for b, c in itertools.combinations(near, 2):
            o = _orient(a, b, c)
            if o == 0:
                continue
            A, B, Cc = (a, b, c) if o > 0 else (a, c, b)
            ok = True
            for d in pts:
                if d is A or d is B or d is Cc:
                    continue
                if _incircle(A, B, Cc, d) > 0:
                    ok = False
                    break
            if ok:
                ux, uy = _circumcentre(A, B, Cc)
                if math.hypot(ux - A[0], uy - A[1]) >= P / 2:
                    raise ValueError("referee: circumradius >= P/2, input too sparse")
                tris.add(_canon((A[2:], B[2:], Cc[2:])))
    def xy(v):
        return (int(sx[v[0]]) + v[1] * P, int(sy[v[0]]) + v[2] * P)

    edges = set()
    by_edge = {}
    for t in tris:
        cc = _circumcentre(*(xy(v) for v in t))
        for u, v in ((t[0], t[1]), (t[1], t[2]), (t[2], t[0])):
            if u[0] != v[0]:
                edges.add((min(u[0], v[0]), max(u[0], v[0])))
            # canonical key of the geometric edge: smaller endpoint translated into the base image
            e = tuple(sorted((u, v)))
            ox, oy = e[0][1], e[0][2]
            key = ((e[0][0], 0, 0), (e[1][0], e[1][1] - ox, e[1][2] - oy))
            by_edge.setdefault(key, []).append((cc[0] - ox * P, cc[1] - oy * P))
    min_ve = math.inf
    for ccs in by_edge.values():
        for c1, c2 in itertools.combinations(ccs, 2):
            min_ve = min(min_ve, math.hypot(c1[0] - c2[0], c1[1] - c2[1]))
    return edges, sorted(tris), min_ve
