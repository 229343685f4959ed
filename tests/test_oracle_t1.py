"""Pins for oracle O8 (couples of active vertices, breaking / arising class, bulk / boundary edges by
common neighbours, T1 pairing; PAPER.md:238, 248-252, 258-266 and Fig. 8)."""
import numpy as np

import oracle
from helpers import pack, read_golden, rhombus_sites

NONE = np.uint64(0xFFFFFFFFFFFFFFFF)


def key(i, j):
    return (min(i, j) << 32) | max(i, j)


def brute(prev_pairs, now_pairs, n):
    """Python sets, straight from the sentences of the paper."""
    def rows(ps):
        r = [set() for _ in range(n)]
        for i, j in ps:
            if i < n and j < n:
                r[i].add(j); r[j].add(i)
        return r
    rp, rn = rows(prev_pairs), rows(now_pairs)
    act = [rp[i] != rn[i] for i in range(n)]
    out = []
    for i in range(n):
        for j in range(i + 1, n):
            if not (act[i] and act[j]):
                continue
            in_p, in_n = j in rp[i], j in rn[i]
            if not (in_p or in_n):
                continue
            sp, sn = sorted(rp[i] & rp[j]), sorted(rn[i] & rn[j])
            pt = None
            if in_p and not in_n and len(sp) == 2 and sp[1] in rn[sp[0]] and sp[1] not in rp[sp[0]]:
                pt = key(*sp)
            if in_n and not in_p and len(sn) == 2 and sn[1] in rp[sn[0]] and sn[1] not in rn[sn[0]]:
                pt = key(*sn)
            out.append((key(i, j), 0 if in_p and in_n else (1 if in_p else 2), len(sp) if in_p else -1,
                        len(sn) if in_n else -1, pt))
    return out


def check(prev_pairs, now_pairs, n):
    r = oracle.t1(pack(prev_pairs), pack(now_pairs), n)
    ref = brute(prev_pairs, now_pairs, n)
    assert r["couples"].tolist() == [c[0] for c in ref]
    assert r["cls"].tolist() == [c[1] for c in ref]
    assert r["common_prev"].tolist() == [c[2] for c in ref] and r["common_now"].tolist() == [c[3] for c in ref]
    assert [None if p == NONE else int(p) for p in r["partner"]] == [c[4] for c in ref]
    return r


def test_single_t1_hand_graph():
    # rhombus 0-1-2-3, diagonal 1-3 flips to 0-2; 4 and 5 are bystanders that close the outer triangles
    common = [(0, 1), (1, 2), (2, 3), (0, 3), (0, 4), (1, 4), (2, 5), (3, 5), (4, 5)]
    r = check(common + [(1, 3)], common + [(0, 2)], 6)
    k = r["couples"].tolist()
    assert k == [key(0, 1), key(0, 2), key(0, 3), key(1, 2), key(1, 3), key(2, 3)]
    assert r["cls"].tolist() == [0, 2, 0, 0, 1, 0]
    assert int(r["partner"][k.index(key(1, 3))]) == key(0, 2)          # breaking <-> arising
    assert int(r["partner"][k.index(key(0, 2))]) == key(1, 3)
    assert r["common_prev"][k.index(key(1, 3))] == 2 and r["common_now"][k.index(key(0, 2))] == 2
    assert all(p == NONE for p, c in zip(r["partner"], r["cls"]) if c == 0)


def test_two_simultaneous_t1_events():
    """Two disjoint rhombi flip in the same frame: every breaking link pairs with the arising link of ITS
    rhombus, never with the other one."""
    def rhombus(o):
        return [(o, o + 1), (o + 1, o + 2), (o + 2, o + 3), (o, o + 3)]
    glue = [(3, 4), (2, 4), (2, 5)]                                     # a strip joining the two rhombi
    prev = rhombus(0) + rhombus(4) + glue + [(1, 3), (4, 6)]
    now = rhombus(0) + rhombus(4) + glue + [(0, 2), (5, 7)]
    r = check(prev, now, 8)
    k = r["couples"].tolist()
    assert int(r["partner"][k.index(key(1, 3))]) == key(0, 2) and int(r["partner"][k.index(key(0, 2))]) == key(1, 3)
    assert int(r["partner"][k.index(key(4, 6))]) == key(5, 7) and int(r["partner"][k.index(key(5, 7))]) == key(4, 6)
    assert sorted(int(c) for c, s in zip(r["couples"], r["cls"]) if s == 1) == [key(1, 3), key(4, 6)]
    assert sorted(int(c) for c, s in zip(r["couples"], r["cls"]) if s == 2) == [key(0, 2), key(5, 7)]


def test_boundary_event_has_a_breaking_link_and_no_partner():
    # PAPER.md Fig. 8 bottom: a boundary link disappears, nothing arises; its end points share ONE neighbour
    r = check([(0, 1), (1, 2), (0, 2)], [(0, 1), (1, 2)], 3)
    assert r["couples"].tolist() == [key(0, 2)] and r["cls"].tolist() == [1]
    assert r["common_prev"].tolist() == [1] and r["common_now"].tolist() == [-1]      # boundary edge, gone now
    assert r["partner"][0] == NONE


def test_breaking_link_whose_common_neighbours_were_already_connected_has_no_partner():
    # tetrahedron 0-1-2-3 loses (0,1): its common neighbours 2, 3 are connected in BOTH frames -> no T1
    full = [(0, 1), (0, 2), (0, 3), (1, 2), (1, 3), (2, 3)]
    r = check(full, full[1:], 4)
    assert r["cls"].tolist() == [1] and r["common_prev"].tolist() == [2] and r["partner"][0] == NONE


def test_nothing_changes_nothing_is_a_couple():
    e = [(0, 1), (1, 2), (2, 3)]
    assert oracle.t1(pack(e), pack(e), 5)["couples"].size == 0
    assert oracle.t1(pack([]), pack([]), 3)["couples"].size == 0


def test_random_graphs_against_python_sets():
    rng = np.random.default_rng(11)
    for n in (3, 6, 15, 30):
        allp = [(i, j) for i in range(n) for j in range(i + 1, n)]
        for _ in range(8):
            a = [p for p in allp if rng.random() < 0.35]
            b = sorted(set([p for p in a if rng.random() < 0.85] + [p for p in allp if rng.random() < 0.05]))
            r = check(a, b, n)
            # breaking / arising couples are exactly the destroyed / created links (both end points of a
            # changed link are active by definition)
            assert sorted(int(c) for c, s in zip(r["couples"], r["cls"]) if s == 1) == sorted(key(*p) for p in set(a) - set(b))
            assert sorted(int(c) for c, s in zip(r["couples"], r["cls"]) if s == 2) == sorted(key(*p) for p in set(b) - set(a))
    # labels >= n are ignored, as in O7
    r = check([(0, 1), (1, 2), (0, 2), (1, 5)], [(0, 1), (1, 2), (2, 6)], 3)
    assert r["couples"].tolist() == [key(0, 2)]


def test_rhombus_construction_golden():
    g = read_golden("rhombus_flip.txt")
    L = g["L"][0]
    lists = []
    for h in (g["h_prev"][0], g["h_now"][0]):
        sx, sy = rhombus_sites(L, h)
        lists.append(oracle.edges(oracle.label_brute(L, sx, sy)))
    r = oracle.t1(lists[0], lists[1], g["n_sites"][0])
    c = g["couples"]
    assert r["couples"].tolist() == [key(c[2 * k], c[2 * k + 1]) for k in range(len(c) // 2)]
    assert r["cls"].tolist() == g["couple_class"]
    k = r["couples"].tolist()
    b, a = key(*g["destroyed"]), key(*g["created"])
    assert int(r["partner"][k.index(b)]) == key(*g["breaking_partner"]) == a
    assert int(r["partner"][k.index(a)]) == key(*g["arising_partner"]) == b
    assert r["common_prev"][k.index(b)] == g["breaking_common_prev"][0]
    assert r["common_now"][k.index(a)] == g["arising_common_now"][0]
    assert (r["common_prev"][r["cls"] == 0] == 2).all() and (r["common_now"][r["cls"] == 0] == 2).all()


# ------------------------------------------------------------------ O10: bulk / boundary vertices of an event
def brute_vertices(prev_pairs, now_pairs, n):
    def rows(ps):
        r = [set() for _ in range(n)]
        for i, j in ps:
            if i < n and j < n:
                r[i].add(j); r[j].add(i)
        return r
    R = [rows(prev_pairs), rows(now_pairs)]
    act = [R[0][v] != R[1][v] for v in range(n)]
    bnd = [[int(any(len(r[v] & r[u]) == 1 for u in r[v])) for v in range(n)] for r in R]
    vc = []
    for v in range(n):
        c = 0
        if act[v]:
            for t, r in enumerate(R):
                if sum(act[u] for u in r[v]) >= 3:
                    c |= 1 << (2 * t)
                if any(act[u] and bnd[t][u] for u in r[v]):
                    c |= 2 << (2 * t)
        vc.append(c)
    return bnd[0], bnd[1], vc


def check_vertices(prev_pairs, now_pairs, n):
    r = oracle.event_vertices(pack(prev_pairs), pack(now_pairs), n)
    bp, bn, vc = brute_vertices(prev_pairs, now_pairs, n)
    assert r["boundary_prev"].tolist() == bp and r["boundary_now"].tolist() == bn and r["vclass"].tolist() == vc
    return r


def test_event_vertices_bulk_t1_and_boundary_event():
    # Fig. 8 top: the T1 of the rhombus 0-1-2-3 inside closed triangles.  In D_P the end points of the breaking
    # link (1, 3) see three active points, in D_N those of the arising link (0, 2) do: bulk events, no boundary
    common = [(0, 1), (1, 2), (2, 3), (0, 3), (0, 4), (1, 4), (2, 5), (3, 5), (4, 5)]
    r = check_vertices(common + [(1, 3)], common + [(0, 2)], 6)
    assert [c & 5 for c in r["vclass"].tolist()[:4]] == [4, 1, 4, 1] and r["vclass"].tolist()[4:] == [0, 0]
    # the same flip inside a triangulation of the torus (the rhombus construction): no boundary anywhere, so the
    # four points carry exactly the bulk bit of the triangulation in which they see three active points
    g = read_golden("rhombus_flip.txt")
    lists = []
    for h in (g["h_prev"][0], g["h_now"][0]):
        sx, sy = rhombus_sites(g["L"][0], h)
        lists.append(oracle.edges(oracle.label_brute(g["L"][0], sx, sy)))
    t = oracle.event_vertices(lists[0], lists[1], g["n_sites"][0])
    assert t["boundary_prev"].sum() == 0 and t["boundary_now"].sum() == 0
    assert t["vclass"].tolist()[:4] == [4, 1, 4, 1] and t["vclass"][4:].sum() == 0
    # Fig. 8 bottom: a triangle loses one side.  All three sides are boundary edges (one common neighbour); the
    # two active end points are connected in D_P to an active boundary point (each other): a boundary event
    r = check_vertices([(0, 1), (1, 2), (0, 2)], [(0, 1), (1, 2)], 3)
    assert r["boundary_prev"].tolist() == [1, 1, 1] and r["boundary_now"].tolist() == [0, 0, 0]
    assert r["vclass"].tolist() == [2, 0, 2]
    # the zig-zag strip of triangles: every vertex lies on the boundary; nothing active, no class
    strip = [(0, 1), (0, 2), (1, 2), (1, 3), (2, 3), (2, 4), (3, 4), (3, 5), (4, 5)]
    r = check_vertices(strip, strip, 6)
    assert r["boundary_prev"].tolist() == [1] * 6 and r["vclass"].tolist() == [0] * 6
    # a vertex in both kinds of event at once (Fig. 9): hub 0 of a fan loses two spokes of its rim
    fan = [(0, k) for k in range(1, 7)] + [(k, k + 1) for k in range(1, 6)]
    r = check_vertices(fan, [e for e in fan if e not in ((0, 1), (0, 3))], 7)
    assert r["vclass"][0] & 1 == 0 and r["vclass"][0] & 2                     # D_P: two active neighbours, on the rim


def test_event_vertices_random_graphs_and_torus():
    rng = np.random.default_rng(31)
    for n in (4, 9, 20, 40):
        allp = [(i, j) for i in range(n) for j in range(i + 1, n)]
        for _ in range(6):
            a = [p for p in allp if rng.random() < 0.3]
            b = sorted(set([p for p in a if rng.random() < 0.85] + [p for p in allp if rng.random() < 0.04]))
            check_vertices(a, b, n)
    check_vertices([(0, 1), (1, 2), (0, 2), (1, 5)], [(0, 1), (1, 2), (2, 6)], 3)     # labels >= n are ignored
    # a well-resolved triangulation of the torus has no boundary vertex (every edge has two common neighbours)
    from helpers import hex_sites
    L = 256
    sx, sy = hex_sites(L, 16, 18, 0.8, seed=3)
    e = oracle.edges(oracle.label_brute(L, sx, sy))
    r = oracle.event_vertices(e, e, len(sx))
    assert r["boundary_prev"].sum() == 0 and r["vclass"].sum() == 0
