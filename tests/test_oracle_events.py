"""Pins for oracle O7 (trigger, eventsIndices, eventsCount)."""
import numpy as np

import oracle
from helpers import pack, pairs, read_golden, rhombus_sites


def brute(prev_pairs, now_pairs, n):
    """Python-set brute force on tiny inputs: rows as sets, straight from the definitions."""
    def rows(ps):
        r = [set() for _ in range(n)]
        for i, j in ps:
            r[i].add(j); r[j].add(i)
        return r
    rp, rn = rows(prev_pairs), rows(now_pairs)
    trig = [int(rp[i] != rn[i]) for i in range(n)]
    cp = [sum(trig[j] for j in rp[i]) if trig[i] else 0 for i in range(n)]
    cn = [sum(trig[j] for j in rn[i]) if trig[i] else 0 for i in range(n)]
    return trig, [i for i in range(n) if trig[i]], cp, cn


def check(prev_pairs, now_pairs, n):
    ev = oracle.events(pack(prev_pairs), pack(now_pairs), n)
    trig, idx, cp, cn = brute(prev_pairs, now_pairs, n)
    assert ev["trigger"].tolist() == trig and ev["events_indices"].tolist() == idx
    assert ev["count_prev"].tolist() == cp and ev["count_now"].tolist() == cn
    assert ev["global_trigger"] == int(any(trig))
    return ev


def test_t1_hand_graph_matches_paper_statement():
    # rhombus 0-1-2-3 with diagonal 1-3 flipping to 0-2, plus a bystander ring 4,5
    common = [(0, 1), (1, 2), (2, 3), (0, 3), (0, 4), (1, 4), (2, 5), (3, 5), (4, 5)]
    ev = check(common + [(1, 3)], common + [(0, 2)], 6)
    assert ev["events_indices"].tolist() == [0, 1, 2, 3]
    assert ev["count_prev"].tolist() == [2, 3, 2, 3, 0, 0]          # >= 3 at the breaking link
    assert ev["count_now"].tolist() == [3, 2, 3, 2, 0, 0]


def test_boundary_type_event_one_breaking_link():
    # PAPER.md Fig. 8 bottom: only a breaking link; the two endpoints trigger, coordination not conserved
    ev = check([(0, 1), (1, 2), (0, 2)], [(0, 1), (1, 2)], 3)
    assert ev["trigger"].tolist() == [1, 0, 1]
    assert ev["count_prev"].tolist() == [1, 0, 1] and ev["count_now"].tolist() == [0, 0, 0]


def test_identical_and_empty():
    e = [(0, 1), (1, 2), (2, 3)]
    ev = check(e, e, 5)
    assert ev["global_trigger"] == 0 and ev["events_indices"].size == 0
    check([], [], 3)
    check([], [(0, 2)], 3)


def test_random_lists_against_brute_force_and_invariants():
    rng = np.random.default_rng(7)
    for n in (2, 5, 17, 40):
        allp = [(i, j) for i in range(n) for j in range(i + 1, n)]
        for _ in range(6):
            a = [p for p in allp if rng.random() < 0.3]
            b = [p for p in a if rng.random() < 0.8] + [p for p in allp if rng.random() < 0.05]
            b = sorted(set(b))
            ev = check(a, b, n)
            sym = set(a) ^ set(b)
            ends = sorted({v for p in sym for v in p})
            assert ev["events_indices"].tolist() == ends                      # endpoints of the changed links
            t = ev["trigger"]
            assert ev["count_prev"].sum() == 2 * sum(1 for i, j in a if t[i] and t[j])
            assert ev["count_now"].sum() == 2 * sum(1 for i, j in b if t[i] and t[j])


def test_rhombus_construction_golden():
    g = read_golden("rhombus_flip.txt")
    L = g["L"][0]
    lists = []
    for h in (g["h_prev"][0], g["h_now"][0]):
        sx, sy = rhombus_sites(L, h)
        lists.append(oracle.edges(oracle.label_brute(L, sx, sy)))
    ev = oracle.events(lists[0], lists[1], g["n_sites"][0])
    assert ev["events_indices"].tolist() == g["events_indices"]
    assert ev["count_prev"][:4].tolist() == g["count_prev"] and ev["count_now"][:4].tolist() == g["count_now"]
    assert ev["global_trigger"] == 1 and ev["trigger"].sum() == 4


def test_keys_with_a_label_beyond_n_are_ignored():
    """vor.h: "keys with a label >= n_labels are ignored" - pinned against the python-set brute force on
    the lists with those keys removed by hand."""
    prev = [(0, 1), (1, 2), (0, 2), (1, 5), (2, 7), (5, 7)]
    now = [(0, 1), (1, 2), (2, 6), (0, 5), (5, 7)]
    n = 4
    ev = oracle.events(pack(prev), pack(now), n)
    trig, idx, cp, cn = brute([p for p in prev if max(p) < n], [p for p in now if max(p) < n], n)
    assert trig == [1, 0, 1, 0]                    # only (0,2) disappeared among the labels < 4
    assert ev["trigger"].tolist() == trig and ev["events_indices"].tolist() == idx
    assert ev["count_prev"].tolist() == cp == [1, 0, 1, 0] and ev["count_now"].tolist() == cn == [0, 0, 0, 0]
