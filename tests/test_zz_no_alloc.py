"""vor_diff_rows_static: the row-by-row edge diff for callers that are not allowed to allocate GPU memory.

Some programs that embed this library cannot let it call cudaMalloc: the GPU's memory is owned by the host
application's pool and a plug-in only ever sees the buffers it was handed, or the process fixed its memory
budget at start-up, or the call sits on a latency path where an allocation (which synchronises the whole
device) is not acceptable.  For them include/vor.h has one context-free entry point whose working memory is a
fixed 4 MiB array inside libvor.so (at most 2^20 rows).  These tests check that it returns exactly what the
ordinary path (Vor.vor_diff_rows, which allocates through its context) returns - integer keys, so the
tolerance is bit-exact as everywhere in tests/test_gpu_parity.py - on calls issued back to back, whose second
call finds the first call's leftovers in the shared array.

The file name sorts last on purpose: `pytest -x` stops at the first failure, and a failure here must not hide
the parity tests.  It passes alone in a fresh process (the first call does the per-device set-up) and after
the rest of the suite.
"""
import ctypes as C

import numpy as np
import pytest

import oracle
from paper_1607_00908_b200 import workloads as W

torch = pytest.importorskip("torch")


def row_offsets(keys, n_rows):
    """row_ptr by definition: offset of the first key whose smaller label is >= a."""
    return np.searchsorted(keys >> np.uint64(32), np.arange(n_rows + 1, dtype=np.uint64), side="left")


def random_graph(rng, n, m, hub):
    i = rng.integers(0, n, m); j = rng.integers(0, n, m)
    if hub and n > 100:                                # vertex 3 touches about half of the others: a long row
        i = np.concatenate([i, np.full(n // 2, 3)]); j = np.concatenate([j, rng.integers(0, n, n // 2)])
    keep = i != j
    lo, hi = np.minimum(i, j)[keep].astype(np.uint64), np.maximum(i, j)[keep].astype(np.uint64)
    return np.unique((lo << np.uint64(32)) | hi)


class Case:
    """Device copies of two key lists with their row offsets, and output buffers with guard regions."""

    def __init__(self, prev, now, n_rows, cap=None):
        dev = lambda a, t: torch.from_numpy(np.ascontiguousarray(a).view(t)).cuda()
        keys = lambda a: dev(a, np.int64) if len(a) else torch.empty(1, dtype=torch.int64, device="cuda")
        ptr = lambda a: dev(row_offsets(a, n_rows).astype(np.uint32), np.int32)
        self.prev, self.now, self.n_rows = prev, now, n_rows
        self.d_prev, self.d_now, self.p_prev, self.p_now = keys(prev), keys(now), ptr(prev), ptr(now)
        self.cap = max(1, len(prev) + len(now)) if cap is None else cap
        new = lambda: torch.full((self.cap + 64,), -7, dtype=torch.int64, device="cuda")
        self.out = {k: (new(), new(), torch.zeros(1, dtype=torch.int64, device="cuda"),
                        torch.zeros(1, dtype=torch.int64, device="cuda")) for k in ("ctx", "static")}

    def args(self, which):
        c, d, nc, nd = self.out[which]
        return (self.d_prev, self.p_prev, self.d_now, self.p_now, self.n_rows, c[:self.cap], d[:self.cap], nc, nd)

    def result(self, which):
        c, d, nc, nd = self.out[which]
        assert (c[self.cap:] == -7).all() and (d[self.cap:] == -7).all(), "write past the capacity"
        nc, nd = int(nc.item()), int(nd.item())
        u = lambda t, n: t[:min(n, self.cap)].cpu().numpy().view(np.uint64)
        return nc, nd, u(c, nc), u(d, nd)


def same(a, b):
    return a[0] == b[0] and a[1] == b[1] and np.array_equal(a[2], b[2]) and np.array_equal(a[3], b[3])


@pytest.mark.gpu
def test_static_entry_point_equals_the_context_path_on_calls_in_a_row():
    from paper_1607_00908_b200.binding import Vor, vor_diff_rows_static
    rng = np.random.default_rng(20261106)
    # two snapshots of a scaled config 5 (961 sites, rows of ~3 keys), then random graphs: hubs (rows longer than
    # the in-register path), several blocks with a ragged tail, a large one, and a small one LAST so that it
    # runs on top of the large call's leftovers in the shared array
    w = W.scaled(5, 512)
    labs = [oracle.label_cells(w.L, sx, sy, 16) for sx, sy in w.frames(2)]
    e0, e1 = oracle.edges(labs[0]), oracle.edges(labs[1])
    cases = [Case(e0, e1, w.n_sites), Case(e1, e0, w.n_sites), Case(np.empty(0, np.uint64), e1, w.n_sites)]
    for n, m in ((5, 6), (3000, 9000), (1300, 40000), (700001, 2000000), (513, 900)):
        a = random_graph(rng, n, m, True)
        b = np.unique(np.concatenate([a[rng.random(len(a)) < 0.9], random_graph(rng, n, max(1, m // 10), False)]))
        cases.append(Case(a, b, n))
    v = Vor(64, 64)
    for c in cases:                                    # the existing path: one call and one check per case
        v.vor_diff_rows(*c.args("ctx"))
        v.vor_sync_status()
    # the new entry point: ALL calls enqueued back to back on one stream, no synchronisation in between
    vor_diff_rows_static(*cases[0].args("static"))     # (the first call on the device also does the set-up)
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    for c in cases:
        vor_diff_rows_static(*c.args("static"))
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free_before, "the calls changed the amount of free device memory"
    for k, c in enumerate(cases):
        got, ref = c.result("static"), c.result("ctx")
        assert same(got, ref), f"case {k}: static entry point differs from vor_diff_rows"
        rc, rd = oracle.diff(c.prev, c.now)
        assert got[0] == len(rc) and got[1] == len(rd) and np.array_equal(got[2], rc) and np.array_equal(got[3], rd)
    # twice the same call in a row gives twice the same answer
    c = cases[4]
    first = c.result("static")
    vor_diff_rows_static(*c.args("static")); vor_diff_rows_static(*c.args("static"))
    torch.cuda.synchronize()
    assert same(c.result("static"), first)
    v.close()


@pytest.mark.gpu
def test_static_entry_point_reports_required_counts_when_the_outputs_are_too_small():
    from paper_1607_00908_b200.binding import vor_diff_rows_static
    rng = np.random.default_rng(7)
    a, b = random_graph(rng, 2000, 6000, True), random_graph(rng, 2000, 6000, False)
    rc, rd = oracle.diff(a, b)
    c = Case(a, b, 2000, cap=100)
    vor_diff_rows_static(*c.args("static"))
    torch.cuda.synchronize()
    nc, nd, gc, gd = c.result("static")                # also checks the guard regions behind cap
    assert (nc, nd) == (len(rc), len(rd)) and min(nc, nd) > 100
    assert np.array_equal(gc, rc[:100]) and np.array_equal(gd, rd[:100])


def test_static_entry_point_rejects_sizes_beyond_its_array_without_a_device():
    """The size check comes before any CUDA call, so it needs no GPU: dummy non-null pointers are never read."""
    from paper_1607_00908_b200 import binding
    lib = binding.load_library()
    p = C.c_void_p(256)
    lim = binding.VOR_DIFF_ROWS_STATIC_MAX_ROWS
    assert lim == 1 << 20
    assert lib.vor_diff_rows_static(p, p, p, p, lim + 1, p, p, 10, p, p, None) == binding.VOR_ELIMIT
    assert lib.vor_diff_rows_static(p, p, p, p, 2 ** 31 - 1, p, p, 10, p, p, None) == binding.VOR_ELIMIT
    assert lib.vor_diff_rows_static(None, p, p, p, 10, p, p, 10, p, p, None) == binding.VOR_EINVAL
    assert lib.vor_diff_rows_static(p, p, p, p, 0, p, p, 10, p, p, None) == binding.VOR_EINVAL
    assert lib.vor_diff_rows_static(p, p, p, p, 10, p, p, -1, p, p, None) == binding.VOR_EINVAL
