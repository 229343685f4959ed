"""CPU oracle — TEST INFRASTRUCTURE ONLY (numpy in, numpy out).

Thin ctypes wrapper around oracle/vor_oracle.cpp.  Only tests/,
__graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package; the product path (paper_1607_00908_b200) never does.
See vor_oracle.cpp for the definitions and the passages they follow.
"""
from __future__ import annotations

import ctypes as C

import numpy as np

from . import build as _build

_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build.build())
        _lib.orc_edges.restype = C.c_int64
        _lib.orc_centroids.restype = C.c_int32
        _lib.orc_label_cells.restype = C.c_int
        _lib.orc_label_cells_at.restype = C.c_int
        _lib.orc_num_threads.restype = C.c_int
    return _lib


def _p(a, t):
    return a.ctypes.data_as(C.POINTER(t))


def _i32(a):
    a = np.ascontiguousarray(a, dtype=np.int32)
    return a


def num_threads(threads: int = 0) -> int:
    return int(lib().orc_num_threads(C.c_int(threads)))


def label_brute(L, sx, sy, threads=0):
    sx, sy = _i32(sx), _i32(sy)
    out = np.empty((L, L), dtype=np.int32)
    lib().orc_label_brute(C.c_int32(L), C.c_int32(len(sx)), _p(sx, C.c_int32), _p(sy, C.c_int32),
                          _p(out, C.c_int32), C.c_int(threads))
    return out


def label_brute_at(L, sx, sy, cells, threads=0):
    sx, sy = _i32(sx), _i32(sy)
    cells = np.ascontiguousarray(cells, dtype=np.int64)
    out = np.empty(len(cells), dtype=np.int32)
    lib().orc_label_brute_at(C.c_int32(L), C.c_int32(len(sx)), _p(sx, C.c_int32), _p(sy, C.c_int32),
                             C.c_int64(len(cells)), _p(cells, C.c_int64), _p(out, C.c_int32),
                             C.c_int(threads))
    return out


def label_cells(L, sx, sy, bucket_cells, threads=0):
    sx, sy = _i32(sx), _i32(sy)
    out = np.empty((L, L), dtype=np.int32)
    rc = lib().orc_label_cells(C.c_int32(L), C.c_int32(len(sx)), _p(sx, C.c_int32), _p(sy, C.c_int32),
                               C.c_int32(bucket_cells), _p(out, C.c_int32), C.c_int(threads))
    if rc != 0:
        raise ValueError("bucket_cells must divide L")
    return out


def label_cells_at(L, sx, sy, bucket_cells, cells, threads=0):
    sx, sy = _i32(sx), _i32(sy)
    cells = np.ascontiguousarray(cells, dtype=np.int64)
    out = np.empty(len(cells), dtype=np.int32)
    rc = lib().orc_label_cells_at(C.c_int32(L), C.c_int32(len(sx)), _p(sx, C.c_int32),
                                  _p(sy, C.c_int32), C.c_int32(bucket_cells), C.c_int64(len(cells)),
                                  _p(cells, C.c_int64), _p(out, C.c_int32), C.c_int(threads))
    if rc != 0:
        raise ValueError("bucket_cells must divide L")
    return out


def edges(labels):
    labels = _i32(labels)
    L = labels.shape[0]
    assert labels.shape == (L, L)
    cap = 2 * L * L
    # first call with a modest buffer; the function returns the true count
    buf = np.empty(min(cap, max(1024, L * L // 8)), dtype=np.uint64)
    m = lib().orc_edges(C.c_int32(L), _p(labels, C.c_int32), _p(buf, C.c_uint64), C.c_int64(len(buf)))
    if m > len(buf):
        buf = np.empty(m, dtype=np.uint64)
        m = lib().orc_edges(C.c_int32(L), _p(labels, C.c_int32), _p(buf, C.c_uint64), C.c_int64(len(buf)))
    return buf[:m].copy()


def diff(prev, now, p2n=None, n2p=None):
    prev = np.ascontiguousarray(prev, dtype=np.uint64)
    now = np.ascontiguousarray(now, dtype=np.uint64)
    cap = max(1, len(prev) + len(now))
    created = np.empty(cap, dtype=np.uint64)
    destroyed = np.empty(cap, dtype=np.uint64)
    nc, nd = C.c_int64(0), C.c_int64(0)
    pp = nn = None
    if p2n is not None:
        p2n = _i32(p2n); pp = _p(p2n, C.c_int32)
    if n2p is not None:
        n2p = _i32(n2p); nn = _p(n2p, C.c_int32)
    lib().orc_diff(_p(prev, C.c_uint64), C.c_int64(len(prev)), _p(now, C.c_uint64), C.c_int64(len(now)),
                   pp, nn, _p(created, C.c_uint64), _p(destroyed, C.c_uint64), C.c_int64(cap),
                   C.byref(nc), C.byref(nd))
    return created[:nc.value].copy(), destroyed[:nd.value].copy()


def threshold_ccl(field, thr, above=True):
    field = np.ascontiguousarray(field, dtype=np.float32)
    L = field.shape[0]
    assert field.shape == (L, L)
    out = np.empty((L, L), dtype=np.int32)
    lib().orc_threshold_ccl(C.c_int32(L), _p(field, C.c_float), C.c_float(thr), C.c_int(1 if above else 0),
                            _p(out, C.c_int32))
    return out


def centroids(ccl, min_size):
    ccl = _i32(ccl)
    L = ccl.shape[0]
    cap = max(1, (L * L + 1) // 2)
    cx = np.empty(cap); cy = np.empty(cap)
    sx = np.empty(cap, dtype=np.int32); sy = np.empty(cap, dtype=np.int32)
    size = np.empty(cap, dtype=np.int32); root = np.empty(cap, dtype=np.int32)
    K = lib().orc_centroids(C.c_int32(L), _p(ccl, C.c_int32), C.c_int32(min_size),
                            _p(cx, C.c_double), _p(cy, C.c_double), _p(sx, C.c_int32), _p(sy, C.c_int32),
                            _p(size, C.c_int32), _p(root, C.c_int32), C.c_int32(cap))
    return dict(cx=cx[:K].copy(), cy=cy[:K].copy(), sx=sx[:K].copy(), sy=sy[:K].copy(),
                size=size[:K].copy(), root=root[:K].copy())


def match(L, px, py, nx, ny, radius_fp):
    px, py, nx, ny = _i32(px), _i32(py), _i32(nx), _i32(ny)
    p2n = np.empty(len(px), dtype=np.int32)
    n2p = np.empty(len(nx), dtype=np.int32)
    lib().orc_match(C.c_int32(L), _p(px, C.c_int32), _p(py, C.c_int32), C.c_int32(len(px)),
                    _p(nx, C.c_int32), _p(ny, C.c_int32), C.c_int32(len(nx)), C.c_int32(radius_fp),
                    _p(p2n, C.c_int32), _p(n2p, C.c_int32))
    return p2n, n2p


def events(prev, now, n):
    """O7: trigger[n], events_indices, count_prev[n], count_now[n], global_trigger."""
    prev = np.ascontiguousarray(prev, dtype=np.uint64)
    now = np.ascontiguousarray(now, dtype=np.uint64)
    trig = np.zeros(n, np.int32); idx = np.zeros(max(n, 1), np.int32)
    cp = np.zeros(n, np.int32); cn = np.zeros(n, np.int32)
    m = C.c_int32(0)
    lib().orc_events.restype = C.c_int32
    g = lib().orc_events(_p(prev, C.c_uint64), C.c_int64(len(prev)), _p(now, C.c_uint64), C.c_int64(len(now)),
                         C.c_int32(n), _p(trig, C.c_int32), _p(idx, C.c_int32), C.byref(m),
                         _p(cp, C.c_int32), _p(cn, C.c_int32))
    return dict(trigger=trig, events_indices=idx[:m.value].copy(), count_prev=cp, count_now=cn,
                global_trigger=int(g))


def t1(prev, now, n):
    """O8: couples of active vertices, their class, common-neighbour counts and T1 partner."""
    prev = np.ascontiguousarray(prev, dtype=np.uint64)
    now = np.ascontiguousarray(now, dtype=np.uint64)
    cap = max(1, len(prev) + len(now))
    couples = np.empty(cap, np.uint64); partner = np.empty(cap, np.uint64)
    cls = np.empty(cap, np.int32); cp = np.empty(cap, np.int32); cn = np.empty(cap, np.int32)
    lib().orc_t1.restype = C.c_int64
    m = lib().orc_t1(_p(prev, C.c_uint64), C.c_int64(len(prev)), _p(now, C.c_uint64), C.c_int64(len(now)),
                     C.c_int32(n), _p(couples, C.c_uint64), _p(cls, C.c_int32), _p(cp, C.c_int32),
                     _p(cn, C.c_int32), _p(partner, C.c_uint64), C.c_int64(cap))
    assert m <= cap
    return dict(couples=couples[:m].copy(), cls=cls[:m].copy(), common_prev=cp[:m].copy(),
                common_now=cn[:m].copy(), partner=partner[:m].copy())


# ---- O9: the same definitions on a rectangular lattice with periodic or walled axes (see vor_oracle.cpp)
def label_brute_g(Lx, Ly, per_x, per_y, sx, sy, threads=0):
    sx, sy = _i32(sx), _i32(sy)
    out = np.empty((Ly, Lx), dtype=np.int32)
    lib().orc_label_brute_g(C.c_int32(Lx), C.c_int32(Ly), C.c_int(per_x), C.c_int(per_y), C.c_int32(len(sx)),
                            _p(sx, C.c_int32), _p(sy, C.c_int32), _p(out, C.c_int32), C.c_int(threads))
    return out


def label_brute_at_g(Lx, Ly, per_x, per_y, sx, sy, cells, threads=0):
    sx, sy = _i32(sx), _i32(sy)
    cells = np.ascontiguousarray(cells, dtype=np.int64)
    out = np.empty(len(cells), dtype=np.int32)
    lib().orc_label_brute_at_g(C.c_int32(Lx), C.c_int32(Ly), C.c_int(per_x), C.c_int(per_y), C.c_int32(len(sx)),
                               _p(sx, C.c_int32), _p(sy, C.c_int32), C.c_int64(len(cells)), _p(cells, C.c_int64),
                               _p(out, C.c_int32), C.c_int(threads))
    return out


def label_cells_g(Lx, Ly, per_x, per_y, sx, sy, bucket_cells, threads=0):
    sx, sy = _i32(sx), _i32(sy)
    out = np.empty((Ly, Lx), dtype=np.int32)
    lib().orc_label_cells_g.restype = C.c_int
    rc = lib().orc_label_cells_g(C.c_int32(Lx), C.c_int32(Ly), C.c_int(per_x), C.c_int(per_y), C.c_int32(len(sx)),
                                 _p(sx, C.c_int32), _p(sy, C.c_int32), C.c_int32(bucket_cells),
                                 _p(out, C.c_int32), C.c_int(threads))
    if rc != 0:
        raise ValueError("bucket_cells must divide Lx and Ly")
    return out


def edges_g(labels, per_x=1, per_y=1, exclude=-1):
    labels = _i32(labels)
    Ly, Lx = labels.shape
    buf = np.empty(2 * Lx * Ly + 1, dtype=np.uint64)
    lib().orc_edges_g.restype = C.c_int64
    m = lib().orc_edges_g(C.c_int32(Lx), C.c_int32(Ly), C.c_int(per_x), C.c_int(per_y), C.c_int32(exclude),
                          _p(labels, C.c_int32), _p(buf, C.c_uint64), C.c_int64(len(buf)))
    return buf[:m].copy()


def apply_obstacles(labels, obstacle_mask, colour):
    """obstacle sites take a fixed large colour (MAXLINK) instead of a bubble's label."""
    return np.where(np.asarray(obstacle_mask) != 0, np.int32(colour), _i32(labels)).astype(np.int32)


def threshold_ccl_g(field, thr, above=True, per_x=1, per_y=1, connectivity=4):
    field = np.ascontiguousarray(field, dtype=np.float32)
    Ly, Lx = field.shape
    out = np.empty((Ly, Lx), dtype=np.int32)
    lib().orc_threshold_ccl_g.restype = C.c_int
    rc = lib().orc_threshold_ccl_g(C.c_int32(Lx), C.c_int32(Ly), C.c_int(per_x), C.c_int(per_y),
                                   _p(field, C.c_float), C.c_float(thr), C.c_int(1 if above else 0),
                                   C.c_int(connectivity), _p(out, C.c_int32))
    if rc != 0:
        raise ValueError("connectivity must be 4 or 8")
    return out


def centroids_g(ccl, min_size, per_x=1, per_y=1, field=None):
    ccl = _i32(ccl)
    Ly, Lx = ccl.shape
    cap = max(1, (Lx * Ly + 1) // 2)
    cx = np.empty(cap); cy = np.empty(cap)
    sx = np.empty(cap, dtype=np.int32); sy = np.empty(cap, dtype=np.int32)
    size = np.empty(cap, dtype=np.int32); root = np.empty(cap, dtype=np.int32)
    fp = None
    if field is not None:
        field = np.ascontiguousarray(field, dtype=np.float32)
        assert field.shape == ccl.shape
        fp = _p(field, C.c_float)
    lib().orc_centroids_g.restype = C.c_int32
    K = lib().orc_centroids_g(C.c_int32(Lx), C.c_int32(Ly), C.c_int(per_x), C.c_int(per_y), _p(ccl, C.c_int32), fp,
                              C.c_int32(min_size), _p(cx, C.c_double), _p(cy, C.c_double), _p(sx, C.c_int32),
                              _p(sy, C.c_int32), _p(size, C.c_int32), _p(root, C.c_int32), C.c_int32(cap))
    return dict(cx=cx[:K].copy(), cy=cy[:K].copy(), sx=sx[:K].copy(), sy=sy[:K].copy(),
                size=size[:K].copy(), root=root[:K].copy())


def match_g(Lx, Ly, per_x, per_y, px, py, nx, ny, radius_fp):
    px, py, nx, ny = _i32(px), _i32(py), _i32(nx), _i32(ny)
    p2n = np.empty(len(px), dtype=np.int32)
    n2p = np.empty(len(nx), dtype=np.int32)
    lib().orc_match_g(C.c_int32(Lx), C.c_int32(Ly), C.c_int(per_x), C.c_int(per_y), _p(px, C.c_int32),
                      _p(py, C.c_int32), C.c_int32(len(px)), _p(nx, C.c_int32), _p(ny, C.c_int32),
                      C.c_int32(len(nx)), C.c_int32(radius_fp), _p(p2n, C.c_int32), _p(n2p, C.c_int32))
    return p2n, n2p


def size_histogram(size, bin_width, n_bins):
    size = _i32(size)
    hist = np.zeros(n_bins, dtype=np.int64)
    lib().orc_size_histogram(_p(size, C.c_int32), C.c_int32(len(size)), C.c_int32(bin_width), C.c_int32(n_bins),
                             _p(hist, C.c_int64))
    return hist


def edge_commons(edges, n):
    edges = np.ascontiguousarray(edges, dtype=np.uint64)
    out = np.empty(len(edges), dtype=np.int32)
    lib().orc_edge_commons(_p(edges, C.c_uint64), C.c_int64(len(edges)), C.c_int32(n), _p(out, C.c_int32))
    return out


def event_vertices(prev, now, n):
    """O10: boundary vertices of both triangulations and the bulk / boundary event class of every active vertex
    (PAPER.md:248-256)."""
    prev = np.ascontiguousarray(prev, dtype=np.uint64)
    now = np.ascontiguousarray(now, dtype=np.uint64)
    bp = np.zeros(n, np.int32); bn = np.zeros(n, np.int32); vc = np.zeros(n, np.int32)
    lib().orc_event_vertices(_p(prev, C.c_uint64), C.c_int64(len(prev)), _p(now, C.c_uint64), C.c_int64(len(now)),
                             C.c_int32(n), _p(bp, C.c_int32), _p(bn, C.c_int32), _p(vc, C.c_int32))
    return dict(boundary_prev=bp, boundary_now=bn, vclass=vc)


def unpack(keys):
    """uint64 packed keys -> (i, j) int64 arrays."""
    keys = np.asarray(keys, dtype=np.uint64)
    return (keys >> np.uint64(32)).astype(np.int64), (keys & np.uint64(0xffffffff)).astype(np.int64)
