"""ctypes binding of libvor.so — argument marshalling only.

Every step of the hot path runs inside the CUDA kernels of libvor.so (include/vor.h); this module
turns torch CUDA tensors into raw device pointers and the current torch stream into a cudaStream_t.
There is no CPU fallback: a missing library or a failing call raises.  This package never imports
`oracle/`.
"""
from __future__ import annotations

import ctypes as C
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libvor.so")

VOR_OK, VOR_EINVAL, VOR_ECAPACITY, VOR_ECUDA, VOR_ESTATE, VOR_ELIMIT = 0, -1, -2, -3, -4, -5
_STATUS = {0: "VOR_OK", -1: "VOR_EINVAL", -2: "VOR_ECAPACITY", -3: "VOR_ECUDA", -4: "VOR_ESTATE", -5: "VOR_ELIMIT"}
VOR_DIFF_ROWS_STATIC_MAX_ROWS = 1 << 20      # include/vor.h

# name -> (restype, argtypes); mirrors include/vor.h one to one
_P = C.c_void_p
SIGNATURES = {
    "vor_create": (C.c_int, [C.POINTER(_P), C.c_int32, C.c_int32, C.c_int64]),
    "vor_create_geom": (C.c_int, [C.POINTER(_P), C.c_int32, C.c_int32, C.c_int32, C.c_int32, C.c_int32, C.c_int64]),
    "vor_destroy": (C.c_int, [_P]),
    "vor_last_error": (C.c_char_p, [_P]),
    "vor_sync_status": (C.c_int, [_P, _P]),
    "vor_launch_count": (C.c_int64, [_P]),
    "vor_download": (C.c_int, [_P, _P, _P, C.c_int64, _P]),
    "vor_set_option": (C.c_int, [_P, C.c_char_p, C.c_int64]),
    "vor_stat": (C.c_int64, [_P, C.c_char_p]),
    "vor_profile_begin": (C.c_int, [_P]),
    "vor_profile_end": (C.c_int, [_P, _P, C.c_char_p, C.c_int32, C.POINTER(C.c_float), C.c_int32]),
    "vor_build_cells": (C.c_int, [_P, _P, _P, C.c_int32, _P]),
    "vor_build_cells_dev": (C.c_int, [_P, _P, _P, _P, C.c_int32, C.c_int32, _P]),
    "vor_label": (C.c_int, [_P, _P, _P]),
    "vor_label_rows": (C.c_int, [_P, C.c_int32, C.c_int32, _P, _P]),
    "vor_paint_obstacles": (C.c_int, [_P, _P, C.c_int32, _P, C.c_int32, _P]),
    "vor_edges_image": (C.c_int, [_P, _P, C.c_int32, C.c_int32, C.c_int32, _P, C.c_int64, _P, _P, _P]),
    "vor_event_vertices": (C.c_int, [_P, _P, _P, _P, _P, C.c_int64, C.c_int64, _P, C.c_int32, _P, _P, _P, _P]),
    "vor_merge_lists": (C.c_int, [_P, _P, C.c_int64, _P, C.c_int32, C.c_int32, _P, C.c_int64, _P, _P]),
    "vor_edge_commons": (C.c_int, [_P, _P, _P, C.c_int64, C.c_int32, _P, _P]),
    "field_threshold_ccl_conn": (C.c_int, [_P, _P, C.c_float, C.c_int, C.c_int32, _P, _P]),
    "field_centroids_weighted": (C.c_int, [_P, _P, _P, C.c_int32, _P, _P, _P, _P, _P, _P, C.c_int32, _P, _P]),
    "field_size_histogram": (C.c_int, [_P, _P, _P, C.c_int32, C.c_int32, C.c_int32, _P, _P]),
    "vor_edges": (C.c_int, [_P, _P, _P, C.c_int64, _P, _P]),
    "vor_edges_rows": (C.c_int, [_P, _P, _P, C.c_int64, _P, _P, _P]),
    "vor_diff": (C.c_int, [_P, _P, _P, _P, _P, C.c_int64, C.c_int64, _P, _P, C.c_int32, C.c_int32, _P, _P, C.c_int64, _P, _P, _P]),
    "vor_diff_rows": (C.c_int, [_P, _P, _P, _P, _P, C.c_int32, _P, _P, C.c_int64, _P, _P, _P]),
    "vor_diff_rows_static": (C.c_int, [_P, _P, _P, _P, C.c_int32, _P, _P, C.c_int64, _P, _P, _P]),
    "vor_events": (C.c_int, [_P, _P, _P, _P, _P, C.c_int64, C.c_int64, _P, _P, _P, _P, C.c_int64, C.c_int64, C.c_int32,
                             _P, _P, _P, _P, _P, _P, _P]),
    "vor_t1_events": (C.c_int, [_P, _P, _P, _P, _P, C.c_int64, C.c_int64, _P, _P, _P, _P, C.c_int64, C.c_int64, _P, C.c_int32,
                                _P, _P, _P, _P, _P, C.c_int64, _P, _P]),
    "field_threshold_ccl": (C.c_int, [_P, _P, C.c_float, C.c_int, _P, _P]),
    "field_centroids": (C.c_int, [_P, _P, C.c_int32, _P, _P, _P, _P, _P, _P, C.c_int32, _P, _P]),
    "match_sites": (C.c_int, [_P, _P, _P, _P, _P, _P, _P, C.c_int32, C.c_int32, C.c_int32, _P, _P, _P]),
    "vor_frame_host": (C.c_int, [_P, _P, _P, C.c_int32, _P, _P, C.c_int64, _P, _P]),
    "vor_frame_device": (C.c_int, [_P, _P, _P, C.c_int32, _P]),
    "vor_frame_submit": (C.c_int, [_P, _P, _P, C.c_int32, _P]),
    "vor_frame_collect": (C.c_int, [_P, _P, _P, C.c_int64, _P]),
    "vor_frame_reset": (C.c_int, [_P]),
    "vor_frame_options": (C.c_int, [_P, C.c_int32, C.c_int32, _P, C.c_int32]),
    "vor_frame_results": (C.c_int, [_P, C.POINTER(_P), C.POINTER(_P), C.POINTER(_P), C.POINTER(_P), C.POINTER(_P)]),
    "field_frame_device": (C.c_int, [_P, _P, C.c_float, C.c_int, C.c_int32, C.c_int32, _P]),
    "field_frame_submit": (C.c_int, [_P, _P, C.c_float, C.c_int, C.c_int32, C.c_int32, _P]),
    "field_frame_collect": (C.c_int, [_P, _P, _P, C.c_int64, _P]),
    "field_frame_results": (C.c_int, [_P] + [C.POINTER(_P)] * 14),
}

_lib = None


def load_library() -> C.CDLL:
    """dlopen libvor.so (no GPU needed for this step) and declare every prototype."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(
                f"{LIB_PATH} is missing: build it with `python -m paper_1607_00908_b200.build` "
                "(there is no CPU fallback)")
        lib = C.CDLL(LIB_PATH)
        for name, (res, args) in SIGNATURES.items():
            fn = getattr(lib, name)          # AttributeError if the symbol is not exported
            fn.restype, fn.argtypes = res, args
        _lib = lib
    return _lib


class VorError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__(f"{_STATUS.get(status, status)}: {msg}")
        self.status = status


def _ptr(t, dtype=None):
    if t is None:
        return None
    if not isinstance(t, torch.Tensor) or not t.is_cuda:
        raise TypeError("expected a CUDA tensor")
    if dtype is not None and t.dtype != dtype:
        raise TypeError(f"expected dtype {dtype}, got {t.dtype}")
    if not t.is_contiguous():
        raise ValueError("tensor must be contiguous")
    return C.c_void_p(t.data_ptr())


def _stream():
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


def vor_diff_rows_static(prev, prev_row_ptr, now, now_row_ptr, n_rows, created, destroyed, n_created, n_destroyed):
    """vor_diff_rows without a context and without any device allocation inside the library.

    For programs that cannot let a library call cudaMalloc: the GPU's memory belongs to someone else's pool
    (you only hold the tensors you were given), the memory budget was fixed at start-up, or the call sits on a
    path where an allocation's device-wide synchronisation is unacceptable.  The working memory is a fixed
    4 MiB array inside libvor.so, so n_rows is limited to VOR_DIFF_ROWS_STATIC_MAX_ROWS (2^20); more raises
    VorError(VOR_ELIMIT).  All tensors are the caller's; same result as Vor.vor_diff_rows.  An overflow of
    created / destroyed is NOT latched anywhere: compare the counts with the capacities.  The array is shared
    by all calls on a device - keep them on one stream.  Make the first call on a device before any stream
    capture (it looks up the array's address)."""
    lib = load_library()
    assert min(prev_row_ptr.numel(), now_row_ptr.numel()) >= n_rows + 1
    cap = min(created.numel(), destroyed.numel())
    rc = lib.vor_diff_rows_static(
        _ptr(prev, torch.int64), _ptr(prev_row_ptr, torch.int32), _ptr(now, torch.int64),
        _ptr(now_row_ptr, torch.int32), n_rows, _ptr(created, torch.int64), _ptr(destroyed, torch.int64),
        cap, _ptr(n_created, torch.int64), _ptr(n_destroyed, torch.int64), _stream())
    if rc == VOR_ELIMIT:
        raise VorError(rc, f"vor_diff_rows_static: n_rows = {n_rows} exceeds the built-in maximum "
                           f"VOR_DIFF_ROWS_STATIC_MAX_ROWS = {VOR_DIFF_ROWS_STATIC_MAX_ROWS}; use Vor.vor_diff_rows")
    if rc != VOR_OK:
        raise VorError(rc, "vor_diff_rows_static: null pointer, cap < 0 or n_rows < 1" if rc == VOR_EINVAL
                       else "vor_diff_rows_static: a CUDA call failed")


class Vor:
    """One libvor context on the current CUDA device.  Methods carry the C names."""

    def __init__(self, L: int, max_sites: int, max_raw_keys: int = 0, Ly: int | None = None,
                 periodic: tuple = (1, 1)):
        """L x L periodic lattice (vor_create), or with Ly / periodic given: L x Ly cells, each axis periodic
        (1) or walled (0) (vor_create_geom)."""
        self.lib = load_library()
        if not torch.cuda.is_available():
            raise RuntimeError("libvor needs a CUDA device; there is no CPU fallback")
        torch.cuda.init()
        torch.zeros(1, device="cuda")        # make sure the primary context exists
        h = C.c_void_p()
        if Ly is None and tuple(periodic) == (1, 1):
            rc = self.lib.vor_create(C.byref(h), L, max_sites, max_raw_keys)
        else:
            rc = self.lib.vor_create_geom(C.byref(h), L, L if Ly is None else Ly, int(periodic[0]), int(periodic[1]),
                                          max_sites, max_raw_keys)
        if rc != VOR_OK:
            raise VorError(rc, "vor_create failed")
        self.h = h
        self.L = self.Lx = L
        self.Ly = L if Ly is None else Ly
        self.cells = self.Lx * self.Ly
        self.periodic = (int(periodic[0]), int(periodic[1]))
        self.max_sites = max_sites

    def close(self):
        if getattr(self, "h", None):
            self.lib.vor_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, rc):
        if rc != VOR_OK:
            raise VorError(rc, self.lib.vor_last_error(self.h).decode())

    # ---- plumbing
    def vor_sync_status(self):
        self._check(self.lib.vor_sync_status(self.h, _stream()))

    def vor_download(self, d_ptr: int, h_array):
        """Copy len(h_array) elements from the raw device pointer d_ptr into the HOST numpy array h_array."""
        self._check(self.lib.vor_download(self.h, C.c_void_p(d_ptr), h_array.ctypes.data_as(_P), h_array.nbytes, _stream()))
        return h_array

    def vor_launch_count(self) -> int:
        return int(self.lib.vor_launch_count(self.h))

    def vor_profile_begin(self):
        self._check(self.lib.vor_profile_begin(self.h))

    def vor_profile_end(self):
        """-> list of (kernel name, milliseconds) for every launch since vor_profile_begin()."""
        cap = 256
        names = C.create_string_buffer(64 * cap)
        ms = (C.c_float * cap)()
        n = self.lib.vor_profile_end(self.h, _stream(), names, len(names), ms, cap)
        if n < 0:
            self._check(n)
        return list(zip(names.value.decode().split("\n")[:n], [float(ms[i]) for i in range(n)]))

    def vor_stat(self, name: str) -> int:
        v = int(self.lib.vor_stat(self.h, name.encode()))
        if v < 0:
            self._check(v)
        return v

    def vor_set_option(self, name: str, value: int):
        self._check(self.lib.vor_set_option(self.h, name.encode(), int(value)))

    # ---- site path
    def vor_build_cells(self, sx, sy):
        assert sx.shape == sy.shape and sx.dim() == 1
        self._check(self.lib.vor_build_cells(self.h, _ptr(sx, torch.int32), _ptr(sy, torch.int32),
                                             sx.numel(), _stream()))

    def vor_build_cells_dev(self, sx, sy, n_sites, n_hint=0):
        """n_sites: int32[1] device scalar; sx/sy sized to the capacity."""
        cap = min(sx.numel(), sy.numel())
        self._check(self.lib.vor_build_cells_dev(self.h, _ptr(sx, torch.int32), _ptr(sy, torch.int32),
                                                 _ptr(n_sites, torch.int32), cap, n_hint, _stream()))

    def vor_label(self, labels):
        assert labels.numel() == self.cells
        self._check(self.lib.vor_label(self.h, _ptr(labels, torch.int32), _stream()))

    def vor_label_rows(self, y0: int, n_rows: int, labels):
        assert labels.numel() == n_rows * self.Lx
        self._check(self.lib.vor_label_rows(self.h, y0, n_rows, _ptr(labels, torch.int32), _stream()))

    def vor_paint_obstacles(self, mask, colour: int, labels):
        """mask: uint8 tensor, labels: int32 tensor of the same size (whole rows of Lx cells)."""
        assert mask.numel() == labels.numel() and labels.numel() % self.Lx == 0
        self._check(self.lib.vor_paint_obstacles(self.h, _ptr(mask, torch.uint8), colour, _ptr(labels, torch.int32),
                                                 labels.numel() // self.Lx, _stream()))

    def vor_edges_image(self, labels, wrap_y: bool, exclude: int, edges, n_edges, row_ptr=None):
        """labels: whole rows of Lx cells (the domain or a strip); exclude: obstacle colour or -1."""
        assert labels.numel() % self.Lx == 0 and n_edges.numel() >= 1
        self._check(self.lib.vor_edges_image(self.h, _ptr(labels, torch.int32), labels.numel() // self.Lx,
                                             1 if wrap_y else 0, exclude, _ptr(edges, torch.int64), edges.numel(),
                                             _ptr(n_edges, torch.int64), _ptr(row_ptr, torch.int32), _stream()))

    def vor_event_vertices(self, prev, n_prev, now, n_now, trigger, boundary_prev, boundary_now, vclass):
        n_labels = min(t.numel() for t in (trigger, boundary_prev, boundary_now, vclass))
        i64, i32 = torch.int64, torch.int32
        self._check(self.lib.vor_event_vertices(
            self.h, _ptr(prev, i64), _ptr(n_prev, i64), _ptr(now, i64), _ptr(n_now, i64), prev.numel(), now.numel(),
            _ptr(trigger, i32), n_labels, _ptr(boundary_prev, i32), _ptr(boundary_now, i32), _ptr(vclass, i32), _stream()))

    def vor_merge_lists(self, lists, counts, n_labels: int, out, n_out):
        """lists: int64[n_lists, stride] (row l = list l), counts: int64[n_lists] device."""
        assert lists.dim() == 2 and counts.numel() == lists.shape[0]
        self._check(self.lib.vor_merge_lists(self.h, _ptr(lists, torch.int64), lists.shape[1], _ptr(counts, torch.int64),
                                             lists.shape[0], n_labels, _ptr(out, torch.int64), out.numel(),
                                             _ptr(n_out, torch.int64), _stream()))

    def vor_edge_commons(self, edges, n_edges, n_labels: int, commons):
        assert commons.numel() >= edges.numel()
        self._check(self.lib.vor_edge_commons(self.h, _ptr(edges, torch.int64), _ptr(n_edges, torch.int64),
                                              edges.numel(), n_labels, _ptr(commons, torch.int32), _stream()))

    def vor_edges(self, labels, edges, n_edges):
        """edges: int64/uint64 tensor viewed as packed keys; n_edges: int64[1] device scalar."""
        assert labels.numel() == self.cells and n_edges.numel() >= 1
        self._check(self.lib.vor_edges(self.h, _ptr(labels, torch.int32), _ptr(edges, torch.int64),
                                       edges.numel(), _ptr(n_edges, torch.int64), _stream()))

    def vor_edges_rows(self, labels, edges, n_edges, row_ptr):
        """As vor_edges, plus row_ptr: int32 tensor (viewed as uint32) of n_rows + 1 row offsets."""
        assert labels.numel() == self.cells and n_edges.numel() >= 1
        self._check(self.lib.vor_edges_rows(self.h, _ptr(labels, torch.int32), _ptr(edges, torch.int64),
                                            edges.numel(), _ptr(n_edges, torch.int64),
                                            _ptr(row_ptr, torch.int32), _stream()))

    def vor_diff_rows(self, prev, prev_row_ptr, now, now_row_ptr, n_rows, created, destroyed, n_created,
                      n_destroyed):
        assert min(prev_row_ptr.numel(), now_row_ptr.numel()) >= n_rows + 1
        cap = min(created.numel(), destroyed.numel())
        self._check(self.lib.vor_diff_rows(
            self.h, _ptr(prev, torch.int64), _ptr(prev_row_ptr, torch.int32), _ptr(now, torch.int64),
            _ptr(now_row_ptr, torch.int32), n_rows, _ptr(created, torch.int64), _ptr(destroyed, torch.int64),
            cap, _ptr(n_created, torch.int64), _ptr(n_destroyed, torch.int64), _stream()))

    def vor_diff(self, prev, n_prev, now, n_now, created, destroyed, n_created, n_destroyed,
                 p2n=None, n2p=None, n_prev_labels=0, n_now_labels=0):
        cap = min(created.numel(), destroyed.numel())
        self._check(self.lib.vor_diff(
            self.h, _ptr(prev, torch.int64), _ptr(n_prev, torch.int64), _ptr(now, torch.int64),
            _ptr(n_now, torch.int64), prev.numel(), now.numel(),
            _ptr(p2n, torch.int32), _ptr(n2p, torch.int32),
            n_prev_labels, n_now_labels, _ptr(created, torch.int64), _ptr(destroyed, torch.int64), cap,
            _ptr(n_created, torch.int64), _ptr(n_destroyed, torch.int64), _stream()))

    def vor_events(self, prev, n_prev, now, n_now, created, n_created, destroyed, n_destroyed,
                   trigger, events_indices, events_number, global_trigger, count_prev, count_now):
        n_labels = min(t.numel() for t in (trigger, events_indices, count_prev, count_now))
        i64, i32 = torch.int64, torch.int32
        self._check(self.lib.vor_events(
            self.h, _ptr(prev, i64), _ptr(n_prev, i64), _ptr(now, i64), _ptr(n_now, i64),
            prev.numel(), now.numel(),
            _ptr(created, i64), _ptr(n_created, i64), _ptr(destroyed, i64), _ptr(n_destroyed, i64),
            created.numel(), destroyed.numel(), n_labels,
            _ptr(trigger, i32), _ptr(events_indices, i32), _ptr(events_number, i32), _ptr(global_trigger, i32),
            _ptr(count_prev, i32), _ptr(count_now, i32), _stream()))

    def vor_t1_events(self, prev, n_prev, now, n_now, created, n_created, destroyed, n_destroyed, trigger,
                      couples, cls, common_prev, common_now, partner, n_couples):
        cap = min(t.numel() for t in (couples, cls, common_prev, common_now, partner))
        i64, i32 = torch.int64, torch.int32
        self._check(self.lib.vor_t1_events(
            self.h, _ptr(prev, i64), _ptr(n_prev, i64), _ptr(now, i64), _ptr(n_now, i64),
            prev.numel(), now.numel(),
            _ptr(created, i64), _ptr(n_created, i64), _ptr(destroyed, i64), _ptr(n_destroyed, i64),
            created.numel(), destroyed.numel(), _ptr(trigger, i32), trigger.numel(),
            _ptr(couples, i64), _ptr(cls, i32), _ptr(common_prev, i32), _ptr(common_now, i32),
            _ptr(partner, i64), cap, _ptr(n_couples, i64), _stream()))

    # ---- field path
    def field_threshold_ccl(self, field, thr: float, above: bool, ccl):
        assert field.numel() == self.cells == ccl.numel()
        self._check(self.lib.field_threshold_ccl(self.h, _ptr(field, torch.float32), C.c_float(thr),
                                                 1 if above else 0, _ptr(ccl, torch.int32), _stream()))

    def field_threshold_ccl_conn(self, field, thr: float, above: bool, connectivity: int, ccl):
        assert field.numel() == self.cells == ccl.numel()
        self._check(self.lib.field_threshold_ccl_conn(self.h, _ptr(field, torch.float32), C.c_float(thr),
                                                      1 if above else 0, connectivity, _ptr(ccl, torch.int32), _stream()))

    def field_centroids_weighted(self, ccl, field, min_size: int, cx, cy, sx, sy, size, root, n_comp):
        cap = min(t.numel() for t in (cx, cy, sx, sy, size, root))
        assert field is None or field.numel() == self.cells
        self._check(self.lib.field_centroids_weighted(
            self.h, _ptr(ccl, torch.int32), _ptr(field, torch.float32), min_size, _ptr(cx, torch.float64),
            _ptr(cy, torch.float64), _ptr(sx, torch.int32), _ptr(sy, torch.int32), _ptr(size, torch.int32),
            _ptr(root, torch.int32), cap, _ptr(n_comp, torch.int32), _stream()))

    def field_size_histogram(self, size, n_comp, bin_width: int, hist):
        self._check(self.lib.field_size_histogram(self.h, _ptr(size, torch.int32), _ptr(n_comp, torch.int32),
                                                  size.numel(), bin_width, hist.numel(), _ptr(hist, torch.int64), _stream()))

    def field_centroids(self, ccl, min_size: int, cx, cy, sx, sy, size, root, n_comp):
        cap = min(t.numel() for t in (cx, cy, sx, sy, size, root))
        self._check(self.lib.field_centroids(
            self.h, _ptr(ccl, torch.int32), min_size, _ptr(cx, torch.float64), _ptr(cy, torch.float64),
            _ptr(sx, torch.int32), _ptr(sy, torch.int32), _ptr(size, torch.int32), _ptr(root, torch.int32),
            cap, _ptr(n_comp, torch.int32), _stream()))

    def match_sites(self, px, py, n_prev, nx, ny, n_now, radius_fp: int, p2n, n2p):
        cap_prev = min(px.numel(), py.numel(), p2n.numel())
        cap_now = min(nx.numel(), ny.numel(), n2p.numel())
        self._check(self.lib.match_sites(
            self.h, _ptr(px, torch.int32), _ptr(py, torch.int32), _ptr(n_prev, torch.int32),
            _ptr(nx, torch.int32), _ptr(ny, torch.int32), _ptr(n_now, torch.int32),
            cap_prev, cap_now, radius_fp, _ptr(p2n, torch.int32), _ptr(n2p, torch.int32), _stream()))

    # ---- frame pipeline
    def vor_frame_reset(self):
        self._check(self.lib.vor_frame_reset(self.h))

    def vor_frame_options(self, connectivity: int = 4, weighted: bool = False, obstacles=None, obstacle_colour: int = -1):
        """obstacles: uint8 CUDA tensor of Lx*Ly entries (keep it alive) or None."""
        self._obstacles = obstacles
        self._check(self.lib.vor_frame_options(self.h, connectivity, 1 if weighted else 0, _ptr(obstacles, torch.uint8),
                                               obstacle_colour))

    def vor_frame_device(self, sx, sy):
        self._check(self.lib.vor_frame_device(self.h, _ptr(sx, torch.int32), _ptr(sy, torch.int32),
                                              sx.numel(), _stream()))

    def vor_frame_host(self, h_sx, h_sy, h_created, h_destroyed, h_counts):
        """All arguments are HOST numpy arrays (int32 sites, uint64 lists, int64[3] counts)."""
        cap = min(len(h_created), len(h_destroyed))
        self._check(self.lib.vor_frame_host(
            self.h, h_sx.ctypes.data_as(_P), h_sy.ctypes.data_as(_P), len(h_sx),
            h_created.ctypes.data_as(_P), h_destroyed.ctypes.data_as(_P), cap,
            h_counts.ctypes.data_as(_P), _stream()))

    def vor_frame_submit(self, h_sx, h_sy):
        """Enqueue one frame (HOST numpy int32 arrays; keep them alive and unchanged until collected)."""
        self._check(self.lib.vor_frame_submit(self.h, h_sx.ctypes.data_as(_P), h_sy.ctypes.data_as(_P),
                                              len(h_sx), _stream()))

    def vor_frame_collect(self, h_created, h_destroyed, h_counts):
        cap = min(len(h_created), len(h_destroyed))
        self._check(self.lib.vor_frame_collect(self.h, h_created.ctypes.data_as(_P),
                                               h_destroyed.ctypes.data_as(_P), cap, h_counts.ctypes.data_as(_P)))

    def vor_frame_results(self):
        """Raw device pointers (ints) of the context-owned results: labels, edges, created,
        destroyed, counts."""
        ps = [C.c_void_p() for _ in range(5)]
        self._check(self.lib.vor_frame_results(self.h, *[C.byref(p) for p in ps]))
        return tuple(p.value for p in ps)

    # ---- field-driven frames
    def field_frame_device(self, field, thr: float, above: bool, min_size: int, radius_fp: int):
        assert field.numel() == self.cells
        self._check(self.lib.field_frame_device(self.h, _ptr(field, torch.float32), C.c_float(thr),
                                                1 if above else 0, min_size, radius_fp, _stream()))

    def field_frame_submit(self, h_field, thr: float, above: bool, min_size: int, radius_fp: int):
        """h_field: HOST float32 numpy array (L*L, C order); keep it alive and unchanged until collected."""
        assert h_field.size == self.cells and h_field.dtype.name == "float32" and h_field.flags.c_contiguous
        self._check(self.lib.field_frame_submit(self.h, h_field.ctypes.data_as(_P), C.c_float(thr),
                                                1 if above else 0, min_size, radius_fp, _stream()))

    def field_frame_collect(self, h_created, h_destroyed, h_counts):
        """h_counts: int64[4] = bubbles, edges, created, destroyed."""
        cap = min(len(h_created), len(h_destroyed))
        self._check(self.lib.field_frame_collect(self.h, h_created.ctypes.data_as(_P),
                                                 h_destroyed.ctypes.data_as(_P), cap, h_counts.ctypes.data_as(_P)))

    FIELD_RESULTS = ("ccl", "labels", "cx", "cy", "sx", "sy", "size", "root", "p2n", "n2p", "edges", "created",
                     "destroyed", "counts")

    def field_frame_results(self):
        """dict of raw device pointers (ints), keys FIELD_RESULTS."""
        ps = [C.c_void_p() for _ in self.FIELD_RESULTS]
        self._check(self.lib.field_frame_results(self.h, *[C.byref(p) for p in ps]))
        return {k: p.value for k, p in zip(self.FIELD_RESULTS, ps)}
