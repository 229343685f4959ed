"""Helpers for the -m gpu parity tests: thin wrappers that run one libvor call on numpy inputs."""
import ctypes as C

import numpy as np
import torch

from paper_1607_00908_b200.binding import Vor


def dev(a, dtype=None):
    t = torch.from_numpy(np.ascontiguousarray(a))
    if dtype is not None:
        t = t.to(dtype)
    return t.cuda()


def u64(t, n=None):
    a = t.cpu().numpy().view(np.uint64)
    return a if n is None else a[:n]


def gpu_labels(v: Vor, sx, sy):
    dsx, dsy = dev(sx), dev(sy)
    lab = torch.empty(v.cells, dtype=torch.int32, device="cuda")
    v.vor_build_cells(dsx, dsy)
    v.vor_label(lab)
    v.vor_sync_status()
    return lab.cpu().numpy().reshape(v.Ly, v.Lx)


def gpu_label_rows(v: Vor, y0, n_rows):
    """vor_label_rows on the cell list built last -> (n_rows, Lx) array; guard rows around the strip."""
    buf = torch.full(((n_rows + 2) * v.Lx,), -9, dtype=torch.int32, device="cuda")
    v.vor_label_rows(y0, n_rows, buf[v.Lx:(n_rows + 1) * v.Lx])
    v.vor_sync_status()
    out = buf.cpu().numpy().reshape(n_rows + 2, v.Lx)
    assert (out[0] == -9).all() and (out[-1] == -9).all(), "write outside the strip"
    return out[1:-1].copy()


def gpu_edges_image(v: Vor, labels, wrap_y, exclude=-1, cap=None, n_rows_ptr=None):
    """vor_edges_image on a host image of whole rows -> keys (and row_ptr if n_rows_ptr is given)."""
    cap = cap or max(1024, 8 * v.max_sites)
    d = dev(np.ascontiguousarray(labels, dtype=np.int32).ravel())
    out = torch.empty(cap, dtype=torch.int64, device="cuda")
    n = torch.zeros(1, dtype=torch.int64, device="cuda")
    ptr = None if n_rows_ptr is None else torch.full((n_rows_ptr + 1,), -1, dtype=torch.int32, device="cuda")
    v.vor_edges_image(d, wrap_y, exclude, out, n, ptr)
    v.vor_sync_status()
    keys = u64(out, int(n.item())).copy()
    return keys if ptr is None else (keys, ptr.cpu().numpy().view(np.uint32).astype(np.int64))


def gpu_edge_commons(v: Vor, edges, n_labels):
    e = dev(np.asarray(edges, np.uint64).view(np.int64)) if len(edges) else torch.empty(1, dtype=torch.int64, device="cuda")
    n = torch.tensor([len(edges)], dtype=torch.int64, device="cuda")
    c = torch.full((max(len(edges), 1) + 2,), -9, dtype=torch.int32, device="cuda")
    v.vor_edge_commons(e[:max(len(edges), 1)], n, n_labels, c[:max(len(edges), 1)])
    v.vor_sync_status()
    assert (c[max(len(edges), 1):] == -9).all()
    return c[:len(edges)].cpu().numpy()


def gpu_edges(v: Vor, labels, cap=None):
    L = v.L
    cap = cap or max(1024, 8 * v.max_sites)
    d = dev(labels.astype(np.int32).ravel())
    out = torch.empty(cap, dtype=torch.int64, device="cuda")
    n = torch.zeros(1, dtype=torch.int64, device="cuda")
    v.vor_edges(d, out, n)
    v.vor_sync_status()
    return u64(out, int(n.item())).copy()


def gpu_edges_rows(v: Vor, labels, n_rows, cap=None):
    """vor_edges_rows on a host label image -> (keys, row_ptr[n_rows + 1])."""
    cap = cap or max(1024, 8 * v.max_sites)
    d = dev(labels.astype(np.int32).ravel())
    out = torch.empty(cap, dtype=torch.int64, device="cuda")
    n = torch.zeros(1, dtype=torch.int64, device="cuda")
    ptr = torch.full((n_rows + 1,), -1, dtype=torch.int32, device="cuda")
    v.vor_edges_rows(d, out, n, ptr)
    v.vor_sync_status()
    return u64(out, int(n.item())).copy(), ptr.cpu().numpy().view(np.uint32).astype(np.int64)


def gpu_diff_rows(v: Vor, prev, prev_ptr, now, now_ptr, n_rows):
    cap = max(1, len(prev) + len(now))
    mk = lambda a: dev(np.asarray(a, np.uint64).view(np.int64)) if len(a) else torch.empty(1, dtype=torch.int64, device="cuda")
    mp = lambda a: dev(np.asarray(a, np.int64).astype(np.uint32).view(np.int32))
    c = torch.empty(cap, dtype=torch.int64, device="cuda")
    d = torch.empty(cap, dtype=torch.int64, device="cuda")
    nc = torch.zeros(1, dtype=torch.int64, device="cuda")
    nd = torch.zeros(1, dtype=torch.int64, device="cuda")
    v.vor_diff_rows(mk(prev), mp(prev_ptr), mk(now), mp(now_ptr), n_rows, c, d, nc, nd)
    v.vor_sync_status()
    return u64(c, int(nc.item())).copy(), u64(d, int(nd.item())).copy()


def gpu_diff(v: Vor, prev, now, p2n=None, n2p=None):
    cap = max(1, len(prev) + len(now))
    dp = dev(np.asarray(prev, np.uint64).view(np.int64)) if len(prev) else torch.empty(1, dtype=torch.int64, device="cuda")
    dn = dev(np.asarray(now, np.uint64).view(np.int64)) if len(now) else torch.empty(1, dtype=torch.int64, device="cuda")
    npv = torch.tensor([len(prev)], dtype=torch.int64, device="cuda")
    nnv = torch.tensor([len(now)], dtype=torch.int64, device="cuda")
    c = torch.empty(cap, dtype=torch.int64, device="cuda")
    d = torch.empty(cap, dtype=torch.int64, device="cuda")
    nc = torch.zeros(1, dtype=torch.int64, device="cuda")
    nd = torch.zeros(1, dtype=torch.int64, device="cuda")
    kw = {}
    if p2n is not None:
        kw = dict(p2n=dev(np.asarray(p2n, np.int32)), n2p=dev(np.asarray(n2p, np.int32)),
                  n_prev_labels=len(p2n), n_now_labels=len(n2p))
    v.vor_diff(dp, npv, dn, nnv, c, d, nc, nd, **kw)
    v.vor_sync_status()
    return u64(c, int(nc.item())).copy(), u64(d, int(nd.item())).copy()


def gpu_events(v: Vor, prev, now, n):
    """vor_diff then vor_events on host lists; returns the same dict as oracle.events()."""
    mk = lambda a: dev(np.asarray(a, np.uint64).view(np.int64)) if len(a) else torch.empty(1, dtype=torch.int64, device="cuda")
    dp, dn = mk(prev), mk(now)
    i64 = dict(dtype=torch.int64, device="cuda"); i32 = dict(dtype=torch.int32, device="cuda")
    npv, nnv = torch.tensor([len(prev)], **i64), torch.tensor([len(now)], **i64)
    cap = max(1, len(prev) + len(now))
    c, d = torch.empty(cap, **i64), torch.empty(cap, **i64)
    nc, nd = torch.zeros(1, **i64), torch.zeros(1, **i64)
    v.vor_diff(dp, npv, dn, nnv, c, d, nc, nd)
    trig = torch.full((n,), -5, **i32); idx = torch.full((n,), -5, **i32)
    cp = torch.full((n,), -5, **i32); cn = torch.full((n,), -5, **i32)
    m, g = torch.full((1,), -5, **i32), torch.full((1,), -5, **i32)
    v.vor_events(dp, npv, dn, nnv, c, nc, d, nd, trig, idx, m, g, cp, cn)
    v.vor_sync_status()
    return dict(trigger=trig.cpu().numpy(), events_indices=idx[:int(m.item())].cpu().numpy(),
                count_prev=cp.cpu().numpy(), count_now=cn.cpu().numpy(), global_trigger=int(g.item()))


def gpu_t1(v: Vor, prev, now, n, cap=None):
    """vor_diff -> vor_events -> vor_t1_events on host lists; returns the same dict as oracle.t1()
    plus n_couples (the required number, which may exceed cap)."""
    mk = lambda a: dev(np.asarray(a, np.uint64).view(np.int64)) if len(a) else torch.empty(1, dtype=torch.int64, device="cuda")
    dp, dn = mk(prev), mk(now)
    i64 = dict(dtype=torch.int64, device="cuda"); i32 = dict(dtype=torch.int32, device="cuda")
    npv, nnv = torch.tensor([len(prev)], **i64), torch.tensor([len(now)], **i64)
    lc = max(1, len(prev) + len(now))
    c, d = torch.empty(lc, **i64), torch.empty(lc, **i64)
    nc, nd = torch.zeros(1, **i64), torch.zeros(1, **i64)
    v.vor_diff(dp, npv, dn, nnv, c, d, nc, nd)
    trig, idx, cp, cn = (torch.empty(n, **i32) for _ in range(4))
    m, g = torch.zeros(1, **i32), torch.zeros(1, **i32)
    v.vor_events(dp, npv, dn, nnv, c, nc, d, nd, trig, idx, m, g, cp, cn)
    cap = lc if cap is None else cap
    pad = 3                                                # guard entries behind the capacity
    couples = torch.full((cap + pad,), -7, **i64); partner = torch.full((cap + pad,), -7, **i64)
    cls, kp, kn = (torch.full((cap + pad,), -7, **i32) for _ in range(3))
    nk = torch.full((1,), -7, **i64)
    v.vor_t1_events(dp, npv, dn, nnv, c, nc, d, nd, trig, couples[:cap], cls[:cap], kp[:cap], kn[:cap],
                    partner[:cap], nk)
    try:
        v.vor_sync_status()
        overflow = False
    except Exception as e:                                 # VOR_ECAPACITY: the caller decides whether it was expected
        overflow = "ECAPACITY" in str(e)
        if not overflow:
            raise
    for t in (couples, partner, cls, kp, kn):
        assert (t[cap:] == -7).all(), "write past the capacity"
    k = min(int(nk.item()), cap)
    return dict(couples=u64(couples, k).copy(), cls=cls[:k].cpu().numpy(), common_prev=kp[:k].cpu().numpy(),
                common_now=kn[:k].cpu().numpy(), partner=u64(partner, k).copy(), n_couples=int(nk.item()),
                overflow=overflow)


def gpu_event_vertices(v: Vor, prev, now, n):
    """vor_diff -> vor_events -> vor_event_vertices on host lists; returns the same dict as oracle.event_vertices()."""
    mk = lambda a: dev(np.asarray(a, np.uint64).view(np.int64)) if len(a) else torch.empty(1, dtype=torch.int64, device="cuda")
    dp, dn = mk(prev), mk(now)
    i64 = dict(dtype=torch.int64, device="cuda"); i32 = dict(dtype=torch.int32, device="cuda")
    npv, nnv = torch.tensor([len(prev)], **i64), torch.tensor([len(now)], **i64)
    lc = max(1, len(prev) + len(now))
    c, d = torch.empty(lc, **i64), torch.empty(lc, **i64)
    nc, nd = torch.zeros(1, **i64), torch.zeros(1, **i64)
    v.vor_diff(dp, npv, dn, nnv, c, d, nc, nd)
    trig, idx, cp, cn = (torch.empty(n, **i32) for _ in range(4))
    m, g = torch.zeros(1, **i32), torch.zeros(1, **i32)
    v.vor_events(dp, npv, dn, nnv, c, nc, d, nd, trig, idx, m, g, cp, cn)
    bp, bn, vc = (torch.full((n,), -9, **i32) for _ in range(3))
    v.vor_event_vertices(dp, npv, dn, nnv, trig, bp, bn, vc)
    v.vor_sync_status()
    return dict(boundary_prev=bp.cpu().numpy(), boundary_now=bn.cpu().numpy(), vclass=vc.cpu().numpy())


def gpu_ccl(v: Vor, field, thr, above=True, connectivity=None):
    f = dev(field.astype(np.float32).ravel())
    ccl = torch.empty(v.cells, dtype=torch.int32, device="cuda")
    if connectivity is None:
        v.field_threshold_ccl(f, thr, above, ccl)
    else:
        v.field_threshold_ccl_conn(f, thr, above, connectivity, ccl)
    v.vor_sync_status()
    return ccl


def gpu_centroids(v: Vor, ccl_dev, min_size, cap=None, field=None):
    cap = cap or max(16, v.cells // 2)
    cx = torch.empty(cap, dtype=torch.float64, device="cuda"); cy = torch.empty_like(cx)
    sx = torch.empty(cap, dtype=torch.int32, device="cuda"); sy = torch.empty_like(sx)
    size = torch.empty_like(sx); root = torch.empty_like(sx)
    n = torch.zeros(1, dtype=torch.int32, device="cuda")
    if field is None:
        v.field_centroids(ccl_dev, min_size, cx, cy, sx, sy, size, root, n)
    else:
        v.field_centroids_weighted(ccl_dev, dev(np.ascontiguousarray(field, dtype=np.float32).ravel()), min_size,
                                   cx, cy, sx, sy, size, root, n)
    v.vor_sync_status()
    K = int(n.item())
    g = lambda t: t[:K].cpu().numpy()
    return dict(cx=g(cx), cy=g(cy), sx=g(sx), sy=g(sy), size=g(size), root=g(root))


def gpu_match(v: Vor, px, py, nx, ny, radius_fp, pad=7):
    """pad > 0 exercises capacity > count."""
    P, N = len(px), len(nx)
    mk = lambda a, n: dev(np.concatenate([np.asarray(a, np.int32), np.zeros(pad, np.int32)]))
    dpx, dpy, dnx, dny = mk(px, P), mk(py, P), mk(nx, N), mk(ny, N)
    p2n = torch.full((P + pad,), -7, dtype=torch.int32, device="cuda")
    n2p = torch.full((N + pad,), -7, dtype=torch.int32, device="cuda")
    v.match_sites(dpx, dpy, torch.tensor([P], dtype=torch.int32, device="cuda"),
                  dnx, dny, torch.tensor([N], dtype=torch.int32, device="cuda"), radius_fp, p2n, n2p)
    v.vor_sync_status()
    return p2n[:P].cpu().numpy(), n2p[:N].cpu().numpy()


def from_device_ptr(ptr, count, dtype):
    """Copy `count` elements of torch dtype from a raw device pointer into a new tensor."""
    t = torch.empty(count, dtype=dtype, device="cuda")
    if count:
        cudart = C.CDLL("libcudart.so.12")
        rc = cudart.cudaMemcpy(C.c_void_p(t.data_ptr()), C.c_void_p(ptr),
                               C.c_size_t(count * t.element_size()), C.c_int(3))
        assert rc == 0, rc
    return t
