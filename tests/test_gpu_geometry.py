"""-m gpu: parity of the CUDA path with oracle O9 on the paper's own geometry - rectangular lattices, walled
axes, obstacle colour, 8-connected bubbles, density-weighted centres, size histogram, bulk / boundary edges,
row strips.  Integer / index work: bit-exact.  Centres (float64):
|diff| <= 1e-9 lattice units.
"""
import numpy as np
import pytest

import oracle
from helpers import FP, hex_sites, pack
from paper_1607_00908_b200 import workloads as W

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def G():
    import gpu_util
    return gpu_util


def make(Lx, Ly, per, max_sites, **kw):
    from paper_1607_00908_b200.binding import Vor
    return Vor(Lx, max_sites, Ly=Ly, periodic=per, **kw)


def rand_sites(rng, Lx, Ly, n):
    return rng.integers(0, FP * Lx, n).astype(np.int32), rng.integers(0, FP * Ly, n).astype(np.int32)


def jitter_sites(rng, Lx, Ly, spacing, jitter=0.4):
    """A jittered grid of about one site per spacing^2 cells (the structure of config 5 and of the paper's
    droplets), wrapped into the lattice."""
    nx, ny = max(1, round(Lx / spacing)), max(1, round(Ly / spacing))
    gx, gy = np.meshgrid((np.arange(nx) + 0.5) * Lx / nx, (np.arange(ny) + 0.5) * Ly / ny)
    x = gx.ravel() + rng.uniform(-jitter, jitter, nx * ny) * Lx / nx
    y = gy.ravel() + rng.uniform(-jitter, jitter, nx * ny) * Ly / ny
    fx = (np.floor(np.mod(x, Lx) * FP + 0.5).astype(np.int64) % (FP * Lx)).astype(np.int32)
    fy = (np.floor(np.mod(y, Ly) * FP + 0.5).astype(np.int64) % (FP * Ly)).astype(np.int32)
    return fx, fy


GEOMS = [(96, 48, (1, 1)), (48, 112, (1, 1)), (64, 32, (0, 1)), (40, 72, (1, 0)), (56, 56, (0, 0)),
         (100, 36, (0, 1)), (33, 47, (1, 1)), (257, 130, (0, 0))]


# ------------------------------------------------------------------ labels
@pytest.mark.parametrize("Lx,Ly,per", GEOMS)
def test_labels_every_path_on_rectangles_and_walls(G, Lx, Ly, per):
    rng = np.random.default_rng(Lx * 7 + Ly)
    for n, gen in ((1, None), (9, None), (max(2, Lx * Ly // 64), "jitter"), (Lx * Ly // 12, None)):
        sx, sy = jitter_sites(rng, Lx, Ly, 8.0) if gen else rand_sites(rng, Lx, Ly, n)
        ref = oracle.label_brute_g(Lx, Ly, per[0], per[1], sx, sy)
        v = make(Lx, Ly, per, len(sx))
        for path in (0, 1, 2, 3):
            for fast_off in ((0, 1) if path in (0, 2) else (0,)):
                v.vor_set_option("label_path", path)
                v.vor_set_option("label_fast_off", fast_off)
                got = G.gpu_labels(v, sx, sy)
                bad = np.argwhere(got != ref)
                assert len(bad) == 0, f"{n} sites, path {path}/{fast_off}: {len(bad)} differ, first {bad[:4].tolist()}"
        v.close()


@pytest.mark.parametrize("Lx,Ly,per", [(2048, 1024, (1, 1)), (2048, 1024, (0, 1)), (1024, 2048, (1, 0)), (1536, 640, (0, 0))])
def test_labels_paper_size_lattice(G, Lx, Ly, per):
    """2048 x 1024 sites, about 2000 droplets of 30-35 sites diameter; O1b on the general
    geometry (pinned against O1a in the CPU tests) is the reference at this size."""
    rng = np.random.default_rng(11)
    sx, sy = jitter_sites(rng, Lx, Ly, 32.0)
    ref = oracle.label_cells_g(Lx, Ly, per[0], per[1], sx, sy, 32)
    cells = rng.integers(0, Lx * Ly, 2000)
    assert np.array_equal(ref.ravel()[cells], oracle.label_brute_at_g(Lx, Ly, per[0], per[1], sx, sy, cells))
    v = make(Lx, Ly, per, len(sx))
    got = G.gpu_labels(v, sx, sy)
    assert np.array_equal(got, ref), int((got != ref).sum())
    e = G.gpu_edges_image(v, got, per[1])
    assert np.array_equal(e, oracle.edges_g(ref, per[0], per[1]))
    v.close()


def test_label_rows_strips_cover_the_lattice(G):
    rng = np.random.default_rng(3)
    for Lx, Ly, per, spacing in ((128, 96, (1, 1), 9.0), (96, 200, (0, 1), 12.0), (64, 64, (1, 0), 5.0)):
        sx, sy = jitter_sites(rng, Lx, Ly, spacing)
        ref = oracle.label_brute_g(Lx, Ly, per[0], per[1], sx, sy)
        v = make(Lx, Ly, per, len(sx))
        v.vor_build_cells(G.dev(sx), G.dev(sy))
        for y0, n in ((0, Ly), (0, 1), (Ly - 1, 1), (7, 33), (Ly // 2, Ly - Ly // 2), (31, 32), (5, 3)):
            assert np.array_equal(G.gpu_label_rows(v, y0, n), ref[y0:y0 + n]), (Lx, Ly, y0, n)
        for bad in ((-1, 4), (0, Ly + 1), (Ly - 1, 2), (3, 0)):
            with pytest.raises(Exception):
                G.gpu_label_rows(v, *bad)
        v.close()


# ------------------------------------------------------------------ edges: walls, obstacles, strips
def test_edges_hand_image_walls_and_obstacle_colour(G):
    lab = np.array([[0, 0, 1, 1, 1, 2],
                    [0, 0, 1, 1, 2, 2],
                    [3, 3, 3, 9, 2, 2],
                    [3, 3, 3, 9, 9, 2]], np.int32)
    for per in ((0, 0), (1, 0), (0, 1), (1, 1)):
        for ex in (-1, 9):
            v = make(6, 4, per, 16)
            assert np.array_equal(G.gpu_edges_image(v, lab, per[1], ex), oracle.edges_g(lab, per[0], per[1], ex)), (per, ex)
            v.close()


@pytest.mark.parametrize("Lx,Ly,per", GEOMS + [(512, 256, (0, 1)), (260, 516, (1, 0))])
def test_edges_random_images_rows_and_strips(G, Lx, Ly, per):
    rng = np.random.default_rng(Lx + 3 * Ly)
    n = max(4, Lx * Ly // 80)
    sx, sy = rand_sites(rng, Lx, Ly, n)
    lab = oracle.label_brute_g(Lx, Ly, per[0], per[1], sx, sy)
    noise = rng.integers(0, n, (Ly, Lx)).astype(np.int32)          # every pair differs: the densest case
    v = make(Lx, Ly, per, n)
    for generic in (0, 1):
        v.vor_set_option("edges_generic", generic)
        for img in (lab, noise):
            for ex in (-1, 3):
                ref = oracle.edges_g(img, per[0], per[1], ex)
                keys, ptr = G.gpu_edges_image(v, img, per[1], ex, cap=2 * Lx * Ly + 8, n_rows_ptr=n)
                assert np.array_equal(keys, ref), (generic, ex)
                hi = (ref >> np.uint64(32)).astype(np.int64)
                assert np.array_equal(ptr, np.searchsorted(hi, np.arange(n + 1)))
    # strips: rows [y0, y1] with the first row of the next strip appended, no wrap; the union is the lattice's
    # list (the last strip's extra row is row 0 when the y axis is periodic)
    v.vor_set_option("edges_generic", 0)
    ref = set(oracle.edges_g(lab, per[0], per[1]).tolist())
    for parts in (2, 3, 5):
        cuts = [round(k * Ly / parts) for k in range(parts + 1)]
        got = set()
        for a, b in zip(cuts[:-1], cuts[1:]):
            if b < Ly:
                strip = lab[a:b + 1]
            elif per[1]:
                strip = np.concatenate([lab[a:b], lab[:1]])
            else:
                strip = lab[a:b]
            keys = G.gpu_edges_image(v, strip, False, -1, cap=2 * Lx * Ly + 8)
            assert np.array_equal(keys, oracle.edges_g(strip, per[0], 0))
            got |= set(keys.tolist())
        assert got == ref, parts
    v.close()


def test_obstacles_channel_with_posts(G):
    """The paper's geometry in small: a channel periodic along y, walls in x, a row of posts on
    the left wall; droplets everywhere else.  Obstacle sites take MAXLINK and take part in no edge."""
    rng = np.random.default_rng(21)
    Lx, Ly = 256, 512
    MAXLINK = 0x77777777
    sx, sy = jitter_sites(rng, Lx, Ly, 30.0)
    mask = np.zeros((Ly, Lx), np.uint8)
    for k in range(8):                                            # equally spaced posts of height 40, width 24
        mask[64 * k + 10: 64 * k + 34, :40] = 1
    v = make(Lx, Ly, (0, 1), len(sx))
    lab = G.gpu_labels(v, sx, sy)
    ref_lab = oracle.label_brute_g(Lx, Ly, 0, 1, sx, sy)
    assert np.array_equal(lab, ref_lab)
    d_lab, d_mask = G.dev(lab.ravel()), G.dev(mask.ravel())
    v.vor_paint_obstacles(d_mask, MAXLINK, d_lab)
    v.vor_sync_status()
    col = d_lab.cpu().numpy().reshape(Ly, Lx)
    ref_col = oracle.apply_obstacles(ref_lab, mask, MAXLINK)
    assert np.array_equal(col, ref_col)
    e = G.gpu_edges_image(v, col, True, MAXLINK)
    ref_e = oracle.edges_g(ref_col, 0, 1, MAXLINK)
    assert np.array_equal(e, ref_e) and len(e) > 2 * len(sx)
    plain = oracle.edges_g(ref_lab, 0, 1)
    assert set(e.tolist()) < set(plain.tolist())                  # the posts cut some contacts, add none
    # bulk and boundary edges: the walls and the posts give the triangulation a boundary
    c = G.gpu_edge_commons(v, e, len(sx))
    assert np.array_equal(c, oracle.edge_commons(ref_e, len(sx)))
    assert (c == 1).sum() > 10 and (c == 2).sum() > len(sx)
    v.close()


def test_edge_commons_hand_random_and_torus(G):
    v = make(64, 64, (1, 1), 64)
    e = pack([(0, 1), (0, 2), (1, 2), (1, 3), (2, 3), (2, 4), (3, 4), (3, 5), (4, 5)])
    assert G.gpu_edge_commons(v, e, 6).tolist() == [1, 1, 2, 1, 2, 1, 2, 1, 1]
    assert G.gpu_edge_commons(v, pack([(0, 1), (1, 7)]), 3).tolist() == [0, -1]
    assert len(G.gpu_edge_commons(v, np.empty(0, np.uint64), 3)) == 0
    rng = np.random.default_rng(5)
    for n, p in ((40, 0.2), (600, 0.02), (3000, 0.004)):
        i, j = np.triu_indices(n, 1)
        keep = rng.random(len(i)) < p
        keys = np.sort((i[keep].astype(np.uint64) << np.uint64(32)) | j[keep].astype(np.uint64))
        assert np.array_equal(G.gpu_edge_commons(v, keys, n), oracle.edge_commons(keys, n))
    v.close()
    L = 256
    sx, sy = hex_sites(L, 16, 18, 0.8, seed=3)
    v = make(L, L, (1, 1), len(sx))
    e = G.gpu_edges(v, G.gpu_labels(v, sx, sy))
    assert set(G.gpu_edge_commons(v, e, len(sx)).tolist()) == {2}           # a torus has no boundary
    v.close()


# ------------------------------------------------------------------ bubbles
@pytest.mark.parametrize("Lx,Ly,per", GEOMS + [(640, 200, (0, 1)), (130, 770, (1, 1))])
def test_ccl_connectivity_walls_rectangles(G, Lx, Ly, per):
    rng = np.random.default_rng(Lx * 3 + Ly)
    v = make(Lx, Ly, per, 16)
    for conn, p in ((4, 0.55), (8, 0.38), (8, 0.5), (4, 0.3)):
        f = rng.random((Ly, Lx)).astype(np.float32)
        got = G.gpu_ccl(v, f, 1.0 - p, True, conn).cpu().numpy().reshape(Ly, Lx)
        ref = oracle.threshold_ccl_g(f, 1.0 - p, True, per[0], per[1], conn)
        assert np.array_equal(got, ref), (conn, p, int((got != ref).sum()))
    # long diagonal chains: connected only under 8-connectivity, crossing many tile seams and the wrap
    f = np.zeros((Ly, Lx), np.float32)
    k = np.arange(4 * max(Lx, Ly))
    f[k % Ly, k % Lx] = 2
    f[(k + 7) % Ly, (-k) % Lx] = 2
    for conn in (4, 8):
        got = G.gpu_ccl(v, f, 1.0, True, conn).cpu().numpy().reshape(Ly, Lx)
        assert np.array_equal(got, oracle.threshold_ccl_g(f, 1.0, True, per[0], per[1], conn)), conn
    with pytest.raises(Exception):
        G.gpu_ccl(v, f, 1.0, True, 6)
    v.close()


@pytest.mark.parametrize("Lx,Ly,per", GEOMS[:6] + [(512, 192, (0, 1))])
def test_centroids_weighted_walls_rectangles_and_histogram(G, Lx, Ly, per):
    rng = np.random.default_rng(Lx + Ly)
    v = make(Lx, Ly, per, 16)
    f = rng.random((Ly, Lx)).astype(np.float32)
    rho = (rng.random((Ly, Lx)) * 3 - 0.2).astype(np.float32)       # some negative densities: weight one unit
    rho[rng.random((Ly, Lx)) < 0.01] = np.nan
    rho[rng.random((Ly, Lx)) < 0.01] = 1e9                            # clipped at 2^24
    for conn, thr in ((4, 0.45), (8, 0.62)):
        ccl = G.gpu_ccl(v, f, thr, True, conn)
        ref_ccl = oracle.threshold_ccl_g(f, thr, True, per[0], per[1], conn)
        for field in (None, rho):
            for min_size in (1, 4):
                got = G.gpu_centroids(v, ccl, min_size, field=field)
                ref = oracle.centroids_g(ref_ccl, min_size, per[0], per[1], field)
                for k in ("sx", "sy", "size", "root"):
                    assert np.array_equal(got[k], ref[k]), (k, conn, field is not None)
                assert np.abs(got["cx"] - ref["cx"]).max() <= 1e-9 and np.abs(got["cy"] - ref["cy"]).max() <= 1e-9
        size = G.dev(ref["size"]) if len(ref["size"]) else torch.zeros(1, dtype=torch.int32, device="cuda")
        n = torch.tensor([len(ref["size"])], dtype=torch.int32, device="cuda")
        for width, bins in ((1, 64), (5, 7), (1000, 2)):
            hist = torch.full((bins,), -3, dtype=torch.int64, device="cuda")
            v.field_size_histogram(size, n, width, hist)
            v.vor_sync_status()
            assert np.array_equal(hist.cpu().numpy(), oracle.size_histogram(ref["size"], width, bins))
    v.close()


def test_weighted_centre_closed_form_on_the_gpu(G):
    Lx, Ly = 64, 40
    yy, xx = np.mgrid[0:Ly, 0:Lx]
    v = make(Lx, Ly, (1, 1), 16)
    for cxr, cyr in ((20, 17), (0, 0), (63, 39)):
        dx = (xx - cxr + Lx // 2) % Lx - Lx // 2
        dy = (yy - cyr + Ly // 2) % Ly - Ly // 2
        r2 = dx * dx + dy * dy
        mask = r2 <= 36
        rho = np.where(mask, 1.0 + r2 / 8.0, 0.0).astype(np.float32)
        ccl = G.gpu_ccl(v, mask.astype(np.float32), 0.5, True, 4)
        c = G.gpu_centroids(v, ccl, 1, field=rho)
        assert len(c["cx"]) == 1 and abs(c["cx"][0] - (cxr + 0.5)) < 1e-12 and abs(c["cy"][0] - (cyr + 0.5)) < 1e-12
        assert c["sx"][0] == FP * cxr + 128 and c["sy"][0] == FP * cyr + 128
    v.close()


@pytest.mark.parametrize("Lx,Ly,per", GEOMS[:5])
def test_match_on_rectangles_and_walls(G, Lx, Ly, per):
    rng = np.random.default_rng(Lx * 5 + Ly)
    v = make(Lx, Ly, per, 4096)
    for n, r in ((1, 300), (30, 500), (400, 256), (2000, 700)):
        px, py = rand_sites(rng, Lx, Ly, n)
        nx = ((px.astype(np.int64) + rng.integers(-400, 400, n)) % (FP * Lx)).astype(np.int32)
        ny = ((py.astype(np.int64) + rng.integers(-400, 400, n)) % (FP * Ly)).astype(np.int32)
        keep = rng.random(n) < 0.9
        nx, ny = nx[keep | (np.arange(n) == 0)], ny[keep | (np.arange(n) == 0)]
        a, b = G.gpu_match(v, px, py, nx, ny, r)
        ra, rb = oracle.match_g(Lx, Ly, per[0], per[1], px, py, nx, ny, r)
        assert np.array_equal(a, ra) and np.array_equal(b, rb), (n, r)
    # a pair across the seam is matched only on a periodic axis
    px, py = np.array([FP * Lx - 30], np.int32), np.array([FP * 4], np.int32)
    nx, ny = np.array([40], np.int32), np.array([FP * 4], np.int32)
    assert G.gpu_match(v, px, py, nx, ny, 100)[0].tolist() == ([0] if per[0] else [-1])
    v.close()


# ------------------------------------------------------------------ the whole path on the paper's geometry
def test_channel_sequence_field_to_events(G):
    """Droplets in a 512 x 256 channel (walls in x, periodic in y) over 4 frames: 8-connected bubbles of a
    density field, weighted centres, matching, labels, obstacle colour, edges, diff with the maps, trigger and
    T1 couples - every stage against the oracle chain."""
    rng = np.random.default_rng(33)
    Lx, Ly, per = 512, 256, (0, 1)
    MAXLINK = 0x77777777
    cx0, cy0 = jitter_sites(rng, Lx, Ly, 32.0, jitter=0.25)
    cx0 = cx0 / FP; cy0 = cy0 / FP
    keep = cx0 > 56                                               # room for the posts on the left wall
    cx0, cy0 = cx0[keep], cy0[keep]
    obst = np.zeros((Ly, Lx), np.uint8)
    for k in range(4):
        obst[64 * k + 8: 64 * k + 32, :36] = 1
    yy, xx = np.mgrid[0:Ly, 0:Lx]
    v = make(Lx, Ly, per, 1024)
    prev = None
    for t in range(4):
        cx = cx0 + 0.8 * t * np.sin(cy0 / 17.0) + rng.normal(0, 0.6, len(cx0))
        cy = (cy0 + 1.5 * t * (cx0 / Lx) + rng.normal(0, 0.6, len(cx0))) % Ly
        rho = np.full((Ly, Lx), 1.2, np.float32)
        for a, b in zip(cx, cy):                                  # low density inside a droplet
            x0, x1 = int(max(0, a - 14)), int(min(Lx, a + 15))
            ys = np.arange(int(b) - 14, int(b) + 15) % Ly
            dx = xx[0, x0:x1][None, :] + 0.5 - a
            dy = (ys[:, None] + 0.5 - b + Ly / 2) % Ly - Ly / 2
            d = np.sqrt(dx * dx + dy * dy)
            rho[np.ix_(ys, np.arange(x0, x1))] = np.minimum(rho[np.ix_(ys, np.arange(x0, x1))],
                                                           (0.2 + 1.0 / (1.0 + np.exp(-(d - 11.0)))).astype(np.float32))
        # oracle chain
        r_ccl = oracle.threshold_ccl_g(rho, 0.7, False, per[0], per[1], 8)
        r_c = oracle.centroids_g(r_ccl, 20, per[0], per[1], rho)
        r_lab = oracle.apply_obstacles(oracle.label_brute_g(Lx, Ly, per[0], per[1], r_c["sx"], r_c["sy"]), obst, MAXLINK)
        r_e = oracle.edges_g(r_lab, per[0], per[1], MAXLINK)
        # CUDA chain
        ccl = G.gpu_ccl(v, rho, 0.7, False, 8)
        assert np.array_equal(ccl.cpu().numpy().reshape(Ly, Lx), r_ccl)
        c = G.gpu_centroids(v, ccl, 20, field=rho)
        for k in ("sx", "sy", "size", "root"):
            assert np.array_equal(c[k], r_c[k]), (t, k)
        assert 80 < len(c["sx"]) <= len(cx0)
        lab = G.gpu_labels(v, c["sx"], c["sy"])
        d_lab = G.dev(lab.ravel())
        v.vor_paint_obstacles(G.dev(obst.ravel()), MAXLINK, d_lab)
        v.vor_sync_status()
        assert np.array_equal(d_lab.cpu().numpy().reshape(Ly, Lx), r_lab)
        e = G.gpu_edges_image(v, d_lab.cpu().numpy().reshape(Ly, Lx), True, MAXLINK)
        assert np.array_equal(e, r_e), t
        if prev is not None:
            p_c, p_e = prev
            r_p2n, r_n2p = oracle.match_g(Lx, Ly, per[0], per[1], p_c["sx"], p_c["sy"], r_c["sx"], r_c["sy"], 4 * FP)
            p2n, n2p = G.gpu_match(v, p_c["sx"], p_c["sy"], c["sx"], c["sy"], 4 * FP)
            assert np.array_equal(p2n, r_p2n) and np.array_equal(n2p, r_n2p)
            r_cr, r_de = oracle.diff(p_e, r_e, r_p2n, r_n2p)
            cr, de = G.gpu_diff(v, p_e, e, p2n, n2p)
            assert np.array_equal(cr, r_cr) and np.array_equal(de, r_de)
        prev = (r_c, r_e)
    v.close()


# ------------------------------------------------------------------ row strips of one lattice (NEXT-4)
def test_strip_decomposition_on_one_gpu(G):
    """Every strip of a 1-, 2-, 3- and 5-way decomposition computed by the product class (explicit rank /
    world, no process group), merged by vor_merge_lists: the lattice's list, bit for bit.  The collective
    itself is covered on CPU (tests/test_strips_ranks.py, gloo)."""
    from paper_1607_00908_b200.strips import StripFrame
    rng = np.random.default_rng(8)
    for Lx, Ly, per, spacing in ((256, 512, (1, 1), 12.0), (192, 320, (0, 1), 16.0), (128, 200, (1, 0), 9.0)):
        sx, sy = jitter_sites(rng, Lx, Ly, spacing)
        n = len(sx)
        ref = oracle.edges_g(oracle.label_brute_g(Lx, Ly, per[0], per[1], sx, sy), per[0], per[1])
        v = make(Lx, Ly, per, n)
        dsx, dsy = G.dev(sx), G.dev(sy)
        cap = 8 * n
        for world in (1, 2, 3, 5):
            lists = torch.zeros(world, cap, dtype=torch.int64, device="cuda")
            counts = torch.zeros(world, dtype=torch.int64, device="cuda")
            for r in range(world):
                f = StripFrame(v, n, cap, cap, rank=r, world=world)
                loc, nl = f.compute_local(dsx, dsy)
                lists[r].copy_(loc); counts[r] = nl[0]
            out = torch.empty(cap, dtype=torch.int64, device="cuda")
            n_out = torch.zeros(1, dtype=torch.int64, device="cuda")
            v.vor_merge_lists(lists, counts, n, out, n_out)
            v.vor_sync_status()
            assert np.array_equal(G.u64(out, int(n_out.item())), ref), (Lx, Ly, world)
        f = StripFrame(v, n, cap, cap)                          # no process group: one strip, the whole lattice
        e, ne = f.compute(dsx, dsy)
        v.vor_sync_status()
        assert np.array_equal(G.u64(e, int(ne.item())), ref)
        v.close()


# ------------------------------------------------------------------ seeded random sweep over geometries
def test_random_sweep_frames_on_random_geometries(G):
    """40 seeded draws of (Lx, Ly, periodicity, site count, motion): three frames each through vor_frame_host
    (with and without the fused label -> edge kernel, which applies where Lx % 32 == 0) against the oracle chain on the same geometry -
    labels, edge counts, created / destroyed lists."""
    rng = np.random.default_rng(20260)
    for case in range(40):
        Lx = int(rng.choice([32, 36, 64, 96, 100, 128, 160, 257, 320]))
        Ly = int(rng.choice([32, 40, 64, 96, 128, 130, 192, 288]))
        per = (int(rng.integers(0, 2)), int(rng.integers(0, 2)))
        spacing = float(rng.choice([3.0, 5.0, 8.0, 12.0, 20.0, 40.0]))
        if rng.random() < 0.5:
            sx, sy = jitter_sites(rng, Lx, Ly, spacing)
        else:
            sx, sy = rand_sites(rng, Lx, Ly, max(1, int(Lx * Ly / spacing ** 2)))
        n = len(sx)
        rng.integers(0, 2)                                 # (keeps the draws of earlier rounds' cases)
        sigma = float(rng.choice([0.0, 0.3, 2.0])) * FP
        frames = []
        for t in range(3):
            frames.append((sx, sy))
            sx = ((sx.astype(np.int64) + np.rint(rng.normal(0, sigma, n)).astype(np.int64)) % (FP * Lx)).astype(np.int32)
            sy = ((sy.astype(np.int64) + np.rint(rng.normal(0, sigma, n)).astype(np.int64)) % (FP * Ly)).astype(np.int32)
        refs, prev = [], np.empty(0, np.uint64)
        for fx, fy in frames:
            lab = oracle.label_brute_g(Lx, Ly, per[0], per[1], fx, fy)
            e = oracle.edges_g(lab, per[0], per[1])
            refs.append((lab, e) + oracle.diff(prev, e))
            prev = e
        cap = 2 * Lx * Ly + 16
        for fuse in (0, 1):                                # every geometry with and without the fused kernel
            v = make(Lx, Ly, per, n)
            v.vor_set_option("fuse", fuse)
            hc = np.empty(cap, np.uint64); hd = np.empty(cap, np.uint64); cnt = np.zeros(3, np.int64)
            for t, ((fx, fy), (lab, e, rc, rd)) in enumerate(zip(frames, refs)):
                v.vor_frame_host(fx, fy, hc, hd, cnt)
                pl = v.vor_frame_results()[0]
                got = G.from_device_ptr(pl, Lx * Ly, torch.int32).cpu().numpy().reshape(Ly, Lx)
                assert np.array_equal(got, lab), (case, t, Lx, Ly, per, n, fuse, int((got != lab).sum()))
                assert cnt.tolist() == [len(e), len(rc), len(rd)], (case, t, Lx, Ly, per, n, fuse)
                assert np.array_equal(hc[:cnt[1]], rc) and np.array_equal(hd[:cnt[2]], rd), (case, t, fuse)
            v.close()


def test_random_sweep_field_chain(G):
    """24 seeded draws: threshold + bubbles (4 / 8-connected) + centres (weighted or not) + matching between two
    fields on random geometries, every output against oracle O9."""
    rng = np.random.default_rng(777)
    for case in range(24):
        Lx = int(rng.choice([32, 48, 100, 128, 200, 257]))
        Ly = int(rng.choice([32, 40, 96, 130, 256]))
        per = (int(rng.integers(0, 2)), int(rng.integers(0, 2)))
        conn = int(rng.choice([4, 8]))
        p = float(rng.choice([0.1, 0.3, 0.45, 0.6]))
        weighted = bool(rng.integers(0, 2))
        min_size = int(rng.choice([1, 3, 10]))
        v = make(Lx, Ly, per, max(16, Lx * Ly // 2))
        cents = []
        base = rng.random((Ly, Lx)).astype(np.float32)
        for t in range(2):
            f = np.roll(base, (t, 2 * t), axis=(0, 1)) + (rng.random((Ly, Lx)) * 0.05).astype(np.float32)
            ccl = G.gpu_ccl(v, f, 1.0 - p, True, conn)
            ref_ccl = oracle.threshold_ccl_g(f, 1.0 - p, True, per[0], per[1], conn)
            assert np.array_equal(ccl.cpu().numpy().reshape(Ly, Lx), ref_ccl), (case, t)
            got = G.gpu_centroids(v, ccl, min_size, field=f if weighted else None)
            ref = oracle.centroids_g(ref_ccl, min_size, per[0], per[1], f if weighted else None)
            for k in ("sx", "sy", "size", "root"):
                assert np.array_equal(got[k], ref[k]), (case, t, k)
            if len(ref["cx"]):
                assert np.abs(got["cx"] - ref["cx"]).max() <= 1e-9 and np.abs(got["cy"] - ref["cy"]).max() <= 1e-9
            cents.append(ref)
        a, b = cents
        if len(a["sx"]) and len(b["sx"]):
            R = int(rng.choice([FP, 3 * FP, 6 * FP]))
            p2n, n2p = G.gpu_match(v, a["sx"], a["sy"], b["sx"], b["sy"], R)
            r1, r2 = oracle.match_g(Lx, Ly, per[0], per[1], a["sx"], a["sy"], b["sx"], b["sy"], R)
            assert np.array_equal(p2n, r1) and np.array_equal(n2p, r2), case
        v.close()


# ------------------------------------------------------------------ the frame calls on the paper's set-up
def test_frame_calls_with_walls_obstacles_weights(G):
    """field_frame_device with vor_frame_options(8-connected, weighted, obstacle mask) on a walled channel, and
    vor_frame_host with the same obstacles: counts, maps and flip lists of every frame against the oracle chain."""
    rng = np.random.default_rng(44)
    Lx, Ly, per = 384, 256, (0, 1)
    MAXLINK = 0x77777777
    obst = np.zeros((Ly, Lx), np.uint8)
    for k in range(4):
        obst[64 * k + 8: 64 * k + 32, :30] = 1
    d_obst = G.dev(obst.ravel())
    cx0, cy0 = jitter_sites(rng, Lx, Ly, 32.0, jitter=0.25)
    cx0 = cx0 / FP; cy0 = cy0 / FP
    keep = cx0 > 50
    cx0, cy0 = cx0[keep], cy0[keep]
    yy, xx = np.mgrid[0:Ly, 0:Lx]
    v = make(Lx, Ly, per, 512)
    v.vor_frame_options(8, True, d_obst, MAXLINK)
    R = 4 * FP
    prev = None
    for t in range(4):
        cx = cx0 + 0.7 * t * np.sin(cy0 / 19.0) + rng.normal(0, 0.5, len(cx0))
        cy = (cy0 + 1.2 * t * (cx0 / Lx) + rng.normal(0, 0.5, len(cx0))) % Ly
        rho = np.full((Ly, Lx), 1.2, np.float32)
        for a, b in zip(cx, cy):
            x0, x1 = int(max(0, a - 14)), int(min(Lx, a + 15))
            ys = np.arange(int(b) - 14, int(b) + 15) % Ly
            dx = xx[0, x0:x1][None, :] + 0.5 - a
            dy = (ys[:, None] + 0.5 - b + Ly / 2) % Ly - Ly / 2
            d = np.sqrt(dx * dx + dy * dy)
            sub = np.ix_(ys, np.arange(x0, x1))
            rho[sub] = np.minimum(rho[sub], (0.2 + 1.0 / (1.0 + np.exp(-(d - 11.0)))).astype(np.float32))
        rho = 1.4 - rho                                           # bubbles where the field is ABOVE the threshold
        v.field_frame_device(G.dev(rho.ravel()), 0.7, True, 20, R)
        v.vor_sync_status()
        r_ccl = oracle.threshold_ccl_g(rho, 0.7, True, per[0], per[1], 8)
        r_c = oracle.centroids_g(r_ccl, 20, per[0], per[1], rho)
        r_lab = oracle.apply_obstacles(oracle.label_brute_g(Lx, Ly, per[0], per[1], r_c["sx"], r_c["sy"]), obst, MAXLINK)
        r_e = oracle.edges_g(r_lab, per[0], per[1], MAXLINK)
        res = v.field_frame_results()
        counts = G.from_device_ptr(res["counts"], 4, torch.int64).cpu().tolist()
        K = len(r_c["sx"])
        assert counts[0] == K and counts[1] == len(r_e), (t, counts, K, len(r_e))
        assert np.array_equal(G.from_device_ptr(res["ccl"], Lx * Ly, torch.int32).cpu().numpy().reshape(Ly, Lx), r_ccl)
        assert np.array_equal(G.from_device_ptr(res["labels"], Lx * Ly, torch.int32).cpu().numpy().reshape(Ly, Lx), r_lab)
        assert np.array_equal(G.from_device_ptr(res["sx"], K, torch.int32).cpu().numpy(), r_c["sx"])
        assert np.array_equal(G.u64(G.from_device_ptr(res["edges"], len(r_e), torch.int64)), r_e)
        if prev is not None:
            p_c, p_e = prev
            r_p2n, r_n2p = oracle.match_g(Lx, Ly, per[0], per[1], p_c["sx"], p_c["sy"], r_c["sx"], r_c["sy"], R)
            r_cr, r_de = oracle.diff(p_e, r_e, r_p2n, r_n2p)
            assert counts[2] == len(r_cr) and counts[3] == len(r_de), (t, counts)
            assert np.array_equal(G.u64(G.from_device_ptr(res["created"], len(r_cr), torch.int64)), r_cr)
            assert np.array_equal(G.u64(G.from_device_ptr(res["destroyed"], len(r_de), torch.int64)), r_de)
        prev = (r_c, r_e)
    v.close()
    # site-driven frames with the same obstacles
    sx, sy = jitter_sites(rng, Lx, Ly, 24.0)
    v = make(Lx, Ly, per, len(sx))
    v.vor_frame_options(4, False, d_obst, MAXLINK)
    cap = 16 * len(sx)
    hc = np.empty(cap, np.uint64); hd = np.empty(cap, np.uint64); cnt = np.zeros(3, np.int64)
    pe = np.empty(0, np.uint64)
    for t in range(3):
        v.vor_frame_host(sx, sy, hc, hd, cnt)
        e = oracle.edges_g(oracle.apply_obstacles(oracle.label_brute_g(Lx, Ly, per[0], per[1], sx, sy), obst, MAXLINK),
                           per[0], per[1], MAXLINK)
        rc, rd = oracle.diff(pe, e)
        assert cnt.tolist() == [len(e), len(rc), len(rd)], t
        assert np.array_equal(hc[:cnt[1]], rc) and np.array_equal(hd[:cnt[2]], rd)
        pe = e
        sx = np.clip(sx + rng.integers(-300, 300, len(sx)), 0, FP * Lx - 1).astype(np.int32)
        sy = ((sy.astype(np.int64) + rng.integers(-300, 300, len(sy))) % (FP * Ly)).astype(np.int32)
    v.vor_frame_options(4, False, None, -1)
    v.close()
    with pytest.raises(Exception):
        make(64, 64, (1, 1), 8).vor_frame_options(6, False, None, -1)


def test_merge_lists_many_lists_empty_lists_and_capacity(G):
    rng = np.random.default_rng(91)
    v = make(1024, 1024, (1, 1), 4096, max_raw_keys=1 << 20)
    for n_lists, stride in ((1, 5000), (2, 3000), (7, 2000), (16, 1500), (33, 700), (64, 64)):
        lists = torch.zeros(n_lists, stride, dtype=torch.int64, device="cuda")
        counts = torch.zeros(n_lists, dtype=torch.int64, device="cuda")
        parts = []
        for l in range(n_lists):
            m = 0 if l % 5 == 3 else int(rng.integers(1, stride + 1))
            i = rng.integers(0, 4000, m); j = rng.integers(0, 4000, m)
            ok = i != j
            keys = np.unique((np.minimum(i, j)[ok].astype(np.uint64) << np.uint64(32)) | np.maximum(i, j)[ok].astype(np.uint64))
            lists[l, : len(keys)] = torch.from_numpy(keys.view(np.int64)).cuda()
            counts[l] = len(keys)
            parts.append(keys)
        counts[0] = counts[0] + (stride if n_lists == 7 else 0)          # a count above the buffer is clamped
        if n_lists == 7:
            parts[0] = lists[0].cpu().numpy().view(np.uint64)[:stride]
            lists[0] = torch.sort(lists[0]).values                        # keep the clamped list ascending
            parts[0] = lists[0].cpu().numpy().view(np.uint64)
        ref = np.unique(np.concatenate(parts))
        out = torch.full((len(ref) + 3,), -5, dtype=torch.int64, device="cuda")
        n_out = torch.zeros(1, dtype=torch.int64, device="cuda")
        v.vor_merge_lists(lists, counts, 4096, out[: len(ref)], n_out)
        if n_lists == 7:                               # the truncated list is reported on the merging side too
            with pytest.raises(Exception, match="ECAPACITY"):
                v.vor_sync_status()
        else:
            v.vor_sync_status()
        assert int(n_out.item()) == len(ref) and np.array_equal(G.u64(out, len(ref)), ref), n_lists
        assert (out[len(ref):] == -5).all()
        if len(ref) > 10:                                                 # too small an output: required count + status
            v.vor_merge_lists(lists, counts, 4096, out[:10], n_out)
            with pytest.raises(Exception, match="ECAPACITY"):
                v.vor_sync_status()
            assert int(n_out.item()) == len(ref) and np.array_equal(G.u64(out, 10), ref[:10])
    v.close()
