"""The seeded generators: determinism, ranges and the workload structure DESIGN.md states."""
import numpy as np

from paper_1607_00908_b200 import workloads as W

FP = 256


def test_site_configs_shapes_ranges_determinism():
    for i in (1, 2):
        w = W.config(i)
        a = list(w.frames(3)); b = list(w.frames(3))
        for (ax, ay), (bx, by) in zip(a, b):
            assert ax.dtype == np.int32 and ax.shape == (w.n_sites,)
            assert np.array_equal(ax, bx) and np.array_equal(ay, by)
            assert ax.min() >= 0 and ax.max() < FP * w.L and ay.min() >= 0 and ay.max() < FP * w.L
        assert not np.array_equal(a[0][0], a[1][0])


def test_config2_min_separation():
    w = W.config(2)
    x, y = w.initial_positions()
    from scipy.spatial import cKDTree
    d, _ = cKDTree(np.stack([x, y], 1), boxsize=w.L).query(np.stack([x, y], 1), k=2)
    assert d[:, 1].min() >= 18.0 and len(x) == 2000


def test_config5_scaled_structure():
    w = W.scaled(5, 1024)
    assert w.n_sites == 62 * 62 or w.n_sites == 63 * 63
    sx, sy = next(iter(w.frames(1)))
    # jittered grid: one site per grid square
    sp = w.L / w.grid
    gx = np.floor(sx / FP / sp).astype(int) % w.grid
    gy = np.floor(sy / FP / sp).astype(int) % w.grid
    assert len(np.unique(gy * w.grid + gx)) == w.n_sites
    w5 = W.config(5)
    assert w5.L == 16384 and w5.n_sites == 10**6 and abs(w5.noise_sigma - 0.2 * 16.384) < 1e-12


def test_field_configs_small():
    w = W.scaled(3, 256)
    f = list(w.frames(2))
    assert f[0].dtype == np.float32 and f[0].shape == (256, 256)
    assert 0.85 < f[0].std() < 1.15
    frac = (f[0] > w.threshold).mean()
    assert 0.08 < frac < 0.25
    assert np.array_equal(f[0], next(iter(w.frames(1))))
    w = W.scaled(4, 512)
    g = list(w.frames(2))
    assert g[0].shape == (512, 512) and g[0].min() >= 0.1 - 1e-6 and g[0].max() <= 1.0 + 1e-6
    x, y, r = w.disc_geometry(0)
    area = (g[0] > w.threshold).sum()
    assert abs(area - np.pi * (r ** 2).sum()) < 0.03 * area       # threshold sits on the disc edge (R20)
