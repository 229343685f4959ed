"""Seeded synthetic input generators for the five BASELINE.json configs.

This module holds NONE of the method's arithmetic (no distances to sites, no
labelling, no edges, no CCL): it only draws site positions / scalar fields.
Both the CUDA path and the CPU oracle consume the arrays produced here, so
generator rounding is never a parity concern.

The inputs stand in for the paper's LBM emulsion frames (§IV) and
its "bubbles from a random field" demo (§I); neither is available.
Readings R17-R21 of SURVEY.md §8c (restated in DESIGN.md) fix the details.

Fixed point: 1 lattice unit = 256 fixed-point units (FP_ONE); a coordinate v
(float64, lattice units) becomes floor(v*256 + 0.5) mod (256*L), int32.
"""
from __future__ import annotations

import dataclasses
from typing import Iterator, Tuple

import numpy as np

FP_ONE = 256
BASE_SEED = 160700908


def to_fixed(v: np.ndarray, L: int) -> np.ndarray:
    """float64 lattice coordinates -> int32 fixed point in [0, 256*L)."""
    P = FP_ONE * L
    q = np.floor(np.asarray(v, dtype=np.float64) * FP_ONE + 0.5).astype(np.int64)
    return np.mod(q, P).astype(np.int32)


# --------------------------------------------------------------------------
# site-driven workloads (configs 1, 2, 5)
# --------------------------------------------------------------------------

@dataclasses.dataclass
class SiteWorkload:
    """A sequence of frames of N persistent sites on an L x L periodic lattice."""
    name: str
    L: int
    n_sites: int
    n_frames: int
    seed: int
    kind: str                      # 'uniform' | 'poisson_disk' | 'jittered_grid'
    noise_sigma: float             # per-frame Gaussian displacement, lattice units
    shear: float = 0.0             # per-frame affine increment x += shear * y
    min_sep: float = 0.0           # poisson_disk only
    grid: int = 0                  # jittered_grid only: grid x grid sites
    jitter: float = 0.0            # jittered_grid only: +- fraction of spacing
    bucket_cells: int = 16         # suggested cell-list bucket side

    def initial_positions(self) -> Tuple[np.ndarray, np.ndarray]:
        rng = np.random.default_rng(self.seed)
        L = self.L
        if self.kind == "uniform":
            x = rng.uniform(0.0, L, self.n_sites)
            y = rng.uniform(0.0, L, self.n_sites)
        elif self.kind == "poisson_disk":
            x, y = _poisson_disk(rng, L, self.n_sites, self.min_sep)
        elif self.kind == "jittered_grid":
            g = self.grid
            assert g * g == self.n_sites
            sp = L / g
            gx, gy = np.meshgrid(np.arange(g, dtype=np.float64),
                                 np.arange(g, dtype=np.float64), indexing="xy")
            x = (gx.ravel() + 0.5 + rng.uniform(-self.jitter, self.jitter, g * g)) * sp
            y = (gy.ravel() + 0.5 + rng.uniform(-self.jitter, self.jitter, g * g)) * sp
        else:
            raise ValueError(self.kind)
        return np.mod(x, L), np.mod(y, L)

    def frames(self, n_frames: int | None = None) -> Iterator[Tuple[np.ndarray, np.ndarray]]:
        """Yield (sx, sy) int32 fixed-point arrays, one pair per frame.

        Frame t = frame t-1 sheared (R17: on the current wrapped positions) plus
        fresh Gaussian noise (R18: cumulative random walk), wrapped mod L.
        """
        n_frames = self.n_frames if n_frames is None else n_frames
        x, y = self.initial_positions()
        rng = np.random.default_rng(self.seed + 7919)
        for t in range(n_frames):
            if t > 0:
                if self.shear != 0.0:
                    x = x + self.shear * y
                x = x + rng.normal(0.0, self.noise_sigma, x.shape)
                y = y + rng.normal(0.0, self.noise_sigma, y.shape)
                x = np.mod(x, self.L)
                y = np.mod(y, self.L)
            yield to_fixed(x, self.L), to_fixed(y, self.L)


def _poisson_disk(rng, L: int, n: int, sep: float):
    """Plain periodic dart throwing with a background grid (R21)."""
    cell = sep / np.sqrt(2.0)
    ng = int(np.floor(L / cell))
    cell = L / ng
    grid = -np.ones((ng, ng), dtype=np.int64)
    xs = np.empty(n)
    ys = np.empty(n)
    k = 0
    sep2 = sep * sep
    tries = 0
    while k < n:
        tries += 1
        if tries > 200 * n + 100000:
            raise RuntimeError("poisson disk saturated before reaching n sites")
        px, py = rng.uniform(0.0, L, 2)
        gx, gy = int(px / cell) % ng, int(py / cell) % ng
        ok = True
        for oy in range(-2, 3):
            for ox in range(-2, 3):
                j = grid[(gy + oy) % ng, (gx + ox) % ng]
                if j >= 0:
                    dx = abs(px - xs[j]); dx = min(dx, L - dx)
                    dy = abs(py - ys[j]); dy = min(dy, L - dy)
                    if dx * dx + dy * dy < sep2:
                        ok = False
                        break
            if not ok:
                break
        if ok:
            xs[k], ys[k] = px, py
            grid[gy, gx] = k
            k += 1
    return xs, ys


# --------------------------------------------------------------------------
# field-driven workloads (configs 3, 4)
# --------------------------------------------------------------------------

@dataclasses.dataclass
class FieldWorkload:
    """A sequence of float32 L x L scalar fields (row-major, x fastest)."""
    name: str
    L: int
    n_frames: int
    seed: int
    kind: str                      # 'gaussian_field' | 'emulsion'
    threshold: float
    min_size: int = 20
    match_radius_cells: float = 4.0
    corr_len: float = 8.0          # gaussian_field
    white_noise: float = 0.05      # gaussian_field: per-frame additive noise
    grid_x: int = 0                # emulsion: triangular lattice columns
    grid_y: int = 0                # emulsion: triangular lattice rows
    r_min: float = 8.0
    r_max: float = 14.0
    shear: float = 0.001           # emulsion: strain per frame
    bucket_cells: int = 32

    # ---- gaussian random field (config 3, R19) ----
    def _base_spectrum(self):
        rng = np.random.default_rng(self.seed)
        L = self.L
        w = rng.standard_normal((L, L))
        k = 2.0 * np.pi * np.fft.fftfreq(L)
        k2 = k[:, None] ** 2 + k[None, :] ** 2
        filt = np.exp(-k2 * self.corr_len ** 2 / 4.0)
        spec = np.fft.fft2(w) * filt
        g = np.real(np.fft.ifft2(spec))
        spec /= g.std()
        return spec, k

    # ---- emulsion discs (config 4, R20) ----
    def _emulsion_setup(self):
        rng = np.random.default_rng(self.seed)
        L, gx, gy = self.L, self.grid_x, self.grid_y
        ax, ay = L / gx, L / gy
        ix, iy = np.meshgrid(np.arange(gx), np.arange(gy), indexing="xy")
        x0 = (ix + 0.25 + 0.5 * (iy % 2)) * ax + rng.uniform(-1.0, 1.0, ix.shape)
        y0 = (iy + 0.5) * ay + rng.uniform(-1.0, 1.0, iy.shape)
        x0, y0 = np.mod(x0.ravel(), L), np.mod(y0.ravel(), L)
        r = rng.uniform(self.r_min, self.r_max, x0.shape)
        # cap radii so r_i + r_j + 2 <= d_ij: r_i <= (nearest-neighbour distance - 2) / 2
        dmin = _nearest_neighbour_dist(x0, y0, L)
        r = np.minimum(r, (dmin - 2.0) / 2.0)
        # rows next to the y seam slide past each other under plain-wrap shear: keep them slim
        seam = (iy.ravel() == 0) | (iy.ravel() == gy - 1)
        r = np.where(seam, np.minimum(r, (ay - 4.0) / 2.0 - 1.0), r)
        return x0, y0, r

    def frames(self, n_frames: int | None = None) -> Iterator[np.ndarray]:
        n_frames = self.n_frames if n_frames is None else n_frames
        L = self.L
        if self.kind == "gaussian_field":
            spec, k = self._base_spectrum()
            rng = np.random.default_rng(self.seed + 7919)
            s = np.zeros(2)
            for t in range(n_frames):
                if t > 0:
                    s = s + rng.uniform(-0.5, 0.5, 2)
                phase = np.exp(-1j * (k[None, :] * s[0] + k[:, None] * s[1]))
                g = np.real(np.fft.ifft2(spec * phase))
                g = g + self.white_noise * rng.standard_normal((L, L))
                yield np.ascontiguousarray(g, dtype=np.float32)
        elif self.kind == "emulsion":
            x0, y0, r = self._emulsion_setup()
            for t in range(n_frames):
                x = np.mod(x0 + self.shear * t * y0, L)
                yield render_discs(L, x, y0, r)
        else:
            raise ValueError(self.kind)

    def disc_geometry(self, t: int = 0):
        """(x, y, r) of the emulsion droplets at frame t (for tests and stats)."""
        x0, y0, r = self._emulsion_setup()
        return np.mod(x0 + self.shear * t * y0, self.L), y0, r


def _nearest_neighbour_dist(x, y, L):
    from scipy.spatial import cKDTree
    pts = np.stack([np.mod(x, L), np.mod(y, L)], axis=1)
    # guard against values that round to exactly L
    pts = np.minimum(pts, np.nextafter(float(L), 0.0))
    tree = cKDTree(pts, boxsize=float(L))
    d, _ = tree.query(pts, k=2)
    return d[:, 1]


def render_discs(L: int, x, y, r, width: float = 2.0, rho_in: float = 1.0,
                 rho_out: float = 0.1, cutoff: float = 16.0) -> np.ndarray:
    """rho = rho_out + (rho_in-rho_out) * max_i 0.5*(1 - tanh((|p-c_i| - R_i)/width)).

    p = cell centre (integer + 0.5), minimum-image distance, `max` (not sum) so that
    the mid level sits exactly on each disc's edge (R20).
    """
    prof = np.zeros((L, L), dtype=np.float64)
    for cx, cy, rr in zip(x, y, r):
        h = rr + cutoff
        ix0, ix1 = int(np.floor(cx - h)), int(np.ceil(cx + h))
        iy0, iy1 = int(np.floor(cy - h)), int(np.ceil(cy + h))
        xs = np.arange(ix0, ix1 + 1)
        ys = np.arange(iy0, iy1 + 1)
        dx = (xs + 0.5) - cx
        dy = (ys + 0.5) - cy
        d = np.sqrt(dy[:, None] ** 2 + dx[None, :] ** 2)
        v = 0.5 * (1.0 - np.tanh((d - rr) / width))
        rows = np.mod(ys, L)[:, None]
        cols = np.mod(xs, L)[None, :]
        assert len(xs) <= L and len(ys) <= L, "disc patch wraps onto itself"
        prof[rows, cols] = np.maximum(prof[rows, cols], v)
    return (rho_out + (rho_in - rho_out) * prof).astype(np.float32)


# --------------------------------------------------------------------------
# the five configs (BASELINE.json `configs`, in order) and scaled-down copies
# --------------------------------------------------------------------------

def config(i: int):
    """Config i in 1..5 at BASELINE.json's full size."""
    seed = BASE_SEED + i
    if i == 1:
        return SiteWorkload("cfg1_tiny_uniform", 64, 32, 2, seed, "uniform", 0.5, bucket_cells=8)
    if i == 2:
        return SiteWorkload("cfg2_sheared_packing", 1024, 2000, 100, seed, "poisson_disk", 0.3,
                            shear=0.002, min_sep=18.0, bucket_cells=16)
    if i == 3:
        return FieldWorkload("cfg3_random_field_bubbles", 2048, 50, seed, "gaussian_field",
                             threshold=1.0, bucket_cells=32)
    if i == 4:
        return FieldWorkload("cfg4_emulsion", 4096, 20, seed, "emulsion", threshold=0.55,
                             grid_x=132, grid_y=152, bucket_cells=16)
    if i == 5:
        g = 1000
        return SiteWorkload("cfg5_throughput_stress", 16384, g * g, 10, seed, "jittered_grid",
                            0.2 * (16384 / g), grid=g, jitter=0.4, bucket_cells=16)
    raise ValueError(i)


def scaled(i: int, L: int):
    """Config i shrunk to an L x L lattice at the same site density / structure."""
    w = config(i)
    f = L / w.L
    if isinstance(w, SiteWorkload):
        if w.kind == "jittered_grid":
            g = max(2, int(round(w.grid * f)))
            return dataclasses.replace(w, name=f"{w.name}_L{L}", L=L, grid=g, n_sites=g * g,
                                       noise_sigma=0.2 * (L / g))
        n = max(1, int(round(w.n_sites * f * f)))
        return dataclasses.replace(w, name=f"{w.name}_L{L}", L=L, n_sites=n)
    if w.kind == "emulsion":
        gx = max(2, int(round(w.grid_x * f)))
        gy = max(2, 2 * int(round(w.grid_y * f / 2)))     # even, so the stagger closes
        return dataclasses.replace(w, name=f"{w.name}_L{L}", L=L, grid_x=gx, grid_y=gy)
    return dataclasses.replace(w, name=f"{w.name}_L{L}", L=L)
