"""Shared test constructions (geometry only; no method arithmetic)."""
import math
import os

import numpy as np

FP = 256
GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def read_golden(name):
    out = {}
    with open(os.path.join(GOLDEN, name)) as f:
        for line in f:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            k, *v = line.split()
            out[k] = [float(t) if "." in t else int(t) for t in v]
    return out


def fixed(v, L):
    P = FP * L
    return (np.floor(np.asarray(v, dtype=np.float64) * FP + 0.5).astype(np.int64) % P).astype(np.int32)


def rhombus_sites(L, h):
    """The single-flip construction of tests/golden/rhombus_flip.txt."""
    c = L / 2
    pts = [(c - 24, c), (c, c + h), (c + 24, c), (c, c - h)]
    for k in range(10):
        a = 2 * math.pi * (k + 0.37) / 10
        pts.append((c + 88 * math.cos(a), c + 88 * math.sin(a)))
    return fixed([p[0] for p in pts], L), fixed([p[1] for p in pts], L)


def hex_sites(L, cols, rows, jitter, seed=0):
    """Perturbed triangular lattice of tests/golden/hex_lattice.txt."""
    rng = np.random.default_rng(seed)
    ax, ay = L / cols, L / rows
    ix, iy = np.meshgrid(np.arange(cols), np.arange(rows), indexing="xy")
    x = (ix + 0.25 + 0.5 * (iy % 2)) * ax + rng.uniform(-jitter, jitter, ix.shape)
    y = (iy + 0.5) * ay + rng.uniform(-jitter, jitter, iy.shape)
    return fixed(np.mod(x.ravel(), L), L), fixed(np.mod(y.ravel(), L), L)


def pairs(keys):
    keys = np.asarray(keys, dtype=np.uint64)
    i = (keys >> np.uint64(32)).astype(np.int64)
    j = (keys & np.uint64(0xffffffff)).astype(np.int64)
    return set(zip(i.tolist(), j.tolist()))


def pack(pair_list):
    return np.array(sorted((i << 32) | j for i, j in pair_list), dtype=np.uint64)
