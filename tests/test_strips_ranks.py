"""Row-strip sharding of ONE lattice: the host logic of
paper_1607_00908_b200/strips.py on CPU - the row partition, the extra row, the all-gather of fixed-capacity
lists over gloo (world size 2 and 3) and the order of the merge - with a stand-in for the libvor context whose
methods are the oracle's definitions (test infrastructure; the product path has no such fallback)."""
import os
import sys

import numpy as np
import pytest

torch = pytest.importorskip("torch")
import torch.distributed as dist  # noqa: E402
import torch.multiprocessing as mp  # noqa: E402

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

from paper_1607_00908_b200.strips import StripFrame, strip_rows  # noqa: E402


def test_strip_rows_partition():
    for Ly in (1, 31, 32, 33, 64, 100, 1024, 16384, 1000):
        for world in (1, 2, 3, 5, 8, 64):
            cuts = [strip_rows(Ly, world, r) for r in range(world)]
            assert cuts[0][0] == 0 and cuts[-1][1] == Ly
            assert all(a[1] == b[0] for a, b in zip(cuts[:-1], cuts[1:]))          # contiguous, no overlap
            assert all(y0 <= y1 for y0, y1 in cuts)
            assert all(y0 % 32 == 0 for y0, _ in cuts)                             # cuts on tile rows
            sizes = [y1 - y0 for y0, y1 in cuts]
            if Ly >= 32 * world:
                assert max(sizes) - min(sizes) <= 32 + 31                          # balanced up to one tile row
    with pytest.raises(ValueError):
        strip_rows(64, 2, 2)


class OracleVor:
    """Stand-in for binding.Vor on CPU tensors: the same method names, computed by the oracle."""

    def __init__(self, Lx, Ly, periodic):
        import oracle
        self.o, self.Lx, self.Ly, self.periodic = oracle, Lx, Ly, periodic
        self.full = None

    def vor_build_cells(self, sx, sy):
        self.full = self.o.label_brute_g(self.Lx, self.Ly, self.periodic[0], self.periodic[1], sx.numpy(), sy.numpy())

    def vor_label_rows(self, y0, n_rows, out):
        out.copy_(torch.from_numpy(self.full[y0:y0 + n_rows].ravel().copy()))

    def vor_edges_image(self, labels, wrap_y, exclude, edges, n_edges, row_ptr=None):
        img = labels.numpy().reshape(-1, self.Lx)
        keys = self.o.edges_g(img, self.periodic[0], 1 if wrap_y else 0, exclude)
        edges[: len(keys)] = torch.from_numpy(keys.view(np.int64))
        n_edges[0] = len(keys)

    def vor_merge_lists(self, lists, counts, n_labels, out, n_out):
        parts = [lists[l, : int(counts[l])].numpy().view(np.uint64) for l in range(lists.shape[0])]
        keys = np.unique(np.concatenate(parts))
        out[: len(keys)] = torch.from_numpy(keys.view(np.int64))
        n_out[0] = len(keys)


def sites(Lx, Ly, n, seed):
    rng = np.random.default_rng(seed)
    return (torch.from_numpy(rng.integers(0, 256 * Lx, n).astype(np.int32)),
            torch.from_numpy(rng.integers(0, 256 * Ly, n).astype(np.int32)))


def _worker(rank, world, port, Lx, Ly, periodic, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        from paper_1607_00908_b200.strips import broadcast_sites
        sx, sy = sites(Lx, Ly, 60, 7) if rank == 0 else (torch.zeros(60, dtype=torch.int32), torch.zeros(60, dtype=torch.int32))
        broadcast_sites(sx, sy, 0)                                                 # only rank 0 knows the sites
        f = StripFrame(OracleVor(Lx, Ly, periodic), 60, cap_strip=4096, cap=8192, device="cpu")
        e, n = f.compute(sx, sy)
        out[rank] = dict(rows=(f.y0, f.y1), extra=f.extra, local=int(f.n_local), counts=f.counts.tolist(),
                         edges=e[: int(n)].numpy().view(np.uint64).tolist())
        dist.barrier()
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world,Lx,Ly,periodic", [(2, 96, 128, (1, 1)), (3, 64, 160, (0, 1)), (2, 80, 96, (1, 0)), (3, 64, 64, (1, 1))])
def test_strips_over_gloo_give_the_lattice_list_on_every_rank(world, Lx, Ly, periodic):
    import oracle
    port = 29600 + (os.getpid() + 7 * world + Lx) % 2000
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, port, Lx, Ly, periodic, out), nprocs=world, join=True)
        res = [out[r] for r in range(world)]
    sx, sy = sites(Lx, Ly, 60, 7)
    ref = oracle.edges_g(oracle.label_brute_g(Lx, Ly, periodic[0], periodic[1], sx.numpy(), sy.numpy()), periodic[0], periodic[1])
    for r in res:
        assert r["edges"] == ref.tolist()                                          # identical on every rank
        assert r["counts"] == [q["local"] for q in res]                            # the gathered counts
    assert res[0]["rows"][0] == 0 and res[-1]["rows"][1] == Ly
    # every non-empty strip but the last carries the next strip's first row; the last one row 0 of a periodic lattice
    assert [r["extra"] for r in res[:-1]] == [int(r["rows"][1] > r["rows"][0]) for r in res[:-1]]
    assert res[-1]["extra"] == periodic[1]
    assert sum(r["local"] for r in res) >= len(ref)                                # strips overlap in their seam rows


def test_single_process_strip_is_the_whole_lattice():
    import oracle
    Lx, Ly = 64, 96
    sx, sy = sites(Lx, Ly, 40, 3)
    for periodic in ((1, 1), (1, 0)):
        f = StripFrame(OracleVor(Lx, Ly, periodic), 40, cap_strip=4096, cap=4096, device="cpu")
        e, n = f.compute(sx, sy)
        ref = oracle.edges_g(oracle.label_brute_g(Lx, Ly, periodic[0], periodic[1], sx.numpy(), sy.numpy()), periodic[0], periodic[1])
        assert e[: int(n)].numpy().view(np.uint64).tolist() == ref.tolist() and f.extra == periodic[1]
