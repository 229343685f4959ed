"""One lattice sharded over the ranks of a torch.distributed group by row strips (
the paper lists a multi-GPU implementation as future work).

Labelling is a pure function of (cell, site list): every rank holds all sites (8 B per site, replicated by the
caller or by `broadcast_sites`), labels the rows of its strip plus the FIRST ROW OF THE NEXT STRIP - recomputed
locally, so there is no halo exchange - and extracts the edge keys of that image without a wrap in y.  The
union of the strips' lists is the lattice's list: one all-gather of the fixed-capacity list buffers and their
counts (NCCL over NVLink on GPUs), then a merge-unique on every rank (`vor_merge_lists`).  The frame-to-frame
comparison then runs on the replicated list as on one GPU.

Every step of the path runs in libvor's kernels through the object `vor` (binding.Vor); this module only
partitions rows and moves buffers.  The arithmetic-free host logic (partition, gather, merge order) is covered
on CPU by tests/test_strips_ranks.py with the gloo backend and a stand-in for `vor`.
"""
from __future__ import annotations

import torch
import torch.distributed as dist


def strip_rows(Ly: int, world: int, rank: int, align: int = 32):
    """Rows [y0, y1) of rank `rank`: a balanced partition whose cuts fall on multiples of `align` rows (the
    labelling kernel's tile height) wherever the lattice is tall enough; a rank may get no rows at all."""
    if world < 1 or not 0 <= rank < world:
        raise ValueError("rank outside the group")
    units = (Ly + align - 1) // align
    cut = lambda r: min(Ly, ((units * r) // world) * align)
    return cut(rank), (Ly if rank == world - 1 else cut(rank + 1))


def broadcast_sites(sx, sy, src: int = 0, group=None):
    """Replicate the site arrays of rank `src` ("replicate the site arrays: one broadcast")."""
    dist.broadcast(sx, src, group=group)
    dist.broadcast(sy, src, group=group)


class StripFrame:
    """Edge list of one frame of an Lx x Ly lattice, computed by all ranks of `group` together.

    vor: the rank's libvor context for the WHOLE lattice geometry (or a stand-in with the same methods);
    cap_strip: capacity of one rank's key list (every rank the same: the all-gather moves fixed-size buffers
    and the counts, so no rank waits for a size on the host); cap: capacity of the merged list."""

    def __init__(self, vor, n_sites: int, cap_strip: int, cap: int, group=None, device="cuda", rank=None, world=None):
        self.vor, self.group, self.device = vor, group, torch.device(device)
        live = dist.is_available() and dist.is_initialized()
        # rank / world may be given explicitly to compute one strip of a decomposition without a process group
        self.world = world if world is not None else (dist.get_world_size(group) if live else 1)
        self.rank = rank if rank is not None else (dist.get_rank(group) if live else 0)
        self.collective = live and world is None
        self.n_sites = n_sites
        self.y0, self.y1 = strip_rows(vor.Ly, self.world, self.rank)
        self.rows = self.y1 - self.y0
        # the extra row: the next strip's first row; below the last strip it is row 0 of a periodic lattice
        self.extra = 0 if self.rows == 0 else (1 if self.y1 < vor.Ly or vor.periodic[1] else 0)
        i32 = dict(dtype=torch.int32, device=self.device)
        i64 = dict(dtype=torch.int64, device=self.device)
        self.labels = torch.empty(max(1, (self.rows + self.extra) * vor.Lx), **i32)
        self.local = torch.zeros(cap_strip, **i64)
        self.n_local = torch.zeros(1, **i64)
        self.gathered = torch.zeros(self.world, cap_strip, **i64)
        self.counts = torch.zeros(self.world, **i64)
        self.edges = torch.empty(cap, **i64)
        self.n_edges = torch.zeros(1, **i64)

    def compute_local(self, sx, sy, exclude: int = -1):
        """This rank's part: labels of its rows (+ the extra row) and their key list -> (local, n_local)."""
        v, Lx = self.vor, self.vor.Lx
        v.vor_build_cells(sx, sy)
        if self.rows > 0:
            own = self.labels[: self.rows * Lx]
            v.vor_label_rows(self.y0, self.rows, own)
            if self.extra:
                v.vor_label_rows(self.y1 if self.y1 < v.Ly else 0, 1, self.labels[self.rows * Lx:(self.rows + 1) * Lx])
            v.vor_edges_image(self.labels[: (self.rows + self.extra) * Lx], False, exclude, self.local, self.n_local)
        else:
            self.n_local.zero_()
        return self.local, self.n_local

    def compute(self, sx, sy, exclude: int = -1):
        """sx, sy: ALL sites (replicated).  Returns (edges, n_edges): the lattice's ascending unique key list,
        identical on every rank, in this object's buffers."""
        v = self.vor
        self.compute_local(sx, sy, exclude)
        if self.collective and self.world > 1:
            dist.all_gather_into_tensor(self.gathered, self.local.unsqueeze(0), group=self.group)
            dist.all_gather_into_tensor(self.counts, self.n_local, group=self.group)
        elif self.world == 1:
            self.gathered.copy_(self.local.unsqueeze(0))
            self.counts.copy_(self.n_local)
        else:
            raise RuntimeError("StripFrame.compute needs a process group for world > 1")
        v.vor_merge_lists(self.gathered, self.counts, self.n_sites, self.edges, self.n_edges)
        return self.edges, self.n_edges
