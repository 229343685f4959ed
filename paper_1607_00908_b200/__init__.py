"""B200-native hot path of arXiv:1607.00908 (Voronoi topological-change detection).

The product is the C-ABI library libvor.so (include/vor.h, csrc/*.cu); `binding.Vor` marshals torch
tensors into it.  `workloads` holds the seeded synthetic input generators (no method arithmetic).
"""
from . import workloads  # noqa: F401

__all__ = ["workloads", "binding", "build"]
