"""B200-native hot path of bosonic / xi-particle PIMD (arXiv 2404.02628).

`workloads` holds the seeded synthetic inputs; `binding` is the thin ctypes layer over the
C-ABI library `libpimd.so` built from csrc/ (see include/pimd.h).  There is no CPU fallback:
anything that computes raises if the CUDA library is missing.
"""
from . import workloads  # noqa: F401

__all__ = ["workloads", "binding"]
