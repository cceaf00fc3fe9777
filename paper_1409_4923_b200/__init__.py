"""bm -- B200-native ensemble Langevin integrator for Brownian motors (after arXiv 1409.4923).

The product is the C-ABI library declared in include/bm.h (built from csrc/ into libbm.so); `binding`
holds the thin ctypes layer with the same names.  Nothing here falls back to a CPU implementation:
every compute call raises if the CUDA library is missing.
"""
from . import workloads  # noqa: F401  (parameter tables only; no arithmetic of the method)

__all__ = ["workloads"]
