"""paper_2401_09843_b200 -- B200-native spectral hyperviscosity Navier-Stokes RHS + SSP-RK3 step.

The product is the C-ABI CUDA library `libns.so` (include/ns.h).  `binding` is a thin ctypes layer
with the same entry-point names; `inputs` holds the seeded synthetic workload generators.
"""
from . import inputs  # noqa: F401

__all__ = ["inputs", "binding", "build"]
