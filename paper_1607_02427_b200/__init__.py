"""paper_1607_02427_b200 -- B200-native DEM force field for rounded polytopes (arXiv:1607.02427).

The product is the C-ABI CUDA library libdem_b200.so (include/dem.h, sources in csrc/).  This package holds its
in-tree build step (build.py) and a thin ctypes binding (binding.py).  There is no CPU implementation here.
"""
from .binding import (DEM_F32, DEM_F64, DEM_OK, EXPORTS, EXPORTS_BENCH, Dem, DemError, from_state, lib)  # noqa: F401
from . import build  # noqa: F401  (module: build.build() compiles the library)
