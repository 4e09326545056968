"""B200-native Crank-Nicolson / BiCGSTAB Dirac propagator (hot path of GaDE, arXiv 2512.21697).

The product is libtdde.so (C ABI in include/tdde.h, CUDA kernels in csrc/); this package holds the build script
and a ctypes binding with the same names.  It never imports ``oracle``.
"""
from .binding import Tdde, TddeGroup, nccl_unique_id, snorm_noalloc, snorm_noalloc_setup, NOALLOC_MAX_N, TddeError, eigensolve, load_library, EXPORTS, LIB_PATH, tdde_stats, tdde_config, tdde_term  # noqa: F401
