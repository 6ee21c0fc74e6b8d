"""B200-native MPCD solvent step (arXiv 1801.10187): CUDA kernels behind a C ABI
(include/mpcd.h) with a thin ctypes binding.  No CPU fallback."""
from .binding import MPCD, MPCDError, load_library, test_philox, LIB_PATH, EXPORTS  # noqa: F401
