"""B200-native Wilson-Dirac / Neuberger-Dirac operator (arXiv:1010.5636): hand-written CUDA kernels for sm_100a behind
the C-ABI library `libnd_b200.so` (include/nd_b200.h), with a thin ctypes binding.  See DESIGN.md."""
from .binding import (ERROR_NAMES, LIB_PATH, SIGNATURES, Context, NDError, cheb_coeffs, choose_l, heev, load_library, minmax_coeffs,  # noqa: F401
                      projector_error, shard_layout, dot_static, DOT_STATIC_MAX_SITES, DOT_STATIC_SCRATCH_BYTES)
