"""B200-native positively-split Ewald (PSE) grand mobility with stresslets (arXiv 1709.06946).

The product is libpse.so (hand-written CUDA for sm_100a + cuFFT for the bare transform) behind the C ABI of
include/pse.h; this package is its thin ctypes binding.  Importing it requires the built library:
    python paper_1709_06946_b200/build.py
"""
from .binding import (Context, PSEError, pse_create, pse_suggest_params, pse_version, pse_hard_sphere_forces_noalloc, PSE_NOALLOC_MAX_N, EXPORTS, LIB_PATH, PHASES,  # noqa: F401
                      PSE_OK, PSE_EINVAL, PSE_ENOMEM, PSE_ECUDA, PSE_ECUFFT, PSE_ENOTREADY, PSE_ENOCONV, PSE_EOVERFLOW,
                      PSE_REAL, PSE_WAVE, PSE_BOTH, PSE_WINDOW_GAUSS, PSE_WINDOW_ES)
