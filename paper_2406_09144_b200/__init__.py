"""fast-resolve hot path on B200: thin Python binding of libfrs.so (see include/frs.h).

The package only marshals arguments (torch tensors -> device pointers); every step of the path
runs in the CUDA kernels of libfrs.so.  There is no CPU fallback: if the library is missing or no
CUDA device is present, calls raise.
"""
from .binding import (FrsError, Context, lib, load_library, selftest_fft_host, selftest_tma_geometry, selftest_dif_host, selftest_dif_exchange, selftest_tcgen05_stage, EXPORTS, dot_noalloc, FRS_DOT_NOALLOC_MAX_N,  # noqa: F401
                      FRS_OK, FRS_EINVAL, FRS_ESTATE, FRS_ENOTPSD, FRS_ECUDA, FRS_EBREAKDOWN)
