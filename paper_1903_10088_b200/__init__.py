"""paper_1903_10088_b200 -- B200-native OS-TV statistical iterative reconstruction (arxiv 1903.10088).

Thin ctypes binding over the C-ABI CUDA library ``libosiv.so`` (``include/osiv.h``).  Every step of
the method runs in the CUDA kernels of ``csrc/``; this package only marshals arguments.  There is no
CPU fallback: importing works anywhere, but every compute call raises ``OsivError`` without a CUDA
device, and loading raises if the library has not been built (``python -m paper_1903_10088_b200.build``).
"""
from .binding import (  # noqa: F401
    Geometry, Params, Handle, OsivError, lib, lib_path, version, strerror, default_params, ray_table, probe_peaks, debug_checks,
    OSIV_OK, OSIV_ERR_INVALID_ARG, OSIV_ERR_CUDA, OSIV_ERR_NOT_FINITE, OSIV_ERR_SCRATCH_LIMIT, STATIC_SCRATCH_BYTES,
    EXPORTED_SYMBOLS,
)
