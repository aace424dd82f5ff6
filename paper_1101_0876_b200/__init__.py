"""B200-native checkerboard Metropolis sweep of the 2D q-state Potts model (arXiv 1101.0876).

The product is the C-ABI library ``libpotts_b200.so`` (``include/potts.h``, sources in
``csrc/``); ``binding`` is a thin ctypes layer with the same names.  Importing this package
does not load the library; the first call does, and raises if it has not been built -- there
is no CPU fallback.
"""
from .binding import (  # noqa: F401
    ERR_ARG, ERR_CUDA, ERR_NOMEM, ERR_UNSUPPORTED, EXPORTED_SYMBOLS, INIT_ORDERED, INIT_RANDOM, LAYOUT_PACKED,
    LAYOUT_U8, LIB_PATH, OK, Potts, Potts3D, Potts8, PottsBatch, PottsError, load_library, potts_magnetisation, potts_observables,
    potts_susceptibility, potts_version, potts_workspace_bytes, potts_measure_noalloc, NOALLOC_MAX_L,
)

__all__ = [
    "Potts", "Potts3D", "Potts8", "PottsBatch", "PottsError", "load_library", "potts_observables", "potts_magnetisation", "potts_susceptibility", "potts_version",
    "potts_workspace_bytes", "INIT_ORDERED", "INIT_RANDOM", "LAYOUT_U8", "LAYOUT_PACKED", "LIB_PATH",
    "EXPORTED_SYMBOLS", "OK", "ERR_ARG", "ERR_UNSUPPORTED", "ERR_NOMEM", "ERR_CUDA", "potts_measure_noalloc", "NOALLOC_MAX_L",
]
