"""B200-native (sm_100a) PVFinder inference hot path behind the C ABI of include/pvf.h.

``binding`` is the thin ctypes layer (argument marshalling only); ``build`` compiles csrc/*.cu into
libpvf.so with nvcc.  There is no CPU fallback: the binding raises if the library is missing.
"""
from .binding import (PVFinder, PVFError, load_library, default_config, LIB_PATH, EXPORTS,
                      PVF_OK, PVF_ERR_ARG, PVF_ERR_CONFIG, PVF_ERR_CAPACITY, PVF_ERR_CUDA,
                      PVF_ERR_UNSUPPORTED, PRECISIONS, FLAG_PEAK_OVERFLOW, FLAG_TRACK_DROPPED,
                      FLAG_NONFINITE, FLAG_BAD_OFFSETS, N_INTERVALS, N_BINS, N_GLOBAL_BINS, MAX_PEAKS,
                      NOALLOC_MAX_EVENTS, NOALLOC_MAX_TRACKS)

__all__ = ["PVFinder", "PVFError", "load_library", "default_config", "LIB_PATH", "EXPORTS"]
