"""B200-native Gadep photon-transport hot path (arxiv 2605.25963): thin ctypes binding over libgadep.so.

The Python layer only marshals arguments; every step of the path runs in the CUDA kernels of csrc/.
There is no CPU fallback: importing works without a GPU (symbols can be inspected), creating a context does not.
"""
from .binding import (Gadep, GadepError, load_library, library_path, EXPORTED_SYMBOLS, GadepCounters,
                      F_ESCAPED, F_PEAK, F_LEAK, F_NONSCORING, FILTER_NONE, MAT_KILL)

__all__ = ["Gadep", "GadepError", "load_library", "library_path", "EXPORTED_SYMBOLS", "GadepCounters",
           "F_ESCAPED", "F_PEAK", "F_LEAK", "F_NONSCORING", "FILTER_NONE", "MAT_KILL"]
