"""paper_2606_15846_b200 -- B200-native batched navigation-simulator step of FlashNav.

Thin Python binding over the C-ABI library `libflashnav.so` (include/flashnav.h): argument
marshalling only; every step of the hot path runs in the library's CUDA kernels.  PyTorch supplies
device memory and the stream.  There is no CPU fallback: a missing library or device raises.
"""
from ._binding import (FlashNavError, Map, Robot, Sim, DRIVE_DIFF, DRIVE_OMNI, N_COUNTERS, COUNTER_NAMES,
                       load_library, measure_peak, library_path, EXPORTED_SYMBOLS, observe_noalloc, NOALLOC_MAX_ENVS)

__all__ = ["FlashNavError", "Map", "Robot", "Sim", "DRIVE_DIFF", "DRIVE_OMNI", "N_COUNTERS",
           "COUNTER_NAMES", "load_library", "measure_peak", "library_path", "EXPORTED_SYMBOLS",
           "observe_noalloc", "NOALLOC_MAX_ENVS"]
