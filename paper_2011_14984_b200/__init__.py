"""paper_2011_14984_b200 -- B200-native (sm_100a) hot path of the HHS-FSI integrator (FROST,
arXiv 2011.14984): thin Python binding over the C-ABI library libfrost_b200.so.

Every step of the path runs in the CUDA kernels behind include/frost.h; this package only marshals
arguments (torch tensors -> device pointers).  There is no CPU fallback and no dependency on
oracle/: if the shared library is missing or no CUDA device is usable, calls raise.
"""
from .binding import (ACC, ACCUMULATE, GRAD, MUTUAL, Frost, FrostError, acc_noalloc, exported_symbols,
                      library_path, load_library, noalloc_max_n)

__all__ = ["ACC", "ACCUMULATE", "GRAD", "MUTUAL", "Frost", "FrostError", "acc_noalloc", "exported_symbols",
           "library_path", "load_library", "noalloc_max_n"]
