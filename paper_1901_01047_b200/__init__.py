"""paper_1901_01047_b200 -- B200-native CT-AUX walker (DCA++ hot path, arXiv:1901.01047 sec. 2.3).

Thin Python binding over the C ABI of include/ctaux.h (libctaux_b200.so, hand-written sm_100a
CUDA).  Argument marshalling only: every step of the path runs in the CUDA kernels.  PyTorch is
used for device memory and streams.  There is no CPU fallback: if the extension cannot be loaded
or no CUDA device is present, calls fail loudly.
"""
from .binding import (CtauxError, Walkers, WalkerGroups, colmajor, ctaux_dgemm, debug_philox, exported_symbols, g0_table_from_sigma, g0_table_from_sigma_noalloc, lib_path, probe_fp64,
                      load_library, LOG_DTYPE, STEP_CLASSES)

__all__ = ["CtauxError", "Walkers", "WalkerGroups", "colmajor", "ctaux_dgemm", "debug_philox", "exported_symbols", "g0_table_from_sigma", "g0_table_from_sigma_noalloc", "lib_path", "probe_fp64",
           "load_library", "LOG_DTYPE", "STEP_CLASSES"]
