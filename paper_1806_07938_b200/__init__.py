"""paper_1806_07938_b200 -- B200-native FFT/Toeplitz MMSE tomographic wave-front reconstruction (arXiv:1806.07938).

The product is the C-ABI shared library `libtomo_b200.so` (include/tomo.h) built from csrc/ by build.py; `tomo.py`
is its thin ctypes binding.  Nothing here imports `oracle/`.
"""
from .tomo import (TOMO_F32, TOMO_F32S_F64A, TOMO_F64, TOMO_FRIED, TOMO_HUDGIN, TOMO_SOLVER_MULTIKERNEL,  # noqa: F401
                   TOMO_SOLVER_PERSISTENT, TomoError, TomoPlan, load)
