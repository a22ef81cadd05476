"""afs-b200: batched Walsh-Fourier projected gradient descent for symmetric pseudo-Boolean SAT on NVIDIA B200.

The product is ``libafs_b200.so`` (``csrc/``, C ABI in ``include/afs.h``); this package is its ctypes binding.
"""
from .binding import (  # noqa: F401
    AFS_OR, AFS_XOR, AFS_AMO, AFS_EO, AFS_EK, AFS_NAE, AFS_CARD,
    AfsError, Problem, coeffs, fp32_fma_peak, lib, EXPORTS, LIB_PATH,
)
