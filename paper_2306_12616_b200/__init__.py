"""paper_2306_12616_b200 -- B200-native dense Chebyshev Fermi-operator solver (arXiv 2306.12616).

Thin ctypes binding of the C ABI in include/cheb_dm.h: argument marshalling only, every step of the
path runs in the CUDA kernels of csrc/.  PyTorch is used by callers for device memory and streams;
this module takes raw device pointers (``tensor.data_ptr()``) and stream handles.

There is no CPU fallback: if libcheb_dm.so is missing (and cannot be built) importing the binding
functions raises; without a CUDA device ``Plan`` raises ChebDMError(ECUDA).
"""
from .binding import (  # noqa: F401
    ChebDMError, Options, Plan, lib, lib_path, dmma_peak, bounds_static, STATIC_MAX_N,
    OUTER_CHEBYSHEV, OUTER_POWER, SCHED_GROUPED, SCHED_SERIAL, PAIR_AUTO, PAIR_ALG1, PAIR_SERIAL, PAIR_BALANCED,
    TILE_AUTO, TILE_128x128, TILE_128x64, TILE_64x64, STATUS_NAMES, MAX_BATCH,
)
