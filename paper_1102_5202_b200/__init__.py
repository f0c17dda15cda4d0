"""B200-native HORIZON GRMHD update: thin Python binding of the C-ABI library libhz.so (include/hz.h).

Argument marshalling only; every step of the path runs in the CUDA kernels of csrc/.  There is no CPU
fallback: importing works without a GPU (so the build can be checked), but creating a context fails
loudly if the library or a CUDA device is missing.
"""
from .binding import (HZ_BC_OUTFLOW, HZ_BC_PERIODIC, HZ_F32, HZ_F32_F64, HZ_F64, Horizon, HzDiag, HzError, HzGrid, HzParams,
                      lib, lib_path)  # noqa: F401
from .slab import DistSlabHorizon, SlabGroup  # noqa: F401
