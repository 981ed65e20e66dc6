"""B200-native MEG6 right-hand side + SSP-RK3 step (arXiv 2303.10785) behind a C ABI (include/meg6.h).

The Python layer only marshals arguments: every step of the path runs in the CUDA kernels of
csrc/libmeg6.so.  There is no CPU fallback: a missing library or device raises.
"""
from .binding import (Grid, Meg6Error, Params, lib, lib_path, make_params, EXPORTS, rhs_blocks, rk3_step_blocks, metrics_compute_blocks, fp64_peak)  # noqa: F401
