"""B200-native exact INLA value-and-gradient over BTA precision matrices (ADELIA hot path).

Thin Python binding (argument marshalling only) over the C-ABI library `libbta_b200.so`
declared in `include/bta.h`; every step of the path runs in hand-written sm_100a kernels.
PyTorch is used for device memory and streams only.  There is no CPU fallback: importing
works anywhere (so the symbols can be checked), but every compute call needs a B200.
"""
from .binding import (  # noqa: F401
    BtaError,
    BtaModel,
    Blocks,
    fp64_peak,
    gemm,
    lib,
    lib_path,
)
