"""paper_1009_1380_b200 -- B200-native NUFFT-Radon pair (arXiv 1009.1380 hot path).

Thin binding over the C ABI in include/radon.h (libradon_b200.so, hand-written CUDA for
sm_100a).  Argument marshalling only: every step of the path runs in the library's kernels.
PyTorch is used for device memory and streams, nothing else.  There is no CPU fallback: if
the shared library is missing or no sm_100 device is present the calls raise.
"""
from .binding import (
    RadonError,
    RadonPlan,
    lib,
    lib_path,
    kernel_launch_count,
    schedule_selfcheck,
    schedule_host_stats,
    kb_weights_host,
    density_host,
    filter_basis_host,
    EXPORTED_SYMBOLS,
)

__all__ = ["RadonError", "RadonPlan", "lib", "lib_path", "kernel_launch_count",
           "schedule_selfcheck", "schedule_host_stats", "kb_weights_host", "density_host", "filter_basis_host",
           "EXPORTED_SYMBOLS"]
