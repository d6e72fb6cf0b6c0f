"""paper_1608_05794_b200 -- B200-native batched reactor integration (arXiv 1608.05794 hot path).

Thin binding over the C-ABI library libck.so (include/ck.h): argument marshalling only; every step of
the path runs in the library's CUDA kernels.  There is no CPU fallback: importing works without a GPU
(so the ABI can be inspected), but any compute call without the library or a device raises.
"""
from ._binding import (Mechanism, CkError, lib, lib_path, exported_symbols, fp64_peak, fp64_mma_peak, lu_solve_batched, parse_mechanism,  # noqa: F401
                       CK_OP_ROS, CK_OP_RKF45, CK_OP_JAC, CK_JAC_ANALYTIC, CK_JAC_FD)
