"""paper_1208_3444_b200 -- B200-native (sm_100a) hot path of COLATUS, arXiv 1208.3444.

The product is the C-ABI library `libcolatus.so` (include/colatus.h) built from `csrc/`;
`binding` is a thin ctypes layer with the same names (argument marshalling only -- every step
of the path runs in the library's CUDA kernels), and `inputs` holds the seeded synthetic input
generators shared with the tests.  There is no CPU fallback: calls fail loudly when the
extension or an sm_100 device is missing.
"""
__all__ = ["binding", "inputs", "build"]
