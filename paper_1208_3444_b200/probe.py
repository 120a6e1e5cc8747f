"""ctypes binding of libcolatus_probe (include/colatus_probe.h): device microbenchmarks, NOT the product.

Only `bench.py` (the measured FP32 peak beside the derived one) and `tests/test_gpu_probe.py` load this.
"""
from __future__ import annotations

import ctypes
import os
from ctypes import POINTER, c_double, c_int

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libcolatus_probe.so")
SIGNATURES = {
    "colatus_probe_fp32_peak": (c_int, [c_int, c_int, POINTER(c_double), POINTER(c_double)]),
    "colatus_probe_pipe": (c_int, [c_int, c_int, POINTER(c_double)]),
}
_lib = None


def lib():
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} is missing: run `python -m paper_1208_3444_b200.build`")
        handle = ctypes.CDLL(LIB_PATH)
        for name, (res, args) in SIGNATURES.items():
            fn = getattr(handle, name)
            fn.restype, fn.argtypes = res, args
        _lib = handle
    return _lib


def fp32_peak(packed: bool, device: int = 0):
    """(TFLOP/s, ms) of a register-only FFMA (packed False) / FFMA2 (packed True) loop."""
    t, ms = c_double(0.0), c_double(0.0)
    rc = lib().colatus_probe_fp32_peak(int(device), int(bool(packed)), ctypes.byref(t), ctypes.byref(ms))
    if rc:
        raise RuntimeError(f"colatus_probe_fp32_peak failed ({rc})")
    return t.value, ms.value


def pipe(mode: int, device: int = 0) -> float:
    """SMSP cycles per group of 12 packed FP32 ops (+ the extras of `mode`, see colatus_probe.h) at max clock."""
    c = c_double(0.0)
    rc = lib().colatus_probe_pipe(int(device), int(mode), ctypes.byref(c))
    if rc:
        raise RuntimeError(f"colatus_probe_pipe failed ({rc})")
    return c.value
