"""ctypes loader of libapd_probe.so (include/apd_probe.h): the FP32 microbenchmark bench.py uses as its roofline
denominator.  A measurement tool, not part of the method; nothing in the product path imports it."""
from __future__ import annotations

import ctypes
import os

_PKG = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_PKG, "libapd_probe.so")
EXPORTED_SYMBOLS = ["apd_fp32_probe"]
_lib = None


def load_library() -> ctypes.CDLL:
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} is missing: build it with `python -m paper_2403_03571_b200.build`")
        lib = ctypes.CDLL(LIB_PATH)
        lib.apd_fp32_probe.restype = ctypes.c_int
        lib.apd_fp32_probe.argtypes = [ctypes.c_int32, ctypes.c_int32, ctypes.POINTER(ctypes.c_double),
                                       ctypes.POINTER(ctypes.c_double)]
        _lib = lib
    return _lib


def apd_fp32_probe(variant: int, device: int = 0):
    """(ops_per_s, sm_clock_mhz) of microbenchmark `variant` (include/apd_probe.h)."""
    ops, mhz = ctypes.c_double(0.0), ctypes.c_double(0.0)
    rc = load_library().apd_fp32_probe(device, variant, ctypes.byref(ops), ctypes.byref(mhz))
    if rc != 0:
        raise RuntimeError(f"apd_fp32_probe failed with status {rc}")
    return ops.value, mhz.value
