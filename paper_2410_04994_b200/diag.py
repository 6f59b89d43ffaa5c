"""ctypes binding of libshg_diag (include/shg_diag.h): bench.py's measuring equipment, kept out of libshg."""
from __future__ import annotations

import ctypes as C
import os

LIB_PATH = os.path.join(os.path.dirname(os.path.abspath(__file__)), "libshg_diag.so")
EXPORTS = ("shg_measure_fp32_peak", "shg_measure_fp32_peak_distinct")

_lib = None


def lib():
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError("libshg_diag.so not found at %s -- build it with `python -m paper_2410_04994_b200.build`"
                              % LIB_PATH)
        _lib = C.CDLL(LIB_PATH)
        for name in EXPORTS:
            getattr(_lib, name).argtypes = [C.POINTER(C.c_double)]
    return _lib


def _measure(name) -> float:
    v = C.c_double()
    rc = getattr(lib(), name)(C.byref(v))
    if rc != 0:
        raise RuntimeError("%s failed with code %d" % (name, rc))
    return float(v.value)


def measure_fp32_peak() -> float:
    """Measured fp32 FFMA peak of the current device in TFLOP/s (shg_measure_fp32_peak)."""
    return _measure("shg_measure_fp32_peak")


def measure_fp32_peak_distinct() -> float:
    """The same with three distinct register operands per FFMA (shg_measure_fp32_peak_distinct)."""
    return _measure("shg_measure_fp32_peak_distinct")
