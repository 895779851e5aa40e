"""Binding of libpwfs_peak.so (include/pwfs_peak.h): the measured FP32 peak that bench.py reports beside the
derived one.  A measurement aid in a library of its own -- the sensor library libpwfs.so does not contain it."""
from __future__ import annotations

import ctypes as C
import os
from typing import Tuple

from .pwfs import PWFS_OK, PwfsError, strerror

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libpwfs_peak.so")
EXPORTS = ("pwfs_peak_fp32",)
_lib = None


def load_library() -> C.CDLL:
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise FileNotFoundError(f"{LIB_PATH} is missing: build it with `python -m paper_1607_07624_b200.build`")
        lib = C.CDLL(LIB_PATH)
        lib.pwfs_peak_fp32.argtypes = [C.c_int32, C.c_int32, C.POINTER(C.c_double), C.POINTER(C.c_double)]
        lib.pwfs_peak_fp32.restype = C.c_int
        _lib = lib
    return _lib


def peak_fp32(device: int = 0, packed: bool = True) -> Tuple[float, float]:
    """(TFLOP/s, ms) of the FFMA / FFMA2 stream micro-benchmark (pwfs_peak_fp32)."""
    tf, ms = C.c_double(), C.c_double()
    rc = load_library().pwfs_peak_fp32(device, int(packed), C.byref(tf), C.byref(ms))
    if rc != PWFS_OK:
        raise PwfsError(rc, "pwfs_peak_fp32", strerror(rc))
    return tf.value, ms.value
