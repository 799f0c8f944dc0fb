"""Binding of liblm_probe.so (csrc/fma_probe.cu): the FMA-pipe peak probe bench.py reports beside the nominal
roofline denominator.  A measurement helper with its own library -- not part of liblm.so or of include/lm.h."""
from __future__ import annotations

import ctypes
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
_lib = None


def fma_peak(precision: int, seconds: float = 0.2) -> float:
    """Measured FMA-pipe peak of the current device in lane-operations per second (precision: 0 = fp32, 1 = fp64)."""
    global _lib
    if _lib is None:
        from . import build as _build
        _build.build()
        _lib = ctypes.CDLL(_build.PROBE_LIB)
        _lib.lm_probe_fma_peak.restype = ctypes.c_int
        _lib.lm_probe_fma_peak.argtypes = [ctypes.c_int, ctypes.c_double, ctypes.POINTER(ctypes.c_double)]
    out = ctypes.c_double(0.0)
    rc = _lib.lm_probe_fma_peak(int(precision), float(seconds), ctypes.byref(out))
    if rc != 0:
        raise RuntimeError(f"lm_probe_fma_peak failed with code {rc}")
    return out.value
