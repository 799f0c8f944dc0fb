"""Test hooks: builds and loads tests/hooks/lm_host_hooks.cpp (g++, host only) -- the host-side headers of the
CUDA library behind a tiny C ABI, so that CPU tests can exercise them.  Not product code."""
import ctypes
import os
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "lm_host_hooks.cpp")
_LIB = os.path.join(_HERE, "liblm_host_hooks.so")
_CSRC = os.path.join(os.path.dirname(os.path.dirname(_HERE)), "paper_2510_02135_b200", "csrc")
_DEPS = [_SRC, os.path.join(_CSRC, "lanczos_host.h"), os.path.join(_CSRC, "tridiag_host.h")]
_lib = None


def lib():
    global _lib
    if _lib is None:
        if not os.path.exists(_LIB) or any(os.path.getmtime(d) > os.path.getmtime(_LIB) for d in _DEPS):
            subprocess.run(["g++", "-O2", "-std=c++17", "-shared", "-fPIC", "-o", _LIB, _SRC], check=True)
        L = ctypes.CDLL(_LIB)
        dp = ctypes.POINTER(ctypes.c_double)
        L.hook_tridiag_sqrt_e1.argtypes, L.hook_tridiag_sqrt_e1.restype = [ctypes.c_int, dp, dp, dp], ctypes.c_int
        L.hook_error_estimate.argtypes, L.hook_error_estimate.restype = [dp, ctypes.c_int], ctypes.c_double
        L.hook_stopper_new.argtypes, L.hook_stopper_new.restype = [ctypes.c_int, ctypes.c_double, ctypes.c_double, ctypes.c_int], ctypes.c_void_p
        L.hook_stopper_free.argtypes, L.hook_stopper_free.restype = [ctypes.c_void_p], None
        L.hook_stopper_gram_column.argtypes, L.hook_stopper_gram_column.restype = [ctypes.c_void_p, ctypes.c_int, dp], None
        L.hook_stopper_feed.argtypes, L.hook_stopper_feed.restype = [ctypes.c_void_p, ctypes.c_int, ctypes.c_double, ctypes.c_double], ctypes.c_int
        L.hook_stopper_advance.argtypes, L.hook_stopper_advance.restype = [ctypes.c_void_p], None
        L.hook_stopper_last_measure.argtypes, L.hook_stopper_last_measure.restype = [ctypes.c_void_p], ctypes.c_double
        L.hook_stopper_coefficients.argtypes, L.hook_stopper_coefficients.restype = [ctypes.c_void_p, dp, ctypes.c_int], ctypes.c_int
        L.hook_agree_on_stops.argtypes, L.hook_agree_on_stops.restype = [ctypes.c_uint, EXCHANGE_FN, ctypes.c_int], ctypes.c_uint
        _lib = L
    return _lib


EXCHANGE_FN = ctypes.CFUNCTYPE(None, ctypes.POINTER(ctypes.c_uint))
