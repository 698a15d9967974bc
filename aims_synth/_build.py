"""Compile and load aims_synth/_heavy.c (input generation only; see that file's header)."""
import ctypes
import os
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "_heavy.c")
_LIB = os.path.join(_HERE, "_heavy.so")
_lib = None


def build(force=False):
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".%d.tmp" % os.getpid()
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


def lib():
    global _lib
    if _lib is None:
        L = ctypes.CDLL(build())
        dp = ctypes.POINTER(ctypes.c_double)
        ip = ctypes.POINTER(ctypes.c_int32)
        lp = ctypes.POINTER(ctypes.c_int64)
        L.synth_partition_weights.restype = ctypes.c_int
        L.synth_partition_weights.argtypes = [ctypes.c_int, dp, ctypes.c_int64, dp, ip, ctypes.c_double, dp]
        L.synth_fields.restype = ctypes.c_int
        L.synth_fields.argtypes = [ctypes.c_int, dp, ctypes.c_int, dp, dp, dp, dp, ctypes.c_double,
                                   ctypes.c_int64, dp, dp, dp]
        L.synth_bisect.restype = ctypes.c_int64
        L.synth_bisect.argtypes = [ctypes.c_int64, dp, ctypes.c_int, lp, lp]
        _lib = L
    return _lib
