"""ctypes binding of oracle/topo.c (Betti numbers of a thresholded film).  TEST INFRASTRUCTURE ONLY:
same rules as oracle/tfo.py -- only tests/ may import it; it imports nothing from the CUDA package."""
import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "topo.c")
_LIB = os.path.join(_HERE, "libtopo.so")
_lib = None


def build(force=False):
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-std=c11", "-fPIC", "-shared", "-o", _LIB, _SRC])
    return _LIB


def lib():
    global _lib
    if _lib is None:
        build()
        _lib = ctypes.CDLL(_LIB)
        dp, lp = ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_longlong)
        _lib.tfo_betti.argtypes = [dp, ctypes.c_int, ctypes.c_int, dp, ctypes.c_int, lp, lp]
    return _lib


def betti(h, thresholds):
    """(b0, b1) arrays for the superlevel sets {h > H*} of a [ny][nx] field, one entry per threshold."""
    h = np.ascontiguousarray(h, dtype=np.float64)
    thr = np.ascontiguousarray(np.atleast_1d(thresholds), dtype=np.float64)
    ny, nx = h.shape
    b0 = np.zeros(len(thr), dtype=np.int64)
    b1 = np.zeros(len(thr), dtype=np.int64)
    dp, lp = ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_longlong)
    rc = lib().tfo_betti(h.ctypes.data_as(dp), nx, ny, thr.ctypes.data_as(dp), len(thr), b0.ctypes.data_as(lp),
                         b1.ctypes.data_as(lp))
    if rc != 0:
        raise MemoryError("tfo_betti")
    return b0, b1
