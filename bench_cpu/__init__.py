"""bench_cpu/ -- BENCH-ONLY: the paper's table method restated for the host cores (tablemethod.c).

A second timed CPU baseline beside the Schulten-Gordon oracle: bench.py's `cpu_table_method`
leg and tests/test_cpu_table_method.py are its only callers.  It shares no source with `oracle/` or with the CUDA
library, and the library never calls it (there is no CPU fallback).
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "tablemethod.c")
_SO = os.path.join(_HERE, "libtablemethod.so")
_LIB = None


def build(force: bool = False) -> str:
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        tmp = _SO + ".tmp.%d" % os.getpid()
        subprocess.run(["gcc", "-O2", "-std=c11", "-fopenmp", "-fPIC", "-shared", "-Wall", "-Wextra", "-o", tmp, _SRC, "-lm"],
                       check=True)
        os.replace(tmp, _SO)
    return _SO


def lib() -> ctypes.CDLL:
    global _LIB
    if _LIB is None:
        build()
        L = ctypes.CDLL(_SO)
        dp, ip = ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_int)
        L.tm_build.argtypes = [ctypes.c_int]
        L.tm_build.restype = ctypes.c_void_p
        L.tm_free.argtypes = [ctypes.c_void_p]
        L.tm_free.restype = None
        L.tm_coupling_rows.argtypes = [ctypes.c_void_p, ctypes.c_int, ctypes.c_int, dp, dp, ctypes.c_int, ip, ctypes.c_int, dp, dp]
        L.tm_coupling_rows.restype = ctypes.c_int
        L.tm_num_threads.restype = ctypes.c_int
        _LIB = L
    return _LIB


def num_threads() -> int:
    return int(lib().tm_num_threads())


def coupling_rows(lmax, l3max, Wtt, Wpp, rows=None):
    """K^TT / K^EE rows (all rows and the paper's triangle + mirror when rows is None).  Returns dict name -> array."""
    L = lib()
    full = rows is None
    rows = np.arange(lmax + 1, dtype=np.int32) if full else np.ascontiguousarray(rows, dtype=np.int32)
    dp, ip = ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_int)
    out = {}
    w = {}
    for k, W in (("TT", Wtt), ("EE", Wpp)):
        if W is not None:
            w[k] = np.ascontiguousarray(W, dtype=np.float64)
            assert w[k].shape == (l3max + 1,)
            out[k] = np.zeros((rows.size, lmax + 1))
    t = L.tm_build(int(lmax))
    if not t:
        raise MemoryError("tm_build")
    try:
        rc = L.tm_coupling_rows(t, int(lmax), int(l3max),
                                w["TT"].ctypes.data_as(dp) if "TT" in w else None,
                                w["EE"].ctypes.data_as(dp) if "EE" in w else None,
                                int(rows.size), rows.ctypes.data_as(ip), 1 if full else 0,
                                out["TT"].ctypes.data_as(dp) if "TT" in out else None,
                                out["EE"].ctypes.data_as(dp) if "EE" in out else None)
    finally:
        L.tm_free(t)
    if rc != 0:
        raise RuntimeError("tm_coupling_rows failed: %d" % rc)
    return out
