"""bench_gpu/ -- BENCH-ONLY: the DFMA-chain probe that measures the FP64 roofline denominator (fp64_probe.cu).

bench.py is its only caller; it is not part of libtj (the product ABI holds no microbenchmark) and shares no source
with it.  Built in-tree with nvcc for sm_100a like the library.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "fp64_probe.cu")
_SO = os.path.join(_HERE, "libfp64probe.so")
_LIB = None


def build(force: bool = False) -> str:
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        nvcc = os.environ.get("NVCC") or ("/usr/local/cuda/bin/nvcc" if os.path.exists("/usr/local/cuda/bin/nvcc") else "nvcc")
        tmp = _SO + ".tmp.%d" % os.getpid()
        subprocess.run([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17", "-shared",
                        "-Xcompiler", "-fPIC", "-o", tmp, _SRC], check=True)
        os.replace(tmp, _SO)
    return _SO


def lib() -> ctypes.CDLL:
    global _LIB
    if _LIB is None:
        build()
        L = ctypes.CDLL(_SO)
        L.probe_fp64.argtypes = [ctypes.c_int, ctypes.c_void_p, ctypes.POINTER(ctypes.c_double)]
        L.probe_fp64.restype = ctypes.c_int
        _LIB = L
    return _LIB


def fp64_probe(iters: int, stream_ptr: int | None = None) -> float:
    """Achieved FP64 thread-instructions per second of `iters` iterations of 16 DFMA chains per thread (synchronous)."""
    v = ctypes.c_double()
    rc = lib().probe_fp64(int(iters), ctypes.c_void_p(stream_ptr or 0), ctypes.byref(v))
    if rc != 0:
        raise RuntimeError("probe_fp64 failed: cudaError %d" % rc)
    return v.value
