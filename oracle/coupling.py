"""ctypes front-end of the C oracle (`sg_oracle.c`).  TEST INFRASTRUCTURE -- see oracle/__init__.py.

Every function here only marshals arguments and lays the per-pair results out as
matrices; the arithmetic is in `sg_oracle.c`.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "sg_oracle.c")
_SO = os.path.join(_HERE, "libsg_oracle.so")
_LOCK = threading.Lock()
_LIB = None


def build(force: bool = False) -> str:
    """Compile sg_oracle.c with gcc (-O2, OpenMP, no fast-math) into oracle/libsg_oracle.so."""
    with _LOCK:
        if force or (not os.path.exists(_SO)) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
            tmp = _SO + ".tmp.%d" % os.getpid()
            cmd = ["gcc", "-O2", "-std=c11", "-fopenmp", "-fPIC", "-shared", "-Wall", "-Wextra",
                   "-o", tmp, _SRC, "-lm"]
            subprocess.run(cmd, check=True)
            os.replace(tmp, _SO)
    return _SO


def lib() -> ctypes.CDLL:
    global _LIB
    if _LIB is None:
        build()
        L = ctypes.CDLL(_SO)
        dp = ctypes.POINTER(ctypes.c_double)
        ip = ctypes.POINTER(ctypes.c_int)
        L.oracle_3j_family.argtypes = [ctypes.c_int] * 4 + [dp, ip, ip]
        L.oracle_3j_family.restype = ctypes.c_int
        L.oracle_l3_range.argtypes = [ctypes.c_int] * 4 + [ip, ip, ip]
        L.oracle_l3_range.restype = ctypes.c_int
        L.oracle_coupling_pairs.argtypes = [ctypes.c_int, dp, dp, dp, ctypes.c_long, ip, ip, dp, dp, dp, dp]
        L.oracle_coupling_pairs.restype = ctypes.c_int
        L.oracle_coupling_spin1_pairs.argtypes = [ctypes.c_int, dp, dp, ctypes.c_long, ip, ip, dp, dp, dp]
        L.oracle_coupling_spin1_pairs.restype = ctypes.c_int
        L.oracle_num_threads.restype = ctypes.c_int
        L.oracle_set_num_threads.argtypes = [ctypes.c_int]
        _LIB = L
    return _LIB


def num_threads() -> int:
    return int(lib().oracle_num_threads())


def set_num_threads(n: int) -> None:
    lib().oracle_set_num_threads(int(n))


def _dptr(a):
    return None if a is None else a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def three_j_family(j2: int, j3: int, m2: int, m3: int):
    """(j j2 j3; -m2-m3 m2 m3) for all allowed j.  Returns (jmin, values[jmax-jmin+1])."""
    m1 = -m2 - m3
    jmin = max(abs(j2 - j3), abs(m1))
    jmax = j2 + j3
    if abs(m2) > j2 or abs(m3) > j3 or jmin > jmax:
        return jmin, np.zeros(0)
    out = np.zeros(jmax - jmin + 1)
    a, b = ctypes.c_int(), ctypes.c_int()
    rc = lib().oracle_3j_family(j2, j3, m2, m3, _dptr(out), ctypes.byref(a), ctypes.byref(b))
    if rc != 0:
        raise RuntimeError("oracle_3j_family failed: %d" % rc)
    assert a.value == jmin and b.value == jmax
    return jmin, out


def l3_range(l1: int, l2: int, l3max: int, parity: int):
    lo, hi, n = ctypes.c_int(), ctypes.c_int(), ctypes.c_int()
    rc = lib().oracle_l3_range(l1, l2, l3max, parity, ctypes.byref(lo), ctypes.byref(hi), ctypes.byref(n))
    if rc != 0:
        raise ValueError("oracle_l3_range: bad arguments")
    return lo.value, hi.value, n.value


def _win(w, l3max):
    if w is None:
        return None
    w = np.ascontiguousarray(w, dtype=np.float64)
    if w.shape != (l3max + 1,):
        raise ValueError("window must have l3max+1 = %d entries, got %r" % (l3max + 1, w.shape))
    return w


def coupling_pairs(l3max, Wtt, Wtp, Wpp, l1s, l2s):
    """Entries K^{TT,TE,EE,EB}_{l1 l2} for the given pairs.  Returns dict name -> float64[npairs]
    (a block whose window is None is absent).  BB equals EE."""
    Wtt, Wtp, Wpp = _win(Wtt, l3max), _win(Wtp, l3max), _win(Wpp, l3max)
    l1s = np.ascontiguousarray(l1s, dtype=np.int32)
    l2s = np.ascontiguousarray(l2s, dtype=np.int32)
    n = l1s.size
    assert l2s.size == n
    out = {}
    if Wtt is not None:
        out["TT"] = np.zeros(n)
    if Wtp is not None:
        out["TE"] = np.zeros(n)
    if Wpp is not None:
        out["EE"] = np.zeros(n)
        out["EB"] = np.zeros(n)
    ip = ctypes.POINTER(ctypes.c_int)
    rc = lib().oracle_coupling_pairs(
        int(l3max), _dptr(Wtt), _dptr(Wtp), _dptr(Wpp), n,
        l1s.ctypes.data_as(ip), l2s.ctypes.data_as(ip),
        _dptr(out.get("TT")), _dptr(out.get("TE")), _dptr(out.get("EE")), _dptr(out.get("EB")))
    if rc != 0:
        raise RuntimeError("oracle_coupling_pairs failed: %d" % rc)
    if "EE" in out:
        out["BB"] = out["EE"].copy()
    return out


def coupling_rows(lmax, l3max, Wtt, Wtp, Wpp, rows):
    """Rows l1 in `rows`, all columns l2 = 0..lmax.  Returns dict name -> float64[len(rows), lmax+1]."""
    rows = np.asarray(rows, dtype=np.int32)
    N = lmax + 1
    l1s = np.repeat(rows, N)
    l2s = np.tile(np.arange(N, dtype=np.int32), rows.size)
    res = coupling_pairs(l3max, Wtt, Wtp, Wpp, l1s, l2s)
    return {k: v.reshape(rows.size, N) for k, v in res.items()}


def coupling_full(lmax, l3max, Wtt, Wtp, Wpp):
    """All (lmax+1)^2 entries, each from its own definition (no symmetry used)."""
    return coupling_rows(lmax, l3max, Wtt, Wtp, Wpp, np.arange(lmax + 1))


def coupling_band(lmax, lcut, Wtt, Wtp, Wpp, rows=None):
    """Band-limited matrices: the l3 sum stops at lcut (inclusive), only
    |l1-l2| <= lcut is stored, band[l1][l2-l1+lcut]; slots whose l2 falls outside 0..lmax are 0.
    Windows have lcut+1 entries.  `rows` restricts the l1 values (result rows in that order)."""
    N = lmax + 1
    rows = np.arange(N, dtype=np.int32) if rows is None else np.asarray(rows, dtype=np.int32)
    width = 2 * lcut + 1
    off = np.arange(-lcut, lcut + 1, dtype=np.int64)
    l1g = np.repeat(rows.astype(np.int64), width)
    l2g = l1g + np.tile(off, rows.size)
    ok = (l2g >= 0) & (l2g <= lmax)
    res = coupling_pairs(lcut, Wtt, Wtp, Wpp, l1g[ok].astype(np.int32), l2g[ok].astype(np.int32))
    out = {}
    for k, v in res.items():
        b = np.zeros(rows.size * width)
        b[ok] = v
        out[k] = b.reshape(rows.size, width)
    return out


def spin1_pairs(l3max, W01, W11, l1s, l2s):
    """Spin-1 blocks K^{01}, K^{11+}, K^{11-} (sg_oracle.c: oracle_coupling_spin1_pairs) for the given pairs."""
    W01, W11 = _win(W01, l3max), _win(W11, l3max)
    l1s = np.ascontiguousarray(l1s, dtype=np.int32)
    l2s = np.ascontiguousarray(l2s, dtype=np.int32)
    n = l1s.size
    out = {}
    if W01 is not None:
        out["K01"] = np.zeros(n)
    if W11 is not None:
        out["K11p"] = np.zeros(n)
        out["K11m"] = np.zeros(n)
    ip = ctypes.POINTER(ctypes.c_int)
    rc = lib().oracle_coupling_spin1_pairs(int(l3max), _dptr(W01), _dptr(W11), n, l1s.ctypes.data_as(ip),
                                           l2s.ctypes.data_as(ip), _dptr(out.get("K01")), _dptr(out.get("K11p")),
                                           _dptr(out.get("K11m")))
    if rc != 0:
        raise RuntimeError("oracle_coupling_spin1_pairs failed: %d" % rc)
    return out


def spin1_full(lmax, l3max, W01, W11):
    """All (lmax+1)^2 entries of the spin-1 blocks."""
    N = lmax + 1
    l1s = np.repeat(np.arange(N, dtype=np.int32), N)
    l2s = np.tile(np.arange(N, dtype=np.int32), N)
    return {k: v.reshape(N, N) for k, v in spin1_pairs(l3max, W01, W11, l1s, l2s).items()}


def coupling_binned(lmax, l3max, Wtt, Wtp, Wpp, edges, P, Q, pairs=None):
    """Binned matrices (reading 20; the paper prints no binning operator):

        B^{XY}[b][b'] = sum_{l1 in bin b} sum_{l2 in bin b'} P[l1] K^{XY}[l1][l2] Q[l2],

    bin b = edges[b] <= l < edges[b+1] (ascending, within 0..lmax+1), P and Q per-l weights with lmax+1 entries:
    the sum of the oracle's own entries, written out (every entry from its definition, no symmetry).
    `pairs`: list of (b, b') to evaluate (default: all); the others are returned as NaN.
    Returns dict name -> float64[nbins, nbins]."""
    edges = np.asarray(edges, dtype=np.int64)
    nb = edges.size - 1
    assert nb >= 1 and edges[0] >= 0 and edges[-1] <= lmax + 1 and np.all(np.diff(edges) >= 0)
    P = np.ascontiguousarray(P, dtype=np.float64)
    Q = np.ascontiguousarray(Q, dtype=np.float64)
    assert P.shape == (lmax + 1,) and Q.shape == (lmax + 1,)
    if pairs is None:
        pairs = [(b, c) for b in range(nb) for c in range(nb)]
    names = [k for k, w in (("TT", Wtt), ("TE", Wtp), ("EE", Wpp), ("BB", Wpp), ("EB", Wpp)) if w is not None]
    out = {k: np.full((nb, nb), np.nan) for k in names}
    for b, c in pairs:
        r = np.arange(edges[b], edges[b + 1], dtype=np.int32)
        q = np.arange(edges[c], edges[c + 1], dtype=np.int32)
        if r.size == 0 or q.size == 0:
            for k in names:
                out[k][b, c] = 0.0
            continue
        l1 = np.repeat(r, q.size)
        l2 = np.tile(q, r.size)
        K = coupling_pairs(l3max, Wtt, Wtp, Wpp, l1, l2)
        wgt = (P[r][:, None] * Q[q][None, :]).ravel()
        for k in names:
            out[k][b, c] = float(np.sum(wgt * K[k]))
    return out


def coupling_binned_multi(lmax, l3max, Wtt, Wtp, Wpp, edges, P, Q, pairs=None):
    """coupling_binned for several window sets (windows [nwin, l3max+1] or None): one independent problem per set
    (one coupling matrix per map pair).  Returns dict name -> float64[nwin, nbins, nbins]."""
    first = next(w for w in (Wtt, Wtp, Wpp) if w is not None)
    res = [coupling_binned(lmax, l3max, None if Wtt is None else Wtt[w], None if Wtp is None else Wtp[w],
                           None if Wpp is None else Wpp[w], edges, P, Q, pairs=pairs) for w in range(len(first))]
    return {k: np.stack([r[k] for r in res]) for k in res[0]}
