"""Thin Python binding of libtj (include/tj.h): argument marshalling only.

Every step of the path runs in the library's CUDA kernels; this file converts torch tensors to
device pointers, picks the current CUDA stream and turns error codes into exceptions.  There is
no fallback of any kind: if `libtj.so` is missing or a call fails, a TJError is raised.
"""
from __future__ import annotations

import ctypes
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libtj.so")
_LIB = None

TJ_OK, TJ_EINVAL, TJ_ENOMEM, TJ_ECUDA, TJ_ELIMIT = 0, -1, -2, -3, -4
TJ_STATIC_LMAX = 16384              # include/tj.h: largest lmax tj_coupling_pol_static accepts

# every symbol include/tj.h declares (tests/test_abi.py checks the header against this and the .so)
SYMBOLS = (
    "tj_build_tables", "tj_free_tables", "tj_tables_info", "tj_tables_copy",
    "tj_coupling_tt", "tj_coupling_pol", "tj_coupling_pol_static", "tj_coupling_band", "tj_coupling_multi", "tj_coupling_spin1", "tj_coupling_rows", "tj_coupling_binned", "tj_coupling_binned_multi", "tj_coupling_literal", "tj_coupling_host", "tj_set_host_pipeline", "tj_host_pipeline_info",
    "tj_chunk_plan", "tj_coupling_host_part", "tj_coupling_host_multi",
    "tj_l3_range", "tj_sweep_counts", "tj_profile_enable", "tj_profile_get",
    "tj_profile_last_sweep", "tj_profile_launches", "tj_strerror",
)


class TJError(RuntimeError):
    def __init__(self, code, what):
        self.code = code
        super().__init__("%s failed: %s (code %d)" % (what, _strerror(code), code))


def library_path() -> str:
    return _SO


def load_library() -> ctypes.CDLL:
    """Load libtj.so (built in-tree by `python -m paper_2602_15605_b200.build`).  Fails loudly."""
    global _LIB
    if _LIB is not None:
        return _LIB
    if not os.path.exists(_SO):
        raise TJError(TJ_ECUDA, "loading %s (not built: run `python -m paper_2602_15605_b200.build`; "
                                "there is no CPU fallback)" % _SO)
    L = ctypes.CDLL(_SO)
    vp, ip, dp, ci = ctypes.c_void_p, ctypes.POINTER(ctypes.c_int), ctypes.POINTER(ctypes.c_double), ctypes.c_int
    L.tj_build_tables.argtypes = [ci, ci, vp, ctypes.POINTER(vp)]
    L.tj_free_tables.argtypes = [vp]
    L.tj_free_tables.restype = None
    L.tj_tables_info.argtypes = [vp, ip, ip, ip]
    L.tj_tables_copy.argtypes = [vp, ci, dp, ci]
    L.tj_coupling_tt.argtypes = [vp, vp, ci, vp, vp]
    L.tj_coupling_pol.argtypes = [vp, vp, vp, vp, ci, vp, vp, vp, vp, vp, vp]
    L.tj_coupling_pol_static.argtypes = [vp, vp, vp, vp, ci, vp, vp, vp, vp, vp, vp]
    L.tj_coupling_band.argtypes = [vp, ci, vp, vp, vp, vp, vp, vp, vp, vp, vp]
    L.tj_coupling_multi.argtypes = [vp, ci, vp, vp, vp, ci, vp, vp, vp, vp, vp, vp]
    L.tj_coupling_spin1.argtypes = [vp, vp, vp, vp, ci, vp, vp, vp, vp, vp]
    L.tj_coupling_rows.argtypes = [vp, vp, vp, vp, ci, ci, ci, vp, vp, vp, vp, vp, vp]
    L.tj_coupling_binned.argtypes = [vp, vp, vp, vp, ci, ci, ip, vp, vp, vp, vp, vp, vp, vp, vp]
    L.tj_coupling_binned_multi.argtypes = [vp, ci, vp, vp, vp, ci, ci, ip, vp, vp, vp, vp, vp, vp, vp, vp]
    L.tj_coupling_literal.argtypes = [vp, vp, vp, ci, vp, vp, vp]
    L.tj_coupling_host.argtypes = [vp, ci, ci, vp, vp, vp, vp, vp, vp, vp, vp, vp]
    L.tj_chunk_plan.argtypes = [ci, ci, ci, ip, ip, ip]
    L.tj_coupling_host_part.argtypes = [vp, ci, ci, ci, vp, vp, vp, vp, vp, vp, vp, vp, vp]
    L.tj_coupling_host_multi.argtypes = [ctypes.POINTER(vp), ci, ci, vp, vp, vp, vp, vp, vp, vp, vp, ctypes.POINTER(vp)]
    L.tj_set_host_pipeline.argtypes = [vp, ctypes.c_double, ctypes.c_double]
    L.tj_host_pipeline_info.argtypes = [vp, ip, ip]
    L.tj_l3_range.argtypes = [ci, ci, ci, ci, ip, ip, ip]
    L.tj_sweep_counts.argtypes = [ci, ci, ci, ip, ip, ip, ip]
    L.tj_profile_enable.argtypes = [ci]
    L.tj_profile_get.argtypes = [dp]
    L.tj_profile_last_sweep.argtypes = [ip]
    L.tj_profile_launches.argtypes = [ctypes.POINTER(ctypes.c_longlong)]
    L.tj_strerror.argtypes = [ci]
    L.tj_strerror.restype = ctypes.c_char_p
    for name in SYMBOLS:
        if name not in ("tj_free_tables", "tj_strerror"):
            getattr(L, name).restype = ci
    _LIB = L
    return L


def _strerror(code):
    try:
        return load_library().tj_strerror(code).decode()
    except Exception:
        return {TJ_EINVAL: "invalid argument", TJ_ENOMEM: "out of memory", TJ_ECUDA: "CUDA error"}.get(code, "?")


def _check(code, what):
    if code != TJ_OK:
        raise TJError(code, what)


def _stream_ptr(stream=None):
    import torch
    s = torch.cuda.current_stream() if stream is None else stream
    return ctypes.c_void_p(s.cuda_stream)


def _dev_ptr(t, n, name):
    """Device pointer of a contiguous float64 CUDA tensor with n elements (None -> NULL)."""
    import torch
    if t is None:
        return ctypes.c_void_p(0)
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()):
        raise TJError(TJ_EINVAL, "%s must be a contiguous float64 CUDA tensor" % name)
    if t.numel() != n:
        raise TJError(TJ_EINVAL, "%s must have %d elements, has %d" % (name, n, t.numel()))
    return ctypes.c_void_p(t.data_ptr())


def _host_ptr(t, n, name):
    import torch
    if t is None:
        return ctypes.c_void_p(0)
    if not (isinstance(t, torch.Tensor) and (not t.is_cuda) and t.dtype == torch.float64 and t.is_contiguous()):
        raise TJError(TJ_EINVAL, "%s must be a contiguous float64 CPU tensor" % name)
    if t.numel() != n:
        raise TJError(TJ_EINVAL, "%s must have %d elements, has %d" % (name, n, t.numel()))
    return ctypes.c_void_p(t.data_ptr())


class Tables:
    """Owns a tj_tables handle (tj_build_tables / tj_free_tables)."""

    def __init__(self, lmax: int, l3max: int | None = None, stream=None):
        L = load_library()
        self.lmax = int(lmax)
        self.l3max = 2 * self.lmax if l3max is None else int(l3max)
        h = ctypes.c_void_p()
        _check(L.tj_build_tables(self.lmax, self.l3max, _stream_ptr(stream), ctypes.byref(h)), "tj_build_tables")
        self._h = h
        a, b, c = ctypes.c_int(), ctypes.c_int(), ctypes.c_int()
        _check(L.tj_tables_info(self._h, ctypes.byref(a), ctypes.byref(b), ctypes.byref(c)), "tj_tables_info")
        self.pmax = c.value

    @property
    def handle(self):
        return self._h

    def copy_table(self, which: int, count: int):
        import numpy as np
        out = np.empty(count, dtype=np.float64)
        _check(load_library().tj_tables_copy(self._h, which, out.ctypes.data_as(ctypes.POINTER(ctypes.c_double)), count),
               "tj_tables_copy")
        return out

    def close(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            load_library().tj_free_tables(self._h)
            self._h = ctypes.c_void_p(0)

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def build_tables(lmax: int, l3max: int | None = None, stream=None) -> Tables:
    return Tables(lmax, l3max, stream)


def coupling_tt(tables: Tables, Wtt, TT=None, stream=None):
    """tj_coupling_tt.  Wtt: float64 CUDA tensor [l3max+1].  Returns TT [(lmax+1),(lmax+1)]."""
    import torch
    N = tables.lmax + 1
    if TT is None:
        TT = torch.empty((N, N), dtype=torch.float64, device=Wtt.device)
    nW = tables.l3max + 1
    _check(load_library().tj_coupling_tt(tables.handle, _dev_ptr(Wtt, nW, "Wtt"), nW, _dev_ptr(TT, N * N, "TT"),
                                         _stream_ptr(stream)), "tj_coupling_tt")
    return TT


_BLOCKS = ("TT", "TE", "EE", "BB", "EB")


def coupling_pol(tables: Tables, Wtt, Wtp, Wpp, want=_BLOCKS, out=None, stream=None):
    """tj_coupling_pol.  `want`: which blocks to compute; `out`: optional dict of preallocated
    [(lmax+1),(lmax+1)] float64 CUDA tensors.  Returns dict name -> tensor."""
    import torch
    N = tables.lmax + 1
    nW = tables.l3max + 1
    dev = next(w for w in (Wtt, Wtp, Wpp) if w is not None).device
    out = {} if out is None else dict(out)
    for k in want:
        if k not in out:
            out[k] = torch.empty((N, N), dtype=torch.float64, device=dev)
    args = [_dev_ptr(out.get(k) if k in want else None, N * N, k) for k in _BLOCKS]
    _check(load_library().tj_coupling_pol(tables.handle, _dev_ptr(Wtt, nW, "Wtt"), _dev_ptr(Wtp, nW, "Wtp"),
                                          _dev_ptr(Wpp, nW, "Wpp"), nW, *args, _stream_ptr(stream)), "tj_coupling_pol")
    return {k: out[k] for k in want}


def coupling_pol_static(tables: Tables, Wtt, Wtp, Wpp, out: dict, stream=None):
    """tj_coupling_pol_static: tj_coupling_pol for callers that may not allocate GPU memory (an application that owns
    all of device memory already, a latency-bound loop, a GPU set-up without the stream-ordered pool).  The library's
    scratch sits in a fixed 2 MiB device array instead of coming from cudaMallocAsync, so handles with
    lmax > TJ_STATIC_LMAX are refused (TJError, code TJ_ELIMIT), and calls that overlap on one GPU race on that array:
    keep them in one stream.  `out` is REQUIRED here -- dict name -> preallocated [(lmax+1),(lmax+1)] float64 CUDA
    tensor for every block wanted; this wrapper creates no tensor either.  The first call on a device looks the
    array's address up; make it before any stream capture.  Returns `out`."""
    N = tables.lmax + 1
    nW = tables.l3max + 1
    if not out or any(k not in _BLOCKS for k in out):
        raise TJError(TJ_EINVAL, "coupling_pol_static needs preallocated outputs named from %s" % (_BLOCKS,))
    args = [_dev_ptr(out.get(k), N * N, k) for k in _BLOCKS]
    _check(load_library().tj_coupling_pol_static(tables.handle, _dev_ptr(Wtt, nW, "Wtt"), _dev_ptr(Wtp, nW, "Wtp"),
                                                 _dev_ptr(Wpp, nW, "Wpp"), nW, *args, _stream_ptr(stream)),
           "tj_coupling_pol_static")
    return out


def coupling_band(tables: Tables, lcut: int, Wtt, Wtp, Wpp, want=_BLOCKS, out=None, stream=None):
    """tj_coupling_band.  Windows have lcut+1 entries; outputs are [(lmax+1),(2*lcut+1)] banded."""
    import torch
    N = tables.lmax + 1
    width = 2 * lcut + 1
    dev = next(w for w in (Wtt, Wtp, Wpp) if w is not None).device
    out = {} if out is None else dict(out)
    for k in want:
        if k not in out:
            out[k] = torch.empty((N, width), dtype=torch.float64, device=dev)
    args = [_dev_ptr(out.get(k) if k in want else None, N * width, k) for k in _BLOCKS]
    _check(load_library().tj_coupling_band(tables.handle, int(lcut), _dev_ptr(Wtt, lcut + 1, "Wtt"),
                                           _dev_ptr(Wtp, lcut + 1, "Wtp"), _dev_ptr(Wpp, lcut + 1, "Wpp"),
                                           *args, _stream_ptr(stream)), "tj_coupling_band")
    return {k: out[k] for k in want}


def coupling_multi(tables: Tables, Wtt, Wtp, Wpp, want=_BLOCKS, out=None, stream=None):
    """tj_coupling_multi.  Windows: float64 CUDA tensors [nwin, l3max+1]; outputs [nwin, lmax+1, lmax+1]."""
    import torch
    N = tables.lmax + 1
    nW = tables.l3max + 1
    first = next(w for w in (Wtt, Wtp, Wpp) if w is not None)
    nwin = int(first.shape[0])
    out = {} if out is None else dict(out)
    for k in want:
        if k not in out:
            out[k] = torch.empty((nwin, N, N), dtype=torch.float64, device=first.device)
    args = [_dev_ptr(out.get(k) if k in want else None, nwin * N * N, k) for k in _BLOCKS]
    _check(load_library().tj_coupling_multi(tables.handle, nwin, _dev_ptr(Wtt, nwin * nW, "Wtt"),
                                            _dev_ptr(Wtp, nwin * nW, "Wtp"), _dev_ptr(Wpp, nwin * nW, "Wpp"), nW,
                                            *args, _stream_ptr(stream)), "tj_coupling_multi")
    return {k: out[k] for k in want}


_SPIN1 = ("K00", "K01", "K11p", "K11m")


def coupling_spin1(tables: Tables, W00, W01, W11, want=_SPIN1, out=None, stream=None):
    """tj_coupling_spin1.  Returns dict name -> [(lmax+1),(lmax+1)] tensor for the blocks in `want`."""
    import torch
    N = tables.lmax + 1
    nW = tables.l3max + 1
    dev = next(w for w in (W00, W01, W11) if w is not None).device
    out = {} if out is None else dict(out)
    for k in want:
        if k not in out:
            out[k] = torch.empty((N, N), dtype=torch.float64, device=dev)
    args = [_dev_ptr(out.get(k) if k in want else None, N * N, k) for k in _SPIN1]
    _check(load_library().tj_coupling_spin1(tables.handle, _dev_ptr(W00, nW, "W00"), _dev_ptr(W01, nW, "W01"),
                                            _dev_ptr(W11, nW, "W11"), nW, *args, _stream_ptr(stream)),
           "tj_coupling_spin1")
    return {k: out[k] for k in want}


def coupling_rows(tables: Tables, Wtt, Wtp, Wpp, row_lo: int, row_hi: int, want=_BLOCKS, out=None, stream=None):
    """tj_coupling_rows: rows row_lo..row_hi-1 of every block in `want`, each [(row_hi-row_lo), (lmax+1)]."""
    import torch
    N = tables.lmax + 1
    nW = tables.l3max + 1
    nr = int(row_hi) - int(row_lo)
    dev = next(w for w in (Wtt, Wtp, Wpp) if w is not None).device
    out = {} if out is None else dict(out)
    for k in want:
        if k not in out:
            out[k] = torch.empty((nr, N), dtype=torch.float64, device=dev)
    args = [_dev_ptr(out.get(k) if k in want else None, nr * N, k) for k in _BLOCKS]
    _check(load_library().tj_coupling_rows(tables.handle, _dev_ptr(Wtt, nW, "Wtt"), _dev_ptr(Wtp, nW, "Wtp"),
                                           _dev_ptr(Wpp, nW, "Wpp"), nW, int(row_lo), int(row_hi), *args,
                                           _stream_ptr(stream)), "tj_coupling_rows")
    return {k: out[k] for k in want}


def coupling_binned(tables: Tables, Wtt, Wtp, Wpp, edges, P, Q, want=_BLOCKS, out=None, stream=None):
    """tj_coupling_binned.  edges: nbins+1 ascending ints (host); P, Q: float64 CUDA tensors [lmax+1].
    Returns dict name -> [nbins, nbins] tensor."""
    import torch
    N = tables.lmax + 1
    nW = tables.l3max + 1
    edges = [int(x) for x in edges]
    nb = len(edges) - 1
    harr = (ctypes.c_int * (nb + 1))(*edges)
    dev = P.device
    out = {} if out is None else dict(out)
    for k in want:
        if k not in out:
            out[k] = torch.empty((nb, nb), dtype=torch.float64, device=dev)
    args = [_dev_ptr(out.get(k) if k in want else None, nb * nb, k) for k in _BLOCKS]
    _check(load_library().tj_coupling_binned(tables.handle, _dev_ptr(Wtt, nW, "Wtt"), _dev_ptr(Wtp, nW, "Wtp"),
                                             _dev_ptr(Wpp, nW, "Wpp"), nW, nb, harr, _dev_ptr(P, N, "P"), _dev_ptr(Q, N, "Q"),
                                             *args, _stream_ptr(stream)), "tj_coupling_binned")
    return {k: out[k] for k in want}


def coupling_binned_multi(tables: Tables, Wtt, Wtp, Wpp, edges, P, Q, want=_BLOCKS, out=None, stream=None):
    """tj_coupling_binned_multi.  Windows: float64 CUDA tensors [nwin, l3max+1]; returns dict name -> [nwin, nbins, nbins]."""
    import torch
    N = tables.lmax + 1
    nW = tables.l3max + 1
    first = next(w for w in (Wtt, Wtp, Wpp) if w is not None)
    nwin = int(first.shape[0])
    edges = [int(x) for x in edges]
    nb = len(edges) - 1
    harr = (ctypes.c_int * (nb + 1))(*edges)
    out = {} if out is None else dict(out)
    for k in want:
        if k not in out:
            out[k] = torch.empty((nwin, nb, nb), dtype=torch.float64, device=first.device)
    args = [_dev_ptr(out.get(k) if k in want else None, nwin * nb * nb, k) for k in _BLOCKS]
    _check(load_library().tj_coupling_binned_multi(tables.handle, nwin, _dev_ptr(Wtt, nwin * nW, "Wtt"),
                                                   _dev_ptr(Wtp, nwin * nW, "Wtp"), _dev_ptr(Wpp, nwin * nW, "Wpp"), nW,
                                                   nb, harr, _dev_ptr(P, N, "P"), _dev_ptr(Q, N, "Q"), *args,
                                                   _stream_ptr(stream)), "tj_coupling_binned_multi")
    return {k: out[k] for k in want}


def coupling_literal(tables: Tables, Wtt, Wpp, want=("TT", "EE"), stream=None):
    """tj_coupling_literal (ablation: the paper's own per-pair evaluation, Eq. 10 / Eq. 16 literally)."""
    import torch
    N = tables.lmax + 1
    nW = tables.l3max + 1
    dev = next(w for w in (Wtt, Wpp) if w is not None).device
    out = {k: torch.empty((N, N), dtype=torch.float64, device=dev) for k in want}
    _check(load_library().tj_coupling_literal(tables.handle, _dev_ptr(Wtt, nW, "Wtt"), _dev_ptr(Wpp, nW, "Wpp"), nW,
                                              _dev_ptr(out.get("TT"), N * N, "TT"), _dev_ptr(out.get("EE"), N * N, "EE"),
                                              _stream_ptr(stream)), "tj_coupling_literal")
    return out


def coupling_host(tables: Tables, Wtt, Wtp, Wpp, out: dict, band_lcut: int | None = None, stream=None):
    """tj_coupling_host: HOST tensors in, HOST tensors out (`out`: dict name -> preallocated CPU
    float64 tensor, ideally pinned).  Synchronises before returning."""
    N = tables.lmax + 1
    if band_lcut is None:
        band, n, nw, per = 0, tables.l3max + 1, tables.l3max + 1, N * N
    else:
        band, n, nw, per = 1, int(band_lcut), int(band_lcut) + 1, N * (2 * int(band_lcut) + 1)
    args = [_host_ptr(out.get(k), per, k) for k in _BLOCKS]
    _check(load_library().tj_coupling_host(tables.handle, band, n, _host_ptr(Wtt, nw, "Wtt"), _host_ptr(Wtp, nw, "Wtp"),
                                           _host_ptr(Wpp, nw, "Wpp"), *args, _stream_ptr(stream)), "tj_coupling_host")
    return out


def chunk_plan(lmax: int, nparts: int, tt_only: bool = False):
    """tj_chunk_plan (host side, no GPU): (bounds, owner) -- the row chunks of a matrix shared by nparts devices and
    the device each belongs to."""
    cap = 12 * int(nparts) + 1
    b, o, n = (ctypes.c_int * cap)(), (ctypes.c_int * cap)(), ctypes.c_int()
    _check(load_library().tj_chunk_plan(int(lmax), 1 if tt_only else 0, int(nparts), b, o, ctypes.byref(n)), "tj_chunk_plan")
    return [int(b[k]) for k in range(n.value + 1)], [int(o[k]) for k in range(n.value)]


def coupling_host_part(tables: Tables, part: int, nparts: int, Wtt, Wtp, Wpp, out: dict, stream=None):
    """tj_coupling_host_part: this part's share of a dense host-buffer call (HOST tensors; only the regions of the
    part's chunks are written into `out`).  Synchronises before returning."""
    N = tables.lmax + 1
    nW = tables.l3max + 1
    args = [_host_ptr(out.get(k), N * N, k) for k in _BLOCKS]
    _check(load_library().tj_coupling_host_part(tables.handle, int(part), int(nparts), nW, _host_ptr(Wtt, nW, "Wtt"),
                                                _host_ptr(Wtp, nW, "Wtp"), _host_ptr(Wpp, nW, "Wpp"), *args,
                                                _stream_ptr(stream)), "tj_coupling_host_part")
    return out


def coupling_host_multi(tables_list, Wtt, Wtp, Wpp, out: dict, streams=None):
    """tj_coupling_host_multi: one matrix set computed by len(tables_list) handles (one per GPU; distinct handles on
    one GPU also work), every pair swept once, all regions delivered into the one set of HOST tensors `out`."""
    T0 = tables_list[0]
    N = T0.lmax + 1
    nW = T0.l3max + 1
    n = len(tables_list)
    harr = (ctypes.c_void_p * n)(*[t.handle for t in tables_list])
    sarr = None if streams is None else (ctypes.c_void_p * n)(*[s.cuda_stream for s in streams])
    args = [_host_ptr(out.get(k), N * N, k) for k in _BLOCKS]
    _check(load_library().tj_coupling_host_multi(harr, n, nW, _host_ptr(Wtt, nW, "Wtt"), _host_ptr(Wtp, nW, "Wtp"),
                                                 _host_ptr(Wpp, nW, "Wpp"), *args, sarr), "tj_coupling_host_multi")
    return out


def set_host_pipeline(tables: Tables, d2h_bytes_per_s: float = 0.0, fp64_instr_per_s: float = 0.0) -> None:
    """tj_set_host_pipeline: the machine rates behind the regime choice of the dense host-buffer call (0: default)."""
    _check(load_library().tj_set_host_pipeline(tables.handle, float(d2h_bytes_per_s), float(fp64_instr_per_s)),
           "tj_set_host_pipeline")


def host_pipeline_info(tables: Tables):
    """tj_host_pipeline_info: (regime, row chunks) of the handle's most recent dense host-buffer call;
    regime 0 none yet, 1 copy-bound (whole rows), 2 compute-bound (L-shaped regions), 3 pageable outputs."""
    a, b = ctypes.c_int(), ctypes.c_int()
    _check(load_library().tj_host_pipeline_info(tables.handle, ctypes.byref(a), ctypes.byref(b)), "tj_host_pipeline_info")
    return a.value, b.value


def l3_range(l1, l2, l3max, parity):
    lo, hi, n = ctypes.c_int(), ctypes.c_int(), ctypes.c_int()
    _check(load_library().tj_l3_range(l1, l2, l3max, parity, ctypes.byref(lo), ctypes.byref(hi), ctypes.byref(n)),
           "tj_l3_range")
    return lo.value, hi.value, n.value


def sweep_counts(l1, l2, l3max):
    a, b, c, d = (ctypes.c_int() for _ in range(4))
    _check(load_library().tj_sweep_counts(l1, l2, l3max, ctypes.byref(a), ctypes.byref(b), ctypes.byref(c), ctypes.byref(d)),
           "tj_sweep_counts")
    return a.value, b.value, c.value, d.value


def profile_launches() -> int:
    """Kernels this thread's calls have launched so far (take differences)."""
    n = ctypes.c_longlong()
    _check(load_library().tj_profile_launches(ctypes.byref(n)), "tj_profile_launches")
    return int(n.value)


def profile_last_sweep() -> dict:
    """The sweep kernel this thread's most recent coupling call launched (include/tj.h)."""
    g = (ctypes.c_int * 10)()
    _check(load_library().tj_profile_last_sweep(g), "tj_profile_last_sweep")
    keys = ("R", "mask", "TS", "minb", "pipe", "nw", "spin", "rows", "diag", "ctas")
    d = dict(zip(keys, (int(x) for x in g)))
    blocks = "|".join(n for b, n in ((1, "TT"), (2, "TE"), (4, "EE"), (8, "EB")) if d["mask"] & b)
    if d["TS"] == 0:
        d["name"] = "small_kernel<%s,R=%d> x %d CTAs of 128 threads" % (blocks, d["R"], d["ctas"])
    else:
        d["name"] = "sweep_tma_kernel<R=%d,%s,TS=%d,MINB=%d,PIPE=%d,NW=%d,SPIN=%d,ROWS=%d,DIAG=%d> x %d one-warp CTAs" % (
            d["R"], blocks, d["TS"], d["minb"], d["pipe"], d["nw"], d["spin"], d["rows"], d["diag"], d["ctas"])
    return d


def profile_enable(on: bool) -> None:
    _check(load_library().tj_profile_enable(1 if on else 0), "tj_profile_enable")


def profile_get():
    """(prepare_ms, sweep_ms, writer_ms) of this thread's most recent coupling call."""
    arr = (ctypes.c_double * 3)()
    _check(load_library().tj_profile_get(arr), "tj_profile_get")
    return float(arr[0]), float(arr[1]), float(arr[2])
