"""bench_cpu/tablemethod.c (the paper's CPU design restated, a bench-only baseline) against the oracle."""
import numpy as np
import pytest

import bench_cpu
import oracle
from paper_2602_15605_b200 import windows


def _close(a, b, what):
    err = np.abs(a - b)
    big = np.abs(b) >= 1e-4
    assert np.all(err[big] <= 1e-9 * np.abs(b[big])), what
    assert np.all(err[~big] <= 1e-13), what


@pytest.mark.parametrize("lmax,l3max", [(0, 0), (1, 2), (2, 4), (37, 74), (120, 240), (300, 600), (150, 97)])
def test_full_matrices_against_oracle(lmax, l3max):
    wl = windows.config(1, lmax=max(lmax, 2))
    Wtt, Wpp = wl.Wtt[: l3max + 1].copy(), wl.Wpp[: l3max + 1].copy()
    got = bench_cpu.coupling_rows(lmax, l3max, Wtt, Wpp)
    ref = oracle.coupling_full(lmax, l3max, Wtt, None, Wpp)
    _close(got["TT"], ref["TT"], "TT")
    _close(got["EE"], ref["EE"], "EE")


def test_sampled_rows_match_full_and_oracle():
    lmax = 260
    wl = windows.config(2, lmax=lmax)
    rows = np.array([0, 1, 2, 3, 77, 130, 259, 260], dtype=np.int32)
    full = bench_cpu.coupling_rows(lmax, 2 * lmax, wl.Wtt, wl.Wpp)
    part = bench_cpu.coupling_rows(lmax, 2 * lmax, wl.Wtt, wl.Wpp, rows)
    ref = oracle.coupling_rows(lmax, 2 * lmax, wl.Wtt, None, wl.Wpp, rows)
    for k in ("TT", "EE"):
        _close(part[k], ref[k], k)
        _close(full[k][rows], ref[k], k + " (triangle + mirror)")
    only_tt = bench_cpu.coupling_rows(lmax, 2 * lmax, wl.Wtt, None, rows)
    assert set(only_tt) == {"TT"} and np.array_equal(only_tt["TT"], part["TT"])


def test_flat_window_closed_form():
    lmax = 200
    W = np.ones(2 * lmax + 1)
    got = bench_cpu.coupling_rows(lmax, 2 * lmax, W, None)
    expect = np.broadcast_to((2.0 * np.arange(lmax + 1) + 1.0) / (4.0 * np.pi), (lmax + 1, lmax + 1))
    np.testing.assert_allclose(got["TT"], expect, rtol=1e-11)
