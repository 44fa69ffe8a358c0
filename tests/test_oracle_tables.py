"""CPU-side pins of oracle/tables.py, the checker of the table-build kernel (row a1).

PAPER.md:166-170 Eq. 11: g(p) = (2p)!/(2^{2p} (p!)^2) = C(2p,p)/4^p, g(0) = 1, g(p) ~ (pi p)^(-1/2);
PAPER.md:172-184 Eq. 12: g(p) = (p - 1/2)/p * g(p-1);  PAPER.md:186: the stored tables g, 1/g, 1/(J+1).

Every check below goes through something other than the routine under test: Python's binomial
coefficient, mpmath's gamma function at 50 digits, exact Fractions, the convolution identity of the
central binomial coefficients, and Stirling's limit.
"""
from __future__ import annotations

import math
from fractions import Fraction

import numpy as np
import pytest

from oracle import tables

PMAX = 2 * 16000 + 1   # largest table any GPU test builds (lmax = 16000)


@pytest.fixture(scope="module")
def numden():
    return list(tables._g_num_den(PMAX))


def test_num_den_equal_binomial_exactly(numden):
    # integers, not floats: every p up to 1500, then a stride that is coprime to every small period, then the end
    ps = list(range(0, 1501)) + list(range(1501, PMAX + 1, 1009)) + [PMAX - 1, PMAX]
    for p in ps:
        q, num, den = numden[p]
        assert q == p
        assert num == math.comb(2 * p, p), p
        assert den == 4 ** p, p


def test_first_values_and_recurrence_eq12(numden):
    g = [Fraction(n, d) for _, n, d in numden[:400]]
    assert g[0] == 1 and g[1] == Fraction(1, 2) and g[2] == Fraction(3, 8)
    for p in range(1, 400):
        assert g[p] == g[p - 1] * Fraction(2 * p - 1, 2 * p)                      # Eq. 12
        assert g[p] == tables.g_exact_fraction(p)                                 # Eq. 11 via math.comb


def test_convolution_identity_exact(numden):
    # sum_k C(2k,k) C(2n-2k,n-k) = 4^n  <=>  sum_k g(k) g(n-k) = 1: ties every entry to all others
    for n in (0, 1, 2, 3, 17, 64, 255, 600):
        s = sum(numden[k][1] * numden[n - k][1] for k in range(n + 1))
        assert s == 4 ** n


def test_all_entries_against_lgamma(numden):
    # every p: ln g(p) = lgamma(2p+1) - 2 lgamma(p+1) - 2p ln 2.  lgamma carries ~1e-16 of its VALUE (~4e5), so
    # 1e-9 on ln g; an index slip anywhere changes g by 1/(2p) >= 1.5e-5
    g = tables.g_table_float(PMAX)
    for p in range(1, PMAX + 1):
        lg = math.lgamma(2 * p + 1) - 2.0 * math.lgamma(p + 1) - 2.0 * p * math.log(2.0)
        assert abs(math.log(g[p]) - lg) < 1e-9, p
    assert g[0] == 1.0


def test_stirling_limit():
    g = tables.g_table_float(PMAX)
    p = np.arange(1, PMAX + 1, dtype=np.float64)
    r = g[1:] * np.sqrt(np.pi * p)
    # g(p) sqrt(pi p) = 1 - 1/(8p) + O(p^-2)   (PAPER.md:170 gives the leading term)
    assert np.all(np.abs(r - (1.0 - 1.0 / (8.0 * p))) < 1.0 / (64.0 * p * p) + 1e-15)   # next term: +1/(128 p^2)
    assert abs(r[-1] - 1.0) < 1e-5
    assert np.all(np.diff(g) < 0)             # strictly decreasing


def test_table_entries_are_correctly_rounded_definitions_small_p():
    pmax = 300
    t = tables.table_entries_float(pmax)
    for p in range(pmax + 1):
        g = Fraction(math.comb(2 * p, p), 4 ** p)
        assert t["g"][p] == float(g)
        assert t["ginv"][p] == float(1 / g)
        assert t["h"][p] == float(1 / ((2 * p + 1) * g))      # 1/((J+1) g(p)) at J = 2p  (Eq. 10)
        assert t["gA"][p] == float(2 * p * g)
        assert t["gB"][p] == float((2 * p + 1) * g)
    assert t["gA"][0] == 0.0                                  # closes the odd-J branch at t = min(l1,l2)


def test_table_entries_against_mpmath_large_p():
    mp = pytest.importorskip("mpmath")
    t = tables.table_entries_float(PMAX)
    gf = tables.g_table_float(PMAX)
    assert np.array_equal(gf, t["g"])
    with mp.workdps(60):
        for p in list(range(301, PMAX, 487)) + [10000, 20001, PMAX]:
            g = mp.gamma(2 * p + 1) / (mp.gamma(p + 1) ** 2 * mp.mpf(4) ** p)
            ref = {"g": g, "ginv": 1 / g, "h": 1 / ((2 * p + 1) * g), "gA": 2 * p * g, "gB": (2 * p + 1) * g}
            for k, v in ref.items():
                assert t[k][p] == float(v), (k, p)
