"""Definition of the lookup-table entries, in exact integer arithmetic.  TEST INFRASTRUCTURE.

PAPER.md:166-170 Eq. 11:   g(p) = (2p)! / (2^{2p} (p!)^2) = C(2p,p) / 4^p,  g(0) = 1.
PAPER.md:186: the method stores g(p), 1/g(p) and 1/(J+1) (J = 2p on the even-J branch).

The values are exact rationals; `float(Fraction)` / Python's int true division round them
correctly (round-half-even) to float64, so every entry returned here is the correctly rounded
value of its definition.  Nothing here is shared with the CUDA table kernel.

Pins (tests/test_oracle_tables.py, `-m "not gpu"`): numerator/denominator == (math.comb(2p,p), 4^p) as
integers (every p <= 1500, strided to p = 32001); g(0..2) = 1, 1/2, 3/8 and Eq. 12 in exact Fractions;
the convolution identity sum_k g(k) g(n-k) = 1; ln g against lgamma for EVERY p <= 32001; Stirling's limit
g(p) sqrt(pi p) = 1 - 1/(8p) + ...; all five derived entries against exact Fractions (p <= 300) and against
mpmath's gamma function at 60 digits (strided to p = 32001).  No function here is "parity unpinned".
"""
from __future__ import annotations

import math
from fractions import Fraction

import numpy as np


def g_exact_fraction(p: int) -> Fraction:
    """g(p) straight from Eq. 11 (one binomial coefficient per call; slow for large p)."""
    if p < 0:
        raise ValueError("p >= 0")
    return Fraction(math.comb(2 * p, p), 4 ** p)


def _g_num_den(pmax: int):
    """Yield (p, num, den) with g(p) = num/den exactly; C(2p,p) advanced by
    C(2p,p) = C(2p-2,p-1) * 2(2p-1)/p  (exact integer division), den = 4^p."""
    c = 1
    for p in range(0, pmax + 1):
        if p > 0:
            c = c * (2 * (2 * p - 1)) // p
        yield p, c, 1 << (2 * p)


def g_table_float(pmax: int) -> np.ndarray:
    """Correctly rounded float64 g(p), p = 0..pmax."""
    out = np.empty(pmax + 1)
    for p, num, den in _g_num_den(pmax):
        out[p] = num / den
    return out


def table_entries_float(pmax: int) -> dict:
    """Correctly rounded float64 values, p = 0..pmax, of
         g     = g(p)
         ginv  = 1/g(p)
         h     = 1/((2p+1) g(p))      (the 1/(J+1) factor of Eq. 10 at J = 2p, times 1/g(p))
         gA    = 2p g(p)
         gB    = (2p+1) g(p)
    The last three are plain products/quotients of Eq. 10-11 quantities by exact integers."""
    names = ("g", "ginv", "h", "gA", "gB")
    out = {k: np.empty(pmax + 1) for k in names}
    for p, num, den in _g_num_den(pmax):
        out["g"][p] = num / den
        out["ginv"][p] = den / num
        out["h"][p] = den / ((2 * p + 1) * num)
        out["gA"][p] = (2 * p * num) / den
        out["gB"][p] = ((2 * p + 1) * num) / den
    return out
