"""Exact Wigner-3j symbols from the Racah single-sum formula, in rational arithmetic.

Textbook formula (Edmonds 1957 Eq. 3.6.11 / 3.7.3; restated in SURVEY.md 8(c.4)):

  (j1 j2 j3; m1 m2 m3) = (-1)^{j1-j2-m3} sqrt(Delta * prod_i (ji+mi)! (ji-mi)!) * S
  Delta = (j1+j2-j3)! (j1-j2+j3)! (-j1+j2+j3)! / (j1+j2+j3+1)!
  S = sum_k (-1)^k / [ k! (j1+j2-j3-k)! (j1-m1-k)! (j2+m2-k)! (j3-j2+m1+k)! (j3-j1-m2+k)! ]

The SQUARE is the rational Delta*prod*S^2 and the sign is sign(S)*(-1)^{j1-j2-m3}; both are
returned exactly.  This is the pin the oracle's Schulten-Gordon recursion is checked against;
it shares nothing with oracle/ or with the CUDA path.
"""
from fractions import Fraction
from functools import lru_cache
from math import factorial as _f


@lru_cache(maxsize=None)
def fact(n):
    return _f(n)


def threej_sq_sign(j1, j2, j3, m1, m2, m3):
    """Return (square as Fraction, sign in {-1,0,+1})."""
    if m1 + m2 + m3 != 0 or abs(m1) > j1 or abs(m2) > j2 or abs(m3) > j3:
        return Fraction(0), 0
    if j3 > j1 + j2 or j3 < abs(j1 - j2):
        return Fraction(0), 0
    kmin = max(0, j2 - j3 - m1, j1 - j3 + m2)
    kmax = min(j1 + j2 - j3, j1 - m1, j2 + m2)
    S = Fraction(0)
    for k in range(kmin, kmax + 1):
        den = (fact(k) * fact(j1 + j2 - j3 - k) * fact(j1 - m1 - k) * fact(j2 + m2 - k)
               * fact(j3 - j2 + m1 + k) * fact(j3 - j1 - m2 + k))
        S += Fraction(-1 if (k & 1) else 1, den)
    if S == 0:
        return Fraction(0), 0
    delta = Fraction(fact(j1 + j2 - j3) * fact(j1 - j2 + j3) * fact(-j1 + j2 + j3), fact(j1 + j2 + j3 + 1))
    pref = (fact(j1 + m1) * fact(j1 - m1) * fact(j2 + m2) * fact(j2 - m2) * fact(j3 + m3) * fact(j3 - m3))
    sq = delta * pref * S * S
    sign = (1 if S > 0 else -1) * (-1 if ((j1 - j2 - m3) & 1) else 1)
    return sq, sign


def threej_float(j1, j2, j3, m1, m2, m3):
    """Correctly-rounded-square-root float value (sign * sqrt(square))."""
    import math
    sq, sg = threej_sq_sign(j1, j2, j3, m1, m2, m3)
    if sg == 0:
        return 0.0
    # sqrt of a rational: sqrt(num/den) = isqrt-scaled; float(Fraction) is correctly rounded and
    # the subsequent sqrt adds <= 0.5 ulp -- ample for a 1e-13 comparison
    return sg * math.sqrt(float(sq))
