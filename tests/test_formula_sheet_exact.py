"""The formula sheet the CUDA kernels implement (DESIGN.md 3 = SURVEY.md 8(c.1)), checked in EXACT
rational arithmetic against Racah symbols for all l1,l2 <= 12.  This pins the *derived* one-product
forms (the paper prints Eqs. 10, 13-16, B14-B17 but not these collapsed forms) independently of both
the oracle and the GPU code: nothing here is imported from either.

  even step t (l3 = s-2t):  X^2 = h[s-t] g[t] g[l1-t] g[l2-t],  h[p] = 1/((2p+1) g(p))       (Eq. 10)
                            (l1 l2 l3;-2 2 0) = X A / sqrt(D),  A = d(d+2)/2 - u1 u2,
                            d = u3 - u1 - u2,  D = D_l1 D_l2,   A2 = (d+1)^2 - (2 u1 u2 + 1) = 2A
  odd step t (l3 = s-2t-1): (l1 l2 l3;-2 2 0)^2 = ginv[s-t] gB[t] gA[l1-t] gA[l2-t] (d+2)^2/(4D)
"""
from fractions import Fraction
from math import comb

from racah import threej_sq_sign

LMAX = 12


def g(p):
    return Fraction(comb(2 * p, p), 4 ** p) if p >= 0 else Fraction(0)


def u(l):
    return l * (l + 1)


def Dl(l):
    return (l - 1) * l * (l + 1) * (l + 2)


def test_eq10_table_form_of_squared_000():
    for l1 in range(LMAX + 1):
        for l2 in range(LMAX + 1):
            s = l1 + l2
            for t in range(0, min(l1, l2) + 1):
                l3 = s - 2 * t
                X2 = g(t) * g(l1 - t) * g(l2 - t) / ((2 * (s - t) + 1) * g(s - t))
                sq, _ = threej_sq_sign(l1, l2, l3, 0, 0, 0)
                assert X2 == sq, (l1, l2, l3)


def test_even_J_spin2_one_product_form():
    for l1 in range(2, LMAX + 1):
        for l2 in range(2, LMAX + 1):
            s = l1 + l2
            D = Dl(l1) * Dl(l2)
            for t in range(0, min(l1, l2) + 1):
                l3 = s - 2 * t
                d = u(l3) - u(l1) - u(l2)
                A = Fraction(d * (d + 2), 2) - u(l1) * u(l2)
                A2 = (d + 1) ** 2 - (2 * u(l1) * u(l2) + 1)
                assert A2 == 2 * A
                x2, sx = threej_sq_sign(l1, l2, l3, 0, 0, 0)
                y2, sy = threej_sq_sign(l1, l2, l3, -2, 2, 0)
                # squares: (spin-2)^2 = X^2 A^2 / D
                assert y2 == x2 * A * A / D, (l1, l2, l3)
                # product sign: X * (spin-2) = X^2 A / sqrt(D): sign(X)*sign(Y) = sign(A)
                sa = (A > 0) - (A < 0)
                assert sx * sy == sa, (l1, l2, l3, sx, sy, sa)


def test_odd_J_spin2_table_form():
    for l1 in range(2, LMAX + 1):
        for l2 in range(2, LMAX + 1):
            s = l1 + l2
            D = Dl(l1) * Dl(l2)
            for t in range(0, min(l1, l2)):
                l3 = s - 2 * t - 1
                d = u(l3) - u(l1) - u(l2)
                gA1 = 2 * (l1 - t) * g(l1 - t)
                gA2 = 2 * (l2 - t) * g(l2 - t)
                gB = (2 * t + 1) * g(t)
                val = gB * gA1 * gA2 / g(s - t) * Fraction((d + 2) ** 2, 4 * D)
                y2, _ = threej_sq_sign(l1, l2, l3, -2, 2, 0)
                assert val == y2, (l1, l2, l3)
            # the odd branch closes by itself at t = min(l1,l2): gA[0] = 0
            t = min(l1, l2)
            assert 2 * (min(l1, l2) - t) * g(min(l1, l2) - t) == 0


def test_guard_band_zero_outside_triangle():
    # g(p) = 0 for p < 0 makes every step outside the triangle vanish
    for l1, l2 in ((3, 7), (5, 5), (0, 4)):
        for t in range(min(l1, l2) + 1, l1 + l2 + 2):
            assert g(t) * g(l1 - t) * g(l2 - t) == 0


def test_whole_sums_random_rational_windows():
    """Xi sums in table form == definition sums (Eqs. A1-A4) with Racah symbols, incl. negative window
    entries and a truncated l3max; TE compared through its exact square-free part:
    TE sum = sum W' X^2 A / sqrt(D)  => (TE sum)^2 * D is rational on both sides."""
    import random
    random.seed(3)
    L = 8
    for l3max in (2 * L, 9):
        W = [Fraction(random.randint(-9, 30), 7) for _ in range(l3max + 1)]
        for l1 in range(2, L + 1):
            for l2 in range(2, L + 1):
                s = l1 + l2
                D = Dl(l1) * Dl(l2)
                tt = te = ee = eb = Fraction(0)
                for t in range(0, min(l1, l2) + 1):
                    l3 = s - 2 * t
                    if l3 <= l3max:
                        X2 = g(t) * g(l1 - t) * g(l2 - t) / ((2 * (s - t) + 1) * g(s - t))
                        d = u(l3) - u(l1) - u(l2)
                        A2 = (d + 1) ** 2 - (2 * u(l1) * u(l2) + 1)
                        w = (2 * l3 + 1) * W[l3]
                        tt += w * X2
                        te += w * X2 * A2          # times 1/(2 sqrt D)
                        ee += w * X2 * A2 * A2     # times 1/(4 D)
                    l3 = s - 2 * t - 1
                    if t < min(l1, l2) and l3 <= l3max:
                        d = u(l3) - u(l1) - u(l2)
                        Z2 = (2 * t + 1) * g(t) * 2 * (l1 - t) * g(l1 - t) * 2 * (l2 - t) * g(l2 - t) / g(s - t)
                        eb += (2 * l3 + 1) * W[l3] * Z2 * (d + 2) ** 2  # times 1/(4 D)
                rtt = ree = reb = Fraction(0)
                rte_times_sqrtD = Fraction(0)
                for l3 in range(abs(l1 - l2), min(s, l3max) + 1):
                    x2, sx = threej_sq_sign(l1, l2, l3, 0, 0, 0)
                    y2, sy = threej_sq_sign(l1, l2, l3, -2, 2, 0)
                    w = (2 * l3 + 1) * W[l3]
                    rtt += w * x2
                    if (s + l3) % 2 == 0:
                        ree += w * y2
                        # X*Y*sqrt(D) = X^2 * A (rational, by the identity checked above)
                        d = u(l3) - u(l1) - u(l2)
                        A = Fraction(d * (d + 2), 2) - u(l1) * u(l2)
                        assert x2 * A * A == y2 * D
                        rte_times_sqrtD += w * sx * sy * abs(x2 * A)
                    else:
                        reb += w * y2
                assert tt == rtt
                assert ee / (4 * D) == ree
                assert eb / (4 * D) == reb
                assert te / 2 == rte_times_sqrtD


def test_spin1_one_product_forms():
    """Spin-1 analogues (PAPER.md:362-392 Eqs. B1-B6, B10 carried to one table product):
       even J: (l1 l2 l3;-1 1 0) = X d / (2 sqrt(u1 u2)),  d = u3 - u1 - u2   (square and sign)
       odd  J: (l1 l2 l3;-1 1 0)^2 = ginv[s-t] gB[t] gA[l1-t] gA[l2-t] / (4 u1 u2)."""
    for l1 in range(1, LMAX + 1):
        for l2 in range(1, LMAX + 1):
            s = l1 + l2
            for t in range(0, min(l1, l2) + 1):
                l3 = s - 2 * t
                d = u(l3) - u(l1) - u(l2)
                x2, sx = threej_sq_sign(l1, l2, l3, 0, 0, 0)
                y2, sy = threej_sq_sign(l1, l2, l3, -1, 1, 0)
                assert y2 == x2 * Fraction(d * d, 4 * u(l1) * u(l2)), (l1, l2, l3)
                assert sx * sy == (d > 0) - (d < 0), (l1, l2, l3)
            for t in range(0, min(l1, l2)):
                l3 = s - 2 * t - 1
                gB = (2 * t + 1) * g(t)
                gA1 = 2 * (l1 - t) * g(l1 - t)
                gA2 = 2 * (l2 - t) * g(l2 - t)
                y2, _ = threej_sq_sign(l1, l2, l3, -1, 1, 0)
                assert y2 == gB * gA1 * gA2 / g(s - t) / (4 * u(l1) * u(l2)), (l1, l2, l3)
