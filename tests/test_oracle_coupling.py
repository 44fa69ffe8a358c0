"""T0: the oracle's matrices against closed forms, invariants and brute force.

Pins:
  A  full sky W_l = 4 pi delta_{l0}  =>  TT = I; TE = EE = BB = I on l >= 2, 0 for l < 2; EB = 0;
     off-diagonals exactly 0.0 (north_star).
  B  flat W_l = 1, l3max = 2 lmax    =>  TT = (2 l2+1)/(4 pi); TE = 0; EE+EB = (2 l2+1)/(4 pi) on l >= 2
     (orthogonality of the 3j symbols over l3 at fixed m).
  C  spike W_l = delta_{l,L}         =>  each entry is one exact squared symbol (Racah rational).
  D  brute force: every sum re-done in exact rational arithmetic with Racah symbols, l <= 7,
     random rational windows incl. negative entries and a truncated l3max.
  E  Xi symmetric: K[l1][l2]/(2 l2+1) = K[l2][l1]/(2 l1+1)  (PAPER.md:236 as read in SURVEY.md 8(c.3) #8).
  F  band-limited == full sum with the window zero-padded.
"""
import math
from fractions import Fraction

import numpy as np

import oracle
from paper_2602_15605_b200 import windows
from racah import threej_sq_sign

FOUR_PI = 4.0 * math.pi


def test_full_sky_identity():
    lmax = 40
    W = windows.full_sky(2 * lmax)
    K = oracle.coupling_full(lmax, 2 * lmax, W, W, W)
    N = lmax + 1
    I = np.eye(N)
    off = ~np.eye(N, dtype=bool)
    for k in ("TT", "TE", "EE", "BB", "EB"):
        assert np.all(K[k][off] == 0.0), k  # exactly zero
    np.testing.assert_allclose(np.diag(K["TT"]), 1.0, rtol=4e-15)
    Ipol = I.copy()
    Ipol[0, 0] = Ipol[1, 1] = 0.0
    for k in ("TE", "EE", "BB"):
        np.testing.assert_allclose(np.diag(K[k]), np.diag(Ipol), rtol=4e-15, atol=0)
    assert np.all(K["EB"] == 0.0)


def test_flat_window_closed_form():
    lmax = 48
    W = windows.flat(2 * lmax)
    K = oracle.coupling_full(lmax, 2 * lmax, W, W, W)
    N = lmax + 1
    expect = np.broadcast_to((2.0 * np.arange(N) + 1.0) / FOUR_PI, (N, N))
    np.testing.assert_allclose(K["TT"], expect, rtol=2e-13)
    # TE: sum_l3 (2l3+1) (000)(-2 2 0) = delta_{0,-2} delta_{0,2} = 0 (different m: orthogonal)
    assert np.max(np.abs(K["TE"])) < 1e-13
    s = K["EE"] + K["EB"]
    np.testing.assert_allclose(s[2:, 2:], expect[2:, 2:], rtol=2e-13)
    assert np.all(K["EE"][:2] == 0) and np.all(K["EE"][:, :2] == 0)
    assert np.all(K["EB"][:2] == 0) and np.all(K["EB"][:, :2] == 0)
    assert np.all(K["TE"][:2] == 0) and np.all(K["TE"][:, :2] == 0)


def test_spike_windows_isolate_exact_symbols():
    lmax = 14
    for L in (0, 1, 2, 5, 9, 20, 28):
        W = windows.spike(2 * lmax, L)
        K = oracle.coupling_full(lmax, 2 * lmax, W, W, W)
        for l1 in range(lmax + 1):
            for l2 in range(lmax + 1):
                pref = (2 * l2 + 1) * (2 * L + 1) / FOUR_PI
                s0, g0 = threej_sq_sign(l1, l2, L, 0, 0, 0)
                s2, g2 = threej_sq_sign(l1, l2, L, -2, 2, 0)
                even = (l1 + l2 + L) % 2 == 0
                tt = pref * float(s0)
                te = pref * g0 * g2 * math.sqrt(float(s0) * float(s2)) if even else 0.0
                ee = pref * float(s2) if even else 0.0
                eb = pref * float(s2) if not even else 0.0
                for name, ex in (("TT", tt), ("TE", te), ("EE", ee), ("EB", eb)):
                    got = K[name][l1, l2]
                    # accidental zeros of the spin-2 symbol (e.g. (3 3 2;-2 2 0)) come out as ~1e-16 noise
                    assert abs(got - ex) <= 2e-13 * abs(ex) + 2e-16 * pref, (L, l1, l2, name, got, ex)


def test_brute_force_exact_rational():
    lmax = 7
    rng = np.random.default_rng(42)
    for l3max in (2 * lmax, 9, 3):
        num = rng.integers(-20, 40, size=(3, l3max + 1))
        Wf = [[Fraction(int(n), 17) for n in row] for row in num]
        Wd = [np.array([float(x) for x in row]) for row in Wf]
        K = oracle.coupling_full(lmax, l3max, *Wd)
        for l1 in range(lmax + 1):
            for l2 in range(lmax + 1):
                acc = {"TT": Fraction(0), "EE": Fraction(0), "EB": Fraction(0)}
                te = 0.0
                for l3 in range(abs(l1 - l2), min(l1 + l2, l3max) + 1):
                    s0, g0 = threej_sq_sign(l1, l2, l3, 0, 0, 0)
                    s2, g2 = threej_sq_sign(l1, l2, l3, -2, 2, 0)
                    w = 2 * l3 + 1
                    acc["TT"] += w * Wf[0][l3] * s0
                    if (l1 + l2 + l3) % 2 == 0:
                        acc["EE"] += w * Wf[2][l3] * s2
                        te += w * float(Wf[1][l3]) * g0 * g2 * math.sqrt(float(s0 * s2))
                    else:
                        acc["EB"] += w * Wf[2][l3] * s2
                pref = (2 * l2 + 1) / FOUR_PI
                scale = pref * sum(abs(float(x)) for x in Wf[0]) * 0.1
                for name in ("TT", "EE", "EB"):
                    ex = pref * float(acc[name])
                    assert abs(K[name][l1, l2] - ex) <= 1e-13 * abs(ex) + 1e-15 * scale, (l3max, l1, l2, name)
                assert abs(K["TE"][l1, l2] - pref * te) <= 1e-13 * abs(pref * te) + 1e-15 * scale
                assert np.array_equal(K["BB"], K["EE"])


def test_xi_symmetry():
    wl = windows.config(1, lmax=60)
    K = oracle.coupling_full(wl.lmax, wl.l3max, wl.Wtt, wl.Wtp, wl.Wpp)
    w = 2.0 * np.arange(wl.lmax + 1) + 1.0
    for k in ("TT", "TE", "EE", "EB"):
        Xi = K[k] / w[None, :]
        np.testing.assert_allclose(Xi, Xi.T, rtol=1e-12, atol=1e-18)


def test_band_equals_zero_padded_full():
    lmax, lcut = 70, 12
    wl = windows.config(4, lmax=lmax)
    W = wl.Wtt[: lcut + 1].copy()
    band = oracle.coupling_band(lmax, lcut, W, W, W)
    Wpad = np.zeros(2 * lmax + 1)
    Wpad[: lcut + 1] = W
    full = oracle.coupling_full(lmax, 2 * lmax, Wpad, Wpad, Wpad)
    for k in ("TT", "TE", "EE", "BB", "EB"):
        F = full[k]
        for l1 in range(lmax + 1):
            for o in range(-lcut, lcut + 1):
                l2 = l1 + o
                v = band[k][l1, o + lcut]
                if 0 <= l2 <= lmax:
                    assert abs(v - F[l1, l2]) <= 1e-13 * abs(F[l1, l2]) + 1e-18
                else:
                    assert v == 0.0
        # outside the band the full matrix vanishes: |l1-l2| > lcut has no l3 <= lcut in the triangle
        i, j = np.indices(F.shape)
        assert np.all(F[np.abs(i - j) > lcut] == 0.0)


def test_windows_recipe_is_seeded_and_shaped():
    a = windows.config(1, lmax=50)
    b = windows.config(1, lmax=50)
    assert np.array_equal(a.Wtt, b.Wtt) and np.array_equal(a.Wpp, b.Wpp)
    assert a.Wtt.shape == (101,) and np.all(a.Wtt > 0) and np.all(a.Wpp > 0)
    np.testing.assert_allclose(a.Wtp ** 2, a.Wtt * a.Wpp, rtol=1e-14)
    c4 = windows.config(4, lmax=400)
    assert c4.l3max == 300 and c4.band and c4.Wtt.shape == (301,)
    # term counts: brute force on a tiny case
    lmax, l3max = 9, 11
    E = O = P = 0
    for l1 in range(lmax + 1):
        for l2 in range(l1, lmax + 1):
            ne = oracle.l3_range(l1, l2, l3max, 0)[2]
            no = oracle.l3_range(l1, l2, l3max, 1)[2]
            E += ne
            O += no
            P += 1 if ne + no > 0 else 0
    assert windows.term_counts(lmax, l3max) == (E, O, P)


def test_band_row_sum_rule():
    """Orthogonality over the third l at fixed m's (sum_l2 (2 l2+1) (l1 l2 l3; m1 m2 m3)^2 = 1): a row of a band-limited
    matrix that holds its whole triangle (lcut <= l1 <= lmax-lcut) sums to sum_l3 (2 l3+1) W_l3 / 4 pi, for TT with W^TT
    and for EE+EB with W^PP (l1 >= 2), whatever the window -- signed windows included.  (TE has no such rule.)"""
    lmax, lcut = 60, 9
    l = np.arange(lcut + 1, dtype=np.float64)
    Wtt = np.exp(-l * l / 20.0) * (1.0 - 0.3 * l)       # changes sign at l = 4
    Wpp = np.cos(0.7 * l) + 0.2
    Wtp = 0.5 * Wtt + 0.1
    r = oracle.coupling_band(lmax, lcut, Wtt, Wtp, Wpp)
    c = lambda w: float(((2 * l + 1) * w).sum() / (4 * math.pi))   # noqa: E731
    rows = slice(max(lcut, 2), lmax - lcut + 1)
    scale = float(((2 * l + 1) * np.abs(Wtt)).sum() / (4 * math.pi))
    assert np.abs(r["TT"][rows].sum(1) - c(Wtt)).max() < 1e-13 * scale
    scale = float(((2 * l + 1) * np.abs(Wpp)).sum() / (4 * math.pi))
    assert np.abs((r["EE"] + r["EB"])[rows].sum(1) - c(Wpp)).max() < 1e-13 * scale
    # a row that does NOT hold its whole triangle falls short (the rule is not vacuous)
    assert abs(r["TT"][lmax].sum() - c(Wtt)) > 1e-3 * scale
