"""Pins of the oracle's spin-1 blocks (oracle_coupling_spin1_pairs; DESIGN.md 2 reading 19; the (0,-1,1)
symbols of PAPER.md:51-53, :362-392).  Same kinds of pin as the spin-2 blocks (test_oracle_coupling.py):

  A  full sky W_l = 4 pi delta_{l0}: (l l 0;m -m 0) = (-1)^{l-m}/sqrt(2l+1)  =>  K11+ = I on l >= 1,
     K01 = -I on l >= 1 (the (000) and (-1 1 0) symbols at l3 = 0 have opposite signs), K11- = 0,
     off-diagonals exactly 0.0.
  B  flat W_l = 1, l3max = 2 lmax: K11+ + K11- = (2 l2+1)/(4 pi) on l >= 1, K01 = 0 (orthogonality over l3).
  C  brute force in exact rational arithmetic with Racah symbols, l <= 7, signed windows, truncated l3max.
  D  the single symbols themselves: test_oracle_3j.py (Racah, all l <= 30, m = (-1,1)).
"""
import math
from fractions import Fraction

import numpy as np

import oracle
from paper_2602_15605_b200 import windows
from racah import threej_sq_sign

FOUR_PI = 4.0 * math.pi


def test_spin1_full_sky():
    lmax = 40
    W = windows.full_sky(2 * lmax)
    K = oracle.spin1_full(lmax, 2 * lmax, W, W)
    N = lmax + 1
    off = ~np.eye(N, dtype=bool)
    for k in ("K01", "K11p", "K11m"):
        assert np.all(K[k][off] == 0.0), k
    d = np.ones(N)
    d[0] = 0.0
    np.testing.assert_allclose(np.diag(K["K11p"]), d, rtol=4e-15, atol=0)
    np.testing.assert_allclose(np.diag(K["K01"]), -d, rtol=4e-15, atol=0)
    assert np.all(K["K11m"] == 0.0)


def test_spin1_flat_window():
    lmax = 48
    W = windows.flat(2 * lmax)
    K = oracle.spin1_full(lmax, 2 * lmax, W, W)
    N = lmax + 1
    expect = np.broadcast_to((2.0 * np.arange(N) + 1.0) / FOUR_PI, (N, N))
    s = K["K11p"] + K["K11m"]
    np.testing.assert_allclose(s[1:, 1:], expect[1:, 1:], rtol=2e-13)
    assert np.max(np.abs(K["K01"])) < 1e-13
    for k in ("K01", "K11p", "K11m"):
        assert np.all(K[k][0] == 0) and np.all(K[k][:, 0] == 0), k


def test_spin1_brute_force_exact_rational():
    lmax = 7
    rng = np.random.default_rng(43)
    for l3max in (2 * lmax, 9, 3):
        num = rng.integers(-20, 40, size=(2, l3max + 1))
        Wf = [[Fraction(int(n), 17) for n in row] for row in num]
        Wd = [np.array([float(x) for x in row]) for row in Wf]
        K = oracle.spin1_full(lmax, l3max, *Wd)
        for l1 in range(lmax + 1):
            for l2 in range(lmax + 1):
                p = Fraction(0)
                m = Fraction(0)
                x = 0.0
                for l3 in range(abs(l1 - l2), min(l1 + l2, l3max) + 1):
                    s0, g0 = threej_sq_sign(l1, l2, l3, 0, 0, 0)
                    s1, g1 = threej_sq_sign(l1, l2, l3, -1, 1, 0)
                    w = 2 * l3 + 1
                    if (l1 + l2 + l3) % 2 == 0:
                        p += w * Wf[1][l3] * s1
                        x += w * float(Wf[0][l3]) * g0 * g1 * math.sqrt(float(s0 * s1))
                    else:
                        m += w * Wf[1][l3] * s1
                pref = (2 * l2 + 1) / FOUR_PI
                scale = pref * sum(abs(float(v)) for v in Wf[1]) * 0.1
                assert abs(K["K11p"][l1, l2] - pref * float(p)) <= 1e-13 * abs(pref * float(p)) + 1e-15 * scale
                assert abs(K["K11m"][l1, l2] - pref * float(m)) <= 1e-13 * abs(pref * float(m)) + 1e-15 * scale
                assert abs(K["K01"][l1, l2] - pref * x) <= 1e-13 * abs(pref * x) + 1e-15 * scale
