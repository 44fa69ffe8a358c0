"""Pins of oracle.coupling_binned (the binned sum of the oracle's own entries, reading 20).

Closed forms that follow from the pinned matrices: full sky (K = identity, Eq. 3 with W = 4 pi delta_{l0})
and the flat window (K_{l1 l2} = (2 l2+1)/4 pi); plus brute force against the full matrices, empty bins, bins that
leave multipoles out, and the additivity of merged bins."""
import math

import numpy as np

import oracle
from paper_2602_15605_b200 import windows


def _weights(lmax, seed):
    rng = np.random.default_rng(seed)
    return rng.uniform(0.5, 1.5, lmax + 1), rng.uniform(0.5, 1.5, lmax + 1)


def test_full_sky_gives_weighted_identity():
    lmax = 40
    W = np.zeros(2 * lmax + 1)
    W[0] = 4.0 * math.pi
    edges = [0, 2, 5, 5, 17, 30, 41]          # one empty bin
    P, Q = _weights(lmax, 1)
    B = oracle.coupling_binned(lmax, 2 * lmax, W, W, W, edges, P, Q)
    nb = len(edges) - 1
    for k in ("TT", "TE", "EE", "BB"):
        for b in range(nb):
            lo = edges[b] if k == "TT" else max(edges[b], 2)     # polarised identity only for l >= 2
            d = float(np.sum(P[lo:edges[b + 1]] * Q[lo:edges[b + 1]]))
            for c in range(nb):
                want = d if b == c else 0.0
                assert abs(B[k][b, c] - want) <= 1e-13 * max(1.0, abs(want)), (k, b, c)
    assert np.all(B["EB"] == 0.0)


def test_flat_window_closed_form():
    lmax = 60
    W = np.ones(2 * lmax + 1)
    edges = [2, 10, 11, 40, 61]
    P, Q = _weights(lmax, 2)
    B = oracle.coupling_binned(lmax, 2 * lmax, W, None, None, edges, P, Q)
    l = np.arange(lmax + 1)
    for b in range(4):
        for c in range(4):
            want = P[edges[b]:edges[b + 1]].sum() * (Q[edges[c]:edges[c + 1]] * (2 * l[edges[c]:edges[c + 1]] + 1)).sum() / (4 * math.pi)
            assert abs(B["TT"][b, c] - want) <= 1e-12 * want


def test_equals_weighted_sums_of_full_matrices_and_is_additive():
    lmax = 33
    wl = windows.config(1, lmax=lmax)
    K = oracle.coupling_full(lmax, 2 * lmax, wl.Wtt, wl.Wtp, wl.Wpp)
    P, Q = _weights(lmax, 3)
    edges = [1, 4, 9, 20, 34]                 # l = 0 left out
    B = oracle.coupling_binned(lmax, 2 * lmax, wl.Wtt, wl.Wtp, wl.Wpp, edges, P, Q)
    for k in ("TT", "TE", "EE", "BB", "EB"):
        for b in range(4):
            for c in range(4):
                want = sum(P[i] * K[k][i, j] * Q[j] for i in range(edges[b], edges[b + 1]) for j in range(edges[c], edges[c + 1]))
                assert abs(B[k][b, c] - want) <= 1e-12 * max(abs(want), 1e-3), (k, b, c)
    # merging two bins adds their rows / columns
    M = oracle.coupling_binned(lmax, 2 * lmax, wl.Wtt, wl.Wtp, wl.Wpp, [1, 9, 20, 34], P, Q)
    for k in ("TT", "EB"):
        assert np.allclose(M[k][0, 1:], B[k][0, 2:] + B[k][1, 2:], rtol=1e-12, atol=1e-15)
        assert np.allclose(M[k][1:, 0], B[k][2:, 0] + B[k][2:, 1], rtol=1e-12, atol=1e-15)
    assert np.array_equal(B["BB"], B["EE"])
    part = oracle.coupling_binned(lmax, 2 * lmax, wl.Wtt, None, None, edges, P, Q, pairs=[(3, 0)])
    assert part["TT"][3, 0] == B["TT"][3, 0] and np.isnan(part["TT"][0, 0])
