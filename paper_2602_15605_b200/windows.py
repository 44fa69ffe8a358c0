"""Seeded synthetic window power spectra W_l for the BASELINE.json configs.

This module holds NO arithmetic of the method: it only draws the inputs.  It is the one module
the tests hand to both the oracle and the CUDA path (it imports neither).

The paper measures on the ACT DR6 survey window, which is not available here; the
red, log-normally scattered power laws below stand in for it (BASELINE.json `configs`; readings of
the recipe are SURVEY.md 8(c.3) #16-18 and DESIGN.md "Inputs").

  W^X_l = 4 pi f^2 (1 + l/l_c)^(-alpha) exp(sigma N(0,1)),   l = 0..l3max
  RNG: numpy.random.default_rng(seed); standard_normal(l3max+1) drawn for TT first, then PP;
  W^TP = sqrt(W^TT W^PP).
"""
from __future__ import annotations

import math
from dataclasses import dataclass

import numpy as np

FOUR_PI = 4.0 * math.pi


@dataclass(frozen=True)
class Workload:
    name: str
    lmax: int
    l3max: int          # windows have l3max+1 entries; for the band config this is L_cut
    band: bool
    pol: bool
    Wtt: np.ndarray
    Wtp: np.ndarray | None
    Wpp: np.ndarray | None


def power_law(l3max, f, lc, alpha, sigma, noise):
    l = np.arange(l3max + 1, dtype=np.float64)
    return FOUR_PI * f * f * (1.0 + l / lc) ** (-alpha) * np.exp(sigma * noise)


def full_sky(l3max):
    """W_l = 4 pi delta_{l0}: the mask is 1 everywhere, K must be the identity."""
    w = np.zeros(l3max + 1)
    w[0] = FOUR_PI
    return w


def flat(l3max):
    """W_l = 1 for all l: closed form K^TT = (2 l2+1)/(4 pi) by orthogonality."""
    return np.ones(l3max + 1)


def spike(l3max, L):
    """W_l = delta_{l,L}: isolates one squared symbol per matrix entry."""
    w = np.zeros(l3max + 1)
    w[L] = 1.0
    return w


def pol_windows(lmax, tt, pp, sigma, seed, ripple=False, l3max=None):
    l3max = 2 * lmax if l3max is None else l3max
    rng = np.random.default_rng(seed)
    ntt = rng.standard_normal(l3max + 1)
    npp = rng.standard_normal(l3max + 1)
    Wtt = power_law(l3max, *tt, sigma, ntt)
    Wpp = power_law(l3max, *pp, sigma, npp)
    if ripple:
        # multiplicative reading of "plus a 1e-3 sin(l/7) ripple"
        r = 1.0 + 1e-3 * np.sin(np.arange(l3max + 1) / 7.0)
        Wtt = Wtt * r
        Wpp = Wpp * r
    Wtp = np.sqrt(Wtt * Wpp)
    return Wtt, Wtp, Wpp


def config(i: int, lmax: int | None = None) -> Workload:
    """BASELINE.json configs[i].  `lmax` overrides the size (same recipe, smaller problem) for
    tests that need the oracle to finish in seconds."""
    if i == 0:
        lm = 256 if lmax is None else lmax
        rng = np.random.default_rng(0)
        W = power_law(2 * lm, 0.6, 20.0, 2.5, 0.1, rng.standard_normal(2 * lm + 1))
        return Workload("cfg0_tt_lmax%d" % lm, lm, 2 * lm, False, False, W, None, None)
    if i == 1:
        lm = 2000 if lmax is None else lmax
        tt, tp, pp = pol_windows(lm, (0.7, 30.0, 2.5), (0.5, 50.0, 3.0), 0.05, 1)
        return Workload("cfg1_pol_lmax%d" % lm, lm, 2 * lm, False, True, tt, tp, pp)
    if i == 2:
        lm = 5000 if lmax is None else lmax
        tt, tp, pp = pol_windows(lm, (0.6, 40.0, 2.2), (0.45, 60.0, 2.8), 0.05, 2, ripple=True)
        return Workload("cfg2_pol_lmax%d" % lm, lm, 2 * lm, False, True, tt, tp, pp)
    if i == 3:
        lm = 10000 if lmax is None else lmax
        tt, tp, pp = pol_windows(lm, (0.4, 80.0, 2.0), (0.35, 100.0, 2.4), 0.05, 3)
        return Workload("cfg3_pol_lmax%d" % lm, lm, 2 * lm, False, True, tt, tp, pp)
    if i == 4:
        lm = 15000 if lmax is None else lmax
        lcut = 300
        l = np.arange(lcut + 1, dtype=np.float64)
        W = FOUR_PI * 0.5 ** 2 * np.exp(-l * l / (2.0 * 60.0 ** 2))
        # same shape for TT and PP; TP = sqrt(TT*PP) = W (the seed is unused)
        return Workload("cfg4_band_lmax%d_lcut%d" % (lm, lcut), lm, lcut, True, True, W, W.copy(), W.copy())
    raise ValueError("config index 0..4")


def term_counts(lmax: int, l3max: int, lcut_band: bool = False):
    """Number of evaluated l3 terms over the upper triangle l1 <= l2 <= lmax:
    (even-J terms, odd-J terms, pairs).  Pure counting, used by bench.py for the metric.
    With lcut_band only pairs with l2-l1 <= l3max are counted (the stored band)."""
    l1 = np.arange(lmax + 1, dtype=np.int64)[:, None]
    E = O = P = 0
    # row-chunked to bound memory
    step = max(1, 4_000_000 // (lmax + 1))
    l2 = np.arange(lmax + 1, dtype=np.int64)[None, :]
    for a in range(0, lmax + 1, step):
        r = l1[a:a + step]
        lo = l2 - r
        hi = np.minimum(r + l2, l3max)
        m = (l2 >= r) & (hi >= lo)
        ne = np.where(m, (hi - ((r + l2 + hi) & 1) - lo) // 2 + 1, 0)
        lo1 = lo + 1
        hi1 = hi - (1 - ((r + l2 + hi) & 1))
        no = np.where(m & (hi1 >= lo1), (hi1 - lo1) // 2 + 1, 0)
        E += int(ne.sum())
        O += int(no.sum())
        P += int(m.sum())
    return E, O, P
