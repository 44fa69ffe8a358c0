"""Parity of the STAGED dense sweep -- the kernels bench.py times -- against the oracle, through the C ABI.  -m gpu.

Dense one-window spin-2 calls at lmax <= 800 take the single-launch kernel (tj_small.cu), so the small-size tests of
tests/test_gpu_parity.py pin that kernel.  The sizes here lie above the threshold and select, by themselves, the plain
staged instantiations sweep_tma_kernel<R, blocks, TS> (NW = 1, SPIN = 2, ROWS = 0, DIAG = 0) plus prepare_kernel and
writer_kernel; every test asserts through tj_profile_last_sweep which instantiation ran:

    lmax < 2600:   <8, TT|TE|EE|EB, 96>   <8, TE|EE|EB, 96>   <16, TT, 48>
    lmax >= 2600:  <12, TT|TE|EE|EB, 96>  <12, TE|EE|EB, 96>  (the headline kernel)      lmax >= 4096: <32, TT, 64>

Bar: that of tests/test_gpu_parity.py (north_star).
"""
import numpy as np
import pytest

import oracle
from paper_2602_15605_b200 import binding, build, windows
from test_gpu_parity import BLOCKS, _expected_support, _oracle_ranges, _t, assert_parity

pytestmark = pytest.mark.gpu

POL = ("TE", "EE", "EB")


@pytest.fixture(scope="module", autouse=True)
def _lib():
    build.build()
    binding.load_library()


def _staged(R, mask, TS):
    g = binding.profile_last_sweep()
    assert (g["R"], g["mask"], g["TS"], g["nw"], g["spin"], g["rows"], g["diag"]) == (R, mask, TS, 1, 2, 0, 0), g


def _three_requests(T, W):
    """All five blocks, the polarised blocks alone, TT alone: the three dense instantiations of one size."""
    import torch
    Wd = [_t(w) for w in W]
    lo = T.lmax < 2600
    out = {}
    out["all"] = {k: v.cpu().numpy() for k, v in binding.coupling_pol(T, *Wd).items()}
    _staged(8 if lo else 12, 15, 96)
    out["pol"] = {k: v.cpu().numpy() for k, v in binding.coupling_pol(T, None, Wd[1], Wd[2], want=POL).items()}
    _staged(8 if lo else 12, 14, 96)
    out["tt"] = {"TT": binding.coupling_tt(T, Wd[0]).cpu().numpy()}
    _staged(16 if T.lmax < 4096 else 32, 1, 48 if T.lmax < 4096 else 64)
    torch.cuda.synchronize()
    return out


# ---------------------------------------------------------------- (a) full matrices, element by element
@pytest.mark.parametrize("lmax,cfg", [(801, 1), (1337, 2)])
def test_staged_sweep_full_matrices_all_requests(lmax, cfg):
    """Just above the single-launch threshold (801 = 100 bands of 8 rows + 1 row, 25 writer tiles + 1 column) and at a
    size with ragged tails in every geometry (1338 = 167*8 + 2 = 83*16 + 10 = 41*32 + 26)."""
    wl = windows.config(cfg, lmax=lmax)
    T = binding.build_tables(wl.lmax)
    got = _three_requests(T, (wl.Wtt, wl.Wtp, wl.Wpp))
    T.close()
    ref = oracle.coupling_full(wl.lmax, wl.l3max, wl.Wtt, wl.Wtp, wl.Wpp)
    worst = {}
    for k in BLOCKS:
        worst[k] = assert_parity(got["all"][k], ref[k], "lmax %d all/%s" % (lmax, k))
        if k != "TT":
            assert np.all(got["all"][k][:2] == 0.0) and np.all(got["all"][k][:, :2] == 0.0), k
    for k in POL:
        assert_parity(got["pol"][k], ref[k], "lmax %d pol/%s" % (lmax, k))
    assert_parity(got["tt"]["TT"], ref["TT"], "lmax %d tt/TT" % lmax)
    assert np.array_equal(got["all"]["BB"], got["all"]["EE"])
    print("lmax %d worst (rel, abs-small):" % lmax, worst)


def test_staged_sweep_truncated_l3max_signed_windows():
    """l3max = 777 < 2 lmax = 2000: the sweep of a pair with l1+l2 > l3max starts at a step t > 0 (the tables' lower
    guard band is never reached from there), and every entry with |l1-l2| > l3max is exactly 0.  Signed windows: the
    sums cancel.  Amplitude 1e-3 so that the bar's absolute branch (1e-14 where |K| < 1e-4) stays well above the
    rounding of the sum of |terms| (sum |terms| <= (2 l2+1)/(4 pi) max|W| < 1 here, i.e. ~1e-16 per entry;
    PAPER.md:251, :261); nine entries in ten are still judged by the relative branch."""
    lmax, l3max = 1000, 777
    rng = np.random.default_rng(777)
    W = [1e-3 * rng.standard_normal(l3max + 1) for _ in range(3)]
    T = binding.build_tables(lmax, l3max)
    got = _three_requests(T, W)
    T.close()
    ref = oracle.coupling_full(lmax, l3max, *W)
    i, j = np.indices((lmax + 1, lmax + 1))
    far = np.abs(i - j) > l3max
    assert far.any()
    for k in BLOCKS:
        assert_parity(got["all"][k], ref[k], "truncated all/%s" % k)
        assert np.all(got["all"][k][far] == 0.0), k
        # the relative branch of the bar is exercised, not only the absolute one
        assert (np.abs(ref[k]) >= 1e-4).mean() > 0.8, k
    for k in POL:
        assert_parity(got["pol"][k], ref[k], "truncated pol/%s" % k)
        assert np.all(got["pol"][k][far] == 0.0), k
    assert_parity(got["tt"]["TT"], ref["TT"], "truncated tt/TT")
    assert np.all(got["tt"]["TT"][far] == 0.0)


# ---------------------------------------------------------------- (b) the kernels' own l3 bookkeeping, whole matrix
@pytest.mark.parametrize("lmax,l3max,Ls", [(820, 1640, (0, 1, 2, 3, 410, 411, 821, 1639, 1640)),
                                           (820, 777, (0, 1, 388, 389, 776, 777))])
def test_staged_sweep_spike_windows_zero_pattern(lmax, l3max, Ls):
    """W = delta_{l,L}: an entry is non-zero iff l3 = L is one of the terms the sweep adds for that pair, so the zero
    pattern of the WHOLE matrix is the staged kernel's l3 bookkeeping (triangle, parity, l3max cut), compared with the
    oracle's integer ranges for every pair.  Integers only; values are sampled rows."""
    T = binding.build_tables(lmax, l3max)
    l1, l2 = np.indices((lmax + 1, lmax + 1))
    pol = (l1 >= 2) & (l2 >= 2)
    ranges = _oracle_ranges(lmax, l3max)
    rows = np.array([0, 1, 2, 7, 8, 9, 95, 96, 97, 409, 410, 411, 799, 800, 801, 819, 820], dtype=np.int32)
    for L in Ls:
        Wn = windows.spike(l3max, L)
        got = _three_requests(T, (Wn, Wn, Wn))
        ev, od = _expected_support(ranges, L)
        for req in ("all", "tt"):
            TT = got[req]["TT"]
            assert np.all(TT[~ev] == 0.0) and np.all(TT[ev] > 0.0), (req, L)
        for req in ("all", "pol"):
            K = got[req]
            for k in ("TE", "EE"):
                assert np.all(K[k][~(ev & pol)] == 0.0), (req, k, L)
            assert np.all(K["EB"][~(od & pol)] == 0.0), (req, L)
            assert np.all(K["EE"][ev & pol] >= 0.0) and np.all(K["EB"][od & pol] >= 0.0), (req, L)
        # inside the support the spin-2 symbol has accidental zeros: checked through the oracle's values on sampled rows
        ref = oracle.coupling_rows(lmax, l3max, Wn, Wn, Wn, rows)
        for k in BLOCKS:
            g = got["all"][k][rows]
            assert_parity(g, ref[k], "spike L=%d %s" % (L, k))
            assert np.all((g != 0.0) | (np.abs(ref[k]) < 1e-13)), (k, L)
    T.close()


# ---------------------------------------------------------------- (c) the R = 8 / R = 12 switch
@pytest.mark.parametrize("lmax", [2599, 2600, 2700])
def test_staged_sweep_rows_at_the_geometry_switch(lmax):
    """lmax = 2599 is the last size on 8-row bands, 2600 the first on the headline geometry (12-row bands, 96-step
    stages).  Full rows against the oracle at band and stage seams: multiples of 8, 12, 32 and 96, +-1, the last rows."""
    import torch
    wl = windows.config(2, lmax=lmax)
    T = binding.build_tables(wl.lmax)
    Wd = [_t(w) for w in (wl.Wtt, wl.Wtp, wl.Wpp)]
    out = binding.coupling_pol(T, *Wd)
    _staged(8 if lmax < 2600 else 12, 15, 96)
    pol = binding.coupling_pol(T, None, Wd[1], Wd[2], want=POL)
    _staged(8 if lmax < 2600 else 12, 14, 96)
    torch.cuda.synchronize()
    rows = np.array(sorted({0, 2, 11, 12, 13, 95, 96, 97, 191, 192, 193, 1151, 1152, 1153, 1200, 2015, 2016, 2017,
                            2591, 2592, 2593, lmax - 12, lmax - 1, lmax}), dtype=np.int32)
    ref = oracle.coupling_rows(wl.lmax, wl.l3max, wl.Wtt, wl.Wtp, wl.Wpp, rows)
    ridx = torch.as_tensor(rows.astype(np.int64)).cuda()
    for k in BLOCKS:
        assert_parity(out[k][ridx].cpu().numpy(), ref[k], "lmax %d rows %s" % (lmax, k))
        # the same rows read as columns: the mirrored writer's half
        w = (2.0 * np.arange(lmax + 1) + 1.0)
        col = out[k][:, ridx].cpu().numpy().T            # K[l2][l1] for l1 in rows
        xi_row = ref[k] / w[None, :]                      # Xi(l1, l2)
        assert_parity(col, xi_row * (2.0 * rows[:, None] + 1.0), "lmax %d columns %s" % (lmax, k))
    for k in POL:
        assert torch.equal(pol[k], out[k]), k            # same arithmetic per entry with or without the TT block
    T.close()


# ---------------------------------------------------------------- (d) the compute-bound host pipeline (the e2e number's path)
@pytest.mark.parametrize("lmax,keys", [(6400, BLOCKS), (7600, ("TT",))])
def test_host_pipeline_compute_bound_regime_bitwise(lmax, keys):
    """tj_coupling_host at sizes where the arithmetic outlasts the copies: after every row chunk the L-shaped region it
    made final goes to the host as two pitched rectangles (chunk bounds at multiples of lcm(R, 32) = 96 rows).  Every
    entry of every output (pre-filled with NaN) must be bit-identical to tj_coupling_pol on device buffers, which
    tests/test_gpu_parity.py::test_full_size_configs_sampled and the tests above hold against the oracle."""
    import torch
    wl = windows.config(3, lmax=lmax)
    T = binding.build_tables(wl.lmax)
    N = wl.lmax + 1
    hw = [torch.as_tensor(w).pin_memory() for w in (wl.Wtt, wl.Wtp, wl.Wpp)]
    out = {k: torch.full((N, N), float("nan"), dtype=torch.float64).pin_memory() for k in keys}
    if keys == ("TT",):
        binding.coupling_host(T, hw[0], None, None, out)
    else:
        binding.coupling_host(T, *hw, out)
    dev = [w.cuda() for w in hw]
    ref = binding.coupling_pol(T, dev[0], dev[1] if len(keys) > 1 else None, dev[2] if len(keys) > 1 else None, want=keys)
    torch.cuda.synchronize()
    for k in keys:
        assert torch.equal(out[k].cuda(), ref[k]), k
    # and the device result itself against the oracle, on a few rows
    rows = np.array([0, 2, 95, 96, 97, 1919, 1920, lmax // 2, lmax - 1, lmax], dtype=np.int32)
    r = oracle.coupling_rows(wl.lmax, wl.l3max, wl.Wtt, wl.Wtp if len(keys) > 1 else None,
                             wl.Wpp if len(keys) > 1 else None, rows)
    for k in keys:
        assert_parity(out[k][torch.as_tensor(rows.astype(np.int64))].numpy(), r[k], "host lmax %d %s" % (lmax, k))
    del out, ref
    T.close()
