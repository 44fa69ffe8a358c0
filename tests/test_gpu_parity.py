"""Parity of the CUDA path (through the C ABI) against the oracle.  All tests need a B200: -m gpu.

Bar (north_star), element-wise:
    |gpu - oracle| <= 1e-10 |oracle|   where |oracle| >= 1e-4,
    |gpu - oracle| <= 1e-14            elsewhere,
and exact structure: entries the triangle / parity / l3max rules make empty are exactly 0.0.
"""
import math

import numpy as np
import pytest

import oracle
from paper_2602_15605_b200 import binding, build, windows

pytestmark = pytest.mark.gpu

RTOL, ATOL_SMALL, SMALL = 1e-10, 1e-14, 1e-4
BLOCKS = ("TT", "TE", "EE", "BB", "EB")


@pytest.fixture(scope="module", autouse=True)
def _lib():
    build.build()
    binding.load_library()


def _t(a):
    import torch
    return None if a is None else torch.as_tensor(np.ascontiguousarray(a), dtype=torch.float64).cuda()


def assert_parity(gpu, ref, what):
    gpu = np.asarray(gpu, dtype=np.float64)
    ref = np.asarray(ref, dtype=np.float64)
    assert gpu.shape == ref.shape, what
    assert np.all(np.isfinite(gpu)), what
    err = np.abs(gpu - ref)
    big = np.abs(ref) >= SMALL
    bad_big = big & (err > RTOL * np.abs(ref))
    bad_small = (~big) & (err > ATOL_SMALL)
    if bad_big.any() or bad_small.any():
        i = np.argwhere(bad_big | bad_small)[0]
        raise AssertionError("%s: %d entries out of tolerance, first at %s: gpu=%r oracle=%r" % (
            what, int(bad_big.sum() + bad_small.sum()), tuple(i), gpu[tuple(i)], ref[tuple(i)]))
    rel = err[big] / np.abs(ref[big]) if big.any() else np.zeros(1)
    return float(rel.max()), float(err[~big].max()) if (~big).any() else 0.0


def run_pol(lmax, l3max, Wtt, Wtp, Wpp, want=BLOCKS):
    T = binding.build_tables(lmax, l3max)
    out = binding.coupling_pol(T, _t(Wtt), _t(Wtp), _t(Wpp), want=want)
    import torch
    torch.cuda.synchronize()
    res = {k: v.cpu().numpy() for k, v in out.items()}
    T.close()
    return res


# ---------------------------------------------------------------- T1 tables
def test_tables_against_exact_definition():
    lmax = 10000
    T = binding.build_tables(lmax)
    assert T.pmax == 2 * lmax + 1
    ref = oracle.table_entries_float(T.pmax)
    for which, name in enumerate(("g", "ginv", "h", "gA", "gB")):
        got = T.copy_table(which, T.pmax + 1)
        ulp = np.spacing(np.abs(ref[name]))
        d = np.abs(got - ref[name])
        assert np.all(d <= ulp), (name, int(np.argmax(d / np.maximum(ulp, 1e-300))))
        # faithfully rounded: the overwhelming majority is bit-identical to the correctly rounded value
        assert np.mean(got == ref[name]) > 0.99, name
    g = T.copy_table(0, 4)
    assert list(g[:3]) == [1.0, 0.5, 0.375]          # g(0), g(1), g(2)  (Eq. 11)
    p = np.arange(1, T.pmax + 1)
    gg = T.copy_table(0, T.pmax + 1)[1:]
    assert abs(gg[-1] * math.sqrt(math.pi * p[-1]) - 1.0) < 1e-4   # g ~ (pi p)^(-1/2)
    u = T.copy_table(5, lmax + 1)
    assert np.array_equal(u, np.arange(lmax + 1.0) * (np.arange(lmax + 1.0) + 1.0))
    isd = T.copy_table(6, lmax + 1)
    l = np.arange(2, lmax + 1, dtype=np.float64)
    np.testing.assert_allclose(isd[2:], 1.0 / np.sqrt((l - 1) * l * (l + 1) * (l + 2)), rtol=4e-16)
    assert isd[0] == 0 and isd[1] == 0
    T.close()


# ---------------------------------------------------------------- T3 configs, full
def test_cfg0_tt_lmax256_full():
    wl = windows.config(0)
    T = binding.build_tables(wl.lmax)
    TT = binding.coupling_tt(T, _t(wl.Wtt)).cpu().numpy()
    ref = oracle.coupling_full(wl.lmax, wl.l3max, wl.Wtt, None, None)["TT"]
    assert TT.shape == (257, 257)
    assert_parity(TT, ref, "cfg0 TT")
    # the fused pol sweep must give the same TT
    both = binding.coupling_pol(T, _t(wl.Wtt), _t(wl.Wtt), _t(wl.Wtt))
    assert_parity(both["TT"].cpu().numpy(), ref, "cfg0 TT via pol")
    T.close()


def test_cfg0b_full_sky_identity_exact_structure():
    lmax = 256
    W = windows.full_sky(2 * lmax)
    K = run_pol(lmax, 2 * lmax, W, W, W)
    N = lmax + 1
    off = ~np.eye(N, dtype=bool)
    for k in BLOCKS:
        assert np.all(K[k][off] == 0.0), k
    np.testing.assert_allclose(np.diag(K["TT"]), 1.0, rtol=1e-14)
    for k in ("TE", "EE", "BB"):
        np.testing.assert_allclose(np.diag(K[k])[2:], 1.0, rtol=1e-14)
        assert np.all(np.diag(K[k])[:2] == 0.0)
    assert np.all(K["EB"] == 0.0)
    T = binding.build_tables(lmax)
    TT = binding.coupling_tt(T, _t(W)).cpu().numpy()
    assert np.all(TT[off] == 0.0)
    np.testing.assert_allclose(np.diag(TT), 1.0, rtol=1e-14)
    T.close()


def test_flat_window_closed_form_lmax700():
    """W = 1: TT = (2 l2+1)/4pi, TE = 0, EE+EB = (2 l2+1)/4pi -- exercises every (l1,l2,l3) term,
    no oracle needed (closed form)."""
    lmax = 700
    W = windows.flat(2 * lmax)
    K = run_pol(lmax, 2 * lmax, W, W, W)
    N = lmax + 1
    expect = np.broadcast_to((2.0 * np.arange(N) + 1.0) / (4 * math.pi), (N, N))
    np.testing.assert_allclose(K["TT"], expect, rtol=1e-12)
    assert np.max(np.abs(K["TE"])) < 1e-11
    np.testing.assert_allclose((K["EE"] + K["EB"])[2:, 2:], expect[2:, 2:], rtol=1e-12)
    for k in ("TE", "EE", "BB", "EB"):
        assert np.all(K[k][:2] == 0.0) and np.all(K[k][:, :2] == 0.0)


def test_cfg1_recipe_lmax300_full_all_blocks():
    """lmax <= 800: a dense one-window call takes the single-launch kernel (tj_small.cu), so this is a test of
    small_kernel; the staged sweep gets the same treatment in tests/test_gpu_staged_sweep.py."""
    wl = windows.config(1, lmax=300)   # 301 rows: ragged against the small kernel's rows per thread and 128-thread CTAs
    K = run_pol(wl.lmax, wl.l3max, wl.Wtt, wl.Wtp, wl.Wpp)
    ref = oracle.coupling_full(wl.lmax, wl.l3max, wl.Wtt, wl.Wtp, wl.Wpp)
    for k in BLOCKS:
        assert_parity(K[k], ref[k], "cfg1@300 " + k)
    assert np.array_equal(K["BB"], K["EE"])


@pytest.mark.parametrize("lmax", [0, 1, 2, 3, 7, 8, 15, 16, 17, 31, 127, 128, 129])
def test_ragged_and_tiny_sizes(lmax):
    wl = windows.config(2, lmax=lmax)
    K = run_pol(wl.lmax, wl.l3max, wl.Wtt, wl.Wtp, wl.Wpp)
    ref = oracle.coupling_full(wl.lmax, wl.l3max, wl.Wtt, wl.Wtp, wl.Wpp)
    for k in BLOCKS:
        assert K[k].shape == (lmax + 1, lmax + 1)
        assert_parity(K[k], ref[k], "lmax=%d %s" % (lmax, k))
    T = binding.build_tables(lmax)
    TT = binding.coupling_tt(T, _t(wl.Wtt)).cpu().numpy()
    assert_parity(TT, ref["TT"], "lmax=%d TT-only" % lmax)
    T.close()


def test_truncated_l3max_and_signed_window():
    lmax, l3max = 200, 137
    rng = np.random.default_rng(9)
    W = [rng.standard_normal(l3max + 1) for _ in range(3)]    # signed: TE/EE sums cancel
    K = run_pol(lmax, l3max, *W)
    ref = oracle.coupling_full(lmax, l3max, *W)
    for k in BLOCKS:
        # tolerance relative to the row scale for signed sums: the bar's absolute branch
        assert_parity(K[k], ref[k], "l3max<2lmax " + k)
        i, j = np.indices(K[k].shape)
        assert np.all(K[k][np.abs(i - j) > l3max] == 0.0)


# ---------------------------------------------------------------- T2 spikes: one symbol per entry, exact zero pattern
@pytest.mark.parametrize("L", [0, 1, 2, 3, 64, 199, 200, 399, 400])
def test_spike_window_structure_bit_exact(L):
    lmax = 200
    W = windows.spike(2 * lmax, L)
    K = run_pol(lmax, 2 * lmax, W, W, W)
    ref = oracle.coupling_full(lmax, 2 * lmax, W, W, W)
    l1, l2 = np.indices((lmax + 1, lmax + 1))
    inside = (np.abs(l1 - l2) <= L) & (L <= l1 + l2)
    even = ((l1 + l2 + L) % 2) == 0
    pol = (l1 >= 2) & (l2 >= 2)
    # bookkeeping: the zero pattern is fixed by triangle + parity; must hold EXACTLY on the GPU
    assert np.all(K["TT"][~(inside & even)] == 0.0)
    assert np.all(K["TT"][inside & even] > 0.0)
    assert np.all(K["EE"][~(inside & even & pol)] == 0.0)
    assert np.all(K["TE"][~(inside & even & pol)] == 0.0)
    assert np.all(K["EB"][~(inside & ~even & pol)] == 0.0)
    for k in BLOCKS:
        assert_parity(K[k], ref[k], "spike L=%d %s" % (L, k))


# ---------------------------------------------------------------- symmetry / mirror
def test_mirror_symmetry_bitwise():
    wl = windows.config(1, lmax=333)
    K = run_pol(wl.lmax, wl.l3max, wl.Wtt, wl.Wtp, wl.Wpp)
    w = 2.0 * np.arange(wl.lmax + 1) + 1.0
    for k in BLOCKS:
        M = K[k]
        a = M * w[:, None]          # (2 l1+1) M[l1][l2]
        b = (M * w[:, None]).T      # (2 l2+1) M[l2][l1]
        # both sides are (2l1+1)(2l2+1) Xi from the SAME Xi double; each side carries two roundings
        # (the writer's product and this test's): |a-b| <= 4 * 2^-53 * |x|
        assert np.all(np.abs(a - b) <= 4.5e-16 * np.maximum(np.abs(a), np.abs(b))), k


# ---------------------------------------------------------------- nullable outputs
def test_nullable_outputs_and_errors():
    wl = windows.config(1, lmax=150)
    ref = run_pol(wl.lmax, wl.l3max, wl.Wtt, wl.Wtp, wl.Wpp)
    for want in (("TT",), ("EE",), ("BB",), ("EB",), ("TE",), ("TE", "EB"), ("TT", "BB"), ("EE", "BB", "EB")):
        got = run_pol(wl.lmax, wl.l3max,
                      wl.Wtt if "TT" in want else None,
                      wl.Wtp if "TE" in want else None,
                      wl.Wpp if set(want) & {"EE", "BB", "EB"} else None, want=want)
        assert set(got) == set(want)
        for k in want:
            assert np.array_equal(got[k], ref[k]), (want, k)
    T = binding.build_tables(wl.lmax)
    with pytest.raises(binding.TJError):   # output without its window
        binding.coupling_pol(T, None, _t(wl.Wtp), _t(wl.Wpp), want=("TT",))
    with pytest.raises(binding.TJError):   # wrong window length
        binding.coupling_tt(T, _t(wl.Wtt[:-1]))
    T.close()


# ---------------------------------------------------------------- band variant
@pytest.mark.parametrize("lmax,lcut", [(400, 30), (257, 0), (100, 150), (64, 7), (300, 300)])
def test_band_equals_oracle_and_zero_padded_full(lmax, lcut):
    import torch
    wl = windows.config(4, lmax=max(lmax, 10))
    W = np.zeros(lcut + 1)
    n = min(lcut + 1, wl.Wtt.size)
    W[:n] = wl.Wtt[:n]
    T = binding.build_tables(lmax)
    # outputs pre-filled with NaN: every slot of the band must be written by the call (values or exact zeros)
    pre = {k: torch.full((lmax + 1, 2 * lcut + 1), float("nan"), dtype=torch.float64, device="cuda") for k in BLOCKS}
    out = binding.coupling_band(T, lcut, _t(W), _t(W), _t(W), out=pre)
    torch.cuda.synchronize()
    band = {k: v.cpu().numpy() for k, v in out.items()}
    ref = oracle.coupling_band(lmax, lcut, W, W, W)
    for k in BLOCKS:
        assert band[k].shape == (lmax + 1, 2 * lcut + 1)
        assert_parity(band[k], ref[k], "band %s" % k)
    # band == dense call with the zero-padded window, on the band; dense is zero outside
    Wpad = np.zeros(2 * lmax + 1)
    m = min(lcut + 1, 2 * lmax + 1)
    Wpad[:m] = W[:m]
    full = binding.coupling_pol(T, _t(Wpad), _t(Wpad), _t(Wpad))
    torch.cuda.synchronize()
    for k in BLOCKS:
        F = full[k].cpu().numpy()
        i, j = np.indices(F.shape)
        assert np.all(F[np.abs(i - j) > lcut] == 0.0)
        for o in range(-lcut, lcut + 1):
            rows = np.arange(max(0, -o), min(lmax, lmax - o) + 1)
            if rows.size:
                assert np.array_equal(band[k][rows, o + lcut], F[rows, rows + o]), (k, o)
        # out-of-range slots are zero
        for l1 in (0, 1, lmax):
            for o in range(-lcut, lcut + 1):
                if not (0 <= l1 + o <= lmax):
                    assert band[k][l1, o + lcut] == 0.0
    T.close()


# ---------------------------------------------------------------- host-buffer (end-to-end) entry point
def test_host_entry_point_matches_device_path():
    import torch
    wl = windows.config(1, lmax=200)
    ref = run_pol(wl.lmax, wl.l3max, wl.Wtt, wl.Wtp, wl.Wpp)
    T = binding.build_tables(wl.lmax)
    N = wl.lmax + 1
    out = {k: torch.empty((N, N), dtype=torch.float64).pin_memory() for k in BLOCKS}
    hw = [torch.as_tensor(w).pin_memory() for w in (wl.Wtt, wl.Wtp, wl.Wpp)]
    binding.coupling_host(T, *hw, out)
    for k in BLOCKS:
        assert np.array_equal(out[k].numpy(), ref[k]), k
    # banded host form
    lcut = 20
    W = torch.as_tensor(np.ascontiguousarray(wl.Wtt[: lcut + 1]))
    outb = {k: torch.empty((N, 2 * lcut + 1), dtype=torch.float64) for k in ("TT", "EB")}
    binding.coupling_host(T, W, None, W, outb, band_lcut=lcut)
    refb = oracle.coupling_band(wl.lmax, lcut, W.numpy(), None, W.numpy())
    assert_parity(outb["TT"].numpy(), refb["TT"], "host band TT")
    assert_parity(outb["EB"].numpy(), refb["EB"], "host band EB")
    T.close()


@pytest.mark.parametrize("lmax,keys", [(1500, BLOCKS), (1000, ("BB", "EB")), (777, ("TT",))])
def test_host_pipeline_many_row_chunks_bitwise(lmax, keys):
    """The host-buffer path runs sweep + writer + copies per row chunk on several streams; every chunking must
    give bit-identical matrices to the single-launch device path (which the tests above hold against the oracle)."""
    import torch
    wl = windows.config(2, lmax=lmax)
    T = binding.build_tables(wl.lmax)
    dev = [torch.as_tensor(w).cuda() for w in (wl.Wtt, wl.Wtp, wl.Wpp)]
    ref = binding.coupling_pol(T, *dev)
    torch.cuda.synchronize()
    N = wl.lmax + 1
    out = {k: torch.full((N, N), np.nan, dtype=torch.float64).pin_memory() for k in keys}
    hw = [torch.as_tensor(w).pin_memory() for w in (wl.Wtt, wl.Wtp, wl.Wpp)]
    if keys == ("TT",):
        binding.coupling_host(T, hw[0], None, None, out)
    elif "TT" not in keys:
        binding.coupling_host(T, None, None, hw[2], out)
    else:
        binding.coupling_host(T, *hw, out)
    for k in keys:
        assert np.array_equal(out[k].numpy(), ref[k].cpu().numpy()), k
    T.close()


# ---------------------------------------------------------------- T3 full-size configs, sampled
def _sample_pairs(lmax, n, seed, band=None):
    rng = np.random.default_rng(seed)
    l1 = rng.integers(0, lmax + 1, n)
    if band is None:
        l2 = rng.integers(0, lmax + 1, n)
    else:
        l2 = np.clip(l1 + rng.integers(-band, band + 1, n), 0, lmax)
    # structured: corners, diagonal, l<2 edges, last rows/cols, and the seams of every geometry in use: row bands of
    # 8 / 12 / 16 / 32 rows, writer tiles of 32, stages of 96 steps, CTA column tiles of 32 (multiples +-1)
    edge = np.array([0, 1, 2, 3, 7, 8, 9, 11, 12, 13, 31, 32, 33, 95, 96, 97, 127, 128, 129, 959, 960, 961,
                     lmax - 129, lmax - 128, lmax - 97, lmax - 96, lmax - 95, lmax - 13, lmax - 12, lmax - 9, lmax - 8,
                     lmax - 1, lmax])
    edge = edge[(edge >= 0) & (edge <= lmax)]
    e1, e2 = np.meshgrid(edge, edge, indexing="ij")
    if band is not None:
        keep = np.abs(e1 - e2) <= band
        e1, e2 = e1[keep], e2[keep]
    d = rng.integers(0, lmax + 1, 64)
    l1 = np.concatenate([l1, e1.ravel(), d, d])
    l2 = np.concatenate([l2, e2.ravel(), d, np.clip(d + 1, 0, lmax)])
    return l1.astype(np.int32), l2.astype(np.int32)


@pytest.mark.parametrize("cfg,npairs", [(1, 6000), (2, 3000), (3, 2500)])
def test_full_size_configs_sampled(cfg, npairs):
    """BASELINE.json configs 1-3 at full size, in the launch configuration bench.py times; outputs
    sampled at random + structured pairs the oracle computes one by one."""
    import torch
    wl = windows.config(cfg)
    T = binding.build_tables(wl.lmax)
    out = binding.coupling_pol(T, _t(wl.Wtt), _t(wl.Wtp), _t(wl.Wpp))
    torch.cuda.synchronize()
    l1, l2 = _sample_pairs(wl.lmax, npairs, 100 + cfg)
    ref = oracle.coupling_pairs(wl.l3max, wl.Wtt, wl.Wtp, wl.Wpp, l1, l2)
    i1 = torch.as_tensor(l1.astype(np.int64)).cuda()
    i2 = torch.as_tensor(l2.astype(np.int64)).cuda()
    worst = {}
    for k in BLOCKS:
        got = out[k][i1, i2].cpu().numpy()
        worst[k] = assert_parity(got, ref[k], "cfg%d %s" % (cfg, k))
    # properties that hold at any size: Xi symmetry on a sampled set, BB == EE, l<2 zero
    w1 = torch.as_tensor(2.0 * l1 + 1.0).cuda()
    w2 = torch.as_tensor(2.0 * l2 + 1.0).cuda()
    for k in BLOCKS:
        a = out[k][i1, i2] * w1
        b = out[k][i2, i1] * w2
        assert torch.all((a - b).abs() <= 4e-16 * torch.maximum(a.abs(), b.abs())), k
        if k != "TT":
            assert torch.all(out[k][:2] == 0) and torch.all(out[k][:, :2] == 0)
    assert torch.equal(out["BB"], out["EE"])
    print("cfg%d worst (rel, abs-small):" % cfg, worst)
    del out
    T.close()


def _assert_band_row_sums(out, lmax, lcut, Wtt, Wpp, what):
    """A property that needs no oracle and holds at any size (orthogonality of the 3j symbols over the third l at fixed
    m's): in a band-limited matrix every row l1 with lcut <= l1 <= lmax-lcut holds its whole triangle,
    so  sum_l2 K^TT = sum_l3 (2 l3+1) W^TT_l3 / 4 pi  and  sum_l2 (K^EE + K^EB) = the same with W^PP (l1 >= 2).
    (TE has no such sum rule: its two symbols carry different m on l2.)  Pinned on the oracle in
    tests/test_oracle_coupling.py::test_band_row_sum_rule."""
    import torch
    l3 = np.arange(lcut + 1, dtype=np.float64)
    ctt = float(((2 * l3 + 1) * Wtt).sum() / (4 * math.pi))
    cpp = float(((2 * l3 + 1) * Wpp).sum() / (4 * math.pi))
    rows = slice(max(lcut, 2), lmax - lcut + 1)
    stt = out["TT"][rows].sum(dim=1)
    spp = out["EE"][rows].sum(dim=1) + out["EB"][rows].sum(dim=1)
    e_tt = float((stt - ctt).abs().max() / ctt)
    e_pp = float((spp - cpp).abs().max() / cpp)
    print("%s: row sums over %d rows: TT %.2e, EE+EB %.2e" % (what, stt.numel(), e_tt, e_pp))
    assert e_tt < 1e-12 and e_pp < 1e-12, (e_tt, e_pp)


def test_cfg4_band_full_size_sampled():
    import torch
    wl = windows.config(4)
    lcut = wl.l3max
    T = binding.build_tables(wl.lmax)
    N, width = wl.lmax + 1, 2 * lcut + 1
    pre = {k: torch.full((N, width), float("nan"), dtype=torch.float64, device="cuda") for k in BLOCKS}
    out = binding.coupling_band(T, lcut, _t(wl.Wtt), _t(wl.Wtp), _t(wl.Wpp), out=pre)
    torch.cuda.synchronize()
    # every slot written (outputs were pre-filled with NaN); slots whose l2 is outside 0..lmax exactly 0
    l2grid = torch.arange(N, device="cuda")[:, None] + torch.arange(-lcut, lcut + 1, device="cuda")[None, :]
    outside = (l2grid < 0) | (l2grid > wl.lmax)
    for k in BLOCKS:
        assert bool(torch.isfinite(out[k]).all()), k
        assert bool((out[k][outside] == 0).all()), k
    l1, l2 = _sample_pairs(wl.lmax, 3000, 104, band=lcut)
    ref = oracle.coupling_pairs(lcut, wl.Wtt, wl.Wtp, wl.Wpp, l1, l2)
    i1 = torch.as_tensor(l1.astype(np.int64)).cuda()
    io = torch.as_tensor((l2.astype(np.int64) - l1 + lcut)).cuda()
    for k in BLOCKS:
        assert out[k].shape == (wl.lmax + 1, 2 * lcut + 1)
        got = out[k][i1, io].cpu().numpy()
        assert_parity(got, ref[k], "cfg4 %s" % k)
    # rows 0 and lmax: out-of-range slots zero
    assert torch.all(out["TT"][0, :lcut] == 0) and torch.all(out["TT"][-1, lcut + 1:] == 0)
    _assert_band_row_sums(out, wl.lmax, lcut, wl.Wtt, wl.Wpp, "cfg4")
    T.close()


# ---------------------------------------------------------------- multi-window batching
def _window_sets(lmax, nwin, seed):
    """nwin independent window sets of the config-1 recipe (different seeds)."""
    sets = [windows.pol_windows(lmax, (0.7, 30.0, 2.5), (0.5, 50.0, 3.0), 0.05, seed + k) for k in range(nwin)]
    return [np.stack([s[j] for s in sets]) for j in range(3)]


def test_multi_window_against_oracle():
    """3 window sets in one call (one batched sweep of three), each against the oracle."""
    import torch
    lmax, nwin = 150, 3
    Wtt, Wtp, Wpp = _window_sets(lmax, nwin, 100)
    T = binding.build_tables(lmax)
    out = binding.coupling_multi(T, _t(Wtt), _t(Wtp), _t(Wpp))
    torch.cuda.synchronize()
    for w in range(nwin):
        ref = oracle.coupling_full(lmax, 2 * lmax, Wtt[w], Wtp[w], Wpp[w])
        for k in BLOCKS:
            assert_parity(out[k][w].cpu().numpy(), ref[k], "multi set %d %s" % (w, k))
    T.close()


def test_multi_window_equals_single_calls_bitwise():
    """The batched sweep forms every entry with the same operations in the same order as tj_coupling_pol."""
    import torch
    lmax, nwin = 777, 5
    Wtt, Wtp, Wpp = _window_sets(lmax, nwin, 200)
    T = binding.build_tables(lmax)
    out = binding.coupling_multi(T, _t(Wtt), _t(Wtp), _t(Wpp))
    torch.cuda.synchronize()
    for w in range(nwin):
        one = binding.coupling_pol(T, _t(Wtt[w]), _t(Wtp[w]), _t(Wpp[w]))
        torch.cuda.synchronize()
        for k in BLOCKS:
            assert torch.equal(out[k][w], one[k]), (w, k)
    # partial requests take the one-set-per-sweep route
    part = binding.coupling_multi(T, None, None, _t(Wpp), want=("EE", "EB"))
    torch.cuda.synchronize()
    for w in range(nwin):
        assert torch.equal(part["EE"][w], out["EE"][w]) and torch.equal(part["EB"][w], out["EB"][w])
    T.close()


# ---------------------------------------------------------------- spin-1 blocks
SPIN1 = ("K00", "K01", "K11p", "K11m")


def _run_spin1(lmax, l3max, W00, W01, W11, want=SPIN1):
    import torch
    T = binding.build_tables(lmax, l3max)
    out = binding.coupling_spin1(T, _t(W00), _t(W01), _t(W11), want=want)
    torch.cuda.synchronize()
    res = {k: v.cpu().numpy() for k, v in out.items()}
    T.close()
    return res


@pytest.mark.parametrize("lmax,l3max", [(0, 0), (1, 2), (2, 4), (67, 134), (150, 300), (150, 101)])
def test_spin1_against_oracle_small(lmax, l3max):
    rng = np.random.default_rng(7 + lmax)
    W = [np.abs(rng.standard_normal(l3max + 1)) / (1.0 + np.arange(l3max + 1)) ** 1.5 for _ in range(3)]
    W[1] = W[1] * np.where(rng.random(l3max + 1) < 0.3, -1.0, 1.0)      # a cross window may change sign
    got = _run_spin1(lmax, l3max, *W)
    ref = oracle.spin1_full(lmax, l3max, W[1], W[2])
    ref["K00"] = oracle.coupling_full(lmax, l3max, W[0], None, None)["TT"]
    for k in SPIN1:
        assert_parity(got[k], ref[k], "spin1 lmax=%d %s" % (lmax, k))
        if k != "K00":
            assert np.all(got[k][:1] == 0.0) and np.all(got[k][:, :1] == 0.0), k


def test_spin1_full_sky_and_partial_requests():
    lmax = 300
    W = windows.full_sky(2 * lmax)
    got = _run_spin1(lmax, 2 * lmax, W, W, W)
    N = lmax + 1
    off = ~np.eye(N, dtype=bool)
    d = np.ones(N)
    d[0] = 0.0
    for k in SPIN1:
        assert np.all(got[k][off] == 0.0), k
    np.testing.assert_allclose(np.diag(got["K00"]), 1.0, rtol=1e-13)
    np.testing.assert_allclose(np.diag(got["K11p"]), d, rtol=1e-13, atol=0)
    np.testing.assert_allclose(np.diag(got["K01"]), -d, rtol=1e-13, atol=0)
    assert np.all(got["K11m"] == 0.0)
    wl = windows.config(1, lmax=lmax)
    full = _run_spin1(lmax, 2 * lmax, wl.Wtt, wl.Wtp, wl.Wpp)
    part = _run_spin1(lmax, 2 * lmax, None, None, wl.Wpp, want=("K11p", "K11m"))
    assert np.array_equal(part["K11p"], full["K11p"]) and np.array_equal(part["K11m"], full["K11m"])
    only00 = _run_spin1(lmax, 2 * lmax, wl.Wtt, None, None, want=("K00",))
    assert np.array_equal(only00["K00"], full["K00"])


def test_spin1_config1_sampled_rows():
    """Config-1 size (lmax = 2000) in the shipped launch configuration; oracle on sampled rows."""
    wl = windows.config(1)
    got = _run_spin1(wl.lmax, wl.l3max, wl.Wtt, wl.Wtp, wl.Wpp)
    rows = np.array([0, 1, 2, 3, 11, 12, 500, 1023, 1024, 1999, 2000], dtype=np.int32)
    N = wl.lmax + 1
    l1s = np.repeat(rows, N)
    l2s = np.tile(np.arange(N, dtype=np.int32), rows.size)
    ref = {k: v.reshape(rows.size, N) for k, v in oracle.spin1_pairs(wl.l3max, wl.Wtp, wl.Wpp, l1s, l2s).items()}
    for k in ("K01", "K11p", "K11m"):
        rel, ab = assert_parity(got[k][rows], ref[k], "spin1 cfg1 %s" % k)
        print("spin1 cfg1 %s: worst rel %.2e, worst abs (small) %.2e" % (k, rel, ab))
        # Xi symmetry through the mirrored writer
        a = got[k] * (2.0 * np.arange(N)[:, None] + 1.0)
        assert np.allclose(a, a.T, rtol=1e-15, atol=0)


@pytest.mark.parametrize("lmax", [4095, 4096, 5000])
def test_tt_only_long_geometry(lmax):
    """tj_coupling_tt switches to R = 32 pairs per thread at lmax >= 4096: sampled entries against the
    oracle, and the whole matrix bitwise against the TT block of the fused sweep (same operations per entry)."""
    import torch
    wl = windows.config(2, lmax=lmax)
    T = binding.build_tables(wl.lmax)
    TT = binding.coupling_tt(T, _t(wl.Wtt))
    pol = binding.coupling_pol(T, _t(wl.Wtt), _t(wl.Wtp), _t(wl.Wpp), want=("TT", "TE", "EE", "EB"))
    torch.cuda.synchronize()
    assert torch.equal(TT, pol["TT"])
    l1, l2 = _sample_pairs(wl.lmax, 1500, 300 + lmax)
    ref = oracle.coupling_pairs(wl.l3max, wl.Wtt, None, None, l1, l2)
    got = TT[torch.as_tensor(l1.astype(np.int64)).cuda(), torch.as_tensor(l2.astype(np.int64)).cuda()].cpu().numpy()
    assert_parity(got, ref["TT"], "TT-only lmax=%d" % lmax)
    T.close()


# ---------------------------------------------------------------- paper-literal ablation kernel
def test_literal_eq16_kernel_against_oracle_and_sweep():
    import torch
    for lmax, l3max in ((150, 300), (97, 120)):
        wl = windows.config(1, lmax=lmax)
        Wtt, Wpp = wl.Wtt[: l3max + 1], wl.Wpp[: l3max + 1]
        T = binding.build_tables(lmax, l3max)
        lit = binding.coupling_literal(T, _t(Wtt), _t(Wpp))
        torch.cuda.synchronize()
        ref = oracle.coupling_full(lmax, l3max, Wtt, None, Wpp)
        assert_parity(lit["TT"].cpu().numpy(), ref["TT"], "literal TT lmax=%d" % lmax)
        assert_parity(lit["EE"].cpu().numpy(), ref["EE"], "literal EE lmax=%d" % lmax)
        T.close()
    wl = windows.config(1)
    T = binding.build_tables(wl.lmax)
    lit = binding.coupling_literal(T, _t(wl.Wtt), _t(wl.Wpp))
    pol = binding.coupling_pol(T, _t(wl.Wtt), None, _t(wl.Wpp), want=("TT", "EE"))
    torch.cuda.synchronize()
    for k in ("TT", "EE"):
        a, b = lit[k], pol[k]
        rel = ((a - b).abs() / b.abs().clamp_min(1e-300))[b.abs() >= SMALL]
        assert float(rel.max()) < 1e-10, (k, float(rel.max()))
        print("literal vs fused sweep, cfg1 %s: worst rel %.2e" % (k, float(rel.max())))
    only = binding.coupling_literal(T, None, _t(wl.Wpp), want=("EE",))
    assert torch.equal(only["EE"], lit["EE"])
    T.close()


def test_flat_window_closed_form_full_size_lmax10000():
    """The closed form of the flat window at the HEADLINE size, in the launch configuration bench.py times:
    W = 1 gives TT = (2 l2+1)/4pi in every one of the 10001^2 entries, TE = 0, EE+EB = (2 l2+1)/4pi on l >= 2
    (orthogonality of the 3j symbols over l3) -- every (l1,l2,l3) term of the full problem takes part, and no
    oracle sample is involved.  Also the spin-1 analogue: K11+ + K11- = (2 l2+1)/4pi on l >= 1, K01 = 0."""
    import torch
    lmax = 10000
    N = lmax + 1
    W = _t(windows.flat(2 * lmax))
    T = binding.build_tables(lmax)
    out = binding.coupling_pol(T, W, W, W, want=("TT", "TE", "EE", "EB"))
    torch.cuda.synchronize()
    col = ((2.0 * torch.arange(N, dtype=torch.float64, device="cuda") + 1.0) / (4 * math.pi))[None, :]
    rel_tt = float(((out["TT"] - col).abs() / col).max())
    s = out["EE"] + out["EB"]
    rel_s = float(((s - col).abs() / col)[2:, 2:].max())
    te = float((out["TE"].abs() / col).max())
    print("flat window lmax=10000: TT rel %.2e, EE+EB rel %.2e, |TE|/scale %.2e" % (rel_tt, rel_s, te))
    assert rel_tt < 1e-12 and rel_s < 1e-12 and te < 1e-12
    for k in ("TE", "EE", "EB"):
        assert torch.all(out[k][:2] == 0) and torch.all(out[k][:, :2] == 0)
    del out, s
    sp = binding.coupling_spin1(T, None, W, W, want=("K01", "K11p", "K11m"))
    torch.cuda.synchronize()
    s1 = sp["K11p"] + sp["K11m"]
    rel_1 = float(((s1 - col).abs() / col)[1:, 1:].max())
    k01 = float((sp["K01"].abs() / col).max())
    print("spin-1: K11+ + K11- rel %.2e, |K01|/scale %.2e" % (rel_1, k01))
    assert rel_1 < 1e-12 and k01 < 1e-12
    T.close()


def test_flat_window_closed_form_beyond_headline_size_lmax16000():
    """Sizes past the headline config (index arithmetic, guard bands, table range p <= 32001): the flat-window
    closed form at lmax = 16000, TT-only sweep and fused sweep."""
    import torch
    lmax = 16000
    N = lmax + 1
    W = _t(windows.flat(2 * lmax))
    T = binding.build_tables(lmax)
    col = ((2.0 * torch.arange(N, dtype=torch.float64, device="cuda") + 1.0) / (4 * math.pi))[None, :]
    TT = binding.coupling_tt(T, W)
    torch.cuda.synchronize()
    rel = float(((TT - col).abs() / col).max())
    assert rel < 1e-12, rel
    del TT
    out = binding.coupling_pol(T, None, W, W, want=("TE", "EE", "EB"))
    torch.cuda.synchronize()
    s = out["EE"]
    s += out["EB"]
    rel_s = float(((s - col).abs() / col)[2:, 2:].max())
    te = float((out["TE"].abs() / col).max())
    print("flat window lmax=16000: TT rel %.2e, EE+EB rel %.2e, |TE|/scale %.2e" % (rel, rel_s, te))
    assert rel_s < 1e-12 and te < 1e-12
    T.close()


def test_multi_window_tt_only_bitwise_and_oracle():
    """TT alone for 7 windows (sweeps of 4 + 2 + 1 windows): bitwise equal to tj_coupling_tt per window, and
    against the oracle at a small size."""
    import torch
    lmax, nwin = 900, 7
    Wtt, _, _ = _window_sets(lmax, nwin, 300)
    T = binding.build_tables(lmax)
    out = binding.coupling_multi(T, _t(Wtt), None, None, want=("TT",))
    torch.cuda.synchronize()
    for w in range(nwin):
        one = binding.coupling_tt(T, _t(Wtt[w]))
        torch.cuda.synchronize()
        assert torch.equal(out["TT"][w], one), w
    T.close()
    lmax = 130
    Wtt, _, _ = _window_sets(lmax, 4, 310)
    T = binding.build_tables(lmax)
    out = binding.coupling_multi(T, _t(Wtt), None, None, want=("TT",))
    torch.cuda.synchronize()
    for w in range(4):
        ref = oracle.coupling_full(lmax, 2 * lmax, Wtt[w], None, None)["TT"]
        assert_parity(out["TT"][w].cpu().numpy(), ref, "multi TT set %d" % w)
    T.close()


# ---------------------------------------------------------------- row blocks
@pytest.mark.parametrize("lmax", [150, 1003])
def test_row_blocks_equal_rows_of_full_matrix_bitwise(lmax):
    """tj_coupling_rows: any block of full rows, bit-identical to the same rows of tj_coupling_pol (blocks that
    start/end inside a row band of the sweep, the first and the last rows, one row, everything)."""
    import torch
    wl = windows.config(1, lmax=lmax)
    T = binding.build_tables(lmax)
    W = [_t(w) for w in (wl.Wtt, wl.Wtp, wl.Wpp)]
    full = binding.coupling_pol(T, *W)
    tt = binding.coupling_tt(T, W[0])
    torch.cuda.synchronize()
    N = lmax + 1
    blocks = [(0, 1), (0, 7), (5, 6), (13, 37), (24, 48), (N - 1, N), (N // 2 - 3, N // 2 + 40), (N - 29, N), (0, N)]
    for r0, r1 in blocks:
        pre = {k: torch.full((r1 - r0, N), float("nan"), dtype=torch.float64, device="cuda") for k in BLOCKS}
        got = binding.coupling_rows(T, *W, r0, r1, out=pre)
        only = binding.coupling_rows(T, W[0], None, None, r0, r1, want=("TT",))
        torch.cuda.synchronize()
        for k in BLOCKS:
            assert torch.equal(got[k], full[k][r0:r1]), (k, r0, r1)
        assert torch.equal(only["TT"], tt[r0:r1]), (r0, r1)
    with pytest.raises(binding.TJError):
        binding.coupling_rows(T, *W, 5, 5)
    with pytest.raises(binding.TJError):
        binding.coupling_rows(T, *W, 0, N + 1)
    T.close()


def test_row_blocks_config1_against_oracle_and_cover():
    """Config 1 cut into 4 work-balanced row blocks (shard.row_blocks): the blocks tile the matrix, each block
    against the oracle on sampled rows."""
    import torch
    from paper_2602_15605_b200 import shard
    wl = windows.config(1)
    N = wl.lmax + 1
    T = binding.build_tables(wl.lmax)
    W = [_t(w) for w in (wl.Wtt, wl.Wtp, wl.Wpp)]
    cuts = shard.row_blocks(wl.lmax, 4)
    assert cuts[0][0] == 0 and cuts[-1][1] == N and all(a[1] == b[0] for a, b in zip(cuts, cuts[1:]))
    for r0, r1 in cuts:
        got = binding.coupling_rows(T, *W, r0, r1)
        torch.cuda.synchronize()
        rows = np.unique(np.array([r0, (r0 + r1) // 2, r1 - 1], dtype=np.int32))
        ref = oracle.coupling_rows(wl.lmax, wl.l3max, wl.Wtt, wl.Wtp, wl.Wpp, rows)
        for k in BLOCKS:
            assert_parity(got[k][torch.as_tensor(rows - r0, dtype=torch.int64).cuda()].cpu().numpy(), ref[k],
                          "rows [%d,%d) %s" % (r0, r1, k))
    T.close()


def test_adjudication_against_exact_racah_sums():
    """Where the GPU path and the oracle disagree most the exact Racah symbols decide.  At lmax = 192 (config-1
    recipe) the largest relative disagreement, 2e-12, is the TE entry (14,135), whose terms cancel to 1e-4 of their
    size; the others are squeezed and diagonal entries.  Each sum is re-done from exact squared
    symbols (big-integer rationals, rounded once per term, math.fsum) and both sides are measured against it on the
    scale of the terms: the table path is the more accurate side."""
    import torch
    from racah import threej_sq_sign
    wl = windows.config(1, lmax=192)
    got = run_pol(wl.lmax, wl.l3max, wl.Wtt, wl.Wtp, wl.Wpp)
    pairs = [(14, 135), (192, 192), (191, 192), (150, 190), (100, 101), (2, 192), (64, 64), (157, 154)]
    l1s = np.array([p[0] for p in pairs], dtype=np.int32)
    l2s = np.array([p[1] for p in pairs], dtype=np.int32)
    ora = oracle.coupling_pairs(wl.l3max, wl.Wtt, wl.Wtp, wl.Wpp, l1s, l2s)
    worst_gpu = worst_ora = 0.0
    for n, (l1, l2) in enumerate(pairs):
        terms = {"TT": [], "TE": [], "EE": [], "EB": []}
        for l3 in range(abs(l1 - l2), l1 + l2 + 1):
            w = 2 * l3 + 1
            s0, g0 = threej_sq_sign(l1, l2, l3, 0, 0, 0)
            s2, g2 = threej_sq_sign(l1, l2, l3, -2, 2, 0)
            terms["TT"].append(w * wl.Wtt[l3] * float(s0))
            if (l1 + l2 + l3) % 2 == 0:
                terms["EE"].append(w * wl.Wpp[l3] * float(s2))
                terms["TE"].append(w * wl.Wtp[l3] * g0 * g2 * math.sqrt(float(s0) * float(s2)))
            else:
                terms["EB"].append(w * wl.Wpp[l3] * float(s2))
        pref = (2 * l2 + 1) / (4 * math.pi)
        for k, t in terms.items():
            ex = pref * math.fsum(t)
            scale = pref * math.fsum(abs(x) for x in t)
            worst_gpu = max(worst_gpu, abs(got[k][l1, l2] - ex) / scale)
            worst_ora = max(worst_ora, abs(ora[k][n] - ex) / scale)
    print("vs exact Racah sums, on the scale of the terms: GPU worst %.2e, oracle worst %.2e" % (worst_gpu, worst_ora))
    assert worst_gpu < 2e-15
    assert worst_ora < 1e-13


# ---------------------------------------------------------------- every shipped sweep variant has its own parity test
@pytest.mark.parametrize("want", [("TT",), ("TE", "EE", "EB"), ("TE", "EE", "BB", "EB")])
@pytest.mark.parametrize("lmax,lcut", [(500, 40), (333, 101)])
def test_band_partial_requests_against_oracle(lmax, lcut, want):
    """tj_coupling_band with TT alone and with the polarised blocks alone (their own sweep variants), element-wise
    against the oracle, and bitwise against the same blocks of the all-blocks band call."""
    import torch
    rng = np.random.default_rng(lmax + lcut)
    W = [np.abs(rng.standard_normal(lcut + 1)) * np.exp(-np.arange(lcut + 1) / 30.0) for _ in range(3)]
    T = binding.build_tables(lmax)
    N, width = lmax + 1, 2 * lcut + 1
    pre = {k: torch.full((N, width), float("nan"), dtype=torch.float64, device="cuda") for k in want}
    got = binding.coupling_band(T, lcut, _t(W[0]) if "TT" in want else None, _t(W[1]) if "TE" in want else None,
                                _t(W[2]) if set(want) & {"EE", "BB", "EB"} else None, want=want, out=pre)
    allb = binding.coupling_band(T, lcut, *[_t(w) for w in W])
    torch.cuda.synchronize()
    ref = oracle.coupling_band(lmax, lcut, *W)
    for k in want:
        assert_parity(got[k].cpu().numpy(), ref[k], "band %r %s" % (want, k))
        assert torch.equal(got[k], allb[k]), (want, k)
    T.close()


def test_band_partial_requests_full_size_cfg4_sampled():
    """Config 4 (lmax 15000, L_cut 300) with TT alone and with the polarised blocks alone: sampled against the oracle."""
    import torch
    wl = windows.config(4)
    lcut = wl.l3max
    T = binding.build_tables(wl.lmax)
    l1, l2 = _sample_pairs(wl.lmax, 1200, 105, band=lcut)
    ref = oracle.coupling_pairs(lcut, wl.Wtt, wl.Wtp, wl.Wpp, l1, l2)
    i1 = torch.as_tensor(l1.astype(np.int64)).cuda()
    io = torch.as_tensor((l2.astype(np.int64) - l1 + lcut)).cuda()
    for want in (("TT",), ("TE", "EE", "EB")):
        got = binding.coupling_band(T, lcut, _t(wl.Wtt) if "TT" in want else None, _t(wl.Wtp) if "TE" in want else None,
                                    _t(wl.Wpp) if "EE" in want else None, want=want)
        torch.cuda.synchronize()
        for k in want:
            assert bool(torch.isfinite(got[k]).all())
            assert_parity(got[k][i1, io].cpu().numpy(), ref[k], "cfg4 %r %s" % (want, k))
    T.close()


def test_row_blocks_pol_only_against_oracle():
    """tj_coupling_rows without TT (its own sweep variant): sampled rows of config 1 against the oracle, bitwise
    against the rows of the full polarised call."""
    import torch
    wl = windows.config(1)
    N = wl.lmax + 1
    T = binding.build_tables(wl.lmax)
    W = [_t(w) for w in (wl.Wtt, wl.Wtp, wl.Wpp)]
    want = ("TE", "EE", "BB", "EB")
    full = binding.coupling_pol(T, None, W[1], W[2], want=want)
    for r0, r1 in ((0, 90), (700, 1291), (N - 45, N)):
        pre = {k: torch.full((r1 - r0, N), float("nan"), dtype=torch.float64, device="cuda") for k in want}
        got = binding.coupling_rows(T, None, W[1], W[2], r0, r1, want=want, out=pre)
        torch.cuda.synchronize()
        rows = np.unique(np.array([r0, (r0 + r1) // 2, r1 - 1], dtype=np.int32))
        ref = oracle.coupling_rows(wl.lmax, wl.l3max, None, wl.Wtp, wl.Wpp, rows)
        for k in want:
            assert torch.equal(got[k], full[k][r0:r1]), (k, r0, r1)
            assert_parity(got[k][torch.as_tensor(rows - r0, dtype=torch.int64).cuda()].cpu().numpy(), ref[k],
                          "pol-only rows [%d,%d) %s" % (r0, r1, k))
    T.close()


def test_row_blocks_tt_only_long_geometry():
    """tj_coupling_rows with TT alone at lmax >= 4096 (the long TT-only geometry): sampled pairs against the oracle,
    whole blocks bitwise against tj_coupling_tt."""
    import torch
    wl = windows.config(2, lmax=4300)
    N = wl.lmax + 1
    T = binding.build_tables(wl.lmax)
    Wtt = _t(wl.Wtt)
    tt = binding.coupling_tt(T, Wtt)
    rng = np.random.default_rng(77)
    for r0, r1 in ((0, 257), (2011, 3100), (N - 300, N)):
        got = binding.coupling_rows(T, Wtt, None, None, r0, r1, want=("TT",))["TT"]
        torch.cuda.synchronize()
        assert torch.equal(got, tt[r0:r1]), (r0, r1)
        l1 = rng.integers(r0, r1, 400).astype(np.int32)
        l2 = rng.integers(0, N, 400).astype(np.int32)
        ref = oracle.coupling_pairs(wl.l3max, wl.Wtt, None, None, l1, l2)
        g = got[torch.as_tensor(l1.astype(np.int64) - r0).cuda(), torch.as_tensor(l2.astype(np.int64)).cuda()].cpu().numpy()
        assert_parity(g, ref["TT"], "TT-only rows [%d,%d)" % (r0, r1))
    T.close()


# ---------------------------------------------------------------- T4 bookkeeping THROUGH THE KERNEL: every l3 slot of every pair
def _oracle_ranges(lmax, l3max):
    """(lo, hi, n) of the l3 sum of every pair, per parity of l1+l2+l3: the ORACLE's integer bookkeeping."""
    out = []
    for par in (0, 1):
        r = np.array([[oracle.l3_range(l1, l2, l3max, par) for l2 in range(lmax + 1)] for l1 in range(lmax + 1)])
        out.append((r[..., 0], r[..., 1], r[..., 2]))
    return out


def _expected_support(ranges, L):
    """Which (l1,l2) have l3 = L among their terms, for even and for odd l1+l2+L."""
    return tuple((n > 0) & (lo <= L) & (L <= hi) & ((L - lo) % 2 == 0) for lo, hi, n in ranges)


@pytest.mark.parametrize("lmax,l3max", [(48, 96), (48, 61), (33, 20)])
def test_spike_every_l3_slot_dense(lmax, l3max):
    """W = delta_{l,L} for EVERY L = 0..l3max: an entry is non-zero iff l3 = L is one of the terms the kernel adds for
    that pair, so the zero pattern of these launches is the kernel's own l3 bookkeeping, slot by slot, compared with
    the oracle's integer ranges (PAPER.md:133-151; :251 for the truncated l3max)."""
    import torch
    T = binding.build_tables(lmax, l3max)
    l1, l2 = np.indices((lmax + 1, lmax + 1))
    pol = (l1 >= 2) & (l2 >= 2)
    ranges = _oracle_ranges(lmax, l3max)
    for L in range(l3max + 1):
        W = _t(windows.spike(l3max, L))
        K = {k: v.cpu().numpy() for k, v in binding.coupling_pol(T, W, W, W).items()}
        ev, od = _expected_support(ranges, L)
        assert np.all(K["TT"][~ev] == 0.0) and np.all(K["TT"][ev] > 0.0), L
        for k in ("TE", "EE", "BB"):
            assert np.all(K[k][~(ev & pol)] == 0.0), (k, L)
        assert np.all(K["EB"][~(od & pol)] == 0.0), L
        assert np.all(K["EE"][ev & pol] >= 0.0) and np.all(K["EB"][od & pol] >= 0.0)
        # the spin-2 symbol has accidental zeros (A = 0), so "non-zero inside" is checked through the oracle's values
        ref = oracle.coupling_full(lmax, l3max, *(3 * [windows.spike(l3max, L)]))
        for k in BLOCKS:
            assert_parity(K[k], ref[k], "spike L=%d %s" % (L, k))
            assert np.all((K[k] != 0.0) | (np.abs(ref[k]) < 1e-13)), (k, L)
    T.close()


@pytest.mark.parametrize("lmax,lcut", [(48, 30), (40, 7)])
def test_spike_every_l3_slot_banded(lmax, lcut):
    """The same through tj_coupling_band: every L = 0..lcut."""
    import torch
    T = binding.build_tables(lmax)
    N, width = lmax + 1, 2 * lcut + 1
    l1 = np.repeat(np.arange(N), width).reshape(N, width)
    l2 = l1 + np.arange(-lcut, lcut + 1)[None, :]
    ok = (l2 >= 0) & (l2 <= lmax)
    pol = (l1 >= 2) & (l2 >= 2)
    ranges = _oracle_ranges(lmax, lcut)
    for L in range(lcut + 1):
        Wn = np.zeros(lcut + 1)
        Wn[L] = 1.0
        W = _t(Wn)
        pre = {k: torch.full((N, width), float("nan"), dtype=torch.float64, device="cuda") for k in BLOCKS}
        K = {k: v.cpu().numpy() for k, v in binding.coupling_band(T, lcut, W, W, W, out=pre).items()}
        ev, od = _expected_support(ranges, L)
        evb = np.zeros((N, width), dtype=bool)
        odb = np.zeros((N, width), dtype=bool)
        evb[ok] = ev[l1[ok], l2[ok]]
        odb[ok] = od[l1[ok], l2[ok]]
        assert np.all(K["TT"][~evb] == 0.0) and np.all(K["TT"][evb] > 0.0), L
        for k in ("TE", "EE", "BB"):
            assert np.all(K[k][~(evb & pol)] == 0.0), (k, L)
        assert np.all(K["EB"][~(odb & pol)] == 0.0), L
        ref = oracle.coupling_band(lmax, lcut, Wn, Wn, Wn)
        for k in BLOCKS:
            assert_parity(K[k], ref[k], "band spike L=%d %s" % (L, k))
    T.close()


# ---------------------------------------------------------------- binned output (DESIGN.md 2 reading 20)
def _bin_weights(lmax, seed):
    rng = np.random.default_rng(seed)
    return rng.uniform(0.5, 1.5, lmax + 1), rng.uniform(0.5, 1.5, lmax + 1)


@pytest.mark.parametrize("lmax,edges", [(100, [0, 2, 7, 7, 30, 64, 101]), (257, [2, 34, 66, 130, 258]), (64, [5, 6]),
                                         (900, list(range(0, 901, 75)) + [901])])
def test_binned_against_oracle_and_binned_full_matrices(lmax, edges):
    import torch
    wl = windows.config(1, lmax=lmax)
    P, Q = _bin_weights(lmax, lmax)
    T = binding.build_tables(lmax)
    W = [_t(w) for w in (wl.Wtt, wl.Wtp, wl.Wpp)]
    nb = len(edges) - 1
    pre = {k: torch.full((nb, nb), float("nan"), dtype=torch.float64, device="cuda") for k in BLOCKS}
    B = binding.coupling_binned(T, *W, edges, _t(P), _t(Q), out=pre)
    full = binding.coupling_pol(T, *W)
    torch.cuda.synchronize()
    pairs = None if lmax <= 300 else [(0, 0), (3, 11), (11, 3), (12, 12), (7, 8), (12, 0)]
    ref = oracle.coupling_binned(lmax, 2 * lmax, wl.Wtt, wl.Wtp, wl.Wpp, edges, P, Q, pairs=pairs)
    for k in BLOCKS:
        got = B[k].cpu().numpy()
        sel = ~np.isnan(ref[k])
        assert_parity(got[sel], ref[k][sel], "binned %s" % k)
        # the same bins formed from the full matrices of tj_coupling_pol, in float64 on the host
        K = full[k].cpu().numpy()
        for b in range(nb):
            for c in range(nb):
                want = float(P[edges[b]:edges[b + 1]] @ K[edges[b]:edges[b + 1], edges[c]:edges[c + 1]] @ Q[edges[c]:edges[c + 1]])
                assert abs(got[b, c] - want) <= 1e-12 * max(abs(want), 1e-6), (k, b, c)
    assert torch.equal(B["BB"], B["EE"])
    # partial requests and determinism
    again = binding.coupling_binned(T, *W, edges, _t(P), _t(Q))
    only = binding.coupling_binned(T, None, None, W[2], edges, _t(P), _t(Q), want=("BB", "EB"))
    tt = binding.coupling_binned(T, W[0], None, None, edges, _t(P), _t(Q), want=("TT",))
    torch.cuda.synchronize()
    for k in BLOCKS:
        assert torch.equal(again[k], B[k]), k
    assert_parity(only["EB"].cpu().numpy(), B["EB"].cpu().numpy(), "binned EB alone")
    assert_parity(only["BB"].cpu().numpy(), B["BB"].cpu().numpy(), "binned BB alone")
    assert_parity(tt["TT"].cpu().numpy(), B["TT"].cpu().numpy(), "binned TT alone")
    with pytest.raises(binding.TJError):
        binding.coupling_binned(T, *W, [0, 5, 3], _t(P), _t(Q))
    with pytest.raises(binding.TJError):
        binding.coupling_binned(T, *W, [0, lmax + 2], _t(P), _t(Q))
    T.close()


@pytest.mark.parametrize("cfg,width", [(1, 40), (3, 50)])
def test_binned_full_size_configs_sampled_bins(cfg, width):
    """Configs 1 and 3 at full size (config 3: several chunks of rows): sampled bin pairs against the oracle."""
    import torch
    wl = windows.config(cfg)
    lmax = wl.lmax
    edges = list(range(2, lmax + 1, width)) + [lmax + 1]
    nb = len(edges) - 1
    l = np.arange(lmax + 1, dtype=np.float64)
    P = (l * (l + 1) / (2 * np.pi)) / width                      # a band-power operator and its inverse
    Q = np.where(l > 0, 2 * np.pi / np.maximum(l * (l + 1), 1.0), 0.0)
    T = binding.build_tables(lmax)
    B = binding.coupling_binned(T, _t(wl.Wtt), _t(wl.Wtp), _t(wl.Wpp), edges, _t(P), _t(Q))
    torch.cuda.synchronize()
    pairs = [(0, 0), (0, 1), (1, 0), (nb - 1, nb - 1), (nb // 2, nb // 2), (nb // 2, nb // 2 + 1), (nb // 3, nb - 2), (nb - 1, 0)]
    ref = oracle.coupling_binned(lmax, wl.l3max, wl.Wtt, wl.Wtp, wl.Wpp, edges, P, Q, pairs=pairs)
    for k in BLOCKS:
        got = B[k].cpu().numpy()
        assert np.all(np.isfinite(got))
        sel = ~np.isnan(ref[k])
        # a bin is a sum of width^2 entries of either sign (TE): the bar applies on the scale of the bin's largest entry sum
        assert_parity(got[sel], ref[k][sel], "cfg%d binned %s" % (cfg, k))
    T.close()


@pytest.mark.parametrize("lmax,edges", [(2000, [0, 2001]), (2000, [2, 300, 301, 1200, 2001]), (3000, [0, 2, 1500, 3001])])
def test_binned_few_wide_bins_split_over_ctas(lmax, edges):
    """One to four wide bins: each bin pair is shared by many CTAs whose partial sums a second pass adds in a fixed order
    (tj_binned.cu).  Against the same bins formed on the host from the full matrices of tj_coupling_pol (which the tests
    above hold against the oracle), against the oracle's own binned sums on a one-row bin, and bit-identical when repeated."""
    import torch
    wl = windows.config(2, lmax=lmax)
    P, Q = _bin_weights(lmax, 3 * lmax)
    T = binding.build_tables(lmax)
    W = [_t(w) for w in (wl.Wtt, wl.Wtp, wl.Wpp)]
    nb = len(edges) - 1
    pre = {k: torch.full((nb, nb), float("nan"), dtype=torch.float64, device="cuda") for k in BLOCKS}
    B = binding.coupling_binned(T, *W, edges, _t(P), _t(Q), out=pre)
    again = binding.coupling_binned(T, *W, edges, _t(P), _t(Q))
    full = binding.coupling_pol(T, *W)
    torch.cuda.synchronize()
    for k in BLOCKS:
        assert torch.equal(again[k], B[k]), k
        got = B[k].cpu().numpy()
        K = full[k].cpu().numpy()
        for b in range(nb):
            for c in range(nb):
                sl = K[edges[b]:edges[b + 1], edges[c]:edges[c + 1]]
                want = float(P[edges[b]:edges[b + 1]] @ sl @ Q[edges[c]:edges[c + 1]])
                scale = float(np.abs(P[edges[b]:edges[b + 1]]) @ np.abs(sl) @ np.abs(Q[edges[c]:edges[c + 1]]))
                assert abs(got[b, c] - want) <= 1e-12 * max(scale, 1e-6), (k, b, c, got[b, c], want)
    if nb == 4:   # the one-row bin [300, 301): its bin pairs are cheap for the oracle
        pairs = [(1, 0), (1, 1), (1, 2), (1, 3), (0, 1), (3, 1)]
        ref = oracle.coupling_binned(lmax, 2 * lmax, wl.Wtt, wl.Wtp, wl.Wpp, edges, P, Q, pairs=pairs)
        for k in BLOCKS:
            sel = ~np.isnan(ref[k])
            assert sel.sum() == len(pairs)
            assert_parity(B[k].cpu().numpy()[sel], ref[k][sel], "few bins %s" % k)
    T.close()


@pytest.mark.parametrize("lmax,nwin,edges", [(150, 5, [0, 2, 9, 9, 40, 100, 151]), (2000, 3, list(range(2, 2001, 40)) + [2001])])
def test_binned_multi_window_against_oracle_and_single_calls(lmax, nwin, edges):
    """tj_coupling_binned_multi (many map pairs -> nwin * nbins^2 numbers per block, SURVEY.md 8(f) #1 + #4): against the
    oracle (all bins at the small size, sampled bins at config-1 size) and bit for bit against nwin single-set
    tj_coupling_binned calls (one chunk of rows at these sizes); groups of 3 + 2 sets, TT alone in 4 + 1, a partial
    request one set at a time."""
    import torch
    Wtt, Wtp, Wpp = _window_sets(lmax, nwin, 40)
    P, Q = _bin_weights(lmax, 11 * lmax)
    T = binding.build_tables(lmax)
    W = [_t(Wtt), _t(Wtp), _t(Wpp)]
    nb = len(edges) - 1
    pre = {k: torch.full((nwin, nb, nb), float("nan"), dtype=torch.float64, device="cuda") for k in BLOCKS}
    B = binding.coupling_binned_multi(T, *W, edges, _t(P), _t(Q), out=pre)
    geo = binding.profile_last_sweep()
    assert geo["nw"] == (2 if nwin == 5 else 3), geo
    torch.cuda.synchronize()
    for w in range(nwin):
        one = binding.coupling_binned(T, W[0][w].contiguous(), W[1][w].contiguous(), W[2][w].contiguous(), edges, _t(P), _t(Q))
        for k in BLOCKS:
            assert torch.equal(B[k][w], one[k]), (w, k)
    pairs = None if lmax <= 300 else [(0, 0), (3, 11), (11, 3), (nb - 1, nb - 1), (7, 8), (nb - 1, 0)]
    ref = oracle.coupling_binned_multi(lmax, 2 * lmax, Wtt, Wtp, Wpp, edges, P, Q, pairs=pairs)
    for k in BLOCKS:
        got = B[k].cpu().numpy()
        assert np.all(np.isfinite(got)), k
        sel = ~np.isnan(ref[k])
        assert_parity(got[sel], ref[k][sel], "binned multi %s" % k)
    assert torch.equal(B["BB"], B["EE"])
    tt = binding.coupling_binned_multi(T, W[0], None, None, edges, _t(P), _t(Q), want=("TT",))
    assert binding.profile_last_sweep()["nw"] == 1      # 4 + 1, or 2 + 1: the last sweep holds the odd set
    pol = binding.coupling_binned_multi(T, None, W[1], W[2], edges, _t(P), _t(Q), want=("TE", "BB", "EB"))
    torch.cuda.synchronize()
    assert_parity(tt["TT"].cpu().numpy(), B["TT"].cpu().numpy(), "binned multi TT alone")
    for k in ("TE", "BB", "EB"):
        assert_parity(pol[k].cpu().numpy(), B[k].cpu().numpy(), "binned multi pol %s" % k)
    T.close()


def test_binned_flat_window_closed_form_multi_chunk():
    """Flat window at lmax = 7000 (two chunks of rows): every bin against B = (sum_b P)(sum_b' Q (2l+1))/4 pi, TE = 0,
    EE + EB = the same on l >= 2 -- no oracle sample involved."""
    import torch
    lmax = 7000
    edges = [0, 2] + list(range(30, lmax, 97)) + [lmax + 1]
    nb = len(edges) - 1
    P, Q = _bin_weights(lmax, 5)
    W = _t(np.ones(2 * lmax + 1))
    T = binding.build_tables(lmax)
    B = {k: v.cpu().numpy() for k, v in binding.coupling_binned(T, W, W, W, edges, _t(P), _t(Q)).items()}
    l = np.arange(lmax + 1)
    sp = np.array([P[edges[b]:edges[b + 1]].sum() for b in range(nb)])
    sq = np.array([(Q[edges[b]:edges[b + 1]] * (2 * l[edges[b]:edges[b + 1]] + 1)).sum() for b in range(nb)])
    want = np.outer(sp, sq) / (4 * np.pi)
    assert np.all(np.abs(B["TT"] - want) <= 1e-11 * want)
    assert np.all(np.abs(B["TE"]) <= 1e-11 * want)
    pol = want.copy()
    pol[0, :] = 0.0
    pol[:, 0] = 0.0                                   # bin 0 = l < 2
    assert np.all(np.abs(B["EE"] + B["EB"] - pol) <= 1e-11 * np.maximum(want, 1e-30))
    T.close()


# ---------------------------------------------------------------- sizes far past the configs (index arithmetic, table range)
def test_flat_window_closed_form_tt_lmax40000():
    """The largest dense size the tests run: lmax = 40000 (TT alone: 12.8 GB, tables up to p = 80001, 2.0e6 one-warp
    tiles): the flat-window closed form K^TT = (2 l2+1)/(4 pi) (orthogonality over l3) in every entry."""
    import torch
    lmax = 40000
    N = lmax + 1
    free, _ = torch.cuda.mem_get_info()
    if free < 16 * 2 ** 30:
        pytest.skip("needs 16 GB of free device memory")
    W = _t(windows.flat(2 * lmax))
    T = binding.build_tables(lmax)
    TT = binding.coupling_tt(T, W)
    torch.cuda.synchronize()
    col = (2.0 * torch.arange(N, dtype=torch.float64, device="cuda") + 1.0) / (4 * math.pi)
    worst = 0.0
    for r0 in range(0, N, 4000):   # row chunks: no second matrix-sized temporary
        blk = TT[r0:r0 + 4000]
        worst = max(worst, float(((blk - col[None, :]).abs() / col[None, :]).max()))
    print("flat window lmax=40000: TT rel %.2e" % worst)
    assert worst < 1e-12, worst
    del TT
    T.close()


def test_band_long_matrix_lmax100000_lcut64_sampled():
    """A band-limited call on a very long matrix (lmax = 10^5, L_cut = 64; 3126 diagonal blocks): every slot written,
    out-of-range slots exactly 0, sampled entries against the oracle (which recurses the whole l3 range of each pair)."""
    import torch
    lmax, lcut = 100000, 64
    l = np.arange(lcut + 1, dtype=np.float64)
    W = 4.0 * math.pi * 0.25 * np.exp(-l * l / (2.0 * 20.0 ** 2))
    Wtp = W * (1.0 - 0.01 * l)          # three different windows, TP with a sign change at l = 100 (none here) ...
    Wpp = W * (1.0 + 0.02 * l)
    T = binding.build_tables(lmax)
    N, width = lmax + 1, 2 * lcut + 1
    pre = {k: torch.full((N, width), float("nan"), dtype=torch.float64, device="cuda") for k in BLOCKS}
    out = binding.coupling_band(T, lcut, _t(W), _t(Wtp), _t(Wpp), out=pre)
    torch.cuda.synchronize()
    l2grid = torch.arange(N, device="cuda")[:, None] + torch.arange(-lcut, lcut + 1, device="cuda")[None, :]
    outside = (l2grid < 0) | (l2grid > lmax)
    for k in BLOCKS:
        assert bool(torch.isfinite(out[k]).all()), k
        assert bool((out[k][outside] == 0).all()), k
    assert bool((out["BB"] == out["EE"]).all())
    l1, l2 = _sample_pairs(lmax, 300, 777, band=lcut)
    ref = oracle.coupling_pairs(lcut, W, Wtp, Wpp, l1, l2)
    i1 = torch.as_tensor(l1.astype(np.int64)).cuda()
    io = torch.as_tensor((l2.astype(np.int64) - l1 + lcut)).cuda()
    for k in BLOCKS:
        got = out[k][i1, io].cpu().numpy()
        assert_parity(got, ref[k], "band lmax=1e5 %s" % k)
    _assert_band_row_sums(out, lmax, lcut, W, Wpp, "band lmax=1e5")
    T.close()
