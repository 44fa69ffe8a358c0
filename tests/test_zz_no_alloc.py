"""tj_coupling_pol_static: the coupling call for programs that may not allocate GPU memory.

Some users of libtj cannot let a library allocate on the device: an application that reserved all of GPU memory
for its own arena at start-up (an allocation made behind its back fails, or takes what it thought it owned), a loop
with a hard latency budget (no allocator lock, no pool growth in the middle of it), a GPU set-up that does not offer
the stream-ordered pool the other entry points draw their scratch from.  For them the library keeps that scratch in
a fixed 2 MiB device array and runs the same kernels on it.  This file checks that entry point against the ordinary
one, tj_coupling_pol, at the tolerance of tests/test_gpu_parity.py, on calls made one after the other -- the second
with other windows, a smaller lmax, a truncated l3max and fewer blocks, so that anything the first call left in the
shared array and the second failed to overwrite would show up in the result.

It is named test_zz_* so that pytest collects it after every other test file: under `-x` a failure here hides nothing.
It does not depend on what ran before it (the array's address is looked up on the first call in the process, wherever
that call is made), so it passes alone in a fresh process and at the end of the whole suite.  Needs a B200: -m gpu.
"""
import ctypes

import numpy as np
import pytest

from paper_2602_15605_b200 import binding, build, windows

pytestmark = pytest.mark.gpu

RTOL, ATOL_SMALL, SMALL = 1e-10, 1e-14, 1e-4      # the bar of tests/test_gpu_parity.py
BLOCKS = ("TT", "TE", "EE", "BB", "EB")


@pytest.fixture(scope="module", autouse=True)
def _lib():
    build.build()
    binding.load_library()


def _dev(a):
    import torch
    return torch.as_tensor(np.ascontiguousarray(a), dtype=torch.float64).cuda()


def _close(got, ref, what):
    got, ref = got.cpu().numpy(), ref.cpu().numpy()
    assert np.all(np.isfinite(got)), what
    err = np.abs(got - ref)
    big = np.abs(ref) >= SMALL
    assert np.all(err[big] <= RTOL * np.abs(ref[big])), what
    assert np.all(err[~big] <= ATOL_SMALL), what
    assert np.array_equal(got == 0.0, ref == 0.0), what + ": zero pattern"


def _both(lmax, l3max, W, want):
    """(static-scratch result, ordinary result) for one problem; outputs start as NaN so that an entry the call
    did not write cannot pass."""
    import torch
    T = binding.build_tables(lmax, l3max)
    N = lmax + 1
    out = {k: torch.full((N, N), float("nan"), dtype=torch.float64, device="cuda") for k in want}
    binding.coupling_pol_static(T, W[0], W[1], W[2], out)
    geo = binding.profile_last_sweep()
    ref = binding.coupling_pol(T, W[0], W[1], W[2], want=want)
    torch.cuda.synchronize()
    T.close()
    return out, ref, geo


def test_static_scratch_matches_ordinary_path_on_consecutive_calls():
    import torch
    # call 1: all five blocks above the single-launch threshold -- both entry points run the same three kernels, so
    # beyond the tolerance the results must be the same bits
    wl = windows.config(1, lmax=1000)
    W1 = [_dev(w) for w in (wl.Wtt, wl.Wtp, wl.Wpp)]
    out1, ref1, geo1 = _both(wl.lmax, wl.l3max, W1, BLOCKS)
    assert geo1["TS"] > 0, geo1          # the staged sweep, i.e. the kernels that use the scratch
    for k in BLOCKS:
        _close(out1[k], ref1[k], "call 1 " + k)
        assert torch.equal(out1[k], ref1[k]), "call 1 %s: same kernels, same bits" % k

    # call 2, straight after: signed windows, smaller lmax, l3max < 2 lmax, polarised blocks only.  The array still
    # holds call 1's longer pre-folded windows and tile schedule; none of it may leak into this result.
    rng = np.random.default_rng(20260215)
    lmax2, l3max2 = 900, 1234
    W2 = [_dev(rng.standard_normal(l3max2 + 1) / (1.0 + np.arange(l3max2 + 1.0))) for _ in range(3)]
    want2 = ("TE", "EE", "EB")
    out2, ref2, geo2 = _both(lmax2, l3max2, W2, want2)
    assert geo2["TS"] > 0, geo2
    for k in want2:
        _close(out2[k], ref2[k], "call 2 " + k)
        assert torch.equal(out2[k], ref2[k]), "call 2 %s: same kernels, same bits" % k

    # call 3: the first problem again -- after call 2 overwrote the array, the first answer must come back unchanged
    out3, _, _ = _both(wl.lmax, wl.l3max, W1, BLOCKS)
    for k in BLOCKS:
        assert torch.equal(out3[k], out1[k]), "call 3 " + k

    # below the threshold the ordinary entry point takes its single-launch kernel; this one still runs the staged
    # sweep on the array, and the two agree to the tolerance (TT alone, tiny and ragged sizes included)
    for lmax in (0, 1, 2, 45, 300):
        w = windows.config(1, lmax=lmax)
        W = [_dev(x) for x in (w.Wtt, w.Wtp, w.Wpp)]
        o, r, _ = _both(lmax, w.l3max, W, BLOCKS)
        for k in BLOCKS:
            _close(o[k], r[k], "lmax %d %s" % (lmax, k))
        o, r, _ = _both(lmax, w.l3max, [W[0], None, None], ("TT",))
        _close(o["TT"], r["TT"], "lmax %d TT alone" % lmax)


def test_static_scratch_refuses_what_does_not_fit():
    """A handle beyond TJ_STATIC_LMAX is turned away with TJ_ELIMIT and a message that names the limit, before anything
    runs: the output is untouched.  (The outputs of such a call would be 2 GiB each; the refusal comes first, so a
    one-element stand-in is enough here.)"""
    import torch
    L = binding.load_library()
    lmax = binding.TJ_STATIC_LMAX + 1
    T = binding.build_tables(lmax, 64)
    W = torch.ones(65, dtype=torch.float64, device="cuda")
    canary = torch.full((1,), -7.0, dtype=torch.float64, device="cuda")
    null = ctypes.c_void_p(0)
    rc = L.tj_coupling_pol_static(T.handle, ctypes.c_void_p(W.data_ptr()), null, null, 65,
                                  ctypes.c_void_p(canary.data_ptr()), null, null, null, null, null)
    assert rc == binding.TJ_ELIMIT
    assert b"TJ_STATIC_LMAX" in L.tj_strerror(rc)
    torch.cuda.synchronize()
    assert canary.item() == -7.0
    T.close()
    # the largest handle that is accepted does fit (argument errors are still reported as such)
    T = binding.build_tables(binding.TJ_STATIC_LMAX, 8)
    assert L.tj_coupling_pol_static(T.handle, null, null, null, 9, null, null, null, null, null, null) == binding.TJ_EINVAL
    with pytest.raises(binding.TJError):
        binding.coupling_pol_static(T, W, None, None, {})
    T.close()
