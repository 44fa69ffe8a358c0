"""The host-buffer call's row-chunk pipeline in each of its regimes, pageable outputs, and the handle-sharing promises
of include/tj.h (one handle used from several threads and streams; one handle per device).  -m gpu.

The regimes are forced through tj_set_host_pipeline at a size the suite finishes in a second (the sizes at which
they arise by themselves are covered in tests/test_gpu_staged_sweep.py and tests/test_gpu_parity.py); every output entry,
pre-filled with NaN, must carry the bits of the device-buffer call, which those files hold against the oracle.
"""
import threading

import numpy as np
import pytest

from paper_2602_15605_b200 import binding, build, windows

pytestmark = pytest.mark.gpu

BLOCKS = ("TT", "TE", "EE", "BB", "EB")


@pytest.fixture(scope="module", autouse=True)
def _lib():
    build.build()
    binding.load_library()


def _problem(lmax, cfg=2):
    import torch
    wl = windows.config(cfg, lmax=lmax)
    hw = [torch.as_tensor(w, dtype=torch.float64) for w in (wl.Wtt, wl.Wtp, wl.Wpp)]
    return wl, hw


def _nan_out(N, keys, pinned=True):
    import torch
    out = {k: torch.full((N, N), float("nan"), dtype=torch.float64) for k in keys}
    return {k: v.pin_memory() for k, v in out.items()} if pinned else out


@pytest.mark.parametrize("keys", [BLOCKS, ("TT",), ("TE", "BB")])
def test_each_regime_forced_bitwise(keys):
    import torch
    lmax = 1000
    wl, hw = _problem(lmax)
    N = lmax + 1
    T = binding.build_tables(lmax)
    dev = [w.cuda() for w in hw]
    pol = len(keys) > 1 or keys[0] != "TT"
    ref = binding.coupling_pol(T, dev[0] if "TT" in keys else None, dev[1] if "TE" in keys else None,
                               dev[2] if pol else None, want=keys)
    torch.cuda.synchronize()
    pw = [w.pin_memory() for w in hw]
    args = (pw[0] if "TT" in keys else None, pw[1] if "TE" in keys else None, pw[2] if pol else None)
    assert binding.host_pipeline_info(T) == (0, 0)
    seen = {}
    # a copy rate of 1 byte/s makes any call copy-bound, an absurdly fast link makes it compute-bound; (0, 0) = defaults
    for copy_rate, want_regime in ((1.0, 1), (1e18, 2), (0.0, None)):
        binding.set_host_pipeline(T, copy_rate, 0.0)
        out = _nan_out(N, keys)
        binding.coupling_host(T, *args, out)
        regime, nchunks = binding.host_pipeline_info(T)
        if want_regime is not None:
            assert regime == want_regime, (copy_rate, regime)
        assert regime in (1, 2) and 1 <= nchunks <= 24
        seen[regime] = nchunks
        for k in keys:
            assert torch.equal(out[k].cuda(), ref[k]), (copy_rate, k)
    assert set(seen) == {1, 2} and seen[1] > seen[2], seen    # many small row chunks vs a few L-shaped ones
    with pytest.raises(binding.TJError):
        binding.set_host_pipeline(T, -1.0, 0.0)
    with pytest.raises(binding.TJError):
        binding.set_host_pipeline(T, float("nan"), 0.0)
    T.close()


def test_pageable_outputs_take_the_plain_path_bitwise():
    """Pageable host buffers: copies into them block the calling thread, so the call computes first and copies each
    matrix in one piece (regime 3).  Same bits as the device path; pageable windows as well."""
    import torch
    lmax = 1200
    wl, hw = _problem(lmax, cfg=1)
    N = lmax + 1
    T = binding.build_tables(lmax)
    ref = binding.coupling_pol(T, *[w.cuda() for w in hw])
    torch.cuda.synchronize()
    out = _nan_out(N, BLOCKS, pinned=False)
    binding.coupling_host(T, *hw, out)
    assert binding.host_pipeline_info(T) == (3, 1)
    for k in BLOCKS:
        assert torch.equal(out[k].cuda(), ref[k]), k
    # one pageable output among pinned ones is enough to take that path
    mixed = _nan_out(N, ("TT", "EB"))
    mixed["TE"] = torch.full((N, N), float("nan"), dtype=torch.float64)
    binding.coupling_host(T, *[w.pin_memory() for w in hw], mixed)
    assert binding.host_pipeline_info(T)[0] == 3
    for k in mixed:
        assert torch.equal(mixed[k].cuda(), ref[k]), k
    T.close()


def test_one_handle_from_two_threads_host_and_device_calls():
    """include/tj.h: the tables are immutable after the build, so one handle may be used from several threads and
    streams at once; host-buffer calls that share a handle are serialised inside the library.  Two threads, each on
    its own stream, each with its own windows, run host-buffer and device-buffer calls on ONE handle at the same time,
    several times over; every result must carry the bits of the same call made alone."""
    import torch
    lmax = 1100
    N = lmax + 1
    T = binding.build_tables(lmax)
    probs = [_problem(lmax, cfg=c)[1] for c in (1, 2)]
    alone = []
    for hw in probs:
        alone.append(binding.coupling_pol(T, *[w.cuda() for w in hw]))
    torch.cuda.synchronize()
    errors = []
    barrier = threading.Barrier(2)

    def worker(i):
        try:
            torch.cuda.set_device(0)
            s = torch.cuda.Stream()
            hw = [w.pin_memory() for w in probs[i]]
            with torch.cuda.stream(s):
                dw = [w.cuda(non_blocking=True) for w in hw]
                barrier.wait()
                for rep in range(4):
                    hout = _nan_out(N, BLOCKS)
                    binding.coupling_host(T, *hw, hout, stream=s)          # synchronises its stream
                    dout = {k: torch.full((N, N), float("nan"), dtype=torch.float64, device="cuda") for k in BLOCKS}
                    binding.coupling_pol(T, *dw, out=dout, stream=s)
                    s.synchronize()
                    for k in BLOCKS:
                        if not torch.equal(hout[k].cuda(), alone[i][k]):
                            errors.append("thread %d rep %d host %s" % (i, rep, k))
                        if not torch.equal(dout[k], alone[i][k]):
                            errors.append("thread %d rep %d device %s" % (i, rep, k))
        except Exception as e:   # noqa: BLE001 -- reported to the main thread
            errors.append("thread %d: %r" % (i, e))
            try:
                barrier.abort()
            except Exception:
                pass

    th = [threading.Thread(target=worker, args=(i,)) for i in range(2)]
    for t in th:
        t.start()
    for t in th:
        t.join()
    torch.cuda.synchronize()
    assert not errors, errors
    T.close()


# ---------------------------------------------------------------- one matrix on several devices, every pair swept once
def _plan_mask(lmax, nparts, part, tt_only=False):
    import torch
    bounds, owner = binding.chunk_plan(lmax, nparts, tt_only=tt_only)
    N = lmax + 1
    m = torch.zeros((N, N), dtype=torch.bool)
    for k, g in enumerate(owner):
        if g == part:
            r0, r1 = bounds[k], bounds[k + 1]
            m[r0:r1, r0:] = True
            m[r1:, r0:r1] = True
    return m


@pytest.mark.parametrize("lmax,nparts,keys", [(1000, 2, BLOCKS), (2700, 4, BLOCKS), (1500, 3, ("TT",)), (300, 2, ("EE", "EB"))])
def test_host_parts_one_after_the_other_complete_the_matrix_bitwise(lmax, nparts, keys):
    """tj_coupling_host_part for part = 0..nparts-1 into ONE set of host matrices (here one after the other on one GPU;
    on nparts GPUs the same calls run side by side): each call writes exactly the regions of its own chunks and nothing
    else, and together they give the bits of the whole-matrix call."""
    import torch
    wl, hw = _problem(lmax)
    N = lmax + 1
    T = binding.build_tables(lmax)
    dev = [w.cuda() for w in hw]
    tt_only = keys == ("TT",)
    pol = not tt_only
    ref = binding.coupling_pol(T, dev[0] if "TT" in keys else None, dev[1] if "TE" in keys else None,
                               dev[2] if pol else None, want=keys)
    torch.cuda.synchronize()
    ref = {k: v.cpu() for k, v in ref.items()}
    pw = [w.pin_memory() for w in hw]
    args = (pw[0] if "TT" in keys else None, pw[1] if "TE" in keys else None, pw[2] if pol else None)
    out = _nan_out(N, keys)
    done = torch.zeros((N, N), dtype=torch.bool)
    for part in range(nparts):
        binding.coupling_host_part(T, part, nparts, *args, out)
        assert binding.host_pipeline_info(T)[0] == 4
        mine = _plan_mask(lmax, nparts, part, tt_only=tt_only)
        assert not bool((done & mine).any())
        done |= mine
        for k in keys:
            assert bool(torch.isnan(out[k][~done]).all()), (part, k)          # nothing outside the parts run so far
            assert torch.equal(out[k][mine], ref[k][mine]), (part, k)
    assert bool(done.all())
    for k in keys:
        assert torch.equal(out[k], ref[k]), k
    with pytest.raises(binding.TJError):
        binding.coupling_host_part(T, nparts, nparts, *args, out)
    T.close()


def test_host_multi_with_three_handles_on_one_gpu_bitwise():
    """tj_coupling_host_multi with three handles ("virtual ranks": all on this one GPU, each with its own stream and side
    streams), running side by side: the one set of host matrices is complete and carries the bits of the single call."""
    import torch
    lmax = 2700
    wl, hw = _problem(lmax, cfg=3)
    N = lmax + 1
    Ts = [binding.build_tables(lmax) for _ in range(3)]
    ref = binding.coupling_pol(Ts[0], *[w.cuda() for w in hw])
    torch.cuda.synchronize()
    pw = [w.pin_memory() for w in hw]
    for streams in (None, [torch.cuda.Stream() for _ in range(3)]):
        out = _nan_out(N, BLOCKS)
        binding.coupling_host_multi(Ts, *pw, out, streams=streams)
        for k in BLOCKS:
            assert torch.equal(out[k].cuda(), ref[k]), k
        assert [binding.host_pipeline_info(t)[0] for t in Ts] == [4, 4, 4]
    with pytest.raises(binding.TJError):      # the same handle twice
        binding.coupling_host_multi([Ts[0], Ts[0]], *pw, _nan_out(N, BLOCKS))
    for t in Ts:
        t.close()


def test_profiled_calls_keep_their_status_and_times_per_thread():
    """Per-kernel profiling is per thread: a thread that has made no profiled call gets TJ_EINVAL from tj_profile_get,
    and profiling never changes a call's result."""
    import torch
    lmax = 900
    wl, hw = _problem(lmax, cfg=1)
    T = binding.build_tables(lmax)
    dw = [w.cuda() for w in hw]
    ref = binding.coupling_pol(T, *dw)
    binding.profile_enable(True)
    try:
        got = binding.coupling_pol(T, *dw)
        ms = binding.profile_get()
        assert all(m >= 0.0 for m in ms) and ms[1] > 0.0
        for k in BLOCKS:
            assert torch.equal(got[k], ref[k]), k
        res = []
        t = threading.Thread(target=lambda: res.append(_raises_einval()))
        t.start()
        t.join()
        assert res == [True]
    finally:
        binding.profile_enable(False)
    T.close()


def _raises_einval():
    try:
        binding.profile_get()
    except binding.TJError as e:
        return e.code == binding.TJ_EINVAL
    return False


# ---------------------------------------------------------------- one handle per device (needs two GPUs; skipped on one)
def _two_gpus():
    import torch
    return torch.cuda.device_count() >= 2


def test_handle_is_bound_to_its_device():
    import torch
    if not _two_gpus():
        pytest.skip("needs two GPUs")
    lmax = 900
    wl, hw = _problem(lmax, cfg=1)
    with torch.cuda.device(0):
        T0 = binding.build_tables(lmax)
        ref = binding.coupling_pol(T0, *[w.cuda() for w in hw])
        torch.cuda.synchronize()
    with torch.cuda.device(1):
        d1 = [w.cuda() for w in hw]
        with pytest.raises(binding.TJError) as ei:
            binding.coupling_pol(T0, *d1)            # handle of device 0, device 1 current
        assert ei.value.code == binding.TJ_EINVAL
        T1 = binding.build_tables(lmax)
        binding.profile_enable(True)                 # profiling events are per (thread, device)
        try:
            got = binding.coupling_pol(T1, *d1)
            torch.cuda.synchronize()
            assert binding.profile_get()[1] > 0.0
        finally:
            binding.profile_enable(False)
        for k in BLOCKS:
            assert torch.equal(got[k].cpu(), ref[k].cpu()), k
        # the no-allocation entry point looks its array up per device
        out = {k: torch.full((lmax + 1, lmax + 1), float("nan"), dtype=torch.float64, device="cuda") for k in BLOCKS}
        binding.coupling_pol_static(T1, *d1, out)
        torch.cuda.synchronize()
        for k in BLOCKS:
            assert torch.equal(out[k].cpu(), ref[k].cpu()), k
        T1.close()
    with torch.cuda.device(0):
        T0.close()


def test_two_devices_from_two_threads():
    import torch
    if not _two_gpus():
        pytest.skip("needs two GPUs")
    lmax = 1100
    N = lmax + 1
    wl, hw = _problem(lmax, cfg=2)
    with torch.cuda.device(0):
        T = binding.build_tables(lmax)
        ref = {k: v.cpu() for k, v in binding.coupling_pol(T, *[w.cuda() for w in hw]).items()}
        T.close()
    errors = []

    def worker(dev):
        try:
            with torch.cuda.device(dev):
                Td = binding.build_tables(lmax)
                hout = _nan_out(N, BLOCKS)
                binding.coupling_host(Td, *[w.pin_memory() for w in hw], hout)
                for k in BLOCKS:
                    if not torch.equal(hout[k], ref[k]):
                        errors.append("device %d %s" % (dev, k))
                Td.close()
        except Exception as e:   # noqa: BLE001
            errors.append("device %d: %r" % (dev, e))

    th = [threading.Thread(target=worker, args=(d,)) for d in (0, 1)]
    for t in th:
        t.start()
    for t in th:
        t.join()
    assert not errors, errors


def test_host_multi_on_two_devices():
    """tj_coupling_host_multi with one handle per GPU: the one set of host matrices carries the bits of the single call."""
    import torch
    if not _two_gpus():
        pytest.skip("needs two GPUs")
    lmax = 2700
    N = lmax + 1
    wl, hw = _problem(lmax, cfg=3)
    Ts = []
    for d in (0, 1):
        with torch.cuda.device(d):
            Ts.append(binding.build_tables(lmax))
    with torch.cuda.device(0):
        ref = {k: v.cpu() for k, v in binding.coupling_pol(Ts[0], *[w.cuda() for w in hw]).items()}
        out = _nan_out(N, BLOCKS)
        binding.coupling_host_multi(Ts, *[w.pin_memory() for w in hw], out)
        assert torch.cuda.current_device() == 0
    for k in BLOCKS:
        assert torch.equal(out[k], ref[k]), k
    for d in (0, 1):
        with torch.cuda.device(d):
            Ts[d].close()
