#!/usr/bin/env python
"""bench.py -- the headline measurement (BASELINE.json `metric`).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 3]

One "step" = one pass of the whole hot path (prepare -> fused l3 sweep -> mirrored writer) for
TT+TE+EE+BB+EB on BASELINE.json configs[3] (lmax = 10000, l3 up to 20000, synthetic seeded windows),
through the C ABI (tj_coupling_pol), inputs resident in HBM.  metric = evaluated l3 terms per second
(upper triangle, even-J + odd-J terms).  Prints ONE JSON line (rank 0).

N > 1 (torchrun): the path has no exchange step; every rank runs the same-size problem on its own
window set (seed 3 + rank) -- weak scaling over independent window sets, no data-path collective.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "coupling-matrix l3-terms/sec (FP64) at lmax=10000, fraction of B200 FP64 peak"
UNIT = "l3-terms/s"

# FP64 roofline: 148 SMs x 64 FP64 lanes/clk (GB100: 4 SMSPs x 16 lanes) x SM clock.
SM_COUNT = 148
FP64_LANES_PER_SM = 64
# algorithmic FP64 instructions per evaluated term
INSTR_EVEN_POL, INSTR_ODD, INSTR_EVEN_TT = 8, 5, 2


def _peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as fh:
            return json.load(fh), "measured"
    return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "sm_max_mhz": 1965.0}, "fallback"


def _traffic(workload, geo):
    """DRAM bytes of one sweep launch for this workload from profiles/traffic.csv (written from ncu --set full
    captures; columns: workload, kernel prefix, dram_read_bytes, dram_write_bytes, capture)."""
    p = os.path.join(ROOT, "profiles", "traffic.csv")
    if workload is None or not os.path.exists(p):
        return None, None
    import csv
    with open(p) as fh:
        for row in csv.DictReader(fh):
            if row["workload"] == workload and geo["name"].startswith(row["kernel_prefix"]):
                return float(row["dram_read_bytes"]) + float(row["dram_write_bytes"]), row["capture"]
    return None, None


class ClockSampler:
    """nvidia-smi sampling DURING the timed region (B200_PROFILING.md clocks line)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index=0):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.p = None
        self.gpu = gpu_index

    def start(self):
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(self.gpu), "--query-gpu=" + self.Q,
                                       "--format=csv,noheader,nounits", "-lms", "100"],
                                      stdout=self.f, stderr=subprocess.DEVNULL)
        except Exception:
            self.p = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.p is None:
            return out
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except Exception:
            self.p.kill()
        self.f.flush()
        self.f.seek(0)
        sm, mx, pw, reasons = [], [], [], set()
        for line in self.f.read().splitlines():
            c = [x.strip() for x in line.split(",")]
            if len(c) < 9:
                continue
            try:
                sm.append(float(c[1])); mx.append(float(c[2])); pw.append(float(c[3]))
            except ValueError:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), c[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        try:
            os.unlink(self.f.name)
        except OSError:
            pass
        if sm:
            # "under load" = samples in the upper half of the power range
            thr = 0.5 * (max(pw) + min(pw)) if pw else 0
            load = [s for s, w in zip(sm, pw) if w >= thr] or sm
            out.update(sm_mhz=statistics.median(load), sm_max_mhz=max(mx), reasons=sorted(reasons),
                       samples=len(sm), power_w_max=max(pw))
        return out


def _oracle_sample(lmax, cfg):
    """Deterministic bounded sample of the workload for the CPU legs: every `stride`-th row, all columns."""
    import numpy as np
    stride = 251 if lmax >= 5000 else max(1, lmax // 40)
    rows = np.arange(stride // 2, lmax + 1, stride, dtype=np.int32)
    N = lmax + 1
    l1 = np.repeat(rows, N)
    l2 = np.tile(np.arange(N, dtype=np.int32), rows.size)
    # terms the oracle evaluates: every l3 of the triangle range (both parities), per pair
    lo = np.abs(l1.astype(np.int64) - l2)
    hi = np.minimum(l1.astype(np.int64) + l2, 2 * lmax)
    terms = int((hi - lo + 1).sum())
    return l1, l2, terms, "cfg%d rows %d::%d (%d rows x %d cols, all blocks)" % (cfg, stride // 2, stride, rows.size, N)


def time_oracle(wl, cfg, reps=1):
    import oracle
    l1, l2, terms, what = _oracle_sample(wl.lmax, cfg)
    oracle.lib()
    best = None
    vals = None
    for _ in range(reps):
        t0 = time.perf_counter()
        vals = oracle.coupling_pairs(wl.l3max, wl.Wtt, wl.Wtp, wl.Wpp, l1, l2)
        dt = time.perf_counter() - t0
        best = dt if best is None else min(best, dt)
    return {"value": terms / best, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
            "sample": what, "sample_terms": terms, "sample_seconds": best}, vals


def _sample_rows(lmax, cfg):
    import numpy as np
    return np.unique(_oracle_sample(lmax, cfg)[0]).astype(np.int64)


def parity_against_oracle(vals, lmax, cfg, dev_rows, host_rows, e2e_equal):
    """SURVEY.md 8(d)(vi) (the paper's own accuracy statement): the oracle values of the cpu_baseline
    sample -- full rows of this workload -- against the same rows of the device-buffer outputs and of the
    tj_coupling_host outputs, at the bar of the parity tests (1e-10 relative where |K| >= 1e-4, 1e-14 absolute below).
    Computed outside every timed region."""
    import numpy as np
    rows = _sample_rows(lmax, cfg)
    N = lmax + 1
    res = {"rows": int(rows.size), "entries_per_block": int(rows.size * N), "blocks": sorted(dev_rows),
           "bar": "rel 1e-10 where |oracle| >= 1e-4, abs 1e-14 below"}
    for name, got in (("device", dev_rows), ("e2e", host_rows)):
        if got is None:
            continue
        mr = ma = 0.0
        ok = True
        for k, g in got.items():
            r = vals[k].reshape(rows.size, N)
            err = np.abs(g - r)
            big = np.abs(r) >= 1e-4
            if big.any():
                mr = max(mr, float((err[big] / np.abs(r[big])).max()))
            if (~big).any():
                ma = max(ma, float(err[~big].max()))
            ok = ok and bool(np.all(err[big] <= 1e-10 * np.abs(r[big])) and np.all(err[~big] <= 1e-14))
        pre = "" if name == "device" else "e2e_"
        res[pre + "max_rel"] = mr
        res[pre + "max_abs_small"] = ma
        res[pre + "within_bar"] = ok
    res["e2e_bitwise_equal_device"] = e2e_equal
    return res


def time_table_method(wl, cfg):
    """The paper's own CPU design (bench_cpu/tablemethod.c: lookup tables, OpenMP dynamic over l1) beside the
    Schulten-Gordon oracle on the same host cores and the same row sample, TT and EE separately -- the paper's
    "6-25x over recursion-based pipelines" re-measured on this box."""
    import numpy as np
    import bench_cpu
    import oracle
    l1, l2, _, what = _oracle_sample(wl.lmax, cfg)
    rows = np.unique(l1).astype(np.int32)
    bench_cpu.lib()
    oracle.lib()

    def best(f, reps):
        b = None
        for _ in range(reps):
            t0 = time.perf_counter()
            f()
            dt = time.perf_counter() - t0
            b = dt if b is None else min(b, dt)
        return b
    t_tm_tt = best(lambda: bench_cpu.coupling_rows(wl.lmax, wl.l3max, wl.Wtt, None, rows), 2)
    t_tm_ee = best(lambda: bench_cpu.coupling_rows(wl.lmax, wl.l3max, None, wl.Wpp, rows), 2)
    t_or_tt = best(lambda: oracle.coupling_pairs(wl.l3max, wl.Wtt, None, None, l1, l2), 1)
    t_or_ee = best(lambda: oracle.coupling_pairs(wl.l3max, None, None, wl.Wpp, l1, l2), 1)
    # even-J terms of the sampled rows (what the table method evaluates per matrix)
    lo = np.abs(l1.astype(np.int64) - l2)
    hi = np.minimum(l1.astype(np.int64) + l2, wl.l3max)
    terms_even = int(np.maximum((hi - lo) // 2 + 1, 0).sum())
    return {"kind": "paper's table method on the host cores (bench_cpu/tablemethod.c)", "cores": bench_cpu.num_threads(),
            "sample": what.replace("all blocks", "TT and EE separately"), "unit": UNIT,
            "tt": {"table_method_s": t_tm_tt, "oracle_s": t_or_tt, "speedup": t_or_tt / t_tm_tt, "value": terms_even / t_tm_tt},
            "ee": {"table_method_s": t_tm_ee, "oracle_s": t_or_ee, "speedup": t_or_ee / t_tm_ee, "value": terms_even / t_tm_ee},
            "paper": "TT 25.3x, EE 6.7x over the S-G reference at lmax = 4722 on 8 Apple-M3 cores (PAPER.md:232-234); "
                     "headline 6-25x (PAPER.md:17)"}


def run_reference(args):
    """--impl reference: the oracle as it stands, on the host cores, on a bounded sample per step."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    from paper_2602_15605_b200 import windows
    wl = windows.config(args.config)
    import oracle
    l1, l2, terms, what = _oracle_sample(wl.lmax, args.config)
    oracle.lib()
    for _ in range(min(args.warmup, 1)):
        oracle.coupling_pairs(wl.l3max, wl.Wtt, wl.Wtp, wl.Wpp, l1[: l1.size // 8], l2[: l2.size // 8])
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle.coupling_pairs(wl.l3max, wl.Wtt, wl.Wtp, wl.Wpp, l1, l2)
    dt = time.perf_counter() - t0
    val = terms * args.steps / dt
    line = {
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": wl.name, "lmax": wl.lmax, "l3max": wl.l3max, "blocks": "TT+TE+EE+BB+EB",
                   "note": "each step = the oracle on a bounded row sample of the workload"},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle", "sample": what},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=3, help="BASELINE.json configs index (headline: 3)")
    ap.add_argument("--nwin", type=int, default=1,
                    help="window sets per step through tj_coupling_multi (default 1: the headline tj_coupling_pol step)")
    ap.add_argument("--tt-only", action="store_true",
                    help="time tj_coupling_tt (K^TT alone, 2 FP64 instructions per term) on the config's W^TT instead of all five blocks")
    ap.add_argument("--split-rows", action="store_true",
                    help="N > 1: cut ONE matrix set into N work-balanced row blocks, one per rank (tj_coupling_rows, no "
                         "exchange; strong scaling) instead of one independent window set per rank (the default, weak)")
    ap.add_argument("--ablation", action="store_true",
                    help="also time tj_coupling_literal (the paper's per-pair Eq. 10 / Eq. 16 evaluation) on the same workload")
    ap.add_argument("--spin1", action="store_true",
                    help="variant line: time tj_coupling_spin1 (K00, K01, K11+, K11-; 6 / 2 FP64 instructions per even / odd term)")
    ap.add_argument("--binned", type=int, default=0, metavar="W",
                    help="variant line: time tj_coupling_binned with bins of W multipoles from l = 2 (W >= lmax: one bin)")
    ap.add_argument("--rows", default="", metavar="R0:R1",
                    help="variant line: time tj_coupling_rows on the full rows R0 <= l1 < R1 (one rank's share of --split-rows)")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-cpu-table-method", action="store_true")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)

    import numpy as np
    import torch
    from paper_2602_15605_b200 import binding, build, shard, windows

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    dist = None
    if world > 1:
        import torch.distributed as dist_
        dist = dist_
        torch.cuda.set_device(local_rank)
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    else:
        torch.cuda.set_device(0)
    if rank == 0:
        build.build()
    if dist is not None:
        dist.barrier()
    binding.load_library()   # fails loudly if the CUDA library is missing: no fallback

    base = windows.config(args.config)
    if args.tt_only and base.pol and not base.band:
        # the paper's own TT benchmark (0.63 s on an A100 at lmax = 10^4): same windows, TT block alone
        base = windows.Workload(base.name + "_tt_only", base.lmax, base.l3max, False, False, base.Wtt, None, None)
    split = bool(args.split_rows) and not base.band and base.pol and args.nwin <= 1
    if world > 1 and not base.band and not split and base.pol:
        # each rank: its own window set of the same recipe (independent problems, weak scaling)
        spec = {1: ((0.7, 30.0, 2.5), (0.5, 50.0, 3.0), False), 2: ((0.6, 40.0, 2.2), (0.45, 60.0, 2.8), True),
                3: ((0.4, 80.0, 2.0), (0.35, 100.0, 2.4), False)}.get(args.config)
        if spec is not None:
            seed = shard.window_seed(args.config, shard.assign_window_sets(world, world, rank)[0])
            tt, tp, pp = windows.pol_windows(base.lmax, spec[0], spec[1], 0.05, seed, ripple=spec[2])
            base = windows.Workload(base.name, base.lmax, base.l3max, False, True, tt, tp, pp)
    wl = base
    N = wl.lmax + 1
    E, O, P = windows.term_counts(wl.lmax, wl.l3max)
    terms = E + O
    blocks = ("TT", "TE", "EE", "BB", "EB") if wl.pol else ("TT",)

    T = binding.build_tables(wl.lmax, None if not wl.band else 2 * wl.lmax)
    dW = [None if w is None else torch.as_tensor(w, dtype=torch.float64).cuda() for w in (wl.Wtt, wl.Wtp, wl.Wpp)]
    width = (2 * wl.l3max + 1) if wl.band else N
    nwin = max(1, args.nwin)
    if nwin > 1:
        # multi-window batching: nwin window sets of the same recipe, scaled copies of the
        # seeded set (the throughput does not depend on the values); one tj_coupling_multi call per step
        assert wl.pol and not wl.band, "--nwin needs a dense polarised config"
        args.no_e2e = True
        dW = [torch.stack([w * (1.0 + 0.01 * k) for k in range(nwin)]).contiguous() for w in dW]
        terms *= nwin
        out = {k: torch.empty((nwin, N, width), dtype=torch.float64, device="cuda") for k in blocks}
    else:
        out = {k: torch.empty((N, width), dtype=torch.float64, device="cuda") for k in blocks}
    # variant lines: other entry points on the same workload, one GPU, so that every number DESIGN.md quotes comes from a
    # bench line (no e2e leg, no oracle leg: their parity lives in tests/)
    variant = "spin1" if args.spin1 else "binned" if args.binned > 0 else "rows" if args.rows else None
    bin_edges = bin_P = bin_Q = None
    if variant:
        assert wl.pol and not wl.band and nwin == 1 and world == 1 and not split, "variant lines need a dense polarised config on one GPU"
        args.no_e2e = True
        args.no_cpu_baseline = True
    if variant == "spin1":
        blocks = ("K00", "K01", "K11p", "K11m")
        out = {k: torch.empty((N, N), dtype=torch.float64, device="cuda") for k in blocks}
    elif variant == "binned":
        bin_edges = list(range(2, wl.lmax + 1, args.binned)) + [wl.lmax + 1]
        lv = np.arange(N, dtype=np.float64)
        bin_P = torch.as_tensor(lv * (lv + 1) / (2 * np.pi) / args.binned).cuda()       # a band-power operator and its inverse
        bin_Q = torch.as_tensor(np.where(lv > 0, 2 * np.pi / np.maximum(lv * (lv + 1), 1.0), 0.0)).cuda()
        out = {k: torch.empty((len(bin_edges) - 1,) * 2, dtype=torch.float64, device="cuda") for k in blocks}
    row_lo, row_hi = 0, N
    if variant == "rows":
        row_lo, row_hi = (int(x) for x in args.rows.split(":"))
        assert 0 <= row_lo < row_hi <= N
        out = {k: torch.empty((row_hi - row_lo, N), dtype=torch.float64, device="cuda") for k in blocks}
    if split:
        # one problem, rank r computes the full rows of block r; the e2e leg is not defined for it
        row_lo, row_hi = shard.row_blocks(wl.lmax, world)[rank]
        args.no_e2e = True
        out = {k: torch.empty((max(row_hi - row_lo, 1), N), dtype=torch.float64, device="cuda") for k in blocks}
    flush = torch.empty(512 * 1024 * 1024 // 8, dtype=torch.float64, device="cuda")

    def step():
        if split or variant == "rows":
            if row_hi > row_lo:
                binding.coupling_rows(T, *dW, row_lo, row_hi, want=blocks, out=out)
        elif variant == "spin1":
            binding.coupling_spin1(T, *dW, want=blocks, out=out)
        elif variant == "binned":
            binding.coupling_binned(T, *dW, bin_edges, bin_P, bin_Q, want=blocks, out=out)
        elif nwin > 1:
            binding.coupling_multi(T, *dW, want=blocks, out=out)
        elif wl.band:
            binding.coupling_band(T, wl.l3max, *dW, want=blocks, out=out)
        elif wl.pol:
            binding.coupling_pol(T, *dW, want=blocks, out=out)
        else:
            binding.coupling_tt(T, dW[0], out["TT"])

    def sync_all():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
            torch.cuda.synchronize()

    n0 = binding.profile_launches()
    step()
    launches_per_step = binding.profile_launches() - n0
    binding.profile_enable(True)
    for _ in range(max(args.warmup, 3)):
        step()
    sync_all()
    geo = binding.profile_last_sweep()
    # A step shorter than ~1 ms is launch-bound: the library's five profiling events per call and the Python side
    # of the call would be a visible part of it.  Such a step is timed WITHOUT the profiling events and as the replay of
    # a CUDA graph that holds ONE call (launch-bound inner loops belong in CUDA graphs); the per-kernel times then come
    # from a separate profiled pass of the same steps, by direct calls, right after the timed region.
    ws, we = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ws.record(); step(); we.record(); torch.cuda.synchronize()
    est_ms = ws.elapsed_time(we)
    profile_in_region = est_ms >= 1.0
    use_graph = est_ms < 1.0 and dist is None
    binding.profile_enable(profile_in_region)
    graph = None
    run = step
    if use_graph:
        gs = torch.cuda.Stream()
        gs.wait_stream(torch.cuda.current_stream())
        with torch.cuda.stream(gs):
            step()
            graph = torch.cuda.CUDAGraph()
            with torch.cuda.graph(graph, stream=gs):
                step()
        torch.cuda.current_stream().wait_stream(gs)
        run = graph.replay
        for _ in range(3):
            run()
        sync_all()

    sampler = ClockSampler(local_rank)
    sampler.start()
    time.sleep(0.3)
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    kern = []
    sync_all()
    t_wall0 = time.perf_counter()
    for i in range(args.steps):
        flush.fill_(float(i))            # L2 flush between timed iterations (outside the event pair)
        ev[i][0].record()
        run()
        ev[i][1].record()
        if profile_in_region:
            kern.append(binding.profile_get())   # waits for this step's kernels (per-kernel device times)
    sync_all()
    t_wall = time.perf_counter() - t_wall0
    clocks = sampler.stop()
    step_ms = [a.elapsed_time(b) for a, b in ev]
    if not profile_in_region:
        binding.profile_enable(True)
        for i in range(args.steps):
            flush.fill_(float(i))
            step()
            kern.append(binding.profile_get())
        sync_all()
    direct_ms = None
    if use_graph:
        # the same steps as DIRECT calls of the C ABI (profiling events off): what a caller that does not capture the
        # call pays per step, host side of the three launches and the stream-ordered alloc/free included
        binding.profile_enable(False)
        evd = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
        for i in range(args.steps):
            flush.fill_(float(i))
            evd[i][0].record()
            step()
            evd[i][1].record()
        sync_all()
        direct_ms = float(sum(a.elapsed_time(b) for a, b in evd)) / args.steps
        binding.profile_enable(True)
    total_ms = float(sum(step_ms))
    total_ms = shard.max_over_ranks(total_ms, dist, "cuda")
    # rows of the device-buffer outputs that the oracle leg computes (parity in the bench line, outside the timed region)
    check_rows = rank == 0 and world == 1 and nwin == 1 and not split and not wl.band and not args.no_cpu_baseline
    dev_rows = host_rows = e2e_equal = None
    if check_rows:
        ridx = torch.as_tensor(_sample_rows(wl.lmax, args.config)).cuda()
        dev_rows = {k: out[k][ridx].cpu().numpy() for k in blocks}
    # split rows: the job is ONE matrix set (its terms counted once); else every rank does `terms`
    value = shard.whole_job_throughput(terms, args.steps, total_ms, 1 if split else world)

    # ---- roofline of the dominant kernel (the sweep), timed live with the library's CUDA events ----
    sweep_ms = statistics.mean(k[1] for k in kern)
    prep_ms = statistics.mean(k[0] for k in kern)
    writer_ms = statistics.mean(k[2] for k in kern)
    if (split and world > 1) or variant == "rows":
        # rank 0's launch sweeps its own upper-triangle rows plus the pairs (l1 < row_lo, l2 in the block)
        nb = row_hi - row_lo
        Eb = sum((l + 1) * (N - l) for l in range(row_lo, row_hi)) + nb * (row_lo * (row_lo + 1) // 2)
        Ob = sum(l * (N - l) for l in range(row_lo, row_hi)) + nb * (row_lo * (row_lo - 1) // 2)
        alg_instr = INSTR_EVEN_POL * Eb + INSTR_ODD * Ob
        alg_flops = 12 * Eb + 6 * Ob
        if variant == "rows":
            terms = Eb + Ob
            value = shard.whole_job_throughput(terms, args.steps, total_ms, 1)
    elif variant == "spin1":
        alg_instr = 6 * E + 2 * O          # DESIGN.md 3 item 6: K00 2 + K01 2 + K11+ 2 per even term, K11- 2 per odd term
        alg_flops = 9 * E + 3 * O
    elif wl.pol:
        alg_instr = INSTR_EVEN_POL * E + INSTR_ODD * O
        alg_flops = 12 * E + 6 * O
    else:
        alg_instr = INSTR_EVEN_TT * E
        alg_flops = 3 * E
    unbatched_equiv = None
    if nwin > 1:
        # the per-kernel events cover the LAST sweep of the call (the library's grouping: threes, a remainder of 4 as
        # 2 + 2, of 2 as one pair).  A batched sweep forms the window-independent part of a term once:
        # 5 + 3 nw instructions per even term and 4 + nw per odd term for nw window sets; that is the algorithmic work of
        # the launch.  The work the UNBATCHED method would need for the same matrices ((8E+5O) per window set) is
        # reported beside it as `unbatched_equivalent_frac` (it may exceed 1: that is the point of batching).
        left = nwin
        while left > 0:
            last = 2 if left in (2, 4) else 3 if left >= 3 else 1
            left -= last
        unbatched_equiv = alg_instr * last
        alg_instr = (5 + 3 * last) * E + (4 + last) * O
        alg_flops = (6 + 6 * last) * E + (4 + 2 * last) * O
    peaks, peak_kind = _peaks()
    traffic, traffic_src = _traffic(wl.name if nwin == 1 and not split and not variant else None, geo)
    sm_max = float(clocks.get("sm_max_mhz") or peaks.get("sm_max_mhz", 1965.0))
    peak_instr = SM_COUNT * FP64_LANES_PER_SM * sm_max * 1e6          # thread-instr/s at max boost
    achieved = alg_instr / (sweep_ms * 1e-3)
    # measured DFMA rate (bench_gpu/fp64_probe.cu, bench-only): a register-resident chain kernel on every SM for >= 1 s, clocks sampled
    it = 2000000
    import bench_gpu
    rate = bench_gpu.fp64_probe(it)
    it = int(min(2.0e9, 1.15 * it * rate / (16.0 * it * SM_COUNT * 4 * 256)))   # iterations for ~1.15 s at that rate
    psampler = ClockSampler(local_rank)
    psampler.start()
    time.sleep(0.2)
    tp0 = time.perf_counter()
    probe = bench_gpu.fp64_probe(it)
    probe_s = time.perf_counter() - tp0
    probe_clocks = psampler.stop()
    bytes_out = len(blocks) * N * width * 8
    nmirror = len(blocks) - (1 if "BB" in blocks else 0)
    writer_bytes = int(nmirror * 1.5 * N * width * 8 + (N * width * 8 if "BB" in blocks else 0))
    roofline = {
        # the instantiation the library really launched (tj_profile_last_sweep), not a label typed here
        "bound": "alu", "kernel": geo["name"] + (" (last group of the call)" if nwin > 1 else "")
                                  + (" -- all row chunks of the call, bin kernels included in the time" if variant == "binned" else ""),
        "achieved": achieved / 1e12, "peak": peak_instr / 1e12, "unit": "T FP64 thread-instr/s",
        "frac": achieved / peak_instr,
        # dram__bytes_read.sum + dram__bytes_write.sum of one launch of this kernel, from the committed ncu --set full
        # summaries (profiles/traffic.csv names the capture each row comes from); None if this workload has no capture
        "traffic": traffic, "traffic_source": traffic_src,
        "peak_source": "derived: %d SMs x %d FP64 lanes/clk x %.0f MHz (DESIGN.md 6; MEASURED_PEAKS.json has no FP64 entry)"
                       % (SM_COUNT, FP64_LANES_PER_SM, sm_max),
        "algorithmic_instr_per_launch": alg_instr, "algorithmic_flops_per_launch": alg_flops,
        "achieved_tflops": alg_flops / (sweep_ms * 1e-3) / 1e12,
        "unbatched_equivalent_frac": None if unbatched_equiv is None else unbatched_equiv / (sweep_ms * 1e-3) / peak_instr,
        "measured_dfma_peak": probe / 1e12, "frac_of_measured_dfma": achieved / probe,
        "dfma_probe": {"seconds": probe_s, "iterations": it, "sm_mhz": probe_clocks.get("sm_mhz"),
                       "reasons": probe_clocks.get("reasons"), "power_w_max": probe_clocks.get("power_w_max")},
        "kernel_ms": {"prepare": prep_ms, "sweep": sweep_ms, "writer": writer_ms},
        "kernel_ms_source": "library CUDA events inside the timed region" if profile_in_region
                            else "library CUDA events in a separate profiled pass of the same steps after the timed region",
        "sweep_share_of_step": sweep_ms / (total_ms / args.steps) if world == 1 else None,
        # writer: per mirrored block reads the upper triangle (N^2/2) and writes N^2; BB is one more N^2 write
        "writer": None if (variant in ("rows", "binned") or split or writer_ms <= 0.0) else
                  {"bound": "hbm", "achieved": writer_bytes / (writer_ms * 1e-3) / 1e9, "peak": peaks.get("hbm_gbs"),
                   "unit": "GB/s", "frac": writer_bytes / (writer_ms * 1e-3) / 1e9 / peaks.get("hbm_gbs"),
                   "peak_kind": peak_kind, "algorithmic_bytes": writer_bytes},
    }

    # ---- end to end through the C ABI with HOST buffers (H2D + D2H inside the timed region) ----
    e2e = None
    if not args.no_e2e:
        hW = [None if w is None else torch.as_tensor(w, dtype=torch.float64).pin_memory() for w in (wl.Wtt, wl.Wtp, wl.Wpp)]
        hout = {k: torch.full((N, width), float("nan"), dtype=torch.float64).pin_memory() for k in blocks}
        lc = wl.l3max if wl.band else None
        binding.coupling_host(T, *hW, hout, band_lcut=lc)      # warm-up (pool growth, page faults)
        sync_all()
        n_e2e = max(1, args.steps)
        t0 = time.perf_counter()
        for _ in range(n_e2e):
            binding.coupling_host(T, *hW, hout, band_lcut=lc)  # synchronises internally
        torch.cuda.synchronize()
        dt = time.perf_counter() - t0
        dt = shard.max_over_ranks(dt, dist, "cuda")
        e2e = {"value": world * terms * n_e2e / dt, "unit": UNIT,
               "h2d_bytes_per_step": int(sum(w.numel() * 8 for w in hW if w is not None)),
               "d2h_bytes_per_step": int(sum(v.numel() * 8 for v in hout.values())),
               "ms_per_step": 1e3 * dt / n_e2e, "steps": n_e2e, "api": "tj_coupling_host (pinned host buffers)"}
        if nwin == 1 and not split:
            # every entry the host-buffer call delivered (buffers were pre-filled with NaN) against the device-buffer
            # call's matrices of the last timed step: must be the same bits
            e2e_equal = all(bool(torch.equal(hout[k].cuda(), out[k])) for k in blocks)
            e2e["bitwise_equal_device_path"] = e2e_equal
        if check_rows:
            hidx = torch.as_tensor(_sample_rows(wl.lmax, args.config))
            host_rows = {k: hout[k][hidx].numpy().copy() for k in blocks}
        del hout
    del out

    ablation = None
    if args.ablation and wl.pol and not wl.band and nwin == 1:
        # the paper's own design on this GPU (tj_literal.cu): one thread per pair, Eq. 10 (TT) / Eq. 16 literally (EE)
        ablation = {"kernel": "literal_kernel (one thread per (l1,l2), PAPER.md:240; Eq. 10 / Eq. 16)", "unit": "ms"}
        for name, a in (("TT", (dW[0], None, ("TT",))), ("EE", (None, dW[2], ("EE",)))):
            binding.coupling_literal(T, a[0], a[1], want=a[2])
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            binding.coupling_literal(T, a[0], a[1], want=a[2])
            e1.record()
            torch.cuda.synchronize()
            ablation[name] = e0.elapsed_time(e1)
        ablation["note"] = "fused sweep of this line: all five blocks in %.1f ms" % sweep_ms

    cpu_baseline = None
    parity = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline and not wl.band:
        cpu_baseline, oracle_vals = time_oracle(wl, args.config)
        if check_rows:
            parity = parity_against_oracle(oracle_vals, wl.lmax, args.config, dev_rows, host_rows, e2e_equal)
    cpu_table_method = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline and not args.no_cpu_table_method and not wl.band and wl.pol:
        cpu_table_method = time_table_method(wl, args.config)

    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": total_ms / args.steps, "higher_is_better": True,
            "scaling": "strong" if split else "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": wl.name, "variant": variant, "bins": None if bin_edges is None else len(bin_edges) - 1, "lmax": wl.lmax, "l3max": wl.l3max, "blocks": "+".join(blocks), "window_sets_per_step": nwin,
                       "terms_even": E, "terms_odd": O, "pairs_upper": P,
                       "pairs_per_s": (1 if split else world) * P * args.steps / (total_ms * 1e-3),
                       "l2": "512 MB flush written between timed steps; each step also writes %.1f GB of output" % (bytes_out / 1e9),
                       "parallelism": ("one matrix set cut into %d row blocks (tj_coupling_rows), rank 0 rows [%d,%d)" % (world, row_lo, row_hi))
                       if split else ("1 problem per GPU" if world > 1 else "single GPU")},
            "roofline": roofline, "cpu_baseline": cpu_baseline, "cpu_table_method": cpu_table_method, "e2e": e2e,
            "parity": parity,
            "ablation": ablation,
            # kernels of libtj launched inside the timed region, counted by the library (tj_profile_launches)
            "gpu_launches": launches_per_step * args.steps, "gpu_launches_per_step": launches_per_step,
            "launch": "replay of a CUDA graph holding one call" if use_graph else "direct calls",
            # launch-bound steps: `value` / `ms_per_step` are graph replays; the same steps as direct C-ABI calls beside them
            "ms_per_step_direct_calls": direct_ms if use_graph else total_ms / args.steps,
            "value_direct_calls": (terms / (direct_ms * 1e-3)) if use_graph else value,
            "clocks": clocks, "wall_s_timed_region": t_wall, "step_ms": step_ms,
            "context": {"paper_A100_TT_lmax1e4_s": 0.63, "paper_A100_EE_lmax1e4_s": 3.2,
                        "note": "paper numbers (PAPER.md:242) are another machine's: context, not the target"},
        }
        print(json.dumps(line))
    T.close()
    if dist is not None:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
