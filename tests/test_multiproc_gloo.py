"""World-size-2 CPU test (gloo) of the N > 1 host logic: window-set sharding covers every set exactly
once with no overlap, the timing reduction is a max over ranks, and the whole-job throughput formula
uses it.  No GPU, no kernels: the data path has no collective to test."""
import os
import socket
import sys

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, n_sets, q):
    sys.path.insert(0, ROOT)
    from paper_2602_15605_b200 import shard, windows
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    mine = shard.assign_window_sets(n_sets, world, rank)
    # every rank draws its own window set of the config-1 recipe
    seeds = [shard.window_seed(1, k) for k in mine]
    sums = [float(windows.pol_windows(20, (0.7, 30.0, 2.5), (0.5, 50.0, 3.0), 0.05, sd)[0].sum()) for sd in seeds]
    gathered = [None] * world
    dist.all_gather_object(gathered, (mine, sums))
    fake_ms = 10.0 + 5.0 * rank
    mx = shard.max_over_ranks(fake_ms, dist)
    dist.barrier()
    q.put((rank, gathered, mx, shard.whole_job_throughput(1000.0, 4, mx, world)))
    dist.destroy_process_group()


def test_window_set_sharding_and_timing_reduction_world2():
    world, n_sets = 2, 5
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, n_sets, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = [q.get(timeout=120) for _ in range(world)]
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, gathered, mx, thr in res:
        allsets = sorted(k for mine, _ in gathered for k in mine)
        assert allsets == list(range(n_sets))                      # exact cover, no overlap
        assert mx == 15.0                                          # max over ranks
        assert thr == pytest.approx(2 * 1000.0 * 4 / 15e-3)
        # different sets -> different windows (distinct seeds)
        flat = [s for _, sums in gathered for s in sums]
        assert len(set(flat)) == n_sets


def _rows_worker(rank, world, port, lmax, q):
    sys.path.insert(0, ROOT)
    from paper_2602_15605_b200 import shard
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    N = lmax + 1
    lo, hi = shard.row_blocks(lmax, world)[rank]
    # entries this rank stores (tj_coupling_rows: full rows [lo, hi)), and the upper-triangle pairs it must sweep for
    # them: (l1, l2 >= l1) with l1 in the block (direct) or l2 in the block (mirrored into row l2)
    stored = torch.zeros((N, N), dtype=torch.int32)
    stored[lo:hi, :] = 1
    l1 = torch.arange(N)[:, None]
    l2 = torch.arange(N)[None, :]
    swept = ((l2 >= l1) & (((l1 >= lo) & (l1 < hi)) | ((l2 >= lo) & (l2 < hi)))).to(torch.int32)
    tot_stored, tot_swept = stored.clone(), swept.clone()
    dist.all_reduce(tot_stored)
    dist.all_reduce(tot_swept)
    work = torch.tensor([float(((torch.minimum(l1, l2) + 1) * swept).sum())], dtype=torch.float64)
    works = [torch.zeros(1, dtype=torch.float64) for _ in range(world)]
    dist.all_gather(works, work)
    q.put((rank, (lo, hi), tot_stored, tot_swept, [float(w) for w in works]))
    dist.destroy_process_group()


def test_split_rows_blocks_tile_the_matrix_world2():
    """bench.py --split-rows: the row blocks of the two ranks store every (l1,l2) exactly once; every upper-triangle
    pair is swept by the owner(s) of its two rows (once on the diagonal blocks, twice across blocks); the sweep work
    of the ranks is balanced."""
    world, lmax = 2, 61
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_rows_worker, args=(r, world, port, lmax, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = [q.get(timeout=120) for _ in range(world)]
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    N = lmax + 1
    blocks = sorted(r[1] for r in res)
    assert blocks[0][0] == 0 and blocks[-1][1] == N and blocks[0][1] == blocks[1][0]
    cut = blocks[0][1]
    for rank, _, tot_stored, tot_swept, works in res:
        assert bool((tot_stored == 1).all())                                   # each entry stored by exactly one rank
        l1 = torch.arange(N)[:, None]
        l2 = torch.arange(N)[None, :]
        upper = l2 >= l1
        cross = upper & (l1 < cut) & (l2 >= cut)                               # rows owned by different ranks
        assert bool((tot_swept[upper & ~cross] == 1).all()) and bool((tot_swept[cross] == 2).all())
        assert bool((tot_swept[~upper] == 0).all())
        assert max(works) <= 1.15 * min(works)                                 # balanced (small N: coarse rows)


def test_assign_window_sets_edge_cases():
    from paper_2602_15605_b200 import shard
    assert shard.assign_window_sets(0, 4, 1) == []
    assert shard.assign_window_sets(3, 8, 5) == []
    assert shard.assign_window_sets(3, 8, 2) == [2]
    assert sorted(sum((shard.assign_window_sets(17, 4, r) for r in range(4)), [])) == list(range(17))
    with pytest.raises(ValueError):
        shard.assign_window_sets(3, 2, 2)
    assert shard.max_over_ranks(3.5, None) == 3.5


def test_row_blocks_partition_is_a_balanced_cover():
    from paper_2602_15605_b200 import shard
    for lmax, world in [(0, 1), (2, 5), (100, 3), (2000, 4), (10000, 8)]:
        N = lmax + 1
        cuts = shard.row_blocks(lmax, world)
        assert len(cuts) == world and cuts[0][0] == 0 and cuts[-1][1] == N
        assert all(a[1] == b[0] and a[0] <= a[1] for a, b in zip(cuts, cuts[1:]))
        cost = [(r + 1) * (N - r) + r * (r + 1) // 2 for r in range(N)]
        loads = [sum(cost[a:b]) for a, b in cuts]
        assert sum(loads) == sum(cost)
        if N >= 50 * world:
            assert max(loads) <= 1.02 * sum(cost) / world + max(cost)
    with pytest.raises(ValueError):
        shard.row_blocks(10, 0)


# ---------------------------------------------------------------- one matrix on several GPUs, every pair swept once (tj_chunk_plan)
def _region_mask(N, r0, r1):
    """The L-shaped region chunk [r0, r1) makes final (include/tj.h): its rows from column r0 on, and columns [r0, r1)
    of all rows below."""
    m = torch.zeros((N, N), dtype=torch.int32)
    m[r0:r1, r0:] = 1
    m[r1:, r0:r1] = 1
    return m


def _chunks_worker(rank, world, port, lmax, q):
    sys.path.insert(0, ROOT)
    from paper_2602_15605_b200 import binding, build
    build.build()
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    bounds, owner = binding.chunk_plan(lmax, world)          # host-side entry point of libtj: no GPU involved
    N = lmax + 1
    stored = torch.zeros((N, N), dtype=torch.int32)
    swept = torch.zeros((N, N), dtype=torch.int32)
    l1 = torch.arange(N)[:, None]
    l2 = torch.arange(N)[None, :]
    work = 0
    for k, g in enumerate(owner):
        if g != rank:
            continue
        r0, r1 = bounds[k], bounds[k + 1]
        stored += _region_mask(N, r0, r1)
        swept += ((l1 >= r0) & (l1 < r1) & (l2 >= l1)).to(torch.int32)   # the chunk's sweep: its rows of the upper triangle
        work += sum((a + 1) * (N - a) for a in range(r0, r1))
    tot_stored, tot_swept = stored.clone(), swept.clone()
    dist.all_reduce(tot_stored)
    dist.all_reduce(tot_swept)
    works = [None] * world
    dist.all_gather_object(works, work)
    q.put((rank, tot_stored, tot_swept, works, (bounds, owner)))
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("lmax", [700, 2700])
def test_chunk_ownership_stores_every_entry_once_and_sweeps_every_pair_once_world2(lmax):
    world = 2
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_chunks_worker, args=(r, world, port, lmax, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = [q.get(timeout=180) for _ in range(world)]
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    N = lmax + 1
    assert res[0][4] == res[1][4]                                              # both ranks derive the same plan
    for rank, tot_stored, tot_swept, works, _ in res:
        assert bool((tot_stored == 1).all())                                   # every (l1,l2) delivered by exactly one rank
        upper = torch.arange(N)[None, :] >= torch.arange(N)[:, None]
        assert bool((tot_swept[upper] == 1).all()) and bool((tot_swept[~upper] == 0).all())   # no pair swept twice
        assert max(works) <= 1.05 * min(works)


def test_chunk_plan_is_a_balanced_cover_for_any_device_count():
    from paper_2602_15605_b200 import binding, build
    build.build()
    for lmax, tt in [(0, False), (31, False), (800, False), (2599, False), (2600, False), (5000, True), (10000, False)]:
        N = lmax + 1
        unit = 96 if (lmax >= 2600 and not tt) else 32
        for G in (1, 2, 3, 4, 8, 64):
            bounds, owner = binding.chunk_plan(lmax, G, tt_only=tt)
            assert bounds[0] == 0 and bounds[-1] == N and all(a < b for a, b in zip(bounds, bounds[1:]))
            assert all(b % unit == 0 for b in bounds[:-1])                   # whole row bands and whole writer tile rows
            assert len(owner) == len(bounds) - 1 <= 12 * G and all(0 <= g < G for g in owner)
            per = [sum(1 for g in owner if g == d) for d in range(G)]
            assert max(per) <= 24
            load = [0] * G
            for k, g in enumerate(owner):
                load[g] += sum((a + 1) * (N - a) for a in range(bounds[k], bounds[k + 1]))
            if lmax == 10000 and G <= 8:
                assert max(load) <= 1.01 * sum(load) / G                     # config 3: within 1 % on 8 GPUs
    with pytest.raises(binding.TJError):
        binding.chunk_plan(100, 0)
    with pytest.raises(binding.TJError):
        binding.chunk_plan(100, 65)
