"""Multi-GPU plumbing: the path has no exchange step (every (l1,l2) entry and every window set is
independent), so N GPUs run N independent problems -- one process per GPU, window
sets dealt round-robin, no data-path collective.  The only communication is the timing reduction
(max over ranks) and a barrier, done with torch.distributed (NCCL on GPUs, gloo in the CPU tests).

Nothing here touches the arithmetic of the method.
"""
from __future__ import annotations


def assign_window_sets(n_sets: int, world: int, rank: int) -> list[int]:
    """Indices of the window sets rank `rank` of `world` computes (round-robin deal)."""
    if world <= 0 or not (0 <= rank < world) or n_sets < 0:
        raise ValueError("bad (n_sets, world, rank) = (%r, %r, %r)" % (n_sets, world, rank))
    return list(range(rank, n_sets, world))


def window_seed(config_seed: int, set_index: int) -> int:
    """Seed of window set `set_index` of a config (set 0 is the BASELINE.json seed itself)."""
    return int(config_seed) + int(set_index)


def max_over_ranks(value: float, dist=None, device=None) -> float:
    """MAX all-reduce of a scalar (the device-timed duration) -- identity when not distributed."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(value)
    import torch
    t = torch.tensor([float(value)], dtype=torch.float64, device=device or "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_throughput(units_per_rank: float, steps: int, ms_max: float, world: int) -> float:
    """units all ranks processed / the slowest rank's time (weak scaling, same work per rank)."""
    return world * units_per_rank * steps / (ms_max * 1e-3)


def row_blocks(lmax: int, world: int) -> list[tuple[int, int]]:
    """Cut the rows 0..lmax of ONE matrix into `world` contiguous blocks of (nearly) equal sweep work for
    tj_coupling_rows (each GPU owns a row block, no exchange).  Work of row r = the pairs the
    block sweeps for it: its upper-triangle part, (r+1) steps for each of the N-r columns l2 >= r, plus the mirrored
    part, l+1 steps for each l < r.  Returns [(row_lo, row_hi), ...] covering 0..lmax+1; blocks may be empty
    (row_lo == row_hi) only when world > lmax+1."""
    if lmax < 0 or world <= 0:
        raise ValueError("bad (lmax, world) = (%r, %r)" % (lmax, world))
    N = lmax + 1
    cost = [(r + 1) * (N - r) + r * (r + 1) // 2 for r in range(N)]
    total = sum(cost)
    cuts, acc, r = [0], 0, 0
    for k in range(1, world):
        target = total * k // world
        while r < N and acc + cost[r] <= target:
            acc += cost[r]
            r += 1
        cuts.append(r)
    cuts.append(N)
    return [(cuts[k], cuts[k + 1]) for k in range(world)]
