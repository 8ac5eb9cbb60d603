"""Orbit / trial sharding across ranks (one process per GPU) -- host arithmetic only.

Orbits are independent ("the orbit integration can be perfectly parallelised"), matrix rows partition by
orbit range and the batched mode partitions by trial, so there is NO data-path collective on this path:
every rank calls sm_build_library on its own contiguous range (pointer offsets in the C ABI) and owns those rows.
torch.distributed is used only for the barrier and the max-over-ranks timing of bench.py.
"""


def split_range(n, world, rank):
    """Contiguous near-equal partition of range(n): -> (start, stop).  The first n % world ranks get one extra."""
    if world < 1 or not (0 <= rank < world) or n < 0:
        raise ValueError("bad shard arguments")
    base, extra = divmod(n, world)
    start = rank * base + min(rank, extra)
    return start, start + base + (1 if rank < extra else 0)


def orbit_range(n_orb, world, rank):
    """Strong-scaling shard of one library: this rank's rows [start, stop)."""
    return split_range(n_orb, world, rank)


def trial_range(n_trials, world, rank):
    """Batched-potential mode: this rank's trials [start, stop)."""
    return split_range(n_trials, world, rank)


def rank_seed(seed, rank):
    """Weak scaling (bench.py): every rank builds its own library of the full per-GPU size from its own seed."""
    return seed + 1000 * rank


def max_over_ranks(value, device=None):
    """Max of a host float over all ranks (the timing rule of bench.py); identity without a process group."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device or "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def gather_ranges(n, device=None):
    """All ranks' (start, stop) of split_range(n, world, rank), gathered -- used by callers that assemble a row index."""
    import torch
    import torch.distributed as dist
    world, rank = dist.get_world_size(), dist.get_rank()
    mine = torch.tensor(split_range(n, world, rank), dtype=torch.int64, device=device or "cpu")
    out = [torch.empty_like(mine) for _ in range(world)]
    dist.all_gather(out, mine)
    return [tuple(int(v) for v in t.tolist()) for t in out]
