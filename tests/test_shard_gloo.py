"""World-size-2 gloo tests (CPU) of the N>1 host logic: orbit/trial sharding and the max-over-ranks timing rule.
There is no data-path collective on this path; these are the only distributed pieces."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2607_00117_b200 import inputs, shard


def test_split_range_partitions_exactly():
    for n in (0, 1, 7, 20000, 100003):
        for world in (1, 2, 3, 8):
            r = [shard.split_range(n, world, k) for k in range(world)]
            assert r[0][0] == 0 and r[-1][1] == n
            assert all(r[k][1] == r[k + 1][0] for k in range(world - 1))
            sizes = [b - a for a, b in r]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        shard.split_range(10, 2, 2)


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        n = 20001
        ranges = shard.gather_ranges(n)
        # each rank generates ONLY its shard of the seeded config-0 ICs; gathered, they must equal the unsharded set
        full = inputs.plummer_ics(257, 5)
        a, b = shard.orbit_range(257, world, rank)
        mine = torch.as_tensor(full[a:b].copy())
        sizes = [r[1] - r[0] for r in shard.gather_ranges(257)]
        pad = max(sizes)  # ragged shards (129 + 128): gather through padded buffers
        buf = torch.zeros((pad, 6), dtype=torch.float64)
        buf[:b - a] = mine
        outs = [torch.empty_like(buf) for _ in range(world)]
        dist.all_gather(outs, buf)
        parts = [o[:s] for o, s in zip(outs, sizes)]
        whole = torch.cat(parts).numpy()
        t = shard.max_over_ranks(10.0 + rank)
        q.put((rank, ranges, bool(np.array_equal(whole, full)), t, shard.rank_seed(1, rank), shard.trial_range(64, world, rank)))
    finally:
        dist.destroy_process_group()


def test_world_size_2_gloo():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, ranges, same, t, seed, tr in res:
        assert ranges == [(0, 10001), (10001, 20001)]
        assert same
        assert t == 11.0                      # max over ranks, seen by every rank
        assert seed == 1 + 1000 * rank
    assert [r[5] for r in res] == [(0, 32), (32, 64)]
