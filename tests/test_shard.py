"""Walker sharding: partition arithmetic, and the gather of per-walker energies over
two gloo ranks on CPU -- the only exchange of the multi-GPU path (bench.py --gpus N shards walkers the same way)."""
import os
import socket

import numpy as np
import pytest

from paper_2507_02888_b200 import shard


@pytest.mark.parametrize("n,world", [(0, 1), (1, 2), (7, 2), (1024, 8), (4096, 3), (5, 8)])
def test_walker_ranges_partition(n, world):
    seen = []
    for r in range(world):
        lo, hi = shard.walker_range(n, r, world)
        assert 0 <= lo <= hi <= n
        seen += list(range(lo, hi))
        assert hi - lo in (n // world, n // world + 1)
    assert seen == list(range(n))
    for wk in range(0, n, max(1, n // 13)):
        r, loc = shard.owner_of(wk, n, world)
        assert shard.walker_range(n, r, world)[0] + loc == wk


def test_bad_arguments():
    with pytest.raises(ValueError):
        shard.walker_range(10, 2, 2)
    with pytest.raises(IndexError):
        shard.owner_of(10, 10, 2)


def _worker(rank, world, port, n, q):
    import torch
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    lo, hi = shard.walker_range(n, rank, world)
    local = torch.arange(lo, hi, dtype=torch.float64) * 0.5 - 3.0   # stands for this rank's energies
    got = shard.gather_energies(local, n)
    q.put((rank, got))
    dist.destroy_process_group()


def test_gather_energies_two_gloo_ranks():
    import torch.multiprocessing as mp
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    n, world = 11, 2   # ragged: 6 + 5 walkers
    procs = [ctx.Process(target=_worker, args=(r, world, port, n, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = dict(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    want = np.arange(n) * 0.5 - 3.0
    for r in range(world):
        assert np.array_equal(res[r], want)
