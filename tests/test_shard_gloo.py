"""World-size-2 gloo test of the multi-rank host logic: the seed partition is disjoint and covering,
per-seed outputs concatenate back to caller order, and the bench reductions are max-of-time / sum-of-units."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1609_00724_b200.shard import gather_concat, reduce_job, shard_range


@pytest.mark.parametrize("n,world", [(0, 2), (1, 2), (7, 2), (8, 2), (1047959, 8), (5, 8)])
def test_shard_range_partitions(n, world):
    r = [shard_range(n, k, world) for k in range(world)]
    assert r[0][0] == 0 and r[-1][1] == n
    assert all(a[1] == b[0] for a, b in zip(r, r[1:]))
    sizes = [b - a for a, b in r]
    assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        shard_range(n, world, world)


def _worker(rank, world, port, n, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        lo, hi = shard_range(n, rank, world)
        full = torch.arange(n * 3, dtype=torch.float64).reshape(n, 3)     # stands for a per-seed output in caller order
        got = gather_concat(full[lo:hi] * 2.0, n)
        ms, units = reduce_job(10.0 + rank, float(hi - lo))
        q.put((rank, bool(torch.equal(got, full * 2.0)), ms, units))
    finally:
        dist.destroy_process_group()


def test_two_ranks_gather_and_reduce():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    n, world = 1001, 2
    procs = [ctx.Process(target=_worker, args=(r, world, port, n, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, same, ms, units in res:
        assert same
        assert ms == 11.0 and units == float(n)
