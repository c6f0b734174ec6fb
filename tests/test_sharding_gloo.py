"""The N > 1 plumbing on CPU: world_size-2 gloo processes shard the mode axis, each computes its own
columns (here with a stand-in compute so that no GPU is needed), and the gathered matrix and the
max-over-ranks timing are checked."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2606_07759_b200 import sharding


def test_partition_is_contiguous_balanced_and_complete():
    for n, w in [(0, 3), (5, 8), (5065, 8), (2000, 3), (97, 2), (1, 1)]:
        r = sharding.partition_modes(n, w)
        assert len(r) == w and r[0][0] == 0 and r[-1][1] == n
        assert all(r[k][1] == r[k + 1][0] for k in range(w - 1))
        sizes = [e - b for b, e in r]
        assert max(sizes) - min(sizes) <= 1 and sizes == sorted(sizes, reverse=True)
    with pytest.raises(ValueError):
        sharding.partition_modes(4, 0)
    assert sharding.weak_scaling_plan(30390, 8)["total_units"] == 243120


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, n_modes, rows, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        def compute(b, e):                       # column m of the stand-in matrix is m + r/1000
            m = torch.arange(b, e, dtype=torch.float32)[:, None]
            return m + torch.arange(rows, dtype=torch.float32)[None, :] / 1000.0
        block, (b, e) = sharding.sharded_columns(n_modes, compute, gather=False)
        full, _ = sharding.sharded_columns(n_modes, compute, gather=True)
        slow = sharding.max_over_ranks(1.0 + rank)
        q.put((rank, b, e, block.numpy(), full.numpy(), slow))
    finally:
        dist.destroy_process_group()


@pytest.mark.timeout(120)
def test_two_rank_gloo_sharding_and_gather():
    world, n_modes, rows = 2, 7, 5
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, n_modes, rows, q)) for r in range(world)]
    for p in procs:
        p.start()
    got = [q.get(timeout=90) for _ in range(world)]
    for p in procs:
        p.join(30)
        assert p.exitcode == 0
    expect = np.arange(n_modes, dtype=np.float32)[:, None] + np.arange(rows, dtype=np.float32)[None, :] / 1000.0
    ranges = sharding.partition_modes(n_modes, world)
    for rank, b, e, block, full, slow in got:
        assert (b, e) == ranges[rank]
        assert np.array_equal(block, expect[b:e])
        assert np.array_equal(full, expect)
        assert slow == 2.0
