"""World-size-2 `gloo` test (CPU) of the multi-GPU plumbing: contiguous event shards, K
partial NLLs combined in rank order, max-over-ranks timing.  The local evaluator here is the oracle (this
is a test); on GPUs it is ipa_nll_eval on the rank's shard."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import ipa_inputs as inp
from paper_1706_01420_b200 import sharding

LO, HI = inp.LO, inp.HI


def test_shard_range_partitions_exactly():
    for n in (0, 1, 7, 10, 1000003):
        for world in (1, 2, 3, 8):
            edges = [sharding.shard_range(n, r, world) for r in range(world)]
            assert edges[0][0] == 0 and edges[-1][1] == n
            assert all(edges[r][1] == edges[r + 1][0] for r in range(world - 1))
            sizes = [b - a for a, b in edges]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        sharding.shard_range(10, 2, 2)
    off = np.array([0, 5, 5, 9, 20, 31])
    assert sharding.shard_segments(off, 0, 2) == (0, 3, 0, 9)
    assert sharding.shard_segments(off, 1, 2) == (3, 5, 9, 31)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, n, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        import oracle
        x = oracle.generate_mixture(2, n, inp.GEN, LO, HI)          # every rank regenerates the same seeded input
        batch, _ = inp.fd_batch(inp.GEN)
        a, b = sharding.shard_range(n, rank, world)
        local = torch.from_numpy(oracle.nll(x[a:b], batch, LO, HI))
        total = sharding.combine_nll(local)
        again = sharding.combine_nll(local)
        slow = sharding.max_over_ranks(1.0 + rank)
        if rank == 0:
            out.put((total.numpy(), again.numpy(), slow, oracle.nll(x, batch, LO, HI)))
        else:
            out.put((total.numpy(), again.numpy(), slow, None))
    finally:
        dist.destroy_process_group()


def test_two_rank_shards_combine_to_the_full_nll():
    world, n = 2, 20001
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, n, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = [q.get(timeout=300) for _ in range(world)]
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    full = next(r[3] for r in res if r[3] is not None)
    assert np.array_equal(res[0][0], res[1][0])                    # same bits on every rank
    assert np.array_equal(res[0][0], res[0][1])                    # reproducible
    assert np.all(np.abs(res[0][0] - full) <= 1e-12 * np.abs(full))
    assert res[0][2] == res[1][2] == 2.0                           # slowest rank defines the time
