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


def _cuda_worker(rank, world, port, n, out):
    """The path bench.py --gpus N times: every rank generates ITS shard of one seeded dataset on its own GPU
    (ipa_options.first_slot), evaluates it with ipa_nll_eval and the partial sums are all-gathered over NCCL."""
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    torch.cuda.set_device(rank)
    dist.init_process_group("nccl", rank=rank, world_size=world)
    try:
        import paper_1706_01420_b200 as ipa
        batch, _ = inp.fd_batch(inp.GEN)
        a, b = sharding.shard_range(n, rank, world)
        x, _, _ = ipa.ipa_toy_generate([3], inp.GEN, -1.0, -1.0, LO, HI, b - a, first_slot=a)
        local, _, _ = ipa.ipa_nll_eval(x, batch, LO, HI)
        total = sharding.combine_nll(local)
        torch.cuda.synchronize()
        full = None
        if rank == 0:
            xf, _, _ = ipa.ipa_toy_generate([3], inp.GEN, -1.0, -1.0, LO, HI, n)
            full = ipa.ipa_nll_eval(xf, batch, LO, HI)[0].cpu().numpy()
        out.put((total.cpu().numpy(), full))
    finally:
        dist.destroy_process_group()


@pytest.mark.gpu
def test_two_gpu_shards_combine_to_the_full_nll():
    if torch.cuda.device_count() < 2:
        pytest.skip("needs two GPUs (the GPU pool of this build hands out one)")
    world, n = 2, 1_000_003
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_cuda_worker, args=(r, world, port, n, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = [q.get(timeout=600) for _ in range(world)]
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    full = next(r[1] for r in res if r[1] is not None)
    assert np.array_equal(res[0][0], res[1][0])
    assert np.all(np.abs(res[0][0] - full) <= 1e-12 * np.abs(full))
