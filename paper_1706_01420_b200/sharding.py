"""Multi-GPU plumbing of the path: events are independent units and the result is
a K-vector of sums, so G ranks each own a contiguous shard of the events (toys: whole toys), evaluate
their shard with `ipa_nll_eval`, and the K partial sums are combined in RANK ORDER after one all-gather
(8 K bytes per rank: latency-bound, no data-path collective on the events).  Rank-order addition keeps the
result bitwise reproducible for a fixed world size.  No arithmetic of the likelihood happens here.
"""
import torch
import torch.distributed as dist


def shard_range(n, rank, world):
    """Contiguous shard [begin, end) of n units for `rank` of `world`; sizes differ by at most 1 and the
    first n % world ranks hold the larger shards."""
    n, rank, world = int(n), int(rank), int(world)
    if not (world >= 1 and 0 <= rank < world and n >= 0):
        raise ValueError("shard_range: need world >= 1, 0 <= rank < world, n >= 0")
    q, r = divmod(n, world)
    begin = rank * q + min(rank, r)
    return begin, begin + q + (1 if rank < r else 0)


def shard_segments(offsets, rank, world):
    """Whole segments (toys) per rank: -> (first_segment, last_segment_exclusive, event_begin, event_end)."""
    T = len(offsets) - 1
    a, b = shard_range(T, rank, world)
    return a, b, int(offsets[a]), int(offsets[b])


def combine_nll(nll_local, group=None):
    """All-gather the K partial NLLs of every rank and add them in rank order.  Works on CPU tensors
    (gloo) and CUDA tensors (nccl); returns a tensor like nll_local on every rank."""
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size(group) == 1:
        return nll_local.clone()
    world = dist.get_world_size(group)
    parts = [torch.empty_like(nll_local) for _ in range(world)]
    dist.all_gather(parts, nll_local.contiguous(), group=group)
    total = parts[0].clone()
    for r in range(1, world):
        total += parts[r]
    return total


def max_over_ranks(seconds, device="cpu", group=None):
    """Timing rule of bench.py: the slowest rank defines the step time."""
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size(group) == 1:
        return float(seconds)
    t = torch.tensor([float(seconds)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX, group=group)
    return float(t.item())
