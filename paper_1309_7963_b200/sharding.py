"""Multi-GPU sharding of the event range: events are independent and the
RNG is keyed by the global event index, so ranks take contiguous ranges and never exchange
data on the path.  The only cross-rank datum is the base offset of each rank's secondary
list: one 8-byte all_gather + a host-side exclusive scan."""
from __future__ import annotations


def shard_range(n_events: int, rank: int, world: int):
    """Contiguous, balanced [lo, hi) for `rank` of `world`; the union is exactly [0, n)."""
    base, rem = divmod(int(n_events), int(world))
    lo = rank * base + min(rank, rem)
    hi = lo + base + (1 if rank < rem else 0)
    return lo, hi


def gather_secondary_bases(local_total: int, group=None):
    """all_gather of the per-rank secondary totals -> (this rank's base offset, global total).
    Works on any torch.distributed backend (gloo on CPU for tests, nccl on GPUs)."""
    import torch
    import torch.distributed as dist
    world = dist.get_world_size(group)
    rank = dist.get_rank(group)
    dev = "cuda" if dist.get_backend(group) == "nccl" else "cpu"
    mine = torch.tensor([int(local_total)], dtype=torch.int64, device=dev)
    allv = [torch.zeros_like(mine) for _ in range(world)]
    dist.all_gather(allv, mine, group=group)
    totals = [int(t.item()) for t in allv]
    return sum(totals[:rank]), sum(totals)
