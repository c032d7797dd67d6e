"""Host-side multi-GPU plumbing: the path shards only over batch members (independent
simulations), one process per GPU, no data-path collective.  These helpers hold the rank / shard
arithmetic and the max-over-ranks timing reduction that bench.py uses; they contain none of the method's arithmetic
and work with any torch.distributed backend (nccl on GPUs, gloo in the CPU tests)."""
from __future__ import annotations

from typing import Optional, Tuple


def shard_members(batch: int, rank: int, world: int) -> range:
    """Contiguous, balanced block of batch members owned by `rank`: the first batch % world ranks get one extra."""
    if batch < 0 or world < 1 or not 0 <= rank < world:
        raise ValueError("bad shard arguments: batch=%d rank=%d world=%d" % (batch, rank, world))
    base, extra = divmod(batch, world)
    lo = rank * base + min(rank, extra)
    return range(lo, lo + base + (1 if rank < extra else 0))


def owner_of(member: int, batch: int, world: int) -> int:
    """Inverse of shard_members: the rank that owns `member`."""
    for r in range(world):
        s = shard_members(batch, r, world)
        if s.start <= member < s.stop:
            return r
    raise ValueError("member %d outside a batch of %d" % (member, batch))


def reduce_timing(ms_local: float, units_local: float, device=None, group=None) -> Tuple[float, float]:
    """(max over ranks of the elapsed milliseconds, sum over ranks of the units processed).  Without an initialised
    process group the local values are returned."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size(group) == 1:
        return float(ms_local), float(units_local)
    t = torch.tensor([ms_local], dtype=torch.float64, device=device)
    u = torch.tensor([units_local], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX, group=group)
    dist.all_reduce(u, op=dist.ReduceOp.SUM, group=group)
    return float(t.item()), float(u.item())


def throughput(ms_local: float, units_local: float, device=None, group=None) -> Tuple[float, float]:
    """Whole-job units per second = all ranks' units / slowest rank's time; also returns that time in ms."""
    ms, units = reduce_timing(ms_local, units_local, device, group)
    return units / (ms * 1e-3), ms
