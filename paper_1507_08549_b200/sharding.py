"""Multi-GPU plumbing of the batch path.

Independent solves are partitioned across ranks with NO data-path collective; the only communication is the
reduction of the timing record (max over ranks of the device time, sum of the work).  A single solve does not
shard: it runs as replicas.  Nothing here touches the solver's arithmetic; it works with any torch.distributed
backend (nccl on the GPUs, gloo in the CPU tests).
"""
from __future__ import annotations


def shard_members(n_members: int, rank: int, world: int):
    """Indices of the batch members rank ``rank`` of ``world`` solves, and the scaling mode.

    A batch with at least one member per rank is dealt round-robin ("strong": total work fixed); anything smaller
    runs in full on every rank ("weak": replicas).
    """
    if not (0 <= rank < world):
        raise ValueError("rank out of range")
    if n_members > 1 and n_members >= world:
        return list(range(rank, n_members, world)), "strong"
    return list(range(n_members)), "weak"


def reduce_timing(total_ms: float, counters, world: int, device=None):
    """max over ranks of ``total_ms`` and the element-wise sum over ranks of ``counters``.

    Returns (max_ms, [sums]).  With world == 1 no process group is needed.
    """
    counters = [float(c) for c in counters]
    if world == 1:
        return float(total_ms), counters
    import torch
    import torch.distributed as dist
    tmax = torch.tensor([float(total_ms)], dtype=torch.float64, device=device)
    tsum = torch.tensor(counters, dtype=torch.float64, device=device)
    dist.all_reduce(tmax, op=dist.ReduceOp.MAX)
    dist.all_reduce(tsum, op=dist.ReduceOp.SUM)
    return float(tmax[0]), [float(x) for x in tsum]
