"""Multi-GPU plumbing: planning instances are independent, so the batch is dealt to
ranks with NO data-path collective; only the bench's bookkeeping (units summed, device time max-ed)
crosses ranks.  Host logic only — runs on gloo (CPU tests) and nccl (one process per GPU) alike."""
from __future__ import annotations


def shard_range(n_total: int, rank: int, world: int) -> range:
    """Contiguous, balanced split of n_total instance indices: sizes differ by at most one."""
    if not (0 <= rank < world):
        raise ValueError("rank outside [0, world)")
    q, r = divmod(n_total, world)
    lo = rank * q + min(rank, r)
    return range(lo, lo + q + (1 if rank < r else 0))


def weak_seeds(per_rank: int, rank: int) -> range:
    """Weak scaling: every rank solves per_rank instances of its own (seeds never overlap)."""
    return range(rank * per_rank, (rank + 1) * per_rank)


def aggregate(sums, maxes, device=None):
    """All-reduce bookkeeping scalars: `sums` are added over ranks, `maxes` take the max over ranks
    (device times are reported as the slowest rank's).  No-op without an initialised process group."""
    import torch
    import torch.distributed as dist
    s = torch.tensor([float(v) for v in sums], dtype=torch.float64, device=device)
    m = torch.tensor([float(v) for v in maxes], dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(s, op=dist.ReduceOp.SUM)
        dist.all_reduce(m, op=dist.ReduceOp.MAX)
    return s.tolist(), m.tolist()


def gather_results(local_results: bytes, group=None):
    """Gathers every rank's packed tg_result bytes on all ranks, in rank order (strong-scaled batch)."""
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return [local_results]
    out = [None] * dist.get_world_size()
    dist.all_gather_object(out, local_results, group=group)
    return out
