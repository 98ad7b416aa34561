"""Multi-GPU plumbing for bench.py: the path does not shard ("replicas
only"), so N GPUs run N independent replicas and the only cross-rank operation is the timing
reduction: barrier + max over ranks.  No data-path collective."""
from __future__ import annotations


def make_dist_max(torch, world: int, device):
    """Returns f(seconds) -> max over ranks (also a barrier).  world == 1: identity."""
    if world <= 1:
        return lambda t: float(t)
    import torch.distributed as dist
    backend = dist.get_backend()
    dev = device if backend == "nccl" else "cpu"

    def f(t):
        v = torch.tensor([float(t)], dtype=torch.float64, device=dev)
        dist.all_reduce(v, op=dist.ReduceOp.MAX)
        return float(v.item())

    return f


def whole_job_value(per_rank_units: float, world: int, max_seconds: float) -> float:
    """Weak scaling: every rank processed per_rank_units in at most max_seconds."""
    return per_rank_units * world / max_seconds
