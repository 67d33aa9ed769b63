"""Host-side plumbing of the multi-GPU mode ("replicas only").

The path does not shard (north_star: one GPU, no domain decomposition, no LET exchange), so N ranks
run N independent replicas and there is no collective on the data path.  The only cross-rank step is
the reduction of the timing: the job took as long as its slowest rank and did the work of all of them.
"""
from __future__ import annotations


def replica_seed(base_seed: int, rank: int) -> int:
    """every rank draws its own initial conditions"""
    return int(base_seed) + int(rank)


def aggregate(elapsed_ms: float, units: float, device=None):
    """(max over ranks of elapsed_ms, sum over ranks of units, units per second of the whole job).

    Uses the default torch.distributed process group when one is initialised (nccl on the GPU box,
    gloo in the CPU tests); a single process is its own job."""
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(elapsed_ms)], dtype=torch.float64, device=device)
    u = torch.tensor([float(units)], dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        dist.all_reduce(u, op=dist.ReduceOp.SUM)
    t_ms, total = float(t.item()), float(u.item())
    return t_ms, total, (total / (t_ms * 1e-3) if t_ms > 0 else 0.0)
