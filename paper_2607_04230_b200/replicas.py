"""N > 1: replicas only (north_star: one GPU, no sharding, no collective on the data path).

Every rank renders the same frame on its own GPU. The only cross-rank step is the bench's timing rule:
barrier, then the MAX over ranks of the per-rank elapsed time; the job's throughput is the units all ranks
processed over that time. These helpers hold that host logic so that it can be tested with the gloo backend
on CPU (tests/test_replicas.py); bench.py calls them with NCCL.
"""
from __future__ import annotations


def max_over_ranks(ms_local: float, dist=None, device="cpu") -> float:
    """MAX over ranks of a per-rank time (ms). `dist` = torch.distributed if a process group is up, else None."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(ms_local)
    import torch
    t = torch.tensor([float(ms_local)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_rate(units_per_rank: int, world: int, ms_per_step: float) -> float:
    """Whole-job units per second: `world` replicas each process `units_per_rank` per step ("weak" scaling)."""
    return world * units_per_rank / (ms_per_step * 1e-3)


def same_on_all_ranks(value: int, dist=None, device="cpu") -> bool:
    """True iff every rank holds the same integer (replicas must render the same frame: same segment count)."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return True
    import torch
    lo = torch.tensor([int(value)], dtype=torch.int64, device=device)
    hi = lo.clone()
    dist.all_reduce(lo, op=dist.ReduceOp.MIN)
    dist.all_reduce(hi, op=dist.ReduceOp.MAX)
    return int(lo.item()) == int(hi.item())
