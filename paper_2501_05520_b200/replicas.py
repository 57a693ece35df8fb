"""Multi-GPU = replicas only: events are independent (PAPER.md line 172 scales by sending whole
requests to different GPUs), so N ranks run N contexts with no collective on the data path.  This module holds the
host-side plumbing of that: which rank serves which request, and the max-over-ranks reduction of a device-measured time
(the only communication, outside the timed region).  Works with any torch.distributed backend (nccl on GPUs, gloo in the
CPU tests)."""
from __future__ import annotations


def assign_round_robin(n_requests: int, world: int) -> list[list[int]]:
    """Request i goes to rank i % world (the default load balancer of the paper's server)."""
    if world < 1 or n_requests < 0:
        raise ValueError("world must be >= 1 and n_requests >= 0")
    return [list(range(r, n_requests, world)) for r in range(world)]


def max_over_ranks(value: float, device=None) -> float:
    """MAX all-reduce of one float when a process group is up; the value itself otherwise."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(value: float, device=None) -> float:
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def whole_job_throughput(units_this_rank: float, elapsed_ms_this_rank: float, device=None) -> tuple[float, float]:
    """(units of all ranks) / (slowest rank's time): returns (units per second, max ms)."""
    total = sum_over_ranks(units_this_rank, device)
    ms = max_over_ranks(elapsed_ms_this_rank, device)
    return (total / (ms * 1e-3) if ms > 0 else 0.0), ms
