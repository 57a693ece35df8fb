"""Multi-GPU = replicas only: events are independent (PAPER.md line 172 scales by sending whole
requests to different GPUs), so N GPUs run N contexts with no collective on the data path.  This module is the host side of
that (the analogue of the server's default load balancer):

  * `assign_round_robin`   which replica serves which request;
  * `Dispatcher`           one process, one model instance per visible device (or several per device): takes a list of
                           DISTINCT events, serves event i on the replica round robin chose -- the replicas run concurrently,
                           one host thread each (the C call releases the GIL) -- and returns the per-event results in request
                           order;
  * `serve_distributed`    one process per GPU (torchrun): rank r serves the requests assigned to it, rank 0 collects the
                           results in request order;
  * `max_over_ranks`, `sum_over_ranks`, `whole_job_throughput`   the reductions of device-measured times / unit counts that
                           bench.py needs (the only communication, outside the timed region).

Nothing here computes anything of the method: every event goes through trk_infer_host of one context.  Works with any
torch.distributed backend (nccl on GPUs, gloo in the CPU tests).
"""
from __future__ import annotations

import threading


def assign_round_robin(n_requests: int, world: int) -> list[list[int]]:
    """Request i goes to replica i % world (the default load balancer of the paper's server)."""
    if world < 1 or n_requests < 0:
        raise ValueError("world must be >= 1 and n_requests >= 0")
    return [list(range(r, n_requests, world)) for r in range(world)]


class Dispatcher:
    """Serves lists of events on a fixed set of replicas.

    A replica is any object with `infer_host(hits_host, event_offsets) -> (labels, counts)` (a `Trk`) and, optionally,
    `close()`.  `serve(events)` takes events as (hits fp32 [N,3] host array, event_offsets int32 [B+1]) pairs and returns the
    list of (labels, counts) in request order.  A replica serves its requests in request order, one at a time (a ctx is
    not re-entrant, include/trk.h); different replicas run concurrently.
    """

    def __init__(self, replicas):
        self.replicas = list(replicas)
        if not self.replicas:
            raise ValueError("at least one replica is needed")

    @classmethod
    def from_devices(cls, cfg, model, calib, *, max_hits, devices=None, instances_per_device=1, **trk_kwargs):
        """One `Trk` per (device, instance); devices defaults to every visible CUDA device."""
        from . import trk_from_config
        if devices is None:
            import torch
            devices = list(range(torch.cuda.device_count()))
        reps = []
        try:
            for d in devices:
                for _ in range(instances_per_device):
                    reps.append(trk_from_config(cfg, model, calib, max_hits=max_hits, device=d, **trk_kwargs))
        except Exception:
            for r in reps:
                r.close()
            raise
        return cls(reps)

    def assignment(self, n_requests: int) -> list[list[int]]:
        return assign_round_robin(n_requests, len(self.replicas))

    def serve(self, events):
        events = list(events)
        results = [None] * len(events)
        errors = []

        def work(replica, mine):
            try:
                for i in mine:
                    hits, off = events[i]
                    results[i] = replica.infer_host(hits, off)
            except Exception as e:          # reported to the caller, never swallowed
                errors.append(e)

        threads = [threading.Thread(target=work, args=(rep, mine)) for rep, mine in zip(self.replicas, self.assignment(len(events))) if mine]
        for t in threads:
            t.start()
        for t in threads:
            t.join()
        if errors:
            raise errors[0]
        return results

    def close(self):
        for r in self.replicas:
            if hasattr(r, "close"):
                r.close()
        self.replicas = []


def serve_distributed(events, infer_fn):
    """One process per GPU: rank r serves requests r, r + world, ... with `infer_fn(hits, offsets) -> result`; returns the
    results of ALL requests in request order on rank 0 (None elsewhere).  Results travel as Python objects (gather_object),
    after the compute; there is no collective on the data path."""
    import torch.distributed as dist
    events = list(events)
    up = dist.is_available() and dist.is_initialized()
    world = dist.get_world_size() if up else 1
    rank = dist.get_rank() if up else 0
    mine = assign_round_robin(len(events), world)[rank]
    local = [(i, infer_fn(*events[i])) for i in mine]
    if world == 1:
        gathered = [local]
    else:
        gathered = [None] * world if rank == 0 else None
        dist.gather_object(local, gathered, dst=0)
    if rank != 0:
        return None
    results = [None] * len(events)
    for part in gathered:
        for i, r in part:
            results[i] = r
    return results


def _reduce(value: float, device, op_name: str) -> float:
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=getattr(dist.ReduceOp, op_name))
    return float(t.item())


def max_over_ranks(value: float, device=None) -> float:
    """MAX all-reduce of one float when a process group is up; the value itself otherwise."""
    return _reduce(value, device, "MAX")


def sum_over_ranks(value: float, device=None) -> float:
    return _reduce(value, device, "SUM")


def whole_job_throughput(units_this_rank: float, elapsed_ms_this_rank: float, device=None) -> tuple[float, float]:
    """(units of all ranks) / (slowest rank's time): returns (units per second, max ms)."""
    total = sum_over_ranks(units_this_rank, device)
    ms = max_over_ranks(elapsed_ms_this_rank, device)
    return (total / (ms * 1e-3) if ms > 0 else 0.0), ms
