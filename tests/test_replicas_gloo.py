"""-m "not gpu": the N > 1 path (replicas, no data-path collective) on CPU with the gloo backend, world_size 2."""
import json
import os
import socket
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out_dir):
    import torch.distributed as dist
    from paper_2501_05520_b200.replicas import assign_round_robin, whole_job_throughput
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    mine = assign_round_robin(7, world)[rank]
    ms = 10.0 * (rank + 1) * len(mine)                 # pretend device time: rank 1 is the slow one
    value, max_ms = whole_job_throughput(len(mine), ms)
    with open(os.path.join(out_dir, f"r{rank}.json"), "w") as f:
        json.dump(dict(mine=mine, value=value, max_ms=max_ms), f)
    dist.barrier()
    dist.destroy_process_group()


def test_round_robin_assignment_partitions_requests():
    from paper_2501_05520_b200.replicas import assign_round_robin, max_over_ranks
    for n in (0, 1, 7, 16):
        for w in (1, 2, 3, 8):
            parts = assign_round_robin(n, w)
            assert len(parts) == w and sorted(sum(parts, [])) == list(range(n))
            assert max(len(p) for p in parts) - min(len(p) for p in parts) <= 1
    with pytest.raises(ValueError):
        assign_round_robin(3, 0)
    assert max_over_ranks(3.5) == 3.5                   # no process group: identity


def test_two_ranks_gloo_max_time_and_total_units(tmp_path):
    import torch.multiprocessing as mp
    port = _free_port()
    mp.spawn(_worker, args=(2, port, str(tmp_path)), nprocs=2, join=True)
    r = [json.load(open(tmp_path / f"r{k}.json")) for k in range(2)]
    assert sorted(r[0]["mine"] + r[1]["mine"]) == list(range(7)) and not set(r[0]["mine"]) & set(r[1]["mine"])
    # rank 0: 4 requests, 40 ms; rank 1: 3 requests, 60 ms -> 7 requests / 60 ms on both ranks
    for x in r:
        assert x["max_ms"] == 60.0 and abs(x["value"] - 7 / 0.060) < 1e-9


class _StubReplica:
    """Stands in for a Trk on the CPU box: 'labels' = hit index + 1000 * replica id + first feature, so order and
    assignment are visible in the results."""

    def __init__(self, ident):
        self.ident = ident
        self.served = []

    def infer_host(self, hits, off):
        import numpy as np
        self.served.append(int(hits[0, 0]))
        return np.arange(int(off[-1]), dtype=np.int64) + 1000 * self.ident + int(hits[0, 0]), np.array([len(hits), 0, 0, 0])


def _events(n):
    import numpy as np
    return [(np.full((3 + i, 3), float(i), np.float32), np.array([0, 3 + i], np.int32)) for i in range(n)]


def test_dispatcher_serves_distinct_events_in_request_order():
    from paper_2501_05520_b200.replicas import Dispatcher
    reps = [_StubReplica(k) for k in range(3)]
    d = Dispatcher(reps)
    ev = _events(8)
    res = d.serve(ev)
    assert len(res) == 8
    for i, (labels, counts) in enumerate(res):
        assert len(labels) == 3 + i and counts[0] == 3 + i          # the result of request i, in position i
        assert labels[0] == 1000 * (i % 3) + i                       # ... served by replica i % 3
    for k, r in enumerate(reps):
        assert r.served == list(range(k, 8, 3))                       # each replica took its share, in request order
    assert d.serve([]) == []
    # an error inside a replica reaches the caller
    class Bad(_StubReplica):
        def infer_host(self, hits, off):
            raise RuntimeError("replica failed")
    with pytest.raises(RuntimeError):
        Dispatcher([Bad(0)]).serve(ev[:1])
    with pytest.raises(ValueError):
        Dispatcher([])


def _serve_worker(rank, world, port, out_dir):
    import pickle
    import torch.distributed as dist
    from paper_2501_05520_b200.replicas import serve_distributed
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    rep = _StubReplica(rank)
    res = serve_distributed(_events(5), rep.infer_host)
    with open(os.path.join(out_dir, f"s{rank}.pkl"), "wb") as f:
        pickle.dump(dict(res=res, served=rep.served), f)
    dist.barrier()
    dist.destroy_process_group()


def test_two_ranks_gloo_serve_distributed_collects_results_in_order(tmp_path):
    import pickle
    import torch.multiprocessing as mp
    port = _free_port()
    mp.spawn(_serve_worker, args=(2, port, str(tmp_path)), nprocs=2, join=True)
    r = [pickle.load(open(tmp_path / f"s{k}.pkl", "rb")) for k in range(2)]
    assert r[0]["served"] == [0, 2, 4] and r[1]["served"] == [1, 3] and r[1]["res"] is None
    res = r[0]["res"]
    assert len(res) == 5
    for i, (labels, counts) in enumerate(res):
        assert len(labels) == 3 + i and labels[0] == 1000 * (i % 2) + i


def test_bench_reference_arm_under_torchrun_prints_one_line():
    """N > 1 launch of `bench.py --impl reference`: rank 0 alone prints the JSON line, the other rank exits 0 without work."""
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
           "--master-port", str(_free_port()), os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "6",
           "--warmup", "0", "--config", "toy"]
    p = subprocess.run(cmd, capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert p.returncode == 0, p.stderr[-2000:]
    lines = [l for l in p.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["unit"] == "events/s" and d["value"] > 0
    # the K steps are the K consecutive pieces of ONE oracle pass over the event: K x ms_per_step is the event's wall time
    assert d["steps"] == 6 and abs(d["steps"] * d["ms_per_step"] * 1e-3 - 1.0 / d["value"]) < 1e-6
    assert set(d["cpu_baseline"]["stage_s"]) == {"s1_embed", "s2_frnn", "s3_filter", "s4_gnn", "s5_cc"}
    assert d["cpu_baseline"]["kind"] == "oracle" and d["e2e"]["h2d_bytes_per_step"] == 0
