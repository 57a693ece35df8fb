#!/usr/bin/env python
"""Benchmark of the hot path: one step = one trk_infer call (all five stages) on the pileup-200 event
(BASELINE.json configs[2], the configuration `metric` is quoted on).

    python bench.py --gpus 1 --steps 10 --warmup 3            # our arm (CUDA library through the C ABI)
    python bench.py --impl reference --steps 3 --warmup 1     # the oracle on the host cores

Prints ONE JSON line (see DESIGN.md "Measurement" for every field).  N > 1 runs one replica per GPU
(events are independent, no collective on the data path: "scaling": "weak").
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

FILTER_FLOP_PER_EDGE = 2 * (24 * 1024 + 1024 * 1024 * 2 + 1024)          # 4 245 504
EMBED_FLOP_PER_HIT = 2 * (3 * 1024 + 1024 * 1024 * 2 + 1024 * 12)        # 4 225 024
# DRAM bytes of one full-chunk launch (1 212 416 rows) of the dominant kernel, from the ncu --set full capture summarised in
# profiles/r1_full_v6.md (dram__bytes_read.sum + dram__bytes_write.sum)
NCU_TRAFFIC_BYTES = {"bias_act": 2578.13e6 + 2441.02e6, "relu_dot": 2490.36e6 + 23.02e6}


def gnn_flops(n, e, H=128, T=8):
    """Algorithmic minimum with the exact first-layer split: per node PA|PB and node_net, per edge K=H."""
    enc = n * 2 * (3 * H + H * H) + e * 2 * (4 * H + H * H)
    it = n * 2 * (2 * H * H) + e * 2 * (2 * H * H) + n * 2 * (3 * H * H + H * H)
    dec = n * 2 * (2 * H * H) + e * 2 * (H * H + H)
    return enc + T * it + dec


def gnn_bytes(n, e, H=128, T=8):
    """Algorithmic HBM bytes of S4 with bf16 state: per iteration e in + e out (edge update), e in again
    (the two aggregations share one pass), m_in | m_out out, [h | m_in | m_out] in and h out (node update); encoders write h and e
    once, the decoder reads e and writes a score; indices 8 B/edge per edge pass."""
    row = 2 * H
    it = e * (3 * row + 16) + n * (2 * row + 3 * row + row)
    return (e * (row + 8) + n * (12 + row)) + T * it + e * (row + 12)


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        return dict(hbm_gbs=d["hbm_gbs"], bf16_tflops=d["bf16_tflops"], bf16_sustained=d.get("bf16_tflops_sustained", d["bf16_tflops"]),
                    source="measured (MEASURED_PEAKS.json)")
    return dict(hbm_gbs=6650.0, bf16_tflops=1590.0, bf16_sustained=1400.0, source="fallback (B200_PROFILING.md)")


class ClockSampler:
    FIELDS = "clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown," \
             "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"

    def __init__(self, index):
        self.p = None
        try:
            self.p = subprocess.Popen(["nvidia-smi", f"--id={index}", f"--query-gpu={self.FIELDS}", "--format=csv,noheader,nounits",
                                       "-lms", "20"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except Exception:
            self.p = None

    def stop(self):
        if self.p is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.p.terminate()
        try:
            out, _ = self.p.communicate(timeout=5)
        except Exception:
            self.p.kill()
            out = ""
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in out.strip().splitlines():
            f = [x.strip() for x in line.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1]))
            except ValueError:
                continue
            for nme, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nme)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": float(max(mx)) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def build_workload(name):
    from synth.configs import get_config, load_calibration, make_events
    from synth.weights import make_model
    cfg = get_config(name)
    calib = load_calibration(cfg["calibration"])
    ev = make_events(cfg)
    model = make_model(cfg)
    # reading C-16: decoder bias centred so that the 0.5 cut has edges on both sides (a weight value, not an API change)
    dec = model["edge_dec"]
    dec["bias"][1] = (dec["bias"][1].astype(np.float64) - calib["gnn_logit_median"]).astype(np.float32)
    return cfg, calib, ev, model


def oracle_sample(n_particles, arch_cfg_name="pileup200"):
    """Times the oracle (as it stands) on a bounded sample: the pileup-50-density event of `n_particles` particles through
    all five stages with the headline architecture; returns per-stage seconds and unit counts."""
    from oracle import pipeline as opipe
    from synth.configs import get_config, load_calibration, make_events
    from synth.weights import make_model
    cfg = get_config("pileup50")                       # same architecture as pileup200, its own calibrated radius/cut
    calib = load_calibration("pileup50")
    ev = make_events(cfg, n_particles=n_particles)
    model = make_model(cfg)
    timing = {}
    t0 = time.perf_counter()
    out = opipe.run(cfg, model, calib, ev["hits"], ev["event_offsets"], timing=timing)
    wall = time.perf_counter() - t0
    units = dict(n=len(ev["hits"]), e_c=len(out["cand_src"]), e_k=len(out["src"]))
    return timing, units, wall


def extrapolate_events_per_s(timing, units, target):
    """Per-stage time scaled by the stage's unit count (S1,S2: hits; S3: candidate edges; S4,S5: kept edges)."""
    t = (timing["s1_embed"] + timing["s2_frnn"]) * target["n"] / max(1, units["n"]) \
        + timing["s3_filter"] * target["e_c"] / max(1, units["e_c"]) \
        + (timing["s4_gnn"] + timing["s5_cc"]) * target["e_k"] / max(1, units["e_k"])
    return 1.0 / t, t


def cpu_threads():
    try:
        from threadpoolctl import threadpool_info
        return max([i.get("num_threads", 1) for i in threadpool_info()] + [1])
    except Exception:
        return os.cpu_count() or 1


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from synth.configs import load_calibration
    cal = load_calibration("pileup200")
    target = dict(n=cal["n_hits"], e_c=cal["n_cand_edges"], e_k=cal["n_kept_edges"])
    npart = args.ref_particles
    for _ in range(args.warmup):
        oracle_sample(npart)
    vals, walls = [], []
    for _ in range(args.steps):
        timing, units, wall = oracle_sample(npart)
        v, _ = extrapolate_events_per_s(timing, units, target)
        vals.append(v); walls.append(wall)
    value = float(np.mean(vals))
    sample = (f"oracle (fp64 NumPy) on a {npart}-particle event of the same generator and architecture "
              f"({units['n']} hits, {units['e_c']} candidate, {units['e_k']} kept edges), per-stage times scaled by unit counts "
              f"to the pileup-200 event ({target['n']} hits, {target['e_c']}, {target['e_k']})")
    line = {"impl": "reference", "metric": "events/s (pileup-200 event)", "value": value, "unit": "events/s", "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1000.0 * float(np.mean(walls)), "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": "pileup200", "hits": target["n"], "parallelism": "host cores"},
            "cpu_baseline": {"value": value, "unit": "events/s", "cores": cpu_threads(), "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": "events/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


def run_concurrency_scan(args):
    """SURVEY.md section 8(f) NEXT-2, the shape of PAPER.md Fig. 6/7 (lines 166-180) without Triton: throughput of pileup-50 events
    (a) on 1..7 model instances (contexts) each on its own stream, every instance serving its own copy of the event,
    (b) the same 16 events packed into ONE trk_infer call (BASELINE.json configs[3]), and (c) a CUDA-graph replay of one call.
    Prints one JSON object (not the bench line)."""
    import torch
    from paper_2501_05520_b200 import trk_from_config
    torch.cuda.set_device(0)
    dev = torch.device("cuda", 0)
    cfg, calib, ev, model = build_workload("pileup50")
    n = len(ev["hits"])
    hits = torch.from_numpy(ev["hits"]).to(dev)
    off = ev["event_offsets"]
    rounds = max(args.steps, 5)
    res = {"workload": "pileup50 event per request", "hits_per_event": n, "rounds": rounds, "instances": []}

    def timed(fn, n_events):
        for _ in range(3):
            fn()
        torch.cuda.synchronize()
        s, e = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        s.record()
        for _ in range(rounds):
            fn()
        e.record()
        torch.cuda.synchronize()
        ms = s.elapsed_time(e)
        return n_events * rounds / (ms * 1e-3), ms / rounds

    ctxs, streams, outs = [], [], []
    max_kept = int(calib["n_kept_edges"] * 1.5 + 4096)
    for k in (1, 2, 3, 4, 5, 6, 7):
        while len(ctxs) < k:
            t = trk_from_config(cfg, model, calib, max_hits=n, max_cand_edges=n * cfg["frnn_k"], max_kept_edges=max_kept)
            st = torch.cuda.Stream()
            ctxs.append(t); streams.append(st)
            with torch.cuda.stream(st):
                outs.append(t.infer(hits, off, stream=st))
            torch.cuda.synchronize()

        def step():
            cur = torch.cuda.current_stream()
            for t, st, o in zip(ctxs[:k], streams[:k], outs[:k]):
                st.wait_stream(cur)
                t.infer(hits, off, out=o, stream=st)
            for st in streams[:k]:
                cur.wait_stream(st)
        ev_s, ms = timed(step, k)
        res["instances"].append({"contexts": k, "events_per_s": ev_s, "ms_per_round": ms})
    # CUDA graph of one call on one context
    g = torch.cuda.CUDAGraph()
    cap = torch.cuda.Stream()
    with torch.cuda.stream(cap):
        with torch.cuda.graph(g, stream=cap):
            ctxs[0].infer(hits, off, out=outs[0], stream=cap)
    ev_s, ms = timed(g.replay, 1)
    res["cuda_graph_one_context"] = {"events_per_s": ev_s, "ms_per_event": ms, "launches_in_graph": ctxs[0].last_launch_count}
    for t in ctxs:
        t.close()
    # the packed batch: 16 events in one call
    cfgb, calibb, evb, modelb = build_workload("batch16")
    nb = len(evb["hits"])
    tb = trk_from_config(cfgb, modelb, calibb, max_hits=nb, max_events=16, max_cand_edges=nb * cfgb["frnn_k"],
                         max_kept_edges=int(calibb["n_kept_edges"] * 16 * 1.5 + 4096))
    hb = torch.from_numpy(evb["hits"]).to(dev)
    ob = tb.infer(hb, evb["event_offsets"])
    torch.cuda.synchronize()
    ev_s, ms = timed(lambda: tb.infer(hb, evb["event_offsets"], out=ob), 16)
    res["packed_batch16"] = {"events_per_s": ev_s, "ms_per_call": ms, "hits": nb}
    tb.close()
    print(json.dumps(res))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="pileup200")
    ap.add_argument("--ref-particles", type=int, default=500)
    ap.add_argument("--cpu-baseline-particles", type=int, default=2500)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--scan", action="store_true", help="concurrency scan (model instances x streams, packed batch, CUDA graph)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 0)
    if args.impl == "reference":
        return run_reference(args)
    if args.scan:
        return run_concurrency_scan(args)

    import torch
    import torch.distributed as dist
    from paper_2501_05520_b200 import gemm_bf16, trk_from_config
    from paper_2501_05520_b200.replicas import max_over_ranks

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    warmup = max(args.warmup, 3)

    cfg, calib, ev, model = build_workload(args.config)
    n = len(ev["hits"])
    n_events = len(ev["event_offsets"]) - 1
    # capacities: N*K can never overflow S2; kept edges sized from the calibrated count with head-room
    max_cand = n * cfg["frnn_k"]
    max_kept = int(min(max_cand, calib["n_kept_edges"] * (n / calib["n_hits"]) * 1.5 + 4096))
    trk = trk_from_config(cfg, model, calib, max_hits=n, max_events=n_events, max_cand_edges=max_cand, max_kept_edges=max_kept,
                          device=local)
    hits = torch.from_numpy(ev["hits"]).to(dev)
    out = trk.infer(hits, ev["event_offsets"])          # allocates outputs once
    torch.cuda.synchronize()
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)   # > 126 MB L2

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    trk.profile(True)
    for _ in range(warmup):
        flush.zero_()
        trk.infer(hits, ev["event_offsets"], out=out)
    barrier()
    sampler = ClockSampler(local) if rank == 0 else None
    starts = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps)]
    ends = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps)]
    stage_ms, kernel_ms = [], []
    for i in range(args.steps):
        flush.zero_()
        starts[i].record()
        trk.infer(hits, ev["event_offsets"], out=out)
        ends[i].record()
        stage_ms.append(trk.stage_ms())                 # waits for this step (the next flush is outside the timed pair anyway)
        kernel_ms.append(trk.kernel_ms())
    barrier()
    clocks = sampler.stop() if sampler else None
    step_ms = [s.elapsed_time(e) for s, e in zip(starts, ends)]
    total_ms = float(np.sum(step_ms))
    launches = trk.last_launch_count * args.steps
    counts = out["counts"].cpu().numpy().tolist()
    total_ms = max_over_ranks(total_ms, dev)            # replicas: the slowest rank's device time (no data-path collective)
    events_per_s = world * n_events * args.steps / (total_ms / 1000.0)

    # ---- end to end through the host API: pinned host buffers, H2D + D2H inside the timed region
    e2e = None
    if not args.no_e2e:
        hh = torch.from_numpy(ev["hits"]).pin_memory()
        lh = torch.empty(n, dtype=torch.int32).pin_memory()
        ch = torch.zeros(4, dtype=torch.int32).pin_memory()
        for _ in range(2):
            trk.infer_host(hh, ev["event_offsets"], lh, ch)
        barrier()
        t0 = time.perf_counter()
        for _ in range(args.steps):
            trk.infer_host(hh, ev["event_offsets"], lh, ch)
        torch.cuda.synchronize()
        dt = time.perf_counter() - t0
        dt = max_over_ranks(dt, dev)
        e2e = {"value": world * n_events * args.steps / dt, "unit": "events/s", "h2d_bytes_per_step": n * 12,
               "d2h_bytes_per_step": n * 4 + 16, "api": "trk_infer_host (pinned host hits in, host labels out, sync inside)"}

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- rooflines
    peaks = load_peaks()
    e_c, e_k = counts[0], counts[1]
    st = {k: float(np.mean([s[k] for s in stage_ms])) for k in stage_ms[0]}
    s3_flops = e_c * FILTER_FLOP_PER_EDGE
    s3_tflops = s3_flops / (st["s3_filter"] * 1e-3) / 1e12
    # the dominant kernel inside the timed steps: CUDA-event pairs around every hidden-layer GEMM launch of S3
    # (trk_profile_kernel_ms); chunk c of launch i = c // 2 holds rows [c*chunk, (c+1)*chunk) clipped to E_c
    width = cfg["filter_dims"][1]
    k_flops, k_ms, k_n = 0.0, 0.0, 0
    for ms_list, chunk_rows in kernel_ms:
        per_chunk = max(1, len(cfg["filter_dims"]) - 3)
        for i, ms in enumerate(ms_list):
            rows = min(max(e_c - (i // per_chunk) * chunk_rows, 0), chunk_rows)
            if rows > 0:
                k_flops += 2.0 * rows * width * width
                k_ms += ms
                k_n += 1
    kern_tflops = k_flops / (k_ms * 1e-3) / 1e12 if k_ms > 0 else 0.0
    chunk_rows = kernel_ms[0][1]
    # ... and in isolation, at the per-launch shape of the pipeline (one full chunk, one hidden layer)
    m_chunk = chunk_rows
    a = torch.randn(m_chunk, 1024, device=dev).to(torch.bfloat16)
    w = (torch.randn(1024, 1024, device=dev) / 32).to(torch.bfloat16)
    b = torch.zeros(1024, device=dev)
    for _ in range(3):
        gemm_bf16(a, w, b)
    evs = []
    for _ in range(10):
        flush.zero_()
        s, e = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        s.record(); gemm_bf16(a, w, b); e.record()
        evs.append((s, e))
    torch.cuda.synchronize()
    iso_ms = float(np.mean([s.elapsed_time(e) for s, e in evs]))
    iso_tflops = 2.0 * m_chunk * 1024 * 1024 / (iso_ms * 1e-3) / 1e12
    hbm = peaks["hbm_gbs"]
    stage_roofline = {
        "s1_embed": {"bound": "tensor", "achieved_tflops": n * EMBED_FLOP_PER_HIT / (st["s1_embed"] * 1e-3) / 1e12},
        "s2_frnn": {"bound": "hbm", "achieved_gbs": (n * 56 + e_c * 8 + n * 4) / (st["s2_frnn"] * 1e-3) / 1e9},
        "s3_filter": {"bound": "tensor", "achieved_tflops": s3_tflops},
        "s4_gnn": {"bound": "tensor", "achieved_tflops": gnn_flops(n, e_k, cfg["gnn_hidden"], cfg["gnn_iters"]) / (st["s4_gnn"] * 1e-3) / 1e12},
        "s5_cc": {"bound": "hbm", "achieved_gbs": (e_k * 12 + n * 4) / (st["s5_cc"] * 1e-3) / 1e9},
    }
    s4 = stage_roofline["s4_gnn"]
    s4["hbm_view"] = {"achieved_gbs": gnn_bytes(n, e_k, cfg["gnn_hidden"], cfg["gnn_iters"]) / (st["s4_gnn"] * 1e-3) / 1e9}
    s4["hbm_view"]["frac_of_measured"] = s4["hbm_view"]["achieved_gbs"] / hbm
    stage_roofline["s2_frnn"]["note"] = ("nominally HBM; really instruction-issue bound (tables live in L2/L1, no DRAM traffic): "
                                         "ncu issue 63 %, profiles/r1_full_v4.md")
    stage_roofline["s5_cc"]["note"] = "nominally HBM; really bound by the latency of atomics on the L2-resident parent array"
    s4["note"] = "on the tensor/HBM ridge: the flop count is the split-first-layer minimum, the byte count the bf16-state minimum"
    for k, v in stage_roofline.items():
        v["ms"] = st[k]
        if "achieved_tflops" in v:
            v["frac_of_measured_sustained"] = v["achieved_tflops"] / peaks["bf16_sustained"]
            v["frac_of_nominal_2250"] = v["achieved_tflops"] / 2250.0
        else:
            v["frac_of_measured"] = v["achieved_gbs"] / hbm
            v["frac_of_nominal_8000"] = v["achieved_gbs"] / 8000.0
    # peak: the launches are 0.4 ms kernels inside 14 ms steps of a ~0.2 s timed region, far from the 4 s back-to-back run that
    # defines the "sustained" cuBLAS figure (SM clocks settle near 1.33 GHz there; here they stay near the burst clocks, see
    # `clocks`), so the burst figure is the denominator; the fraction of the sustained figure is given beside it.
    roofline = {"bound": "tensor",
                "kernel": "tc::gemm_tc2_kernel<256,*> (tcgen05.mma.cta_group::2, the 1024x1024 hidden layers of the S3 filter MLP; "
                          f"one launch = one layer of one {chunk_rows}-edge chunk)",
                "achieved": kern_tflops, "peak": peaks["bf16_tflops"], "unit": "TFLOP/s", "frac": kern_tflops / peaks["bf16_tflops"],
                "peak_source": peaks["source"] + ", burst bf16 (short launches at burst clocks)",
                "frac_of_sustained_peak": kern_tflops / peaks["bf16_sustained"], "sustained_peak": peaks["bf16_sustained"],
                "launches_timed": k_n, "avg_launch_ms": k_ms / max(1, k_n), "flop_per_full_launch": 2.0 * chunk_rows * width * width,
                "how": "algorithmic flops of the non-empty launches (2 x rows x 1024 x 1024 each) / their summed durations, CUDA-event pairs "
                       "around each launch on the launch stream inside the timed steps (trk_profile_kernel_ms)",
                # ncu --set full, profiles/r1_full_v6.md: dram__bytes_read.sum + dram__bytes_write.sum of one full-chunk launch
                "traffic": NCU_TRAFFIC_BYTES["bias_act"], "traffic_unit": "bytes per full-chunk launch (EpiBiasActBf16 variant)",
                "traffic_detail": dict(NCU_TRAFFIC_BYTES, algorithmic_bias_act=2 * chunk_rows * width * 2 + width * width * 2,
                                       algorithmic_relu_dot=chunk_rows * width * 2 + width * width * 2 + chunk_rows * 16,
                                       source="profiles/r1_full_v6.md"),
                "whole_stage": {"achieved": s3_tflops, "frac": s3_tflops / peaks["bf16_sustained"],
                                "how": "algorithmic flops of S3 (E_c x 4 245 504) / S3 stage time (gather, 3 GEMMs, finish, compaction)"},
                "isolated_launch": {"shape": [m_chunk, 1024, 1024], "ms": iso_ms, "achieved": iso_tflops,
                                    "frac_of_burst_peak": iso_tflops / peaks["bf16_tflops"]}}

    cpu_baseline = None
    if world == 1 and not args.no_cpu_baseline:
        timing, units, wall = oracle_sample(args.cpu_baseline_particles)
        from synth.configs import load_calibration
        cal = load_calibration("pileup200")
        target = dict(n=cal["n_hits"], e_c=cal["n_cand_edges"], e_k=cal["n_kept_edges"])
        v, t_est = extrapolate_events_per_s(timing, units, target)
        cpu_baseline = {"value": v, "unit": "events/s", "cores": cpu_threads(), "kind": "oracle",
                        "sample": (f"oracle (fp64 NumPy) on the {args.cpu_baseline_particles}-particle pileup-50 event (same architecture; "
                                   f"{units['n']} hits, {units['e_c']} candidate, {units['e_k']} kept edges; {wall:.1f} s wall), per-stage "
                                   f"times scaled by unit counts to the pileup-200 event => {t_est:.0f} s/event"),
                        "stage_s": {k: round(v_, 3) for k, v_ in timing.items()}}

    line = {"metric": "events/s (pileup-200 event)", "value": events_per_s, "unit": "events/s", "n_gpus": world, "steps": args.steps,
            "warmup": warmup, "ms_per_step": total_ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "bf16", "data": "synthetic",
            "config": {"workload": args.config, "hits": n, "events_per_step": n_events, "cand_edges": e_c, "kept_edges": e_k,
                       "gnn_pass_edges": counts[2], "overflow": counts[3], "parallelism": f"replicas x{world}",
                       "l2": "256 MB buffer written between timed steps (L2 flush)", "precision": "bf16 operands, fp32 accumulate",
                       "workspace_gb": trk.workspace_bytes / 2 ** 30},
            "hits_per_s": events_per_s * n / n_events, "stage_ms": st, "stage_roofline": stage_roofline,
            "clocks": clocks, "e2e": e2e, "gpu_launches": launches, "roofline": roofline, "cpu_baseline": cpu_baseline}
    print(json.dumps(line))
    trk.close()
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
