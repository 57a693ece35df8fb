"""-m gpu: empty / ragged / degenerate inputs, capacity overflow, error statuses, the literal (uncentred, LayerNorm-free)
models, stream concurrency and CUDA-graph capture -- all through the C ABI, expected values from the oracle."""
import numpy as np
import pytest

import gpu_common as G
from oracle import pipeline as opipe
from oracle import s2_frnn, s5_cc
from synth.events import generate_event

pytestmark = pytest.mark.gpu


def _dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _toy(precision="fp32", centred=True):
    cfg = G.get_config("toy")
    cfg["precision"] = precision
    calib = G.load_calibration("toy")
    model = G.centred_model(cfg, calib) if centred else G.make_model(cfg)
    return cfg, calib, model


def _make(cfg, calib, model, n, n_events=1, **kw):
    from paper_2501_05520_b200 import trk_from_config
    return trk_from_config(cfg, model, calib, max_hits=max(n, 1), max_events=max(n_events, 1), **kw)


def _ragged_batch():
    """Four events: 50 particles, EMPTY, one hit, 30 particles -- offsets with a repeated entry."""
    a = generate_event(50, 0.10, 0)["hits"]
    c = generate_event(30, 0.10, 5)["hits"]
    one = generate_event(3, 0.0, 9)["hits"][:1]
    hits = np.ascontiguousarray(np.concatenate([a, one, c]))
    off = np.array([0, len(a), len(a), len(a) + 1, len(a) + 1 + len(c)], np.int32)
    return hits, off


@pytest.mark.parametrize("precision", ["fp32", "bf16"])
def test_empty_call_and_empty_events(precision):
    import torch
    cfg, calib, model = _toy(precision)
    hits, off = _ragged_batch()
    n = len(hits)
    trk = _make(cfg, calib, model, n, 4)
    try:
        # no events at all
        res = trk.infer(torch.empty(0, 3, device="cuda"), np.array([0], np.int32))
        torch.cuda.synchronize()
        assert res["counts"].cpu().tolist() == [0, 0, 0, 0] and res["labels"].numel() == 0
        # one event with no hits
        res = trk.infer(torch.empty(0, 3, device="cuda"), np.array([0, 0], np.int32))
        torch.cuda.synchronize()
        assert res["counts"].cpu().tolist() == [0, 0, 0, 0]
        # ragged batch, stage by stage against the oracle
        ref = opipe.run(cfg, model, calib, hits, off)
        emb = trk.stage_embed(_dev(hits)).cpu().numpy()
        assert np.max(np.abs(emb - ref["emb"])) / np.max(np.abs(ref["emb"])) <= G.EMB_TOL[precision]
        src, dst, rowptr, cnt = trk.stage_frnn(_dev(ref["emb"]), _dev(hits), off)
        ec = int(cnt[0])
        assert ec == len(ref["cand_src"]) and np.array_equal(src[:ec].cpu().numpy(), ref["cand_src"])
        assert np.array_equal(dst[:ec].cpu().numpy(), ref["cand_dst"]) and np.array_equal(rowptr.cpu().numpy(), ref["rowptr"])
        lone = int(off[2])                                   # the single-hit event has no neighbour
        assert ref["rowptr"][lone + 1] == ref["rowptr"][lone]
        sc = trk.stage_gnn(_dev(hits), _dev(ref["src"]), _dev(ref["dst"])).cpu().numpy()
        G.check_scores(sc, ref["gnn_score"], precision, "gnn score (ragged batch)")
        lab = trk.stage_cc(n, _dev(ref["src"]), _dev(ref["dst"]), _dev(ref["gnn_score"]), cfg["gnn_cut"]).cpu().numpy()
        assert np.array_equal(lab, ref["labels"]) and lab[lone] == lone
        # the whole call: batch == each event alone + offset (BASELINE.json configs[3])
        res = trk.infer(_dev(hits), off, want_edges=True, want_cand=True)
        torch.cuda.synchronize()
        ec, ek = int(res["counts"][0]), int(res["counts"][1])
        cs, cd = res["cand_src"][:ec].cpu().numpy(), res["cand_dst"][:ec].cpu().numpy()
        labels = res["labels"].cpu().numpy()
        for b in (0, 3):
            lo, hi = int(off[b]), int(off[b + 1])
            one = trk.infer(_dev(hits[lo:hi]), np.array([0, hi - lo], np.int32), want_cand=True)
            torch.cuda.synchronize()
            e1 = int(one["counts"][0])
            m = (cs >= lo) & (cs < hi)
            assert np.array_equal(one["cand_src"][:e1].cpu().numpy() + lo, cs[m]) and np.array_equal(one["cand_dst"][:e1].cpu().numpy() + lo, cd[m])
            assert np.array_equal(one["labels"].cpu().numpy() + lo, labels[lo:hi])
    finally:
        trk.close()


@pytest.mark.parametrize("npart", [1, 3, 12, 19])
def test_ragged_sizes_big_architecture(npart):
    """The 1024-wide bf16 architecture on events far smaller than one 128-row tile, and just over one."""
    run = G.oracle_run("pileup50", "bf16", True, npart)
    o, ev, cfg = run["out"], run["ev"], run["cfg"]
    n = len(ev["hits"])
    trk = G.make_trk(run)
    try:
        emb = trk.stage_embed(_dev(ev["hits"])).cpu().numpy()
        assert np.max(np.abs(emb - o["emb"])) / np.max(np.abs(o["emb"])) <= G.EMB_TOL["bf16"]
        src, dst, _, cnt = trk.stage_frnn(_dev(o["emb"]), _dev(ev["hits"]), ev["event_offsets"])
        ec = int(cnt[0])
        assert ec == len(o["cand_src"]) and np.array_equal(dst[:ec].cpu().numpy(), o["cand_dst"])
        if ec:
            fs = trk.stage_filter(_dev(o["emb"]), _dev(o["cand_src"]), _dev(o["cand_dst"])).cpu().numpy()
            G.check_scores(fs, o["filter_score"], "bf16", "filter score")
        if len(o["src"]):
            sc = trk.stage_gnn(_dev(ev["hits"]), _dev(o["src"]), _dev(o["dst"])).cpu().numpy()
            G.check_scores(sc, o["gnn_score"], "bf16", "gnn score")
        lab = trk.stage_cc(n, _dev(o["src"]), _dev(o["dst"]), _dev(o["gnn_score"]), cfg["gnn_cut"]).cpu().numpy()
        assert np.array_equal(lab, o["labels"])
    finally:
        trk.close()


@pytest.mark.parametrize("k,radius", [(1, None), (128, 1e9), (16, 0.0), (5, 2.0)])
def test_frnn_degenerate_caps_and_radii(k, radius):
    """K = 1 (nearest outer neighbour), r = inf with K >= N-1 (every pair once), r = 0 (no edge), a cap that always bites."""
    cfg, calib, model = _toy()
    ev = generate_event(10, 0.1, 3)                 # ~80 hits: out-degree <= N-1 < 128
    hits = ev["hits"]
    n = len(hits)
    off = np.array([0, n], np.int32)
    emb = G.oracle_run("toy", "fp32")["out"]["emb"][:n].copy()      # any fp32 table will do as the latent space
    cfg = dict(cfg, frnn_k=k)
    calib = dict(calib, frnn_radius=calib["frnn_radius"] if radius is None else radius)
    osrc, odst, orow = s2_frnn.frnn_brute(emb, hits, off, calib["frnn_radius"], k)
    trk = _make(cfg, calib, model, n)
    try:
        src, dst, rowptr, cnt = trk.stage_frnn(_dev(emb), _dev(hits), off)
        ec = int(cnt[0])
        assert ec == len(osrc) and np.array_equal(src[:ec].cpu().numpy(), osrc) and np.array_equal(dst[:ec].cpu().numpy(), odst)
        assert np.array_equal(rowptr.cpu().numpy(), orow)
        if radius == 1e9:
            assert ec == n * (n - 1) // 2
        if radius == 0.0:
            assert ec == 0
    finally:
        trk.close()


@pytest.mark.parametrize("scale", [1.0, 1.0e3, 1.0e-3])
def test_frnn_projection_slack_scales_with_the_data(scale):
    """The fp32 projection P^T e used for binning and for the level-0 pre-filter is inexact; its slack must scale with |e|
    (it is taken from max|e| on the device).  An embedding offset far from the origin and scaled by 1e3 / 1e-3, searched with a
    rotated (non-axis-aligned) orthonormal grid_proj, must still give the oracle's brute-force edge list bit for bit."""
    run = G.oracle_run("pileup50", "bf16", True, 300)
    cfg, calib, ev = run["cfg"], run["calib"], run["ev"]
    hits = ev["hits"]
    n = len(hits)
    off = ev["event_offsets"]
    emb = ((run["out"]["emb"].astype(np.float64) + 37.0) * scale).astype(np.float32)   # |e| ~ 40 scale, neighbours ~0.3 scale apart
    r = np.float32(calib["frnn_radius"] * scale)
    d_e = emb.shape[1]
    rng = np.random.default_rng(5)
    q, _ = np.linalg.qr(rng.standard_normal((d_e, d_e)))
    proj = q[:, :3].astype(np.float32)
    osrc, odst, orow = s2_frnn.frnn_brute(emb, hits, off, r, cfg["frnn_k"])
    assert len(osrc) > 2 * n                                   # a real graph, with the cap biting somewhere
    from paper_2501_05520_b200 import Trk
    trk = Trk(model=run["model"], precision="bf16", frnn_radius=float(r), frnn_k=cfg["frnn_k"], filter_input=cfg["filter_input"],
              filter_cut=calib["filter_cut"], gnn_hidden=cfg["gnn_hidden"], gnn_iters=cfg["gnn_iters"], gnn_cut=cfg["gnn_cut"],
              max_hits=n, grid_proj=proj)
    try:
        src, dst, rowptr, cnt = trk.stage_frnn(_dev(emb), _dev(hits), off)
        ec = int(cnt[0])
        assert int(cnt[1]) == 0 and ec == len(osrc), (ec, len(osrc))
        assert np.array_equal(src[:ec].cpu().numpy(), osrc) and np.array_equal(dst[:ec].cpu().numpy(), odst)
        assert np.array_equal(rowptr.cpu().numpy(), orow)
    finally:
        trk.close()


@pytest.mark.parametrize("width,input_kind", [(256, "raw"), (512, "emb"), (768, "raw")])
def test_fused_filter_kernel_other_shapes(width, input_kind):
    """The fused S3 kernel (filter_fused.cuh) on shapes other than 24 -> 1024^3 -> 1: 1, 2 and 3 column tiles per layer, an odd
    endpoint width (u = 3 raw features, so an operand pair straddles the src | dst boundary) and u = 8 latent features, on a
    ragged number of edges; every score against the oracle, and against the layer-by-layer path."""
    import torch
    from oracle import s3_filter
    cfg, calib, _ = _toy("bf16")
    cfg = dict(cfg, filter_input=input_kind)
    u = 3 if input_kind == "raw" else cfg["embed_dims"][-1]
    cfg["filter_dims"] = [2 * u, width, width, width, 1]
    model = G.make_model(cfg)
    ev = generate_event(120, 0.1, 11)
    hits = ev["hits"]
    n = len(hits)
    rng = np.random.default_rng(1)
    e = 5 * 256 + 77                                            # several row blocks and a ragged tail
    src = rng.integers(0, n, e).astype(np.int32)
    dst = rng.integers(0, n, e).astype(np.int32)
    feat = hits if input_kind == "raw" else rng.standard_normal((n, u)).astype(np.float32)
    ref = s3_filter.filter_scores(feat, src, dst, model["filter"]).astype(np.float32)
    trk = _make(cfg, calib, model, n, max_cand_edges=e)
    try:
        fused = trk.stage_filter(_dev(feat), _dev(src), _dev(dst)).clone()
        trk.set_option("filter_fused", 0)
        layered = trk.stage_filter(_dev(feat), _dev(src), _dev(dst)).clone()
        torch.cuda.synchronize()
        G.check_scores(fused.cpu().numpy(), ref, "bf16", f"fused filter score (W = {width}, {input_kind})")
        G.check_scores(layered.cpu().numpy(), ref, "bf16", "layer-by-layer filter score")
        assert float((fused - layered).abs().max()) < 2e-3
    finally:
        trk.close()


def test_capacity_overflow_is_flagged_and_deterministic():
    import torch
    run = G.oracle_run("toy", "fp32")
    cfg, calib, ev = run["cfg"], run["calib"], run["ev"]
    hits, off = ev["hits"], ev["event_offsets"]
    n = len(hits)
    full = G.make_trk(run)
    small = G.make_trk(run, max_kept_edges=100)
    tiny_cand = G.make_trk(run, max_cand_edges=500)
    try:
        ref = full.infer(_dev(hits), off, want_edges=True, want_cand=True)
        torch.cuda.synchronize()
        ec, ek = int(ref["counts"][0]), int(ref["counts"][1])
        assert ek > 100 and ec > 500 and int(ref["counts"][3]) == 0
        # S3 capacity: the first 100 kept edges in (src,dst) order survive; labels are the components of that graph
        res = small.infer(_dev(hits), off, want_edges=True)
        torch.cuda.synchronize()
        c = res["counts"].cpu().tolist()
        assert c[3] == 1 and c[1] == 100 and c[0] == ec
        es, ed, sc = (res[k][:100].cpu().numpy() for k in ("edge_src", "edge_dst", "edge_score"))
        assert np.array_equal(es, ref["edge_src"][:100].cpu().numpy()) and np.array_equal(ed, ref["edge_dst"][:100].cpu().numpy())
        assert np.array_equal(res["labels"].cpu().numpy(), s5_cc.connected_components(n, es, ed, sc, cfg["gnn_cut"]))
        # S2 capacity: the candidate list is cut after 500 edges
        res = tiny_cand.infer(_dev(hits), off, want_cand=True)
        torch.cuda.synchronize()
        c = res["counts"].cpu().tolist()
        assert c[3] == 1 and c[0] == 500
        assert np.array_equal(res["cand_src"][:500].cpu().numpy(), ref["cand_src"][:500].cpu().numpy())
        assert np.array_equal(res["cand_dst"][:500].cpu().numpy(), ref["cand_dst"][:500].cpu().numpy())
        # an output buffer smaller than the result: flagged, nothing written past it
        out = {"labels": torch.empty(n, dtype=torch.int32, device="cuda"), "counts": torch.zeros(4, dtype=torch.int32, device="cuda"),
               "edge_src": torch.full((ek,), -7, dtype=torch.int32, device="cuda"), "edge_dst": torch.full((ek,), -7, dtype=torch.int32, device="cuda"),
               "edge_score": torch.zeros(ek, device="cuda")}
        view = dict(out, edge_src=out["edge_src"][:50], edge_dst=out["edge_dst"][:50], edge_score=out["edge_score"][:50])
        full.infer(_dev(hits), off, out=view)
        torch.cuda.synchronize()
        assert int(view["counts"][3]) == 1 and torch.all(out["edge_src"][50:] == -7)
        assert torch.equal(out["edge_src"][:50], ref["edge_src"][:50])
    finally:
        full.close(); small.close(); tiny_cand.close()


def test_error_statuses_enqueue_nothing():
    import torch
    from paper_2501_05520_b200 import TrkError
    cfg, calib, model = _toy()
    trk = _make(cfg, calib, model, 100, 2)
    hits = torch.zeros(200, 3, device="cuda")
    try:
        # a valid call first: the launch counter is non-zero and the outputs hold real values
        out = trk.infer(hits[:60] + 0.5, np.array([0, 60], np.int32), want_edges=True)
        torch.cuda.synchronize()
        assert trk.last_launch_count > 0
        sentinel = -123456789
        for t in (out["labels"], out["counts"], out["edge_src"], out["edge_dst"]):
            t.fill_(sentinel)
        out["edge_score"].fill_(-7.5)
        torch.cuda.synchronize()
        for off, status in (([0, 200], 3), ([0, 50, 40], 1), ([1, 50], 1), ([0, 10, 20, 30], 3)):
            with pytest.raises(TrkError) as e:
                trk.infer(hits, np.array(off, np.int32), out=out)
            assert e.value.status == status, (off, e.value.status)
            # include/trk.h: "Host-detectable errors return before anything is enqueued": no launch was counted ...
            assert trk.last_launch_count == 0, (off, trk.last_launch_count)
        # ... and nothing ran on the device: every output still holds the sentinel
        torch.cuda.synchronize()
        for k in ("labels", "counts", "edge_src", "edge_dst"):
            assert bool((out[k] == sentinel).all()), k
        assert bool((out["edge_score"] == -7.5).all())
        with pytest.raises(TrkError):
            trk.stage_embed(hits)                                 # 200 rows > max_hits
        # the context is still usable afterwards
        res = trk.infer(hits[:60] + 0.5, np.array([0, 60], np.int32))
        torch.cuda.synchronize()
        assert int(res["counts"][3]) == 0
    finally:
        trk.close()
    bad = dict(cfg, gnn_hidden=48)                               # bf16 needs H in {64,128}
    bad["precision"] = "bf16"
    with pytest.raises(TrkError) as e:
        _make(bad, calib, G.make_model(bad), 100)
    assert e.value.status == 2


@pytest.mark.parametrize("precision", ["fp32", "bf16"])
def test_literal_model_uncentred_and_without_layernorm(precision):
    """Reading C-16 (the literal 0.5 cut with random weights) and C-13 (gnn_layernorm = 0: the ReLU-only network)."""
    run = G.oracle_run("toy", precision, False)                  # uncentred decoder bias
    o, ev, cfg = run["out"], run["ev"], run["cfg"]
    hits = ev["hits"]
    n = len(hits)
    trk = G.make_trk(run)
    try:
        sc = trk.stage_gnn(_dev(hits), _dev(o["src"]), _dev(o["dst"])).cpu().numpy()
        G.check_scores(sc, o["gnn_score"], precision, "gnn score (literal)")
        lab = trk.stage_cc(n, _dev(o["src"]), _dev(o["dst"]), _dev(o["gnn_score"]), cfg["gnn_cut"]).cpu().numpy()
        assert np.array_equal(lab, o["labels"])
    finally:
        trk.close()
    if precision == "fp32":
        from oracle import s4_gnn
        from oracle.mlp import sigmoid
        logit = s4_gnn.gnn_forward(hits, o["src"], o["dst"], run["model"], cfg["gnn_iters"], layernorm_on=False)
        with np.errstate(over="ignore"):
            ref = sigmoid(logit)
        trk = G.make_trk(run, gnn_layernorm=False)
        try:
            sc = trk.stage_gnn(_dev(hits), _dev(o["src"]), _dev(o["dst"])).cpu().numpy().astype(np.float64)
            # without normalisation the logits are huge (the fp32 error of a logit scales with the largest one) and nearly
            # all scores saturate: scores agree absolutely except where the logit is within 1e-5 of that scale of zero
            scale = np.max(np.abs(logit))
            assert scale > 1e3
            bad = np.abs(sc - ref) > 1e-4
            assert np.all(np.abs(logit[bad]) <= 1e-5 * scale) and np.mean(bad) < 0.02
            solid = np.abs(logit) > 1e-5 * scale
            assert np.array_equal(sc[solid] > 0.5, ref[solid] > 0.5)
        finally:
            trk.close()


def test_two_contexts_on_two_streams_and_graph_replay():
    """Several model instances on several streams give the results of a lone call, bit for bit,
    and trk_infer can be captured into a CUDA graph (include/trk.h: never allocates, never synchronises)."""
    import torch
    run = G.oracle_run("pileup50", "bf16", True, 600)
    ev = run["ev"]
    hits, off = _dev(ev["hits"]), ev["event_offsets"]
    a, b = G.make_trk(run), G.make_trk(run)
    try:
        ref = a.infer(hits, off, want_edges=True)
        torch.cuda.synchronize()
        ek = int(ref["counts"][1])
        ref = {k: v.clone() for k, v in ref.items()}
        s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
        outs = []
        for _ in range(3):
            with torch.cuda.stream(s1):
                ra = a.infer(hits, off, want_edges=True, stream=s1)
            with torch.cuda.stream(s2):
                rb = b.infer(hits, off, want_edges=True, stream=s2)
            outs += [ra, rb]
        torch.cuda.synchronize()
        for r in outs:
            assert torch.equal(r["labels"], ref["labels"]) and torch.equal(r["counts"], ref["counts"])
            assert torch.equal(r["edge_score"][:ek], ref["edge_score"][:ek])
        # CUDA graph: capture one call, replay it twice on fresh inputs of the same size
        out = a.infer(hits, off, want_edges=True)
        torch.cuda.synchronize()
        g = torch.cuda.CUDAGraph()
        cap = torch.cuda.Stream()
        with torch.cuda.stream(cap):
            with torch.cuda.graph(g, stream=cap):
                a.infer(hits, off, out=out, stream=cap)
        for _ in range(2):
            out["labels"].fill_(-1)
            out["counts"].zero_()
            g.replay()
            torch.cuda.synchronize()
            assert torch.equal(out["labels"], ref["labels"]) and torch.equal(out["counts"], ref["counts"])
    finally:
        a.close(); b.close()


def test_infer_host_equals_infer():
    import torch
    run = G.oracle_run("toy", "bf16")
    ev = run["ev"]
    trk = G.make_trk(run)
    try:
        ref = trk.infer(_dev(ev["hits"]), ev["event_offsets"])
        torch.cuda.synchronize()
        hh = torch.from_numpy(ev["hits"]).pin_memory()
        lab, cnt = trk.infer_host(hh, ev["event_offsets"])
        assert np.array_equal(lab, ref["labels"].cpu().numpy()) and np.array_equal(cnt, ref["counts"].cpu().numpy())
    finally:
        trk.close()


def test_dispatcher_two_replicas_serve_four_different_events():
    """SURVEY.md section 8(f) NEXT-4 on one GPU: two model instances on device 0 behind the Dispatcher serve four DIFFERENT
    events concurrently (one host thread per replica) and return, in request order, exactly what one context returns."""
    from paper_2501_05520_b200.replicas import Dispatcher
    cfg = G.get_config("pileup50")
    calib = G.load_calibration("pileup50")
    model = G.centred_model(cfg, calib)
    events = []
    for seed in (3, 4, 5, 6):
        ev = G.make_events(dict(cfg, seeds=[seed]), n_particles=300 + 50 * seed)
        events.append((ev["hits"], ev["event_offsets"]))
    max_hits = max(len(h) for h, _ in events)
    disp = Dispatcher.from_devices(cfg, model, calib, max_hits=max_hits, devices=[0], instances_per_device=2)
    from paper_2501_05520_b200 import trk_from_config
    single = trk_from_config(cfg, model, calib, max_hits=max_hits)
    try:
        assert disp.assignment(4) == [[0, 2], [1, 3]]
        res = disp.serve(events)
        assert len(res) == 4
        for (hits, off), (labels, counts) in zip(events, res):
            want_labels, want_counts = single.infer_host(hits, off)
            assert np.array_equal(labels, want_labels) and np.array_equal(counts, want_counts)
            assert counts[3] == 0 and counts[0] > counts[1] > 0 and len(np.unique(labels)) < len(hits)
        assert len({len(r[0]) for r in res}) == 4                     # four different events indeed
    finally:
        disp.close()
        single.close()
