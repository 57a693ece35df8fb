"""-m gpu: S6 track-candidate lists through the C ABI, bit-exact against oracle/s6_tracks."""
import numpy as np
import pytest

import gpu_common as G
from oracle import s5_cc, s6_tracks
from synth.events import generate_event, truth_edges

pytestmark = pytest.mark.gpu


def _dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _toy_trk(n):
    from paper_2501_05520_b200 import trk_from_config
    cfg = G.get_config("toy")
    cfg["precision"] = "fp32"
    calib = G.load_calibration("toy")
    return trk_from_config(cfg, G.centred_model(cfg, calib), calib, max_hits=max(n, 1), max_cand_edges=1024, max_kept_edges=1024)


def _check(trk, labels, min_hits, capacity=None):
    import torch
    n = len(labels)
    toff, thit, cnt = trk.stage_tracks(_dev(labels.astype(np.int32)) if n else torch.empty(0, dtype=torch.int32, device="cuda"),
                                       min_hits, capacity)
    torch.cuda.synchronize()
    ref_off, ref_hit = s6_tracks.build_tracks(labels, min_hits)
    T, nh, over = cnt.cpu().tolist()
    toff, thit = toff.cpu().numpy(), thit.cpu().numpy()
    cap = capacity if capacity is not None else max(n, 1)
    if len(ref_off) - 1 <= cap:
        assert over == 0 and T == len(ref_off) - 1 and nh == len(ref_hit)
        assert np.array_equal(toff[:T + 1], ref_off) and np.array_equal(thit[:nh], ref_hit)
    else:                                         # truncated deterministically to the first `cap` tracks
        assert over == 1 and T == cap and nh == ref_off[cap]
        assert np.array_equal(toff[:cap + 1], ref_off[:cap + 1]) and np.array_equal(thit[:nh], ref_hit[:nh])
    assert np.all(thit[nh:] == -1)
    return T, nh


def _random_labels(n, e, seed):
    rng = np.random.default_rng(seed)
    return s5_cc.labels_union_find(n, rng.integers(0, n, e), rng.integers(0, n, e))


@pytest.mark.parametrize("n,e", [(1, 0), (255, 100), (256, 300), (257, 90), (5000, 3500), (70001, 45000)])
def test_random_components(n, e):
    """Several radix passes (n > 65 536 needs three), blocks with a ragged tail, all minimum lengths."""
    trk = _toy_trk(n)
    try:
        lab = _random_labels(n, e, n)
        for m in (1, 2, 3, 7):
            _check(trk, lab, m)
    finally:
        trk.close()


def test_degenerate_label_sets():
    n = 3000
    trk = _toy_trk(n)
    try:
        _check(trk, np.zeros(n, np.int64), 3)                    # one giant component
        _check(trk, np.arange(n), 1)                             # all singletons, every one a track
        T, nh = _check(trk, np.arange(n), 2)                     # ... none long enough
        assert T == 0 and nh == 0
        _check(trk, np.zeros(0, np.int64), 3)                    # no hits
        lab = _random_labels(n, 2000, 7)
        ref_off, _ = s6_tracks.build_tracks(lab, 2)
        assert len(ref_off) - 1 > 10
        _check(trk, lab, 2, capacity=10)                         # more tracks than the caller's capacity
        _check(trk, lab, 2, capacity=len(ref_off) - 1)           # exactly enough
    finally:
        trk.close()


def test_truth_graph_tracks_are_particles():
    ev = generate_event(2500, 0.10, 4)
    n = len(ev["hits"])
    s, d = truth_edges(ev["particle_id"], ev["layer"], ev["hits"])
    lab = s5_cc.labels_union_find(n, s, d)
    trk = _toy_trk(n)
    try:
        import torch
        toff, thit, cnt = trk.stage_tracks(_dev(lab), 3)
        torch.cuda.synchronize()
        T, nh, _ = cnt.cpu().tolist()
        toff, thit = toff.cpu().numpy(), thit.cpu().numpy()
        pid = ev["particle_id"]
        assert not np.any(pid[thit[:nh]] < 0)
        for t in range(0, T, 37):
            seg = thit[toff[t]:toff[t + 1]]
            assert len(np.unique(pid[seg])) == 1 and np.array_equal(seg, np.flatnonzero(pid == pid[seg[0]]))
    finally:
        trk.close()


@pytest.mark.parametrize("name,precision", [("toy", "fp32"), ("pileup50", "bf16")])
def test_pipeline_tracks(name, precision):
    """trk_infer with track outputs and trk_infer_host_tracks: the lists are the oracle's S6 of the call's own labels."""
    import torch
    run = G.oracle_run(name, precision, stages=1)
    ev = run["ev"]
    trk = G.make_trk(run, min_track_hits=3)
    try:
        out = trk.infer(_dev(ev["hits"]), ev["event_offsets"], want_tracks=True)
        torch.cuda.synchronize()
        lab = out["labels"].cpu().numpy()
        ref_off, ref_hit = s6_tracks.build_tracks(lab, 3)
        T, nh = out["track_counts"].cpu().tolist()
        assert T == len(ref_off) - 1 and nh == len(ref_hit) and out["counts"].cpu().tolist()[3] == 0
        assert np.array_equal(out["track_offsets"].cpu().numpy()[:T + 1], ref_off)
        assert np.array_equal(out["track_hits"].cpu().numpy()[:nh], ref_hit)
        toff, thit, lab_h, counts = trk.infer_host_tracks(torch.from_numpy(ev["hits"]).pin_memory(), ev["event_offsets"])
        assert np.array_equal(lab_h, lab) and counts[4] == T and counts[5] == nh
        assert np.array_equal(toff, ref_off) and np.array_equal(thit, ref_hit)
    finally:
        trk.close()
