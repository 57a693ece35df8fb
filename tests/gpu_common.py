"""Shared helpers of the -m gpu parity tests: oracle runs (cached per session) and tolerances.

Tolerances (BASELINE.json north_star; derivations in DESIGN.md "Tolerances"):
  bf16 GEMMs : max abs diff 2e-2 on sigmoid scores; embedding max|d| / max|ref| <= 2e-2
  fp32       : 1e-4 relative on scores; embedding max|d| / max|ref| <= 1e-4
  edge lists : bit-exact;  labels: bit-exact given the same kept-edge set;
  a kept edge may differ only if its oracle score lies within the band of the cut.
"""
from __future__ import annotations

import functools

import numpy as np

import oracle
from oracle import pipeline as opipe
from synth.configs import get_config, load_calibration, make_events
from synth.weights import make_model

BAND = {"bf16": 2e-2, "fp32": 1e-4}
EMB_TOL = {"bf16": 2e-2, "fp32": 1e-4}


def centred_model(cfg, calib):
    """Reading C-16: the decoder's final bias is shifted by -median(oracle logit) so both sides of the 0.5 cut occur."""
    model = make_model(cfg)
    dec = model["edge_dec"]
    dec["bias"][1] = (dec["bias"][1].astype(np.float64) - calib["gnn_logit_median"]).astype(np.float32)
    return model


@functools.lru_cache(maxsize=None)
def oracle_run(name: str, precision: str | None = None, centred: bool = True, n_particles: int | None = None, stages: int = 5):
    cfg = get_config(name)
    if precision:
        cfg["precision"] = precision
    calib = load_calibration(cfg["calibration"])
    ev = make_events(cfg, n_particles=n_particles)
    model = centred_model(cfg, calib) if centred else make_model(cfg)
    timing = {}
    out = opipe.run(cfg, model, calib, ev["hits"], ev["event_offsets"], stages=stages, timing=timing)
    return dict(cfg=cfg, calib=calib, ev=ev, model=model, out=out, timing=timing)


def make_trk(run, **kw):
    from paper_2501_05520_b200 import trk_from_config
    cfg, ev = run["cfg"], run["ev"]
    n = len(ev["hits"])
    args = dict(max_hits=n, max_events=len(ev["event_offsets"]) - 1)
    args.update(kw)
    return trk_from_config(cfg, run["model"], run["calib"], **args)


def edge_keys(src, dst):
    return (np.asarray(src, np.int64) << 32) | np.asarray(dst, np.int64)


def check_scores(gpu, ref, precision, what):
    gpu = np.asarray(gpu, np.float64)
    ref = np.asarray(ref, np.float64)
    assert gpu.shape == ref.shape, what
    assert np.all(np.isfinite(gpu)), what
    if precision == "bf16":
        err = np.max(np.abs(gpu - ref)) if len(ref) else 0.0
        assert err <= 2e-2, f"{what}: max abs diff {err:.3e} > 2e-2"
    else:
        err = np.max(np.abs(gpu - ref) / np.maximum(ref, 1e-30)) if len(ref) else 0.0
        assert err <= 1e-4, f"{what}: max rel diff {err:.3e} > 1e-4"
    return err


def check_kept(gpu_keys, ref_keys, all_keys, ref_scores, cut, precision, what):
    """Kept sets may differ only on edges whose oracle score is within the band of the cut."""
    band = BAND[precision] if precision == "bf16" else 1e-4 * max(cut, 1e-6)
    diff = np.setxor1d(gpu_keys, ref_keys)
    if len(diff):
        pos = np.searchsorted(all_keys, diff)
        assert np.all(all_keys[pos] == diff), what
        worst = np.max(np.abs(np.asarray(ref_scores, np.float64)[pos] - cut))
        assert worst <= band, f"{what}: an edge {worst:.3e} from the cut flipped"
    return len(diff)


def same_track_fraction(labels_a, labels_b):
    """Per hit: is the set of hits that share its label the same in both labelings?  (reading C-22, informational.)
    The sets are equal iff the pair (label_a, label_b) occurs exactly |set_a| = |set_b| times."""
    a = np.asarray(labels_a, np.int64)
    b = np.asarray(labels_b, np.int64)
    n = len(a)
    size_a = np.bincount(a, minlength=n)[a]
    size_b = np.bincount(b, minlength=n)[b]
    _, inv, cnt = np.unique(a * n + b, return_inverse=True, return_counts=True)
    pair = cnt[inv]
    return (pair == size_a) & (pair == size_b)
