"""Oracle-side calibration of the hyperparameters BASELINE.json leaves to "the oracle":
FRNN radius for a target mean out-degree D (post-cap, reading C-7), filter cut for a target
keep fraction f (reading C-11), plus two conveniences derived from oracle outputs only:
a PCA grid projection for the CUDA search structure (reading C-21; any orthonormal P gives the
same graph) and the median GNN logit (the "centred" variant of reading C-16).

Run as a script to (re)write synth/calibration.json:
    python -m oracle.calibrate toy pileup50 pileup200 pileup300
It calls only oracle/ and synth/ (never the CUDA path).
"""
from __future__ import annotations

import json
import sys
import time

import numpy as np

from . import s1_embed, s2_frnn, s3_filter, s4_gnn


def calibrate_radius(emb_f32, hits_f32, event_offsets, degree, K, r_start=0.25):
    """Smallest fp32 r with E_c(r)/N >= D where E_c counts emitted (post-cap) edges.

    One search at r_max >= r gives, per query, its K nearest outer neighbours inside r_max; for any
    r <= r_max the emitted edges are exactly those with d2 <= r^2, so E_c(r) is read off the sorted d2."""
    n = len(hits_f32)
    target = int(np.ceil(degree * n))
    r_max = np.float32(r_start)
    while True:
        _, _, _, d2 = s2_frnn.frnn(emb_f32, hits_f32, event_offsets, r_max, K, return_d2=True)
        if len(d2) >= int(target * 1.02) + 1 or r_max > 1e3:
            break
        r_max = np.float32(r_max * 1.3)
    d2 = np.sort(d2)
    if len(d2) < target:
        return float(r_max), len(d2)
    r = np.float32(np.sqrt(0.5 * (d2[target - 1] + d2[min(target, len(d2) - 1)])))
    while s2_frnn.radius_squared(r) < d2[target - 1]:        # fp32 rounding went below the target edge
        r = np.nextafter(r, np.float32(np.inf))
    count = int(np.searchsorted(d2, s2_frnn.radius_squared(r), side="right"))
    return float(r), count


def calibrate_cut(scores, keep_frac):
    """Midpoint between the ceil((1-f)E)-th smallest score and the next one, rounded to fp32."""
    s = np.sort(np.asarray(scores, np.float64))
    k = int(np.ceil((1.0 - keep_frac) * len(s)))
    k = min(max(k, 1), len(s) - 1)
    return float(np.float32(0.5 * (s[k - 1] + s[k])))


def pca_projection(emb_f32, g=3):
    """[d_e, g] orthonormal columns: the g leading principal axes of the embedding."""
    x = np.asarray(emb_f32, np.float64)
    x = x - x.mean(axis=0)
    w, v = np.linalg.eigh(x.T @ x / max(1, len(x)))
    p = v[:, ::-1][:, :min(g, x.shape[1])]
    return np.ascontiguousarray(p)


def calibrate_config(name, log=print):
    from synth.configs import get_config, make_events
    from synth.weights import make_model
    cfg = get_config(name)
    if len(cfg["seeds"]) != 1:
        raise ValueError("calibrate on single-event configs; the batch config reuses pileup50")
    t0 = time.time()
    ev = make_events(cfg)
    model = make_model(cfg)
    hits, off = ev["hits"], ev["event_offsets"]
    emb = s1_embed.embed_f32(hits, model["embed"])
    r, ec = calibrate_radius(emb, hits, off, cfg["degree"], cfg["frnn_k"])
    log(f"[{name}] N={len(hits)} r={r:.7f} E_c={ec} ({ec / len(hits):.3f}/hit) t={time.time() - t0:.0f}s")
    src, dst, _ = s2_frnn.frnn(emb, hits, off, r, cfg["frnn_k"])
    assert len(src) == ec
    feat = emb if cfg["filter_input"] == "emb" else hits
    fs = s3_filter.filter_scores(feat, src, dst, model["filter"])
    cut = calibrate_cut(fs, cfg["keep_frac"])
    keep = s3_filter.keep_mask(fs, cut)
    log(f"[{name}] cut={cut:.7f} E_k={int(keep.sum())} ({keep.mean():.4f}) t={time.time() - t0:.0f}s")
    logit = s4_gnn.gnn_forward(hits, src[keep], dst[keep], model, cfg["gnn_iters"])
    med = float(np.median(logit))
    log(f"[{name}] gnn logit median={med:.5f} frac>0={np.mean(logit > 0):.4f} t={time.time() - t0:.0f}s")
    proj = pca_projection(emb, 3)
    return dict(frnn_radius=r, filter_cut=cut, gnn_logit_median=med, grid_proj=[[float(v) for v in row] for row in proj],
                n_hits=int(len(hits)), n_cand_edges=int(ec), n_kept_edges=int(keep.sum()),
                n_gnn_pass=int(np.sum(logit > 0)))


def main(argv):
    from synth.configs import CALIBRATION_PATH
    names = argv or ["toy", "pileup50", "pileup200", "pileup300"]
    try:
        with open(CALIBRATION_PATH) as f:
            table = json.load(f)
    except FileNotFoundError:
        table = {}
    for name in names:
        table[name] = calibrate_config(name)
        with open(CALIBRATION_PATH, "w") as f:
            json.dump(table, f, indent=1, sort_keys=True)
            f.write("\n")


if __name__ == "__main__":
    main(sys.argv[1:])
