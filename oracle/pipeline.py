"""The five stages in order, with fp32 interchange between stages
(each stage starts from the fp32 values the previous stage wrote)."""
from __future__ import annotations

import time

import numpy as np

from . import s1_embed, s2_frnn, s3_filter, s4_gnn, s5_cc
from .mlp import sigmoid


def run(cfg, model, calib, hits_f32, event_offsets, stages=5, timing=None, layernorm_on=True):
    """Returns dict of per-stage outputs.  `stages` = how many stages to run (1..5)."""
    out = {}
    t = time.perf_counter()

    def lap(name):
        nonlocal t
        now = time.perf_counter()
        if timing is not None:
            timing[name] = timing.get(name, 0.0) + now - t
        t = now

    hits_f32 = np.asarray(hits_f32, np.float32)
    n = hits_f32.shape[0]
    out["emb"] = s1_embed.embed_f32(hits_f32, model["embed"])
    lap("s1_embed")
    if stages < 2:
        return out
    src, dst, rowptr = s2_frnn.frnn(out["emb"], hits_f32, event_offsets, calib["frnn_radius"], cfg["frnn_k"])
    out.update(cand_src=src, cand_dst=dst, rowptr=rowptr)
    lap("s2_frnn")
    if stages < 3:
        return out
    feat = out["emb"] if cfg["filter_input"] == "emb" else hits_f32
    fs = s3_filter.filter_scores(feat, src, dst, model["filter"])
    out["filter_score"] = fs.astype(np.float32)
    keep = s3_filter.keep_mask(out["filter_score"], calib["filter_cut"])
    out.update(src=src[keep], dst=dst[keep])
    lap("s3_filter")
    if stages < 4:
        return out
    logit = s4_gnn.gnn_forward(hits_f32, out["src"], out["dst"], model, cfg["gnn_iters"], layernorm_on)
    out["gnn_logit"] = logit
    out["gnn_score"] = sigmoid(logit).astype(np.float32)
    lap("s4_gnn")
    if stages < 5:
        return out
    out["labels"] = s5_cc.connected_components(n, out["src"], out["dst"], out["gnn_score"], cfg["gnn_cut"])
    lap("s5_cc")
    return out
