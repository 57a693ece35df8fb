"""S3 edge filter ("another MLP to filter out clearly fake edges ... A fixed
threshold is applied to these filtered edge scores").  BASELINE.json configs: 24->1024->1024->1024->1
on the two endpoint embeddings (pileup), 6->64->1 on the two raw feature rows (toy) -- reading
C-10; score = sigmoid(logit); keep iff score > cut (strict, reading C-11); order preserved."""
from __future__ import annotations

import numpy as np

from .mlp import mlp_forward, sigmoid


def filter_logits(feat_f32, src, dst, mlp, chunk=65536):
    """feat fp32 [N,u] (embedding or raw hits); u_edge = [feat[src] ; feat[dst]]."""
    feat = np.asarray(feat_f32, np.float32).astype(np.float64)
    src = np.asarray(src, np.int64)
    dst = np.asarray(dst, np.int64)
    out = np.empty(len(src), dtype=np.float64)
    for a in range(0, len(src), chunk):       # chunking bounds memory only; rows are independent
        u = np.concatenate([feat[src[a:a + chunk]], feat[dst[a:a + chunk]]], axis=1)
        out[a:a + chunk] = mlp_forward(u, mlp)[:, 0]
    return out


def filter_scores(feat_f32, src, dst, mlp):
    return sigmoid(filter_logits(feat_f32, src, dst, mlp))


def keep_mask(scores, cut_f32):
    """The decision is taken on the fp32 interchange value of the score against the fp32 cut."""
    return np.asarray(scores).astype(np.float32) > np.float32(cut_f32)
