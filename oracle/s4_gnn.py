"""S4 interaction-network edge classifier ("The edge classification step uses
the interaction network [28]").  The paper gives no equations; BASELINE.json configs give
H, T and the edge features (dr, dphi, dz, deta).  The network below is reading C-12/C-13/C-14
of SURVEY.md section 8(c), restated in DESIGN.md:

  a_k   = (x_d0 - x_s0, wrap(x_d1 - x_s1) into (-1,1], x_d2 - x_s2, asinh(x_d2/x_d0) - asinh(x_s2/x_s0))
  LNR(v)= ReLU(LayerNorm(v))   (LayerNorm over the H outputs, biased variance, eps 1e-5, no affine;
                                plain ReLU when layernorm=False)
  h0_v  = LNR(W_n2 LNR(W_n1 x_v + b) + b)                              node_enc 3  -> H -> H
  e0_k  = LNR(W_e2 LNR(W_e1 a_k + b) + b)                              edge_enc 4  -> H -> H
  for t = 1..T (shared weights):
     e_k   <- e_k + LNR(W2 LNR(W1 [h_s ; h_d ; e_k] + b) + b)          edge_net 3H -> H -> H
     m_in_v = sum_{k: dst(k)=v} e_k ;  m_out_v = sum_{k: src(k)=v} e_k
     h_v   <- h_v + LNR(W2 LNR(W1 [h_v ; m_in_v ; m_out_v] + b) + b)   node_net 3H -> H -> H
  score_k = sigmoid( w_o2 . LNR(W_o1 [h_s ; h_d ; e_k] + b) + b )      edge_dec 3H -> H -> 1
"""
from __future__ import annotations

import numpy as np

from .mlp import layernorm, linear, relu, sigmoid


def edge_features(hits_f32, src, dst):
    x = np.asarray(hits_f32, np.float32).astype(np.float64)
    s, d = x[np.asarray(src, np.int64)], x[np.asarray(dst, np.int64)]
    dphi = d[:, 1] - s[:, 1]
    dphi = np.where(dphi > 1.0, dphi - 2.0, dphi)
    dphi = np.where(dphi <= -1.0, dphi + 2.0, dphi)
    deta = np.arcsinh(d[:, 2] / d[:, 0]) - np.arcsinh(s[:, 2] / s[:, 0])
    return np.stack([d[:, 0] - s[:, 0], dphi, d[:, 2] - s[:, 2], deta], axis=1)


def _act(v, layernorm_on):
    return relu(layernorm(v)) if layernorm_on else relu(v)


def _mlp2(x, mlp, layernorm_on):
    """Two Linear layers, both followed by LNR."""
    v = _act(linear(x, mlp["weight"][0], mlp["bias"][0]), layernorm_on)
    return _act(linear(v, mlp["weight"][1], mlp["bias"][1]), layernorm_on)


def scatter_sum(values, index, n):
    """out[v] = sum_{k: index[k]=v} values[k]  (the definition; numpy add.at)."""
    out = np.zeros((n, values.shape[1]), dtype=np.float64)
    np.add.at(out, np.asarray(index, np.int64), values)
    return out


def gnn_forward(hits_f32, src, dst, model, n_iters, layernorm_on=True, return_state=False):
    """Returns edge logits fp64 [E] (score = sigmoid(logit)); optionally (h, e) after T iterations."""
    x = np.asarray(hits_f32, np.float32).astype(np.float64)
    n = x.shape[0]
    src = np.asarray(src, np.int64)
    dst = np.asarray(dst, np.int64)
    h = _mlp2(x, model["node_enc"], layernorm_on)
    e = _mlp2(edge_features(hits_f32, src, dst), model["edge_enc"], layernorm_on)
    for _ in range(n_iters):
        e = e + _mlp2(np.concatenate([h[src], h[dst], e], axis=1), model["edge_net"], layernorm_on)
        m_in = scatter_sum(e, dst, n)
        m_out = scatter_sum(e, src, n)
        h = h + _mlp2(np.concatenate([h, m_in, m_out], axis=1), model["node_net"], layernorm_on)
    dec = model["edge_dec"]
    v = _act(linear(np.concatenate([h[src], h[dst], e], axis=1), dec["weight"][0], dec["bias"][0]), layernorm_on)
    logit = linear(v, dec["weight"][1], dec["bias"][1])[:, 0]
    if return_state:
        return logit, h, e
    return logit


def gnn_scores(hits_f32, src, dst, model, n_iters, layernorm_on=True):
    return sigmoid(gnn_forward(hits_f32, src, dst, model, n_iters, layernorm_on))
