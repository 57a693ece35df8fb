"""Pins for the oracle's dense layers, S1 and S3 (SURVEY.md section 8(c) "Pins / S1/S3 MLP")."""
import numpy as np
import torch

from oracle import mlp as om
from oracle import s1_embed, s3_filter
from synth.weights import make_mlp


def test_hand_computed_mlp():
    # 2 -> 2 -> 1 with integer weights, worked by hand:
    # x=(1,2): z1 = (1*1-1*2+0, 2*1+1*2-5) = (-1,-1) -> relu (0,0) -> y = 3*0-2*0+7 = 7
    # x=(3,1): z1 = (3-1, 6+1-5) = (2,2) -> y = 3*2-2*2+7 = 9
    m = dict(weight=[np.array([[1., -1.], [2., 1.]]), np.array([[3., -2.]])], bias=[np.array([0., -5.]), np.array([7.])])
    y = om.mlp_forward(np.array([[1., 2.], [3., 1.]]), m)
    assert np.array_equal(y, np.array([[7.], [9.]]))
    # identity weights pass positive inputs through, kill negative rows
    eye = dict(weight=[np.eye(3), np.eye(3)], bias=[np.zeros(3), np.zeros(3)])
    assert np.array_equal(om.mlp_forward(np.array([[1., 2., 3.], [-1., -2., -3.]]), eye), np.array([[1., 2., 3.], [0., 0., 0.]]))


def test_sigmoid_and_layernorm_closed_forms():
    assert om.sigmoid(0.0) == 0.5
    assert abs(om.sigmoid(np.log(3.0)) - 0.75) < 1e-15
    assert abs(om.sigmoid(-2.0) + om.sigmoid(2.0) - 1.0) < 1e-15
    # LayerNorm of a 2-vector (a,b): +-(delta/sqrt(delta^2+eps)), delta = (a-b)/2
    v = np.array([[3.0, 1.0]])
    d = 1.0
    assert np.allclose(om.layernorm(v), [[d / np.sqrt(d * d + 1e-5), -d / np.sqrt(d * d + 1e-5)]], atol=1e-15)
    x = np.random.default_rng(0).standard_normal((5, 64)) * 3 + 2
    y = om.layernorm(x)
    assert np.max(np.abs(y.mean(axis=1))) < 1e-14 and np.max(np.abs(y.var(axis=1) - x.var(axis=1) / (x.var(axis=1) + 1e-5))) < 1e-12
    t = torch.nn.functional.layer_norm(torch.from_numpy(x), (64,), eps=1e-5).numpy()   # library routine
    assert np.max(np.abs(y - t)) < 1e-12


def test_embed_matches_independent_fp64_library_evaluation():
    m = make_mlp(1, "embed", [3, 64, 64, 8], bf16=False)
    x = np.random.default_rng(1).uniform(-1, 1, (257, 3)).astype(np.float32)
    seq = []
    for l in range(3):
        lin = torch.nn.Linear(m["dims"][l], m["dims"][l + 1]).double()
        lin.weight.data = torch.from_numpy(m["weight"][l]).double()
        lin.bias.data = torch.from_numpy(m["bias"][l]).double()
        seq += [lin] + ([torch.nn.ReLU()] if l < 2 else [])
    ref = torch.nn.Sequential(*seq)(torch.from_numpy(x).double()).detach().numpy()
    out = s1_embed.embed(x, m)
    assert out.dtype == np.float64 and np.max(np.abs(out - ref)) < 1e-12
    assert s1_embed.embed_f32(x, m).dtype == np.float32
    # a transposed weight or a dropped bias must fail: check one entry by explicit loops
    h = x[5].astype(np.float64)
    for l in range(3):
        z = np.array([sum(float(m["weight"][l][o, i]) * h[i] for i in range(len(h))) + float(m["bias"][l][o])
                      for o in range(m["dims"][l + 1])])
        h = np.maximum(z, 0) if l < 2 else z
    assert np.max(np.abs(out[5] - h)) < 1e-12


def test_filter_concat_order_and_first_layer_split():
    rng = np.random.default_rng(2)
    m = make_mlp(2, "filter", [6, 16, 1], bf16=False)
    feat = rng.standard_normal((10, 3)).astype(np.float32)
    src = np.array([0, 1, 2, 9]); dst = np.array([3, 1, 7, 0])
    lg = s3_filter.filter_logits(feat, src, dst, m)
    w1 = m["weight"][0].astype(np.float64)
    f = feat.astype(np.float64)
    # W1 [u_s ; u_d] = W1a u_s + W1b u_d
    z = f[src] @ w1[:, :3].T + f[dst] @ w1[:, 3:].T + m["bias"][0]
    ref = np.maximum(z, 0) @ m["weight"][1].astype(np.float64).T + m["bias"][1]
    assert np.max(np.abs(lg - ref[:, 0])) < 1e-13
    # swapping src and dst changes the result (order of the concat matters)
    assert np.max(np.abs(s3_filter.filter_logits(feat, dst, src, m) - lg)) > 1e-3
    s = s3_filter.filter_scores(feat, src, dst, m)
    assert np.allclose(s, 1 / (1 + np.exp(-lg)))
    # strict inequality and fp32 decision
    assert list(s3_filter.keep_mask(np.array([0.5, 0.50000006, 0.4]), 0.5)) == [False, True, False]


def test_filter_chunking_is_invisible():
    rng = np.random.default_rng(3)
    m = make_mlp(3, "filter", [6, 8, 1], bf16=False)
    feat = rng.standard_normal((50, 3)).astype(np.float32)
    src = rng.integers(0, 50, 1000); dst = rng.integers(0, 50, 1000)
    assert np.max(np.abs(s3_filter.filter_logits(feat, src, dst, m, chunk=7) - s3_filter.filter_logits(feat, src, dst, m))) < 1e-13
