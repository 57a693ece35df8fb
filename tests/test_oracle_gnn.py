"""Pins for the oracle's S4 (SURVEY.md section 8(c) "Pins / S4 GNN")."""
import numpy as np

from oracle import s4_gnn
from oracle.mlp import sigmoid
from synth.weights import make_mlp


def _model(seed, H):
    return dict(node_enc=make_mlp(seed, "node_enc", [3, H, H], False), edge_enc=make_mlp(seed, "edge_enc", [4, H, H], False),
                edge_net=make_mlp(seed, "edge_net", [3 * H, H, H], False), node_net=make_mlp(seed, "node_net", [3 * H, H, H], False),
                edge_dec=make_mlp(seed, "edge_dec", [3 * H, H, 1], False))


def _graph(n, e, seed):
    rng = np.random.default_rng(seed)
    hits = np.stack([rng.integers(1, 6, n) / 10.0, rng.uniform(-1, 1, n), rng.uniform(-1, 1, n)], 1).astype(np.float32)
    return hits, rng.integers(0, n, e).astype(np.int32), rng.integers(0, n, e).astype(np.int32)


def test_edge_features_closed_forms():
    hits = np.array([[0.1, 0.9, 0.2], [0.2, -0.9, 0.4], [0.3, 0.5, -0.3], [0.5, -0.5, 0.5]], dtype=np.float32)
    a = s4_gnn.edge_features(hits, [0, 1, 2, 0], [1, 0, 3, 0])
    h = hits.astype(np.float64)
    # dphi wraps across +-1 (phi/pi units): -0.9 - 0.9 = -1.8 -> +0.2 ; 0.9 + 0.9 = 1.8 -> -0.2
    assert abs(a[0, 1] - (h[1, 1] - h[0, 1] + 2.0)) < 1e-15 and abs(a[0, 1] - 0.2) < 1e-6
    assert abs(a[1, 1] + 0.2) < 1e-6 and a[2, 1] == 1.0       # -0.5 - 0.5 = -1 -> +1 (range (-1, 1])
    assert abs(a[0, 0] - (h[1, 0] - h[0, 0])) < 1e-15 and abs(a[0, 2] - (h[1, 2] - h[0, 2])) < 1e-15
    # deta = 0 for equal z/r (hits 0 and 1 have z/r = 2 up to fp32 rounding of the inputs)
    assert abs(a[0, 3] - (np.arcsinh(h[1, 2] / h[1, 0]) - np.arcsinh(h[0, 2] / h[0, 0]))) < 1e-15 and abs(a[0, 3]) < 1e-6
    # eta of a hit at z/r = 1: asinh(1) = ln(1+sqrt 2)
    assert abs(a[2, 3] - (np.arcsinh(1.0) - np.arcsinh(-1.0))) < 1e-6
    assert np.all(a[3] == 0.0)
    # wrap maps exactly -1 to +1 (range (-1, 1])
    hw = np.array([[0.1, 0.5, 0.0], [0.1, -0.5, 0.0]], dtype=np.float32)
    assert s4_gnn.edge_features(hw, [0], [1])[0, 1] == 1.0 and s4_gnn.edge_features(hw, [1], [0])[0, 1] == 1.0


def test_hand_computed_4_node_graph_integer_weights_no_layernorm():
    """4 nodes, 3 edges, H=2, T=1, LayerNorm off, integer weights: worked by hand below."""
    hits = np.array([[1, 0, 1], [2, 0, 0], [1, 0, -1], [3, 0, 3]], dtype=np.float32)   # (r, phi, z)
    src = np.array([0, 1, 0]); dst = np.array([1, 3, 2])
    I2 = np.eye(2)
    z2 = np.zeros(2)
    model = dict(
        node_enc=dict(weight=[np.array([[1., 0, 0], [0, 0, 1.]]), I2], bias=[z2, z2]),           # h0 = relu((r, z))
        edge_enc=dict(weight=[np.array([[1., 0, 0, 0], [0, 0, 1., 0]]), I2], bias=[z2, z2]),     # e0 = relu((dr, dz))
        edge_net=dict(weight=[np.array([[1., 0, 0, 0, 0, 0], [0, 0, 0, 1., 0, 1.]]), I2], bias=[z2, z2]),  # (h_s[0], h_d[1]+e[1])
        node_net=dict(weight=[np.array([[0, 0, 1., 0, 0, 0], [0, 0, 0, 0, 1., 1.]]), I2], bias=[z2, z2]),  # (m_in[0], m_out[0]+m_out[1])
        edge_dec=dict(weight=[np.array([[1., 0, 0, 0, 0, 0], [0, 0, 0, 1., 0, 0]]), np.array([[1., -1.]])], bias=[z2, np.array([0.5])]),
    )
    # h0 = relu(r,z): n0 (1,1) n1 (2,0) n2 (1,0) n3 (3,3)
    # e0 = relu(dr,dz): k0 0->1 (1,0)   k1 1->3 (1,3)   k2 0->2 (0,0)
    # edge update: e += (h_s[0], h_d[1]+e[1]) : k0 (1,0)+(1,0+0)=(2,0); k1 (1,3)+(2,3+3)=(3,9); k2 (0,0)+(1,0+0)=(1,0)
    # m_in: n1=(2,0) n3=(3,9) n2=(1,0) n0=0 ; m_out: n0=(2,0)+(1,0)=(3,0), n1=(3,9)
    # node update: h += (m_in[0], m_out[0]+m_out[1]): n0 (1,1)+(0,3)=(1,4); n1 (2,0)+(2,12)=(4,12); n2 (1,0)+(1,0)=(2,0); n3 (3,3)+(3,0)=(6,3)
    # decoder: v = relu(h_s[0], h_d[1]); logit = v0 - v1 + 0.5: k0 1-12+.5=-10.5; k1 4-3+.5=1.5; k2 1-0+.5=1.5
    logit, h, e = s4_gnn.gnn_forward(hits, src, dst, model, 1, layernorm_on=False, return_state=True)
    assert np.array_equal(e, np.array([[2., 0], [3, 9], [1, 0]]))
    assert np.array_equal(h, np.array([[1., 4], [4, 12], [2, 0], [6, 3]]))
    assert np.array_equal(logit, np.array([-10.5, 1.5, 1.5]))
    assert np.allclose(s4_gnn.gnn_scores(hits, src, dst, model, 1, False), sigmoid(np.array([-10.5, 1.5, 1.5])))


def test_hand_computed_layernorm_h2():
    """H=2: LayerNorm of (a,b) = +-(d/sqrt(d^2+eps)), d=(a-b)/2; after ReLU one component survives."""
    hits = np.array([[1, 0, 3], [2, 0, 1]], dtype=np.float32)
    I2 = np.eye(2); z2 = np.zeros(2)
    ne = dict(weight=[np.array([[1., 0, 0], [0, 0, 1.]]), I2], bias=[z2, z2])
    zero3 = dict(weight=[np.zeros((2, 6)), np.zeros((2, 2))], bias=[z2, z2])
    model = dict(node_enc=ne, edge_enc=dict(weight=[np.zeros((2, 4)), I2], bias=[z2, z2]), edge_net=zero3, node_net=zero3,
                 edge_dec=dict(weight=[np.array([[1., 0, 0, 0, 0, 0], [0, 1., 0, 0, 0, 0]]), np.array([[1., 1.]])], bias=[z2, np.zeros(1)]))
    _, h, e = s4_gnn.gnn_forward(hits, [0], [1], model, 0, layernorm_on=True, return_state=True)
    eps = 1e-5
    f = lambda a, b: np.maximum(np.array([(a - b) / 2, (b - a) / 2]) / np.sqrt(((a - b) / 2) ** 2 + eps), 0)
    l1 = [f(1., 3.), f(2., 1.)]
    want = np.array([f(*l1[0]), f(*l1[1])])
    assert np.allclose(h, want, atol=1e-15) and h[0, 1] > 0.99 and h[0, 0] == 0 and h[1, 0] > 0.99
    assert np.array_equal(e, np.zeros((1, 2)))            # LN(0) = 0/sqrt(eps) = 0


def test_zero_update_weights_keep_states_and_empty_graph():
    H = 8
    m = _model(0, H)
    hits, src, dst = _graph(20, 50, 0)
    for k in ("edge_net", "node_net"):
        m[k] = dict(weight=[np.zeros_like(w) for w in m[k]["weight"]], bias=[np.zeros_like(b) for b in m[k]["bias"]])
    _, h0, e0 = s4_gnn.gnn_forward(hits, src, dst, m, 0, return_state=True)
    _, h3, e3 = s4_gnn.gnn_forward(hits, src, dst, m, 3, return_state=True)
    assert np.array_equal(h0, h3) and np.array_equal(e0, e3)
    lg, h, e = s4_gnn.gnn_forward(hits, src[:0], dst[:0], _model(0, H), 2, return_state=True)
    assert lg.shape == (0,) and e.shape == (0, H) and h.shape == (20, H) and np.all(np.isfinite(h))


def test_scatter_conservation_and_duplicate_edge():
    rng = np.random.default_rng(0)
    vals = rng.standard_normal((40, 5))
    idx = rng.integers(0, 7, 40)
    out = s4_gnn.scatter_sum(vals, idx, 7)
    assert np.allclose(out.sum(axis=0), vals.sum(axis=0), atol=1e-13)
    for v in range(7):
        assert np.allclose(out[v], vals[idx == v].sum(axis=0), atol=1e-13)
    # duplicating an edge doubles its message: node 1 receives e twice
    hits, _, _ = _graph(4, 0, 1)
    m = _model(1, 4)
    for k in ("edge_net",):
        m[k] = dict(weight=[np.zeros_like(w) for w in m[k]["weight"]], bias=[np.zeros_like(b) for b in m[k]["bias"]])
    m["node_net"]["weight"][0][:, :] = 0
    m["node_net"]["weight"][0][:, 4:8] = np.eye(4)            # reads m_in only
    _, h1, e1 = s4_gnn.gnn_forward(hits, [0], [1], m, 1, layernorm_on=False, return_state=True)
    _, h2, e2 = s4_gnn.gnn_forward(hits, [0, 0], [1, 1], m, 1, layernorm_on=False, return_state=True)
    _, h0, _ = s4_gnn.gnn_forward(hits, [0], [1], m, 0, layernorm_on=False, return_state=True)
    b1 = m["node_net"]["bias"][0].astype(np.float64)
    w2, b2 = m["node_net"]["weight"][1].astype(np.float64), m["node_net"]["bias"][1].astype(np.float64)
    upd = lambda msg: np.maximum(np.maximum(msg + b1, 0) @ w2.T + b2, 0)
    assert np.allclose(h1[1] - h0[1], upd(e1[0]), atol=1e-13) and np.allclose(h2[1] - h0[1], upd(2 * e1[0]), atol=1e-13)


def test_node_and_edge_permutation_equivariance():
    """BASELINE.json north_star: permutation equivariance under hit shuffling, to 1e-12."""
    H = 16
    m = _model(3, H)
    hits, src, dst = _graph(60, 300, 3)
    lg, h, e = s4_gnn.gnn_forward(hits, src, dst, m, 3, return_state=True)
    rng = np.random.default_rng(9)
    perm = rng.permutation(60)                    # new node p is old node perm[p]
    inv = np.argsort(perm)
    eperm = rng.permutation(300)
    lg2, h2, e2 = s4_gnn.gnn_forward(hits[perm], inv[src][eperm], inv[dst][eperm], m, 3, return_state=True)
    assert np.max(np.abs(lg2 - lg[eperm])) < 1e-12 and np.max(np.abs(h2 - h[perm])) < 1e-12 and np.max(np.abs(e2 - e[eperm])) < 1e-12
    # direction matters: reversing edges changes the scores
    lg3 = s4_gnn.gnn_forward(hits, dst, src, m, 3)
    assert np.max(np.abs(lg3 - lg)) > 1e-3


def test_layernorm_keeps_states_bounded():
    """Reading C-13: with LayerNorm the residual stream grows at most linearly in T."""
    H = 32
    m = _model(5, H)
    hits, src, dst = _graph(200, 1600, 5)
    _, h, e = s4_gnn.gnn_forward(hits, src, dst, m, 8, return_state=True)
    assert np.max(np.abs(h)) < 9 * np.sqrt(H) and np.max(np.abs(e)) < 9 * np.sqrt(H)


# ---------------------------------------------------------------------------------------------------------------------
# LayerNorm-on pins with H = 2 (SURVEY.md section 8(c) "Pins / S4 GNN"; reading C-13: LN after every GNN Linear except
# the final logit).  For a 2-vector (a, b): mean (a+b)/2, deviations +-(a-b)/2, biased variance ((a-b)/2)^2, so
# ReLU(LayerNorm((a, b))) = (g(d), 0) if d = (a-b)/2 > 0 else (0, g(-d)) with g(d) = d / sqrt(d^2 + eps).  Everything below
# is scalar arithmetic on Python floats, one line per node / edge, no arrays and nothing imported from oracle/.
# ---------------------------------------------------------------------------------------------------------------------
import math

_EPS = 1e-5


def _g(d):
    return d / math.sqrt(d * d + _EPS)


def _lnr2(a, b):
    d = (a - b) / 2
    if d > 0:
        return (_g(d), 0.0)
    if d < 0:
        return (0.0, _g(-d))
    return (0.0, 0.0)


_S = 0.004      # small weights keep |a-b|/2 near sqrt(eps) = 0.00316, so g() is far from 0 and from 1 (0.3 ... 0.9)


def _ln_model():
    s = _S
    I2 = np.eye(2)
    z2 = np.zeros(2)
    return dict(
        node_enc=dict(weight=[s * np.array([[1., 0, 0], [0, 0, 1.]]), s * I2], bias=[z2, np.array([0, s / 4])]),
        edge_enc=dict(weight=[s * np.array([[1., 0, 0, 0], [0, 0, 1., 0]]), s * I2], bias=[z2, z2]),
        edge_net=dict(weight=[s * np.array([[1., 0, 0, 0, 0, 0], [0, 0, 0, 1., 0, 1.]]), s * I2], bias=[z2, np.array([s / 4, 0])]),
        node_net=dict(weight=[s * np.array([[0, 0, 1., 0, 0, 0], [0, 0, 0, 0, 1., 1.]]), s * I2], bias=[z2, np.array([0, s / 4])]),
        edge_dec=dict(weight=[s * np.array([[1., 0, 0, 0, 1., 0], [0, 0, 0, 1., 0, 0]]), np.array([[1., -1.]])],
                      bias=[np.array([0, s / 8]), np.array([0.5])]),
    )


_LN_HITS = np.array([[1, 0, 3], [2, 0, 1], [1, 0, -1], [3, 0, 2]], dtype=np.float32)      # (r, phi, z)
_LN_SRC = np.array([0, 1, 0])
_LN_DST = np.array([1, 3, 2])


def _ln_hand(T):
    """The network of DESIGN.md C-12 on the 4-node / 3-edge graph above, written out element by element."""
    s = _S
    # node encoder: layer 1 pre-activation s*(r, z), layer 2 pre-activation s*v + (0, s/4)
    def node_enc(r, z):
        v = _lnr2(s * r, s * z)
        return _lnr2(s * v[0], s * v[1] + s / 4)
    h = [node_enc(1, 3), node_enc(2, 1), node_enc(1, -1), node_enc(3, 2)]
    # edge encoder on a = (dr, dphi, dz, deta): layer 1 s*(dr, dz), layer 2 s*v
    def edge_enc(dr, dz):
        v = _lnr2(s * dr, s * dz)
        return _lnr2(s * v[0], s * v[1])
    e = [edge_enc(2 - 1, 1 - 3), edge_enc(3 - 2, 2 - 1), edge_enc(1 - 1, -1 - 3)]     # k0 0->1, k1 1->3, k2 0->2
    def edge_net(hs, hd, ek):          # layer 1 s*(h_s[0], h_d[1] + e[1]); layer 2 s*v + (s/4, 0)
        v = _lnr2(s * hs[0], s * (hd[1] + ek[1]))
        return _lnr2(s * v[0] + s / 4, s * v[1])
    def node_net(hv, mi, mo):          # layer 1 s*(m_in[0], m_out[0] + m_out[1]); layer 2 s*v + (0, s/4)
        v = _lnr2(s * mi[0], s * (mo[0] + mo[1]))
        return _lnr2(s * v[0], s * v[1] + s / 4)
    add = lambda a, b: (a[0] + b[0], a[1] + b[1])
    zero = (0.0, 0.0)
    for _ in range(T):
        e = [add(e[0], edge_net(h[0], h[1], e[0])), add(e[1], edge_net(h[1], h[3], e[1])), add(e[2], edge_net(h[0], h[2], e[2]))]
        m_in = [zero, e[0], e[2], e[1]]                    # n0 none, n1 <- k0, n2 <- k2, n3 <- k1
        m_out = [add(e[0], e[2]), e[1], zero, zero]        # n0 -> k0, k2 ; n1 -> k1
        h = [add(h[v], node_net(h[v], m_in[v], m_out[v])) for v in range(4)]
    def edge_dec(hs, hd, ek):          # v = LNR(s*(h_s[0] + e[0]), s*h_d[1] + s/8); logit = v0 - v1 + 0.5 (no LN on the logit)
        v = _lnr2(s * (hs[0] + ek[0]), s * hd[1] + s / 8)
        return v[0] - v[1] + 0.5
    logit = [edge_dec(h[0], h[1], e[0]), edge_dec(h[1], h[3], e[1]), edge_dec(h[0], h[2], e[2])]
    return logit, h, e


def test_lnr2_closed_form_literals():
    """The helper itself against numbers worked by hand: g(d) = d/sqrt(d^2 + 1e-5)."""
    assert abs(_g(0.004) - 0.004 / math.sqrt(2.6e-5)) < 1e-15 and abs(_g(0.004) - 0.7844645405527362) < 1e-12
    assert abs(_g(0.003) - 0.003 / math.sqrt(1.9e-5)) < 1e-15 and abs(_g(0.003) - 0.6882472016116853) < 1e-12
    assert abs(_g(1.0) - (1 - 0.5e-5)) < 1e-9                 # 1/sqrt(1+eps) = 1 - eps/2 + O(eps^2)
    assert _lnr2(3.0, 1.0) == (_g(1.0), 0.0) and _lnr2(1.0, 3.0) == (0.0, _g(1.0)) and _lnr2(2.0, 2.0) == (0.0, 0.0)


def test_hand_computed_layernorm_decoder_logit_h2():
    """T = 0, LayerNorm on: the *logit* (the decoder's LNR, then the un-normalised final Linear) against hand values."""
    logit, h, e = s4_gnn.gnn_forward(_LN_HITS, _LN_SRC, _LN_DST, _ln_model(), 0, layernorm_on=True, return_state=True)
    want_logit, want_h, want_e = _ln_hand(0)
    assert np.allclose(h, np.array(want_h), rtol=0, atol=1e-13) and np.allclose(e, np.array(want_e), rtol=0, atol=1e-13)
    assert np.allclose(logit, np.array(want_logit), rtol=0, atol=1e-13)
    # one edge spelled out completely, k0 = 0 -> 1, numbers a reader can follow:
    s = _S
    # node 0 (r=1, z=3): layer 1 (s, 3s) -> d = -s -> (0, g(s)); layer 2 (0, s*g(s) + s/4) -> (0, g((s*g(s) + s/4)/2))
    g1 = _g(s)
    h0 = (0.0, _g((s * g1 + s / 4) / 2))
    # node 1 (r=2, z=1): layer 1 (2s, s) -> d = s/2 -> (g(s/2), 0); layer 2 (s*g(s/2), s/4) -> d = (s*g(s/2) - s/4)/2 > 0
    g2 = _g(s / 2)
    h1 = (_g((s * g2 - s / 4) / 2), 0.0)
    assert np.allclose(h[0], h0, atol=1e-13) and np.allclose(h[1], h1, atol=1e-13)
    # edge 0 -> 1: (dr, dz) = (1, -2): layer 1 (s, -2s) -> d = 1.5 s -> (g(1.5 s), 0); layer 2 (s g(1.5 s), 0) -> (g(s g(1.5 s)/2), 0)
    e0 = (_g(s * _g(1.5 * s) / 2), 0.0)
    assert np.allclose(e[0], e0, atol=1e-13)
    # decoder: (s*(h_s[0] + e[0]), s*h_d[1] + s/8) = (s*e0[0], s/8) since h0[0] = 0 and h1[1] = 0
    d = (s * e0[0] - s / 8) / 2
    assert d > 0
    assert abs(logit[0] - (_g(d) + 0.5)) < 1e-13
    # the decoder's LayerNorm is really there: without it the logit would be relu(s*e0[0]) - relu(s/8) + 0.5, about 0.5007
    assert abs(logit[0] - (s * e0[0] - s / 8 + 0.5)) > 0.1
    assert 0.6 < logit[0] < 0.95 and np.allclose(s4_gnn.gnn_scores(_LN_HITS, _LN_SRC, _LN_DST, _ln_model(), 0, True)[0],
                                                   1 / (1 + math.exp(-logit[0])), atol=1e-15)


def test_hand_computed_two_iterations_layernorm_h2():
    """T = 2, LayerNorm on, shared weights: every e, h and logit of both iterations against the scalar hand evaluation."""
    for T in (1, 2, 3):
        logit, h, e = s4_gnn.gnn_forward(_LN_HITS, _LN_SRC, _LN_DST, _ln_model(), T, layernorm_on=True, return_state=True)
        want_logit, want_h, want_e = _ln_hand(T)
        assert np.allclose(e, np.array(want_e), rtol=0, atol=1e-12), T
        assert np.allclose(h, np.array(want_h), rtol=0, atol=1e-12), T
        assert np.allclose(logit, np.array(want_logit), rtol=0, atol=1e-12), T
    # the second iteration is not a no-op and differs from the first (states feed back; weights are shared)
    l1, h1, e1 = _ln_hand(1)
    l2, h2, e2 = _ln_hand(2)
    assert max(abs(a - b) for x, y in zip(e1, e2) for a, b in zip(x, y)) > 0.1
    assert max(abs(a - b) for x, y in zip(h1, h2) for a, b in zip(x, y)) > 0.1
    # first iteration, edge k1 = 1 -> 3, spelled out: e += LNR(s*LNR(s*h1[0], s*(h3[1] + e1[1])) + (s/4, 0))
    _, h0, e0 = _ln_hand(0)
    v = _lnr2(_S * h0[1][0], _S * (h0[3][1] + e0[1][1]))
    u = _lnr2(_S * v[0] + _S / 4, _S * v[1])
    got = s4_gnn.gnn_forward(_LN_HITS, _LN_SRC, _LN_DST, _ln_model(), 1, layernorm_on=True, return_state=True)[2]
    assert np.allclose(got[1], (e0[1][0] + u[0], e0[1][1] + u[1]), atol=1e-13)
