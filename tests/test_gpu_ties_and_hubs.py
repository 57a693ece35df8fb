"""-m gpu: the tie, boundary and hub cases of the method, through the C ABI against the oracle on inputs built here.

Generic float inputs never produce two equal d2, a d2 equal to r^2, a score equal to a cut or a node with hundreds of
in-edges, so the kernels' branches for those cases (frnn.cu: the sort fallback of the top-K selection and `d2 <= r2` at
equality; util_kernels.cu / cc.cu: `score > cut` at equality; graph.cu: in-edge segments longer than 32 and 256) need
inputs of their own.  BASELINE.json cfg 1 ("ties to lower index"), SURVEY.md section 8(c) Pins/S2, S4, S5.
"""
import numpy as np
import pytest

import gpu_common as G
from oracle import s2_frnn, s3_filter, s4_gnn, s5_cc
from oracle.mlp import sigmoid

pytestmark = pytest.mark.gpu


def _dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _toy_trk(n, **over):
    from paper_2501_05520_b200 import trk_from_config
    cfg = dict(G.get_config("toy"), **{k: v for k, v in over.items() if k in ("frnn_k",)})
    calib = dict(G.load_calibration("toy"), **{k: v for k, v in over.items() if k in ("frnn_radius", "filter_cut")})
    return trk_from_config(cfg, G.make_model(cfg), calib, max_hits=n), cfg, calib


def _assert_frnn_equal(trk, emb, hits, off, r, k):
    osrc, odst, orow = s2_frnn.frnn_brute(emb, hits, off, r, k)
    src, dst, rowptr, cnt = trk.stage_frnn(_dev(emb), _dev(hits), off)
    ec = int(cnt[0])
    assert int(cnt[1]) == 0 and ec == len(osrc), (ec, len(osrc))
    assert np.array_equal(src[:ec].cpu().numpy(), osrc) and np.array_equal(dst[:ec].cpu().numpy(), odst)
    assert np.array_equal(rowptr.cpu().numpy(), orow)
    return osrc, odst, orow


@pytest.mark.parametrize("axes", [(3, 7), (0, 1)])
@pytest.mark.parametrize("k", [1, 16, 32, 33, 64, 128])
def test_frnn_integer_lattice_ties_under_the_cap(k, axes):
    """A 6 x 6 integer lattice, every point replicated m >= 2.5 K times, r = 1 exactly.  A query sees only two distinct d2:
    0 (up to m - 1 replicas of its own point) and 1 (up to 4 m replicas of the lattice neighbours, accepted because
    d2 == r^2).  Whenever fewer than K outer replicas of its own point exist the K-th nearest lies inside the d2 = 1 group
    of >= 2.5 K equal values, so no threshold separates K .. CAP - 32 entries: the mid-scan prune and the final prune(K)
    must both fall back to the (d2, index) sort and keep the LOWEST indices of the tied group (K = 1, 16, 32 -> CAP 64;
    33, 64 -> CAP 128; 128 -> CAP 256).  Orientation mixes r, |z| and index ties.  axes (0, 1) puts the lattice on the
    binning coordinates, every point exactly on a cell face; (3, 7) leaves all hits in one cell column."""
    m = max(40, (5 * k) // 2)
    side = 6
    rng = np.random.default_rng(100 + k)
    pts = np.array([[x, y] for x in range(side) for y in range(side)], np.float32)
    n = len(pts) * m
    point_of = np.tile(np.arange(len(pts)), m)                 # replicas interleaved: index order != point order
    emb = np.zeros((n, 8), np.float32)
    emb[:, axes[0]] = pts[point_of, 0]
    emb[:, axes[1]] = pts[point_of, 1]
    hits = np.zeros((n, 3), np.float32)
    hits[:, 0] = rng.choice(np.array([0.1, 0.2], np.float32), n)           # two layers: many r ties
    hits[:, 2] = rng.choice(np.array([0.0, 0.5, -0.5], np.float32), n)      # |z| ties between +0.5 and -0.5
    off = np.array([0, n], np.int32)
    trk, _, _ = _toy_trk(n, frnn_k=k, frnn_radius=1.0)
    try:
        osrc, odst, orow = _assert_frnn_equal(trk, emb, hits, off, np.float32(1.0), k)
        deg = np.diff(orow)
        assert deg.max() == k and (deg == k).mean() > 0.5                   # the cap bites on most queries ...
        cut_through = 0                                                     # ... and cuts through a tied group on many
        for i in np.flatnonzero(deg == k):
            nb = odst[orow[i]:orow[i + 1]]
            own = np.sum(point_of[nb] == point_of[i])
            cut_through += int(own < k)
        assert cut_through > 20
    finally:
        trk.close()
    # one ulp below: the d2 == 1 group is rejected, only exact duplicates remain
    r_lo = np.nextafter(np.float32(1.0), np.float32(0.0))
    trk, _, _ = _toy_trk(n, frnn_k=k, frnn_radius=float(r_lo))
    try:
        osrc, odst, _ = _assert_frnn_equal(trk, emb, hits, off, r_lo, k)
        assert len(osrc) > 0 and np.all(point_of[osrc] == point_of[odst])
    finally:
        trk.close()


@pytest.mark.parametrize("k", [3, 16])
def test_frnn_every_hit_duplicated(k):
    """Every hit of a toy event appears twice (same features, same embedding row): d2 = 0 between the two copies and every
    other d2 occurs at least twice; outer() between copies is decided by the index alone."""
    run = G.oracle_run("toy", "fp32")
    hits = np.repeat(run["ev"]["hits"], 2, axis=0)
    emb = np.repeat(run["out"]["emb"], 2, axis=0)
    n = len(hits)
    off = np.array([0, n], np.int32)
    r = np.float32(run["calib"]["frnn_radius"])
    trk, _, _ = _toy_trk(n, frnn_k=k, frnn_radius=float(r))
    try:
        osrc, odst, orow = _assert_frnn_equal(trk, emb, hits, off, r, k)
        pair = (osrc % 2 == 0) & (odst == osrc + 1)
        assert pair.sum() == n // 2                                          # copy 2i -> 2i+1 is always an edge
    finally:
        trk.close()


def test_scores_equal_to_the_cut_in_compaction_and_components():
    """score > cut is strict in fp32: a score equal to the fp32 cut is dropped, one ulp above is kept (S3 tail and S5)."""
    rng = np.random.default_rng(3)
    n, n_edges = 5000, 20000
    cut32 = np.float32(G.load_calibration("toy")["filter_cut"])
    for cut, stage in ((cut32, "compact"), (np.float32(0.5), "cc")):
        vals = np.array([cut, np.nextafter(cut, np.float32(0)), np.nextafter(cut, np.float32(1)), 0.0, 1.0], np.float32)
        score = vals[rng.integers(0, len(vals), n_edges)]
        src = rng.integers(0, n, n_edges).astype(np.int32)
        dst = rng.integers(0, n, n_edges).astype(np.int32)
        order = np.lexsort((dst, src))
        src, dst = src[order], dst[order]
        trk, cfg, calib = _toy_trk(n, filter_cut=float(cut32))
        try:
            if stage == "compact":
                keep = s3_filter.keep_mask(score, cut)
                assert 0.3 < keep.mean() < 0.5 and np.sum(score == cut) > 1000
                ks, kd, cnt = trk.stage_compact(_dev(src), _dev(dst), _dev(score))
                ek = int(cnt[0])
                assert ek == keep.sum() and int(cnt[1]) == 0
                assert np.array_equal(ks[:ek].cpu().numpy(), src[keep]) and np.array_equal(kd[:ek].cpu().numpy(), dst[keep])
            else:
                # sparse enough that equality matters: ~0.4 n edges pass, so components are small and a wrongly kept
                # "== cut" edge merges two of them
                sel = rng.random(n_edges) < 0.25
                s_, d_, sc_ = src[sel], dst[sel], score[sel]
                ref = s5_cc.connected_components(n, s_, d_, sc_, cut)
                loose = s5_cc.connected_components(n, s_, d_, np.where(sc_ == cut, np.float32(1), sc_), cut)
                assert not np.array_equal(ref, loose)
                lab = trk.stage_cc(n, _dev(s_), _dev(d_), _dev(sc_), float(cut)).cpu().numpy()
                assert np.array_equal(lab, ref)
        finally:
            trk.close()


def _hub_graph(run, in_degrees, out_degree):
    """The kept edges of a pileup-50-architecture event plus star hubs: for each d in in_degrees one node that receives d
    extra in-edges from distinct nodes, one node with out_degree extra out-edges, and a pair of hits half a turn apart
    (dphi = +1 and -1 before wrapping).  Sorted by (src, dst), no duplicate edge."""
    o = run["out"]
    hits = run["ev"]["hits"].copy()
    n = len(hits)
    rng = np.random.default_rng(17)
    free = rng.permutation(n)
    hubs = free[: len(in_degrees) + 1]
    src, dst = [o["src"].astype(np.int64)], [o["dst"].astype(np.int64)]
    for h, d in zip(hubs, in_degrees):
        others = np.setdiff1d(np.arange(n), [h])
        s = rng.choice(others, d, replace=False)
        src.append(s); dst.append(np.full(d, h))
    h = hubs[-1]
    others = np.setdiff1d(np.arange(n), [h])
    t = rng.choice(others, out_degree, replace=False)
    src.append(np.full(out_degree, h)); dst.append(t)
    a, b = free[-1], free[-2]
    hits[a, 1], hits[b, 1] = np.float32(0.5), np.float32(-0.5)
    src.append(np.array([a, b])); dst.append(np.array([b, a]))
    key = np.unique((np.concatenate(src) << 32) | np.concatenate(dst))
    return hits, (key >> 32).astype(np.int32), (key & 0xffffffff).astype(np.int32), hubs, (a, b)


@pytest.mark.parametrize("precision", ["bf16", "fp32"])
def test_gnn_on_hub_nodes(precision):
    """S4 on a graph with in-degrees 33, 256, 257, 300, 1000, 3000 and an out-degree of 2000 (graph.cu: the 33..256 rank
    sort, the > 256 path, a long serial segment sum), a node-update row whose mean dwarfs its spread, and dphi = +-1:
    scores against the oracle at the usual tolerance, twice with identical bits."""
    import torch
    run = G.oracle_run("pileup50", precision, True, 400, 4) if precision == "bf16" else G.oracle_run("toy", "fp32", True, 400, 4)
    cfg, model = run["cfg"], run["model"]
    in_degrees = [33, 256, 257, 300, 1000, 3000]
    hits, src, dst, hubs, (a, b) = _hub_graph(run, in_degrees, 2000)
    n = len(hits)
    assert n > 3001
    indeg = np.bincount(dst, minlength=n)
    assert all(indeg[h] >= d for h, d in zip(hubs, in_degrees))
    logit = s4_gnn.gnn_forward(hits, src, dst, model, cfg["gnn_iters"])
    ref = sigmoid(logit)
    trk = G.make_trk(run, max_hits=n, max_kept_edges=len(src), max_cand_edges=max(len(src), n * cfg["frnn_k"]))
    try:
        sc1 = trk.stage_gnn(_dev(hits), _dev(src), _dev(dst))
        sc2 = trk.stage_gnn(_dev(hits), _dev(src), _dev(dst))
        torch.cuda.synchronize()
        assert torch.equal(sc1, sc2), "run-to-run bits differ"
        sc = sc1.cpu().numpy()
        err = G.check_scores(sc, ref, precision, "gnn score on the hub graph")
        touched = np.isin(dst, hubs) | np.isin(src, hubs)
        assert touched.sum() > 6000
        print(f"hub graph [{precision}]: E={len(src)} max err {err:.3e}, on hub edges "
              f"{np.max(np.abs(sc[touched] - ref[touched])):.3e}")
        # the half-turn pair: both directions exist and were scored
        for s_, d_ in ((a, b), (b, a)):
            k = np.flatnonzero((src == s_) & (dst == d_))
            assert len(k) == 1 and abs(sc[k[0]] - ref[k[0]]) <= (2e-2 if precision == "bf16" else 1e-4)
    finally:
        trk.close()


def test_gnn_scatter_structure_on_hub_nodes():
    """The in-edge lists that fix the summation order of S4 (trk_stage_gnn_csr): ascending edge index inside every segment
    -- segments of length <= 32 (one rank pass), 33..256 (chunked rank passes) and > 256 (in-place sorting network) -- and
    the two row-pointer arrays, bit for bit against a stable argsort, twice."""
    run = G.oracle_run("toy", "fp32", True, 400, 4)
    hits, src, dst, hubs, _ = _hub_graph(run, [33, 256, 257, 300, 1000, 3000], 2000)
    n = len(hits)
    indeg = np.bincount(dst, minlength=n)
    assert np.sum((indeg > 32) & (indeg <= 256)) >= 2 and np.sum(indeg > 256) >= 4 and np.sum((indeg > 1) & (indeg <= 32)) > 100
    want_perm = np.argsort(dst, kind="stable").astype(np.int32)
    want_in = np.concatenate([[0], np.cumsum(indeg)]).astype(np.int32)
    want_out = np.concatenate([[0], np.cumsum(np.bincount(src, minlength=n))]).astype(np.int32)
    trk = G.make_trk(run, max_hits=n, max_kept_edges=len(src), max_cand_edges=max(len(src), n * run["cfg"]["frnn_k"]))
    try:
        for _ in range(2):
            in_rowptr, in_perm, out_rowptr = trk.stage_gnn_csr(_dev(hits), _dev(src), _dev(dst))
            assert np.array_equal(in_rowptr.cpu().numpy(), want_in) and np.array_equal(out_rowptr.cpu().numpy(), want_out)
            assert np.array_equal(in_perm.cpu().numpy(), want_perm)
    finally:
        trk.close()


def test_fused_gnn_without_layernorm_bf16():
    """gnn_layernorm = 0 through the FUSED bf16 kernels (H = 128): the ReLU-only network of reading C-13 with one
    iteration (with more, the un-normalised logits grow by ~20x per iteration and every score saturates).  Without
    LayerNorm nothing rescales the activations, so the error of a logit is relative to the largest logit: bf16 operands
    (2^-9 per rounding, a handful of roundings along the encoder - edge net - decoder chain) give ~1e-2 of that scale.
    Scores must agree to 2e-2 except where the oracle logit lies within 3e-2 x scale of zero, and the side of the 0.5
    cut must agree on every edge outside that band."""
    run = G.oracle_run("pileup50", "bf16", True, 300, 4)
    o, hits, cfg = run["out"], run["ev"]["hits"], run["cfg"]
    logit = s4_gnn.gnn_forward(hits, o["src"], o["dst"], run["model"], 1, layernorm_on=False)
    ref = sigmoid(logit)
    scale = np.max(np.abs(logit))
    assert 10 < scale < 500
    run1 = dict(run, cfg=dict(cfg, gnn_iters=1))
    trk = G.make_trk(run1, gnn_layernorm=False)
    try:
        sc = trk.stage_gnn(_dev(hits), _dev(o["src"]), _dev(o["dst"])).cpu().numpy().astype(np.float64)
        assert np.all(np.isfinite(sc))
        band = np.abs(logit) <= 3e-2 * scale
        bad = np.abs(sc - ref) > 2e-2
        assert np.all(band[bad]), f"{np.sum(bad & ~band)} scores off outside the band, worst {np.max(np.abs(sc - ref)[~band]):.3e}"
        assert np.mean(bad) < 0.05
        assert np.array_equal(sc[~band] > 0.5, ref[~band] > 0.5) and np.mean(~band) > 0.5
    finally:
        trk.close()
