"""-m gpu parity tests: every stage through the C ABI, fed the oracle's own inputs for that stage
(BASELINE.json north_star), compared element by element."""
import numpy as np
import pytest

import gpu_common as G

pytestmark = pytest.mark.gpu

# (config, precision, n_particles or None for the config's own size)
FULL_CASES = [("toy", "fp32", None), ("toy", "bf16", None), ("pileup50", "bf16", 600), ("pileup50", "fp32", 300),
              ("pileup50", "bf16", None)]


def _dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


@pytest.fixture(scope="module", params=FULL_CASES, ids=lambda c: f"{c[0]}-{c[1]}-{c[2] or 'full'}")
def case(request):
    name, precision, npart = request.param
    run = G.oracle_run(name, precision, True, npart)
    trk = G.make_trk(run)
    yield run, trk, precision
    trk.close()


def test_s1_embedding(case):
    run, trk, precision = case
    ref = run["out"]["emb"].astype(np.float64)
    emb = trk.stage_embed(_dev(run["ev"]["hits"])).cpu().numpy().astype(np.float64)
    err = np.max(np.abs(emb - ref)) / np.max(np.abs(ref))
    assert err <= G.EMB_TOL[precision], f"embedding error {err:.3e}"


def test_s2_frnn_bit_exact(case):
    run, trk, _ = case
    o = run["out"]
    src, dst, rowptr, count = trk.stage_frnn(_dev(o["emb"]), _dev(run["ev"]["hits"]), run["ev"]["event_offsets"])
    ec = int(count[0])
    assert int(count[1]) == 0 and ec == len(o["cand_src"])
    assert np.array_equal(src[:ec].cpu().numpy(), o["cand_src"]) and np.array_equal(dst[:ec].cpu().numpy(), o["cand_dst"])
    assert np.array_equal(rowptr.cpu().numpy(), o["rowptr"])


def test_s2_frnn_without_grid_projection_is_identical(case):
    run, _, _ = case
    o = run["out"]
    trk = G.make_trk(run, use_grid_proj=False)
    try:
        src, dst, _, count = trk.stage_frnn(_dev(o["emb"]), _dev(run["ev"]["hits"]), run["ev"]["event_offsets"])
        ec = int(count[0])
        assert ec == len(o["cand_src"]) and np.array_equal(src[:ec].cpu().numpy(), o["cand_src"])
        assert np.array_equal(dst[:ec].cpu().numpy(), o["cand_dst"])
    finally:
        trk.close()


def test_s3_filter_scores_and_kept_set(case):
    run, trk, precision = case
    o, cfg = run["out"], run["cfg"]
    feat = o["emb"] if cfg["filter_input"] == "emb" else run["ev"]["hits"]
    src, dst = _dev(o["cand_src"]), _dev(o["cand_dst"])
    score = trk.stage_filter(_dev(feat), src, dst)
    G.check_scores(score.cpu().numpy(), o["filter_score"], precision, "filter score")
    ks, kd, count = trk.stage_compact(src, dst, score)
    ek = int(count[0])
    keys = G.edge_keys(ks[:ek].cpu().numpy(), kd[:ek].cpu().numpy())
    assert np.all(np.diff(keys) > 0)                                    # stable: still sorted by (src,dst)
    G.check_kept(keys, G.edge_keys(o["src"], o["dst"]), G.edge_keys(o["cand_src"], o["cand_dst"]), o["filter_score"],
                 float(np.float32(run["calib"]["filter_cut"])), precision, "filter kept set")
    # compaction of the ORACLE's scores is bit-exact
    ks, kd, count = trk.stage_compact(src, dst, _dev(o["filter_score"]))
    ek = int(count[0])
    assert ek == len(o["src"]) and np.array_equal(ks[:ek].cpu().numpy(), o["src"]) and np.array_equal(kd[:ek].cpu().numpy(), o["dst"])


def test_s4_gnn_scores(case):
    run, trk, precision = case
    o = run["out"]
    score = trk.stage_gnn(_dev(run["ev"]["hits"]), _dev(o["src"]), _dev(o["dst"]))
    err = G.check_scores(score.cpu().numpy(), o["gnn_score"], precision, "gnn score")
    frac = np.mean(o["gnn_score"] > 0.5)
    assert 0.05 < frac < 0.95, "centred decoder bias should put scores on both sides of the cut"
    print(f"gnn max err {err:.3e}")


def test_s5_labels_bit_exact(case):
    run, trk, _ = case
    o, cfg = run["out"], run["cfg"]
    n = len(run["ev"]["hits"])
    labels = trk.stage_cc(n, _dev(o["src"]), _dev(o["dst"]), _dev(o["gnn_score"]), cfg["gnn_cut"])
    assert np.array_equal(labels.cpu().numpy(), o["labels"])
    assert len(np.unique(o["labels"])) < n                              # the test is not vacuous


def test_end_to_end_invariants(case):
    """trk_infer feeds S2 its own embedding, so only invariants and (fp32) near-identity are claimed (reading C-22)."""
    import torch
    from oracle import s5_cc
    run, trk, precision = case
    o, cfg, ev = run["out"], run["cfg"], run["ev"]
    n = len(ev["hits"])
    res = trk.infer(_dev(ev["hits"]), ev["event_offsets"], want_edges=True, want_cand=True, want_embedding=True)
    torch.cuda.synchronize()
    ec, ek, et, of = [int(v) for v in res["counts"].cpu().numpy()]
    assert of == 0 and 0 < ek <= ec
    cs, cd = res["cand_src"][:ec].cpu().numpy(), res["cand_dst"][:ec].cpu().numpy()
    assert np.all(np.diff(G.edge_keys(cs, cd)) > 0)
    es, ed, sc = res["edge_src"][:ek].cpu().numpy(), res["edge_dst"][:ek].cpu().numpy(), res["edge_score"][:ek].cpu().numpy()
    fsc = res["cand_score"][:ec].cpu().numpy()
    keep = fsc > np.float32(run["calib"]["filter_cut"])
    assert np.array_equal(es, cs[keep]) and np.array_equal(ed, cd[keep])
    assert et == int(np.sum(sc > np.float32(cfg["gnn_cut"])))
    labels = res["labels"].cpu().numpy()
    assert np.array_equal(labels, s5_cc.connected_components(n, es, ed, sc, cfg["gnn_cut"]))
    off = ev["event_offsets"]
    ev_of = np.searchsorted(off, np.arange(n), side="right") - 1
    assert np.all(ev_of[cs] == ev_of[cd])                               # no edge across events
    jac = len(np.intersect1d(G.edge_keys(cs, cd), G.edge_keys(o["cand_src"], o["cand_dst"]))) / max(1, len(
        np.union1d(G.edge_keys(cs, cd), G.edge_keys(o["cand_src"], o["cand_dst"]))))
    print(f"end-to-end candidate-edge Jaccard vs oracle: {jac:.4f}")
    assert jac > (0.999 if precision == "fp32" else 0.9)
    # run-to-run determinism (identical track candidates)
    res2 = trk.infer(_dev(ev["hits"]), ev["event_offsets"], want_edges=True)
    torch.cuda.synchronize()
    assert torch.equal(res2["labels"], res["labels"]) and torch.equal(res2["edge_score"][:ek], res["edge_score"][:ek])


@pytest.mark.parametrize("variant", [0, 1], ids=["layerwise", "fused"])
def test_s4_kernel_variants_agree_with_the_oracle(variant):
    """The two implementations of S4 (trk_set_option 'gnn_fused': layer-by-layer GEMMs with the exact split first layer, or the
    fused two-layer CTA-pair kernels) against the same oracle scores."""
    run = G.oracle_run("pileup50", "bf16", True, 600)
    o = run["out"]
    trk = G.make_trk(run)
    try:
        trk.set_option("gnn_fused", variant)
        score = trk.stage_gnn(_dev(run["ev"]["hits"]), _dev(o["src"]), _dev(o["dst"])).cpu().numpy()
        G.check_scores(score, o["gnn_score"], "bf16", f"gnn score (variant {variant})")
    finally:
        trk.close()


def test_s3_first_layer_variants_are_bit_identical():
    """trk_set_option 'filter_fused' / 'epi_split': the fused S3 kernel against the layer-by-layer path, and the latter's variants
    (four or eight epilogue warps, gather inside the GEMM or before it -- the same arithmetic)."""
    import torch
    run = G.oracle_run("pileup50", "bf16", True, 600)
    o = run["out"]
    trk = G.make_trk(run)
    try:
        feat, src, dst = _dev(o["emb"]), _dev(o["cand_src"]), _dev(o["cand_dst"])
        fused = trk.stage_filter(feat, src, dst).clone()            # default: all layers in one persistent kernel
        for pairs in (1, 5, 62):                                    # 'filter_max_pairs': fewer CTA pairs, the same bits
            trk.set_option("filter_max_pairs", pairs)
            assert torch.equal(trk.stage_filter(feat, src, dst), fused), pairs
        trk.set_option("filter_max_pairs", 0)
        trk.set_option("filter_fused", 0)                           # layer by layer, chunked
        scores = []
        for v in (0, 1, 2):
            trk.set_option("epi_split", v)
            scores.append(trk.stage_filter(feat, src, dst).clone())
        torch.cuda.synchronize()
        assert torch.equal(scores[0], scores[1]) and torch.equal(scores[1], scores[2])
        G.check_scores(scores[1].cpu().numpy(), o["filter_score"], "bf16", "filter score (layer by layer)")
        G.check_scores(fused.cpu().numpy(), o["filter_score"], "bf16", "filter score (fused kernel)")
        # the two implementations round the same quantities at the same places (bf16 activations, fp32 accumulation)
        assert float((fused - scores[1]).abs().max()) < 2e-3
    finally:
        trk.close()
