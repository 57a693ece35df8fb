"""-m gpu: an event of the paper's own size (~350 k spacepoints): the
"paper350k" config, 43 500 particles -> 349 056 hits, E_c = 11.17 M, E_k = 3.19 M, one context sized for the whole event.

The oracle cannot run whole stages at this size in minutes (its S2 alone took 45 min here), so, as for the other full-size
configs, each stage is checked on sampled outputs the oracle computes one by one, plus exact whole-output properties:

  S1  the oracle embedding of all hits (one fp64 pass, ~1 min);
  S2  the whole GPU edge list against (a) the oracle's calibrated edge COUNT (synth/calibration.json, written by
      oracle/calibrate.py: 11 169 792) and (b) the brute-force definition (oracle.s2_frnn._search_block against ALL hits
      of the event) for 192 sampled queries, rows bit-exact; order and degree-cap invariants on every row;
  S3  a SYNTHETIC candidate list of the config's size (every hit -> its 32 successors in (phi, z) order; no GPU value
      enters it): scores of 20 000 sampled edges (+ the chunk seams) against the oracle; exact compaction property;
  S4  a synthetic kept graph of the config's size: the candidates whose two hits share one of 32 phi sectors, thinned by
      a seeded hash; sectors are independent sub-graphs, so the oracle runs one sector alone and the GPU, given the whole
      graph, must reproduce its scores; S5 labels and S6 track lists bit-exact on the whole graph.
"""
import numpy as np
import pytest

import gpu_common as G
from oracle import s1_embed, s2_frnn, s3_filter, s4_gnn, s5_cc, s6_tracks
from oracle.mlp import sigmoid
from synth.rng import Stream

pytestmark = pytest.mark.gpu

NAME = "paper350k"
N_SECTORS = 32
ORACLE_SECTOR = 5
RING = 32


def _dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


class Paper:
    def __init__(self):
        self.cfg = G.get_config(NAME)
        self.calib = G.load_calibration(NAME)
        self.ev = G.make_events(self.cfg)
        self.model = G.centred_model(self.cfg, self.calib)
        self.hits, self.off = self.ev["hits"], self.ev["event_offsets"]
        self.n = len(self.hits)
        self._c = {}

    def memo(self, key, fn):
        if key not in self._c:
            self._c[key] = fn()
        return self._c[key]

    @property
    def emb(self):
        return self.memo("emb", lambda: s1_embed.embed_f32(self.hits, self.model["embed"]))

    @property
    def sector(self):
        return np.minimum(((self.hits[:, 1].astype(np.float64) + 1.0) * (N_SECTORS / 2)).astype(np.int64), N_SECTORS - 1)

    @property
    def ring(self):
        """Synthetic candidate edges sorted by (src, dst): hit -> its RING successors in (phi, z) order."""
        def f():
            order = np.lexsort((self.hits[:, 2], self.hits[:, 1]))
            pos = np.empty(self.n, np.int64)
            pos[order] = np.arange(self.n)
            dst = order[(pos[:, None] + np.arange(1, RING + 1)[None, :]) % self.n]
            dst.sort(axis=1)
            return np.repeat(np.arange(self.n, dtype=np.int32), RING), dst.reshape(-1).astype(np.int32)
        return self.memo("ring", f)

    @property
    def kept(self):
        def f():
            src, dst = self.ring
            same = self.sector[src] == self.sector[dst]
            frac = self.calib["n_kept_edges"] / max(1, int(same.sum()))
            u = Stream(11, "thin:paper350k").uniform(np.arange(len(src), dtype=np.uint64))
            return same & (u < frac)
        return self.memo("kept", f)


@pytest.fixture(scope="module")
def paper():
    from paper_2501_05520_b200 import trk_from_config
    p = Paper()
    trk = trk_from_config(p.cfg, p.model, p.calib, max_hits=p.n, max_cand_edges=p.n * p.cfg["frnn_k"],
                          max_kept_edges=int(1.5 * p.calib["n_kept_edges"]) + 4096)
    yield p, trk
    trk.close()


def test_paper_s1_embedding(paper):
    p, trk = paper
    assert p.n == p.calib["n_hits"] == 349056
    emb = trk.stage_embed(_dev(p.hits)).cpu().numpy().astype(np.float64)
    ref = p.emb.astype(np.float64)
    err = np.max(np.abs(emb - ref)) / np.max(np.abs(ref))
    assert err <= G.EMB_TOL["bf16"], f"embedding error {err:.3e}"


def test_paper_s2_count_invariants_and_sampled_rows(paper):
    p, trk = paper
    K, r = p.cfg["frnn_k"], p.calib["frnn_radius"]
    src, dst, rowptr, count = trk.stage_frnn(_dev(p.emb), _dev(p.hits), p.off)
    ec = int(count[0])
    assert int(count[1]) == 0 and ec == p.calib["n_cand_edges"], (ec, p.calib["n_cand_edges"])     # the oracle's own count
    src, dst, rowptr = src[:ec].cpu().numpy(), dst[:ec].cpu().numpy(), rowptr.cpu().numpy()
    deg = np.diff(rowptr)
    assert rowptr[0] == 0 and rowptr[-1] == ec and deg.max() == K and np.array_equal(src, np.repeat(np.arange(p.n), deg))
    assert np.all(np.diff(G.edge_keys(src, dst)) > 0)                                               # sorted by (src, dst), no duplicate
    # every emitted pair is outer and inside the radius (fp64, the oracle's arithmetic), for a 2 M-edge sample
    idx = np.unique((Stream(3, "s2pairs").uniform(np.arange(2_000_000, dtype=np.uint64)) * ec).astype(np.int64))
    e64 = p.emb.astype(np.float64)
    d2 = np.zeros(len(idx))
    for k in range(e64.shape[1]):
        t = e64[src[idx], k] - e64[dst[idx], k]
        d2 = d2 + t * t
    assert np.all(d2 <= s2_frnn.radius_squared(r))
    hr, hz = p.hits[:, 0], np.abs(p.hits[:, 2])
    s, d = src[idx], dst[idx]
    assert np.all((hr[s] < hr[d]) | ((hr[s] == hr[d]) & ((hz[s] < hz[d]) | ((hz[s] == hz[d]) & (s < d)))))
    # rows of sampled queries against the brute-force definition over all hits of the event
    q = np.unique((Stream(5, "s2queries").uniform(np.arange(192, dtype=np.uint64)) * p.n).astype(np.int64))
    q = np.unique(np.concatenate([q, np.argsort(-deg, kind="stable")[:16], [0, p.n - 1]]))         # + capped rows, ends
    allj = np.arange(p.n)
    for a in range(0, len(q), 32):
        qi = q[a:a + 32]
        for i, (dj, _) in zip(qi, s2_frnn._search_block(e64, p.hits, qi, allj, s2_frnn.radius_squared(r), K)):
            assert np.array_equal(dst[rowptr[i]:rowptr[i + 1]], np.asarray(dj, np.int32)), f"row {i}"


def test_paper_s3_scores_sampled_and_compaction(paper):
    p, trk = paper
    osrc, odst = p.ring
    e = len(osrc)
    assert e == RING * p.n
    src, dst = _dev(osrc), _dev(odst)
    score = trk.stage_filter(_dev(p.emb), src, dst)
    gpu = score.cpu().numpy()
    assert np.all(np.isfinite(gpu))
    idx = np.unique((Stream(7, "sample:paper350k").uniform(np.arange(20000, dtype=np.uint64)) * e).astype(np.int64))
    seams = np.concatenate([np.arange(c * 1212416 - 32, c * 1212416 + 32) for c in range(1, e // 1212416 + 1)])
    idx = np.unique(np.concatenate([idx, [0, e - 1], seams[seams < e]]))
    ref = s3_filter.filter_scores(p.emb, osrc[idx], odst[idx], p.model["filter"]).astype(np.float32)
    G.check_scores(gpu[idx], ref, "bf16", f"filter score ({len(idx)} sampled edges)")
    cut = np.float32(p.calib["filter_cut"])
    ks, kd, count = trk.stage_compact(src, dst, score)
    ek = int(count[0])
    m = gpu > cut
    assert ek == int(m.sum()) and np.array_equal(ks[:ek].cpu().numpy(), osrc[m]) and np.array_equal(kd[:ek].cpu().numpy(), odst[m])


def test_paper_s4_s5_s6(paper):
    import torch
    p, trk = paper
    osrc, odst = p.ring
    ks, kd = osrc[p.kept], odst[p.kept]
    assert 0.95 < len(ks) / p.calib["n_kept_edges"] < 1.05
    score = trk.stage_gnn(_dev(p.hits), _dev(ks), _dev(kd)).cpu().numpy()
    assert np.all(np.isfinite(score))
    nodes = np.nonzero(p.sector == ORACLE_SECTOR)[0]
    remap = np.full(p.n, -1, np.int64)
    remap[nodes] = np.arange(len(nodes))
    pos = np.nonzero(p.sector[ks] == ORACLE_SECTOR)[0]                 # both endpoints are in the sector by construction
    assert len(pos) > 50000 and np.all(remap[kd[pos]] >= 0)
    ref = sigmoid(s4_gnn.gnn_forward(p.hits[nodes], remap[ks[pos]], remap[kd[pos]], p.model, p.cfg["gnn_iters"])).astype(np.float32)
    err = G.check_scores(score[pos], ref, "bf16", f"gnn score (sector {ORACLE_SECTOR})")
    print(f"paper350k: gnn max abs err {err:.3e} over {len(pos)} edges")
    full_ref = np.array(score, copy=True)
    full_ref[pos] = ref
    labels = trk.stage_cc(p.n, _dev(ks), _dev(kd), _dev(full_ref), p.cfg["gnn_cut"])
    lab = labels.cpu().numpy()
    assert np.array_equal(lab, s5_cc.connected_components(p.n, ks, kd, full_ref, p.cfg["gnn_cut"]))
    toff, thit, cnt = trk.stage_tracks(labels, 3)
    torch.cuda.synchronize()
    ref_off, ref_hit = s6_tracks.build_tracks(lab, 3)
    T, nh, over = cnt.cpu().tolist()
    assert over == 0 and T == len(ref_off) - 1 and nh == len(ref_hit)
    assert np.array_equal(toff.cpu().numpy()[:T + 1], ref_off) and np.array_equal(thit.cpu().numpy()[:nh], ref_hit)


def test_paper_infer_invariants(paper):
    import torch
    p, trk = paper
    res = trk.infer(_dev(p.hits), p.off, want_edges=True, want_cand=True, want_tracks=True)
    torch.cuda.synchronize()
    ec, ek, et, of = [int(v) for v in res["counts"].cpu().numpy()]
    assert of == 0 and 0 < et < ek < ec
    assert abs(ec / p.calib["n_cand_edges"] - 1) < 0.02 and abs(ek / p.calib["n_kept_edges"] - 1) < 0.05
    cs, cd, fs = (res[k][:ec].cpu().numpy() for k in ("cand_src", "cand_dst", "cand_score"))
    es, ed, sc = (res[k][:ek].cpu().numpy() for k in ("edge_src", "edge_dst", "edge_score"))
    assert np.all(np.diff(G.edge_keys(cs, cd)) > 0)
    keep = fs > np.float32(p.calib["filter_cut"])
    assert np.array_equal(es, cs[keep]) and np.array_equal(ed, cd[keep])
    lab = res["labels"].cpu().numpy()
    assert np.array_equal(lab, s5_cc.connected_components(p.n, es, ed, sc, p.cfg["gnn_cut"]))
    ref_off, ref_hit = s6_tracks.build_tracks(lab, 3)
    T, nh = res["track_counts"].cpu().tolist()
    assert T == len(ref_off) - 1 and np.array_equal(res["track_hits"].cpu().numpy()[:nh], ref_hit)
    print(f"paper350k: E_c={ec} E_k={ek} E_t={et} tracks={T}")
