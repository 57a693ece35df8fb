"""Pins for the oracle's S2 (SURVEY.md section 8(c) "Pins / S2 FRNN")."""
import numpy as np
import pytest

from oracle import s1_embed, s2_frnn
from synth.configs import get_config, load_calibration, make_events
from synth.events import generate_batch, generate_event
from synth.weights import make_model


def _pure_python_frnn(emb, hits, off, r, K):
    """The definition as explicit loops (tiny inputs only); shares nothing with oracle/."""
    emb = [[float(np.float32(v)) for v in row] for row in emb]
    rr = float(np.float32(r)) ** 2
    edges = []
    for b in range(len(off) - 1):
        for i in range(off[b], off[b + 1]):
            cand = []
            for j in range(off[b], off[b + 1]):
                if j == i:
                    continue
                ki = (float(hits[i][0]), abs(float(hits[i][2])), i)
                kj = (float(hits[j][0]), abs(float(hits[j][2])), j)
                if not ki < kj:
                    continue
                d2 = 0.0
                for k in range(len(emb[i])):
                    df = emb[i][k] - emb[j][k]
                    d2 = d2 + df * df
                if d2 <= rr:
                    cand.append((d2, j))
            cand.sort()
            for _, j in sorted(cand[:K], key=lambda t: t[1]):
                edges.append((i, j))
    return edges


def _pairs(src, dst):
    return list(zip(src.tolist(), dst.tolist()))


def _rand_event(n, d, seed, layers=4):
    rng = np.random.default_rng(seed)
    emb = rng.standard_normal((n, d)).astype(np.float32)
    hits = np.stack([rng.integers(1, layers + 1, n) / 10.0, rng.uniform(-1, 1, n), rng.uniform(-1, 1, n)], 1).astype(np.float32)
    return emb, hits


def test_brute_equals_pure_python_definition():
    emb, hits = _rand_event(60, 5, 0)
    off = np.array([0, 25, 25, 60], dtype=np.int32)            # includes an empty event
    for r, K in [(1.5, 4), (2.5, 3), (0.0, 4), (100.0, 100)]:
        s, d, rp = s2_frnn.frnn_brute(emb, hits, off, r, K)
        assert _pairs(s, d) == _pure_python_frnn(emb, hits, off, r, K)
        assert rp[0] == 0 and rp[-1] == len(s) and np.array_equal(np.diff(rp), np.bincount(s, minlength=60))


def test_grid_equals_brute_on_small_events():
    for seed in range(4):
        emb, hits = _rand_event(700, 6, seed)
        emb[:, 3:] *= 0.1
        off = np.array([0, 300, 700], dtype=np.int32)
        for r, K in [(0.4, 8), (0.9, 5)]:
            a = s2_frnn.frnn_brute(emb, hits, off, r, K, return_d2=True)
            b = s2_frnn.frnn_grid(emb, hits, off, r, K, return_d2=True)
            assert len(a[0]) > 100
            for x, y in zip(a, b):
                assert np.array_equal(x, y)


def test_grid_equals_brute_on_generated_events():
    """BASELINE.json north_star: brute force O(N^2) vs grid on events of 2k hits or fewer."""
    cfg = get_config("pileup50")
    model = make_model(dict(cfg, embed_dims=[3, 64, 64, 12]))
    for seed, npart in [(0, 50), (1, 200)]:
        e = generate_event(npart, 0.1, seed)
        emb = s1_embed.embed_f32(e["hits"], model["embed"])
        off = np.array([0, len(emb)], dtype=np.int32)
        for r, K in [(0.15, 16), (0.5, 8)]:
            a = s2_frnn.frnn_brute(emb, e["hits"], off, r, K)
            b = s2_frnn.frnn_grid(emb, e["hits"], off, r, K)
            assert len(a[0]) > 0
            for x, y in zip(a, b):
                assert np.array_equal(x, y)


def test_radius_zero_and_infinite():
    emb, hits = _rand_event(40, 3, 1)
    off = np.array([0, 15, 40], dtype=np.int32)
    s, d, rp = s2_frnn.frnn_brute(emb, hits, off, 0.0, 8)
    assert len(s) == 0 and np.all(rp == 0)
    s, d, _ = s2_frnn.frnn_brute(emb, hits, off, 1e6, 40)
    assert len(s) == 15 * 14 // 2 + 25 * 24 // 2               # every unordered pair exactly once
    key = lambda i: (hits[i, 0], abs(hits[i, 2]), i)
    assert all(key(i) < key(j) for i, j in _pairs(s, d))
    assert len(set(_pairs(s, d))) == len(s)
    assert all((i < 15) == (j < 15) for i, j in _pairs(s, d))   # never across events


def test_k1_is_nearest_outer_neighbour():
    emb, hits = _rand_event(50, 4, 2)
    off = np.array([0, 50], dtype=np.int32)
    s, d, rp = s2_frnn.frnn_brute(emb, hits, off, 1e6, 1)
    e64 = emb.astype(np.float64)
    for i, j in _pairs(s, d):
        outer = [k for k in range(50) if (hits[i, 0], abs(hits[i, 2]), i) < (hits[k, 0], abs(hits[k, 2]), k)]
        dd = [np.sum((e64[i] - e64[k]) ** 2) for k in outer]
        assert j == outer[int(np.argmin(dd))]


def test_integer_lattice_boundary_and_tie_break():
    """Points on an integer lattice, r = 1 exactly: tests '<=' and the (d2, index) tie-break under the cap."""
    pts = np.array([[x, y] for x in range(4) for y in range(4)], dtype=np.float32)
    emb = np.zeros((16, 12), dtype=np.float32)
    emb[:, 3] = pts[:, 0]; emb[:, 7] = pts[:, 1]
    hits = np.zeros((16, 3), dtype=np.float32)
    hits[:, 0] = 0.1                                           # all on one layer: orientation falls to (|z|, index)
    off = np.array([0, 16], dtype=np.int32)
    s, d, _ = s2_frnn.frnn_brute(emb, hits, off, 1.0, 16)
    # lattice neighbours at distance exactly 1 are accepted; each unordered neighbour pair once, lower index -> higher
    want = sorted((i, j) for i in range(16) for j in range(16) if i < j and np.sum((pts[i] - pts[j]) ** 2) == 1.0)
    assert _pairs(s, d) == want
    s, d, _ = s2_frnn.frnn_brute(emb, hits, off, np.nextafter(np.float32(1.0), np.float32(0.0)), 16)
    assert len(s) == 0
    # cap K=1 with two equidistant candidates: keep the lower index
    s, d, _ = s2_frnn.frnn_brute(emb, hits, off, 1.0, 1)
    assert dict(_pairs(s, d))[0] == 1 and dict(_pairs(s, d))[5] == 6       # 0->{1,4}: keep 1; 5->{6,9}: keep 6
    # orientation by |z| when r ties: give hit 0 the largest |z| -> it becomes outermost and emits nothing
    hits2 = hits.copy(); hits2[0, 2] = -0.9
    s, d, _ = s2_frnn.frnn_brute(emb, hits2, off, 1.0, 16)
    assert 0 not in s.tolist() and (1, 0) in _pairs(s, d) and (4, 0) in _pairs(s, d)


def test_batch_equals_union_of_single_events():
    cfg = get_config("pileup50")
    model = make_model(dict(cfg, embed_dims=[3, 32, 12]))
    b = generate_batch(60, 0.1, [1, 2, 3])
    emb = s1_embed.embed_f32(b["hits"], model["embed"])
    s, d, rp = s2_frnn.frnn(emb, b["hits"], b["event_offsets"], 0.3, 8)
    off = b["event_offsets"]
    got = []
    for i in range(3):
        lo, hi = off[i], off[i + 1]
        si, di, _ = s2_frnn.frnn(emb[lo:hi], b["hits"][lo:hi], np.array([0, hi - lo], np.int32), 0.3, 8)
        got += _pairs(si + lo, di + lo)
    assert got == _pairs(s, d) and len(got) > 50


def test_permutation_equivariance():
    e = generate_event(120, 0.1, 7)
    model = make_model(dict(get_config("pileup50"), embed_dims=[3, 32, 12]))
    emb = s1_embed.embed_f32(e["hits"], model["embed"])
    n = len(emb)
    off = np.array([0, n], np.int32)
    s, d, _ = s2_frnn.frnn(emb, e["hits"], off, 0.35, 6)
    perm = np.random.default_rng(0).permutation(n)          # new position p holds old hit perm[p]
    inv = np.argsort(perm)
    s2, d2, _ = s2_frnn.frnn(emb[perm], e["hits"][perm], off, 0.35, 6)
    # generic event: no exact ties in (r,|z|) among in-radius pairs or in d2, so the edge SET is index-free
    assert set(_pairs(perm[s2], perm[d2])) == set(_pairs(s, d)) and len(s) > 100
    assert inv[perm[0]] == 0


def test_invariants_and_monotone_count():
    e = generate_event(150, 0.1, 4)
    model = make_model(dict(get_config("pileup50"), embed_dims=[3, 32, 12]))
    emb = s1_embed.embed_f32(e["hits"], model["embed"])
    off = np.array([0, len(emb)], np.int32)
    last = -1
    for r in [0.05, 0.1, 0.2, 0.4, 0.8]:
        s, d, rp, d2 = s2_frnn.frnn(emb, e["hits"], off, r, 8, return_d2=True)
        assert len(s) >= last
        last = len(s)
        assert np.all(np.diff(rp) <= 8) and np.all(d2 <= float(np.float32(r)) ** 2)
        key = np.stack([s.astype(np.int64), d.astype(np.int64)])
        assert np.all(np.diff(key[0] * (1 << 32) + key[1]) > 0)            # sorted by (src,dst), no duplicates
        e64 = emb.astype(np.float64)
        assert np.allclose(d2, np.sum((e64[s] - e64[d]) ** 2, axis=1), rtol=1e-14)
        hr, hz = e["hits"][:, 0], np.abs(e["hits"][:, 2])
        assert np.all((hr[s] < hr[d]) | ((hr[s] == hr[d]) & ((hz[s] < hz[d]) | ((hz[s] == hz[d]) & (s < d)))))


def test_toy_calibration_hits_target_degree():
    cfg = get_config("toy")
    cal = load_calibration("toy")
    ev = make_events(cfg)
    emb = s1_embed.embed_f32(ev["hits"], make_model(cfg)["embed"])
    s, d, rp = s2_frnn.frnn(emb, ev["hits"], ev["event_offsets"], cal["frnn_radius"], cfg["frnn_k"])
    assert abs(len(s) / len(emb) - cfg["degree"]) < 0.005 * cfg["degree"] and len(s) == cal["n_cand_edges"]
    assert np.max(np.diff(rp)) == cfg["frnn_k"]               # the cap really bites
