"""Pins for the input generators (SURVEY.md section 8(c) "Pins / Generator")."""
import os

import numpy as np

from synth import events as ev
from synth.configs import get_config, make_events
from synth.rng import Stream
from synth.weights import make_mlp, round_to_bf16

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "helix_worked_values.txt")


def test_worked_helix_values():
    rows = np.loadtxt(GOLDEN, comments="#")
    for pt, phi0, q, eta, z0, r, phi_ref, arc_ref, z_ref in rows:
        phi, z, arc, ok = ev.helix_layer_crossing(pt, eta, phi0, q, z0, r)
        assert ok
        assert abs(phi - phi_ref) < 1e-11
        if not np.isnan(arc_ref):
            assert abs(arc - arc_ref) < 1e-8
        assert abs(z - z_ref) < (1e-8 if abs(z_ref) < 1000 else 1e-2)   # the rejected row is printed to 2 decimals
    assert ev.helix_radius_mm(0.6) == 1000.0


def test_helix_radius_closed_form_every_hit():
    """Every unsmeared true hit lies on the circle of radius R = pT/(0.3 B) about c = qR(sin phi0, -cos phi0)."""
    e = ev.generate_event(300, 0.1, seed=3)
    P = e["particles"]
    m = e["particle_id"] >= 0
    pid = e["particle_id"][m]
    r = ev.LAYER_R_MM[e["layer"][m]]
    R = 1000.0 * P["pt"][pid] / (0.3 * 2.0)
    cx, cy = P["q"][pid] * R * np.sin(P["phi0"][pid]), -P["q"][pid] * R * np.cos(P["phi0"][pid])
    x, y = r * np.cos(e["true_phi"][m]), r * np.sin(e["true_phi"][m])
    assert np.max(np.abs(np.hypot(x - cx, y - cy) - R)) < 1e-9 * np.max(R) / 1000.0 + 1e-9
    # hit radius equals the layer radius exactly (feature r/1000 in fp32)
    assert np.array_equal(e["hits"][:, 0], (ev.LAYER_R_MM[e["layer"]] / 1000.0).astype(np.float32))


def test_straight_line_limit():
    phi, z, arc, ok = ev.helix_layer_crossing(1e9, 0.7, 1.3, 1.0, 5.0, 500.0)
    assert abs(phi - 1.3) < 1e-9 and abs(z - (5.0 + 500.0 * np.sinh(0.7))) < 1e-6 and abs(arc - 500.0) < 1e-6


def test_event_statistics_and_shape():
    e = ev.generate_event(2500, 0.1, seed=0)
    n = len(e["hits"])
    assert e["hits"].dtype == np.float32 and e["hits"].shape == (n, 3)
    assert e["n_noise"] == round(0.1 * e["n_true"]) and n == e["n_true"] + e["n_noise"]
    assert abs(e["n_true"] / 2500 - 7.32) < 0.25                      # SURVEY C-2: 7.32 layers crossed / particle
    assert np.all(np.abs(e["hits"][:, 2]) < 1.005) and np.all(e["hits"][:, 1] > -1.0) and np.all(e["hits"][:, 1] <= 1.0)
    assert set(np.unique(e["hits"][:, 0])) <= set((ev.LAYER_R_MM / 1000).astype(np.float32))
    P = e["particles"]
    assert P["pt"].min() >= 0.5 and P["pt"].max() <= 10.0 and np.all(np.abs(P["eta"]) <= 2.5)
    assert abs(np.mean(np.log(P["pt"] / 0.5) / np.log(20.0)) - 0.5) < 0.03   # log-uniform
    assert abs(np.std(P["z0"]) - 50.0) < 3.0 and set(np.unique(P["q"])) == {-1.0, 1.0}
    # determinism and seed sensitivity
    assert np.array_equal(e["hits"], ev.generate_event(2500, 0.1, seed=0)["hits"])
    assert not np.array_equal(e["hits"][:100], ev.generate_event(2500, 0.1, seed=1)["hits"][:100])


def test_smear_magnitude():
    e = ev.generate_event(2000, 0.0, seed=5)
    r = ev.LAYER_R_MM[e["layer"]]
    dphi = ev.wrap_phi(e["hits"][:, 1].astype(np.float64) * np.pi - e["true_phi"])
    assert abs(np.std(dphi * r) - 0.05) < 0.01           # fp32 storage of phi/pi adds ~1e-7*r
    assert abs(np.std(e["hits"][:, 2] * 1000.0 - e["true_z"]) - 0.5) < 0.03


def test_batch_offsets_and_config_sizes():
    cfg = get_config("batch16")
    b = make_events(cfg, n_particles=40)
    off = b["event_offsets"]
    assert len(off) == 17 and off[0] == 0 and off[-1] == len(b["hits"]) and np.all(np.diff(off) > 0)
    for i, e in enumerate(b["events"]):
        assert np.array_equal(b["hits"][off[i]:off[i + 1]], e["hits"])
    toy = make_events(get_config("toy"))
    assert 300 < len(toy["hits"]) < 600


def test_truth_edges_connect_same_particle():
    e = ev.generate_event(100, 0.1, seed=2)
    s, d = ev.truth_edges(e["particle_id"], e["layer"], e["hits"])
    assert np.all(e["particle_id"][s] == e["particle_id"][d]) and np.all(e["layer"][s] < e["layer"][d])
    assert len(s) == e["n_true"] - len(np.unique(e["particle_id"][e["particle_id"] >= 0]))


def test_rng_streams():
    a = Stream(0, "a")
    u = a.uniform(np.arange(200000))
    assert 0.0 <= u.min() and u.max() < 1.0 and abs(u.mean() - 0.5) < 3e-3 and abs(u.var() - 1 / 12) < 2e-3
    g = a.normal(np.arange(200000))
    assert abs(g.mean()) < 0.01 and abs(g.std() - 1.0) < 0.01
    assert not np.array_equal(a.u64(np.arange(8)), Stream(0, "b").u64(np.arange(8)))
    assert np.array_equal(a.u64(np.arange(8)), Stream(0, "a").u64(np.arange(8)))


def test_weights_kaiming_uniform_and_bf16():
    m = make_mlp(0, "t", [256, 512, 4], bf16=False)
    w, b = m["weight"][0], m["bias"][0]
    assert w.shape == (512, 256) and b.shape == (512,) and w.dtype == np.float32
    bound = np.sqrt(6.0 / 256)
    assert np.abs(w).max() <= bound and abs(w.var() - bound ** 2 / 3) < 0.02 * bound ** 2
    assert np.abs(b).max() <= 1 / 16.0
    x = np.array([1.0, 1.00390625, 1.01171875, -3.1415927, 1e-30], dtype=np.float32)
    r = round_to_bf16(x)
    assert np.all((r.view(np.uint32) & 0xFFFF) == 0)
    assert r[0] == 1.0 and r[1] == 1.0 and r[2] == np.float32(1.015625)        # ties to even: 1+2^-8 -> 1, 1+3*2^-8 -> 1+2^-6
    import torch
    t = torch.from_numpy(np.random.default_rng(0).standard_normal(10000).astype(np.float32))
    assert np.array_equal(round_to_bf16(t.numpy()), t.to(torch.bfloat16).to(torch.float32).numpy())
    mb = make_mlp(0, "t", [256, 512, 4], bf16=True)
    assert np.array_equal(mb["weight"][0], round_to_bf16(w))
