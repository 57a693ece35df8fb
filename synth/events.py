"""Synthetic collider events (BASELINE.json configs[0]; SURVEY.md §8(c) "G", readings C-2..C-6).

Detector: solenoid Bz = 2 T, ten barrel cylinders, |z| < 1000 mm.  Particles
are helices from the beam line; hits are helix-layer intersections with
Gaussian smearing, plus uniform noise hits, shuffled.  These events stand in
for the paper's simulated ttbar <pileup>=200 events, which
are not available; only their shape (three fp32 features per spacepoint) is
kept.  This module makes inputs only and contains none of the pipeline's
arithmetic.
"""
from __future__ import annotations

import numpy as np

from .rng import Stream

LAYER_R_MM = np.array([32.0, 72.0, 116.0, 172.0, 260.0, 360.0, 500.0, 660.0, 820.0, 1020.0])
Z_MAX_MM = 1000.0
B_TESLA = 2.0
SIGMA_RPHI_MM = 0.05
SIGMA_Z_MM = 0.5
PT_MIN_GEV, PT_MAX_GEV = 0.5, 10.0
ETA_MAX = 2.5
VERTEX_SIGMA_Z_MM = 50.0


def helix_radius_mm(pt_gev):
    """R[m] = pT / (0.3 B)  (BASELINE.json north_star), returned in mm."""
    return 1000.0 * np.asarray(pt_gev, dtype=np.float64) / (0.3 * B_TESLA)


def helix_layer_crossing(pt_gev, eta, phi0, q, z0_mm, r_mm):
    """Unsmeared crossing of a helix from (0,0,z0) with the cylinder of radius r.

    Reading C-5: circle through the beam line with centre q*R*(sin phi0, -cos phi0);
    alpha = asin(r / 2R); phi = phi0 - q*alpha; transverse arc s = 2*R*alpha;
    z = z0 + s*sinh(eta).  Returns (phi, z, arc, reachable)."""
    R = helix_radius_mm(pt_gev)
    ratio = np.asarray(r_mm, dtype=np.float64) / (2.0 * R)
    reachable = ratio < 1.0
    alpha = np.arcsin(np.where(reachable, ratio, 0.0))
    phi = phi0 - q * alpha
    arc = 2.0 * R * alpha
    z = z0_mm + arc * np.sinh(eta)
    return phi, z, arc, reachable


def draw_particles(n_particles: int, seed: int):
    """pT log-uniform 0.5-10 GeV (0.5 * 20**U), eta U[-2.5,2.5], phi0 U[0,2pi), q = +-1, z0 ~ N(0, 50 mm)."""
    s = Stream(seed, "particles")
    p = np.arange(n_particles, dtype=np.uint64)
    pt = PT_MIN_GEV * (PT_MAX_GEV / PT_MIN_GEV) ** s.uniform(p * np.uint64(8) + np.uint64(0))
    eta = -ETA_MAX + 2.0 * ETA_MAX * s.uniform(p * np.uint64(8) + np.uint64(1))
    phi0 = 2.0 * np.pi * s.uniform(p * np.uint64(8) + np.uint64(2))
    q = np.where(s.uniform(p * np.uint64(8) + np.uint64(3)) < 0.5, -1.0, 1.0)
    z0 = VERTEX_SIGMA_Z_MM * s.normal(p * np.uint64(4) + np.uint64(2))  # counters 8p+4, 8p+5
    return dict(pt=pt, eta=eta, phi0=phi0, q=q, z0=z0)


def wrap_phi(phi):
    """Wrap to (-pi, pi]."""
    w = np.mod(phi + np.pi, 2.0 * np.pi) - np.pi
    return np.where(w <= -np.pi, w + 2.0 * np.pi, w)


def generate_event(n_particles: int, noise_frac: float, seed: int, smear: bool = True):
    """One event.  Returns dict with
    hits        fp32 [N,3] = (r/1000, phi/pi, z/1000)   (BASELINE.json "Features")
    particle_id int32 [N]  (-1 for noise), layer int32 [N]   -- truth, tests only
    particles   the drawn particle parameters
    true_phi/true_z  fp64 unsmeared crossing per hit (nan for noise)   -- tests only
    """
    P = draw_particles(n_particles, seed)
    nl = len(LAYER_R_MM)
    pid = np.repeat(np.arange(n_particles), nl)
    lay = np.tile(np.arange(nl), n_particles)
    r = LAYER_R_MM[lay]
    phi, z, _, reach = helix_layer_crossing(P["pt"][pid], P["eta"][pid], P["phi0"][pid], P["q"][pid], P["z0"][pid], r)
    ok = reach & (np.abs(z) < Z_MAX_MM)
    pid, lay, r, phi, z = pid[ok], lay[ok], r[ok], phi[ok], z[ok]
    true_phi, true_z = phi.copy(), z.copy()
    if smear:
        sm = Stream(seed, "smear")
        c = (pid * nl + lay).astype(np.uint64)
        phi = phi + SIGMA_RPHI_MM * sm.normal(c * np.uint64(2)) / r
        z = z + SIGMA_Z_MM * sm.normal(c * np.uint64(2) + np.uint64(1))
    n_true = len(pid)
    n_noise = int(round(noise_frac * n_true))
    ns = Stream(seed, "noise")
    k = np.arange(n_noise, dtype=np.uint64)
    nlay = np.minimum((ns.uniform(k * np.uint64(3)) * nl).astype(np.int64), nl - 1)
    nphi = 2.0 * np.pi * ns.uniform(k * np.uint64(3) + np.uint64(1))
    nz = -Z_MAX_MM + 2.0 * Z_MAX_MM * ns.uniform(k * np.uint64(3) + np.uint64(2))
    pid = np.concatenate([pid, -np.ones(n_noise, dtype=np.int64)])
    lay = np.concatenate([lay, nlay])
    r = np.concatenate([r, LAYER_R_MM[nlay]])
    phi = wrap_phi(np.concatenate([phi, nphi]))
    z = np.concatenate([z, nz])
    true_phi = np.concatenate([true_phi, np.full(n_noise, np.nan)])
    true_z = np.concatenate([true_z, np.full(n_noise, np.nan)])
    # shuffle: stable argsort of per-hit random keys (a uniformly random permutation)
    keys = Stream(seed, "shuffle").u64(np.arange(len(pid), dtype=np.uint64))
    perm = np.argsort(keys, kind="stable")
    hits = np.stack([r / 1000.0, phi / np.pi, z / 1000.0], axis=1)[perm].astype(np.float32)
    return dict(hits=np.ascontiguousarray(hits), particle_id=pid[perm].astype(np.int32),
                layer=lay[perm].astype(np.int32), particles=P, n_true=n_true, n_noise=n_noise,
                true_phi=true_phi[perm], true_z=true_z[perm])


def generate_batch(n_particles: int, noise_frac: float, seeds):
    """Concatenate events (BASELINE.json configs[3]): hits [N,3], event_offsets int32 [B+1], truth."""
    evs = [generate_event(n_particles, noise_frac, s) for s in seeds]
    off = np.zeros(len(evs) + 1, dtype=np.int32)
    off[1:] = np.cumsum([len(e["hits"]) for e in evs])
    pid = np.concatenate([np.where(e["particle_id"] >= 0, e["particle_id"] + i * n_particles, -1)
                          for i, e in enumerate(evs)]).astype(np.int32)
    return dict(hits=np.ascontiguousarray(np.concatenate([e["hits"] for e in evs])), event_offsets=off,
                particle_id=pid, layer=np.concatenate([e["layer"] for e in evs]), events=evs)


def truth_edges(particle_id, layer, hits):
    """Consecutive same-particle hits (inner->outer layer): the 'truth graph' of reading C-16."""
    idx = np.nonzero(particle_id >= 0)[0]
    order = idx[np.lexsort((layer[idx], particle_id[idx]))]
    same = particle_id[order[1:]] == particle_id[order[:-1]]
    return order[:-1][same].astype(np.int32), order[1:][same].astype(np.int32)
