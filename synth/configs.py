"""The five workloads of BASELINE.json `configs` as plain dicts.

Hyperparameters that the oracle calibrates (FRNN radius, filter cut, grid projection,
GNN logit median) live in synth/calibration.json, written by oracle/calibrate.py.
"""
from __future__ import annotations

import json
import os

import numpy as np

from .events import generate_batch, generate_event

_HERE = os.path.dirname(os.path.abspath(__file__))
CALIBRATION_PATH = os.path.join(_HERE, "calibration.json")

_BIG_EMBED = [3, 1024, 1024, 1024, 12]
_BIG_FILTER = [24, 1024, 1024, 1024, 1]

CONFIGS = {
    # configs[0]: toy event
    "toy": dict(n_particles=50, noise_frac=0.10, seeds=[0], weight_seed=0, precision="fp32",
                embed_dims=[3, 64, 64, 8], filter_dims=[6, 64, 1], filter_input="raw",
                degree=8, frnn_k=16, keep_frac=0.50, gnn_hidden=64, gnn_iters=4, gnn_cut=0.5,
                calibration="toy"),
    # configs[1]: pileup-50
    "pileup50": dict(n_particles=2500, noise_frac=0.10, seeds=[0], weight_seed=0, precision="bf16",
                     embed_dims=_BIG_EMBED, filter_dims=_BIG_FILTER, filter_input="emb",
                     degree=32, frnn_k=64, keep_frac=0.25, gnn_hidden=128, gnn_iters=8, gnn_cut=0.5,
                     calibration="pileup50"),
    # configs[2]: pileup-200 (headline)
    "pileup200": dict(n_particles=10000, noise_frac=0.10, seeds=[0], weight_seed=0, precision="bf16",
                      embed_dims=_BIG_EMBED, filter_dims=_BIG_FILTER, filter_input="emb",
                      degree=32, frnn_k=64, keep_frac=1.0e6 / 3.5e6, gnn_hidden=128, gnn_iters=8, gnn_cut=0.5,
                      calibration="pileup200"),
    # configs[3]: 16 pileup-50 events in one call, weights/radius/cut of pileup-50
    "batch16": dict(n_particles=2500, noise_frac=0.10, seeds=list(range(1, 17)), weight_seed=0, precision="bf16",
                    embed_dims=_BIG_EMBED, filter_dims=_BIG_FILTER, filter_input="emb",
                    degree=32, frnn_k=64, keep_frac=0.25, gnn_hidden=128, gnn_iters=8, gnn_cut=0.5,
                    calibration="pileup50"),
    # configs[4]: stress, pileup 300
    "pileup300": dict(n_particles=15000, noise_frac=0.15, seeds=[0], weight_seed=0, precision="bf16",
                      embed_dims=_BIG_EMBED, filter_dims=_BIG_FILTER, filter_input="emb",
                      degree=48, frnn_k=128, keep_frac=2.5e6 / 8.0e6, gnn_hidden=128, gnn_iters=8, gnn_cut=0.5,
                      calibration="pileup300"),
    # SURVEY.md section 8(c) reading C-2, secondary "size-matched" run of configs[2]: BASELINE.json's nominal ~110 k hits need
    # 13 600 particles with the literal geometry (7.3 hits per particle); same architecture, its own calibrated radius and cut
    "pileup200_nominal": dict(n_particles=13600, noise_frac=0.10, seeds=[0], weight_seed=0, precision="bf16",
                              embed_dims=_BIG_EMBED, filter_dims=_BIG_FILTER, filter_input="emb",
                              degree=32, frnn_k=64, keep_frac=1.0e6 / 3.5e6, gnn_hidden=128, gnn_iters=8, gnn_cut=0.5,
                              calibration="pileup200_nominal"),
    # an event of the paper's own size (~350 k spacepoints per ttbar
    # <mu>=200 event), same detector, generator and architecture as pileup-200; 43 500 particles x 7.3 hits x 1.10 noise
    "paper350k": dict(n_particles=43500, noise_frac=0.10, seeds=[0], weight_seed=0, precision="bf16",
                      embed_dims=_BIG_EMBED, filter_dims=_BIG_FILTER, filter_input="emb",
                      degree=32, frnn_k=64, keep_frac=1.0e6 / 3.5e6, gnn_hidden=128, gnn_iters=8, gnn_cut=0.5,
                      calibration="paper350k"),
}


def get_config(name: str) -> dict:
    cfg = dict(CONFIGS[name])
    cfg["name"] = name
    return cfg


def make_events(cfg: dict, n_particles: int | None = None):
    """hits fp32 [N,3], event_offsets int32 [B+1], truth arrays."""
    npart = cfg["n_particles"] if n_particles is None else n_particles
    if len(cfg["seeds"]) == 1:
        ev = generate_event(npart, cfg["noise_frac"], cfg["seeds"][0])
        off = np.array([0, len(ev["hits"])], dtype=np.int32)
        return dict(hits=ev["hits"], event_offsets=off, particle_id=ev["particle_id"], layer=ev["layer"])
    return generate_batch(npart, cfg["noise_frac"], cfg["seeds"])


def load_calibration(name: str) -> dict:
    """Stored oracle-calibrated hyperparameters: frnn_radius, filter_cut, grid_proj, gnn_logit_median."""
    with open(CALIBRATION_PATH) as f:
        return json.load(f)[name]
