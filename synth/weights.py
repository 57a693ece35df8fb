"""Seeded network weights (SURVEY.md §8(c) "W", reading C-15).

The paper's trained Exa.TrkX models are not available, so every
Linear(fan_in -> fan_out) gets W ~ U(-b, b), b = sqrt(6/fan_in) (Kaiming-uniform, ReLU
gain) and bias ~ U(+-1/sqrt(fan_in)), drawn in fp64 from a named sub-stream of the
seed and stored fp32.  With bf16=True the fp32 values are rounded (RNE) to
bf16-representable fp32 before anyone sees them, so weight quantisation is not an
error source.  Input maker only: no pipeline arithmetic here.
"""
from __future__ import annotations

import numpy as np

from .rng import Stream


def round_to_bf16(x: np.ndarray) -> np.ndarray:
    """Round fp32 to the nearest bf16 (ties to even), returned as fp32."""
    u = np.ascontiguousarray(x, dtype=np.float32).view(np.uint32).astype(np.uint64)
    u = (u + np.uint64(0x7FFF) + ((u >> np.uint64(16)) & np.uint64(1))) & np.uint64(0xFFFF0000)
    return u.astype(np.uint32).view(np.float32).reshape(np.shape(x))


def make_mlp(seed: int, name: str, dims, bf16: bool):
    """Returns dict(dims=[...], weight=[fp32 [out,in]...], bias=[fp32 [out]...])."""
    dims = [int(d) for d in dims]
    weight, bias = [], []
    for l in range(len(dims) - 1):
        fi, fo = dims[l], dims[l + 1]
        s = Stream(seed, f"w:{name}:{l}")
        bw = np.sqrt(6.0 / fi)
        bb = 1.0 / np.sqrt(fi)
        w = (2.0 * s.uniform(np.arange(fo * fi, dtype=np.uint64)) - 1.0) * bw
        b = (2.0 * s.uniform(np.arange(fo * fi, fo * fi + fo, dtype=np.uint64)) - 1.0) * bb
        w = w.reshape(fo, fi).astype(np.float32)
        b = b.astype(np.float32)
        if bf16:
            w = round_to_bf16(w)
        weight.append(np.ascontiguousarray(w))
        bias.append(np.ascontiguousarray(b))
    return dict(dims=dims, weight=weight, bias=bias)


def make_model(cfg: dict, seed: int | None = None):
    """All five MLP groups of one config (see synth.configs)."""
    seed = cfg["weight_seed"] if seed is None else seed
    bf = cfg["precision"] == "bf16"
    H = cfg["gnn_hidden"]
    return dict(
        embed=make_mlp(seed, "embed", cfg["embed_dims"], bf),
        filter=make_mlp(seed, "filter", cfg["filter_dims"], bf),
        node_enc=make_mlp(seed, "node_enc", [3, H, H], bf),
        edge_enc=make_mlp(seed, "edge_enc", [4, H, H], bf),
        edge_net=make_mlp(seed, "edge_net", [3 * H, H, H], bf),
        node_net=make_mlp(seed, "node_net", [3 * H, H, H], bf),
        edge_dec=make_mlp(seed, "edge_dec", [3 * H, H, 1], bf),
    )
