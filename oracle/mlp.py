"""Dense layers in fp64 (oracle building blocks; "multilayer perceptrons").

Weights are stored (out, in) row-major like the C ABI's trk_mlp (include/trk.h).
"""
from __future__ import annotations

import numpy as np

LN_EPS = 1e-5  # reading C-13/C-18


def linear(x, w, b):
    """y = x W^T + b, all promoted to fp64."""
    return np.asarray(x, np.float64) @ np.asarray(w, np.float64).T + np.asarray(b, np.float64)


def relu(v):
    return np.maximum(v, 0.0)


def sigmoid(v):
    """sigma(x) = 1 / (1 + exp(-x))  (reading C-18)."""
    return 1.0 / (1.0 + np.exp(-np.asarray(v, np.float64)))


def layernorm(v):
    """LayerNorm over the last axis, biased variance, eps = 1e-5, no affine (reading C-13)."""
    mu = v.mean(axis=-1, keepdims=True)
    var = ((v - mu) ** 2).mean(axis=-1, keepdims=True)
    return (v - mu) / np.sqrt(var + LN_EPS)


def mlp_forward(x, mlp):
    """Linear+ReLU for all but the last layer; last layer is a plain Linear (S1, S3 shape)."""
    h = np.asarray(x, np.float64)
    n = len(mlp["weight"])
    for l in range(n):
        h = linear(h, mlp["weight"][l], mlp["bias"][l])
        if l < n - 1:
            h = relu(h)
    return h
