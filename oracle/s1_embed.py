"""S1 embedding MLP ("uses multilayer perceptrons (MLPs) to encode
spacepoint raw features to a new latent space"; BASELINE.json configs: 3->1024->1024->1024->12
ReLU, toy 3->64->64->8; no activation on the output)."""
from __future__ import annotations

import numpy as np

from .mlp import mlp_forward


def embed(hits_f32, mlp):
    """hits fp32 [N,3] -> embedding fp64 [N,d_e]."""
    return mlp_forward(np.asarray(hits_f32, np.float32), mlp)


def embed_f32(hits_f32, mlp):
    """The stage's interchange output: fp64 result rounded (RNE) to fp32."""
    return embed(hits_f32, mlp).astype(np.float32)
