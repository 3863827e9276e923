"""Seeded random-init weights (BASELINE.json: "Xavier-uniform weights from the seed").

Matrices ~ U[-a, a], a = sqrt(6/(fan_in+fan_out)); biases ~ U[-0.05, 0.05];
LayerNorm gamma = 1 + U[-0.1, 0.1], beta = U[-0.1, 0.1] (reading A18: non-trivial
vectors so that a dropped bias / affine term is visible in parity).  fp32 master weights.
"""
from __future__ import annotations
import numpy as np
from .configs import BASE_SEED, CFG_INDEX, ModelCfg, CONFIGS, weight_names


def make_weights(m: ModelCfg | str, seed: int | None = None):
    if isinstance(m, str):
        if seed is None:
            seed = BASE_SEED + 1000 + CFG_INDEX[m]
        m = CONFIGS[m]
    if seed is None:
        seed = BASE_SEED + 1000
    rng = np.random.default_rng(seed)
    W = {}
    for name, shp in weight_names(m):
        leaf = name.split(".")[-1]
        if len(shp) == 2:
            a = np.sqrt(6.0 / (shp[0] + shp[1]))
            w = rng.uniform(-a, a, size=shp)
        elif leaf == "g":
            w = 1.0 + rng.uniform(-0.1, 0.1, size=shp)
        elif leaf == "b" and ("ln" in name):
            w = rng.uniform(-0.1, 0.1, size=shp)
        else:
            w = rng.uniform(-0.05, 0.05, size=shp)
        W[name] = np.ascontiguousarray(w, dtype=np.float32)
    return W


def sharpen(W: dict, m: ModelCfg, factor: float = 4.0):
    """The "sharp" weight set (pin P15): scale the Q rows of every Wqkv/bqkv by `factor`
    so attention is far from uniform and a masking / cross-event leak is visible."""
    out = {k: v.copy() for k, v in W.items()}
    d = m.d_model
    for s in range(m.n_stacks):
        pre = "" if m.n_stacks == 1 else f"enc{s}."
        for l in range(m.n_layers):
            out[f"{pre}layer.{l}.Wqkv"][:d, :] *= factor
            out[f"{pre}layer.{l}.bqkv"][:d] *= factor
    return out
