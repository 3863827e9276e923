"""Seeded synthetic CMS-like events (stand-ins for the paper's simulation samples,
PAPER.md Table 1, which are not available).  Recipe: DESIGN.md "Input recipe".

Row layout (fp32, 55 features): x[0] = element type id (0 pad, 1 track, 2 ECAL,
3 HCAL, 4 HF); x[1] = pT = exp(z); x[2] = eta ~ U[-5,5]; x[3] = phi ~ U[-pi,pi];
x[4] = E = pT*cosh(eta); x[5:55] ~ N(0,1).  Pad rows are all-zero.
"""
from __future__ import annotations
import numpy as np
from .configs import BASE_SEED, CFG_INDEX, N_FEAT

CMS_TYPE_P = (0.60, 0.20, 0.15, 0.05)      # track, ECAL, HCAL, HF
UNIFORM_TYPE_P = (0.25, 0.25, 0.25, 0.25)


def _rows(rng, n, type_p, hard_frac=0.0, pad_frac=0.0):
    x = np.zeros((n, N_FEAT), dtype=np.float64)
    t = rng.choice(np.arange(1, 5), size=n, p=np.asarray(type_p))
    z = rng.standard_normal(n)
    if hard_frac > 0.0:
        hard = (t == 1) & (rng.random(n) < hard_frac)       # 20% of tracks: pT ~ lognormal(1,1)
        z = np.where(hard, z + 1.0, z)
    pt = np.exp(z)
    eta = rng.uniform(-5.0, 5.0, n)
    phi = rng.uniform(-np.pi, np.pi, n)
    x[:, 0] = t
    x[:, 1] = pt
    x[:, 2] = eta
    x[:, 3] = phi
    x[:, 4] = pt * np.cosh(eta)
    x[:, 5:] = rng.standard_normal((n, N_FEAT - 5))
    if pad_frac > 0.0:
        pad = rng.random(n) < pad_frac
        x[pad, :] = 0.0
    return x.astype(np.float32)


def _lengths(name, rng):
    if name == "cfg1":
        return [64, 192]
    if name == "cfg2":
        return [int(v) for v in rng.integers(500, 2001, size=16)]
    if name == "cfg3":
        return [int(v) for v in np.rint(np.clip(rng.normal(5000, 1000, 8), 1000, 9000))]
    if name == "cfg4":
        return [int(v) for v in np.rint(np.clip(rng.lognormal(np.log(3000), 0.5, 64), 200, 12000))]
    if name == "cfg5a":
        return [16384]
    if name == "cfg5b":
        return [8192] * 32
    if name in ("paper", "paper2"):
        return [int(v) for v in np.rint(np.clip(rng.normal(5000, 1000, 4), 1000, 9000))]
    raise KeyError(name)


def make_named_events(name: str, seed: int | None = None, max_events: int | None = None):
    """Return (X[N,55] float32, event_offsets[E+1] int32) for one of the named workloads."""
    if seed is None:
        seed = BASE_SEED + CFG_INDEX[name]
    rng = np.random.default_rng(seed)
    lens = _lengths(name, rng)
    if max_events is not None:
        lens = lens[:max_events]
    if name in ("cfg1", "cfg2"):
        kw = dict(type_p=UNIFORM_TYPE_P)
    elif name in ("cfg3", "cfg4", "paper", "paper2"):
        kw = dict(type_p=CMS_TYPE_P, hard_frac=0.20)
    else:
        kw = dict(type_p=CMS_TYPE_P, hard_frac=0.20, pad_frac=0.10)
    return make_events(lens, rng=rng, **kw)


def make_events(lens, seed: int = 0, rng=None, type_p=UNIFORM_TYPE_P, hard_frac=0.0, pad_frac=0.0):
    """Events with explicit lengths (used by the edge-case tests: empty, ragged, padded)."""
    if rng is None:
        rng = np.random.default_rng(seed)
    xs = [_rows(rng, int(n), type_p, hard_frac, pad_frac) for n in lens]
    off = np.zeros(len(lens) + 1, dtype=np.int32)
    off[1:] = np.cumsum([int(n) for n in lens])
    X = np.concatenate(xs, axis=0) if xs else np.zeros((0, N_FEAT), np.float32)
    return np.ascontiguousarray(X, dtype=np.float32), off
