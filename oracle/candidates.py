"""CPU oracle for candidate building -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

The step right after the encoder forward pass: turn the per-element outputs into the per-event
list of particle candidates that the experiment software consumes ("the module
... builds the particle candidates from the model output").  Written out from the paper:

* PID: the class with the largest logit (multiclass PID head, L130/L156).  Ties -> lowest class.
* Four-momentum: the model predicts the transformed quantities of Eq. 2 (L137-L139)
      pT' = log(pT_target / pT_primary),   E' = log(E_target / E_primary),
  so the candidate's  pT = pT_primary * exp(pT'),  E = E_primary * exp(E'),  with pT_primary = x[1]
  and E_primary = x[4] of the element itself (DESIGN.md input recipe).  eta is the raw output;
  phi = atan2(sin phi, cos phi) ("parameterized through sin phi and cos phi to preserve the
  quadrant information", L126).
* Selection, the paper's rule (L156): "selecting the candidates with a binary classification score
  above 0.5, and assigning them the PID with the largest probability score": with the binary head's
  logit b_i, keep iff sigmoid(b_i) > 0.5 (and the row is not a pad row, reading A2); the PID is the
  argmax over all classes.
  DEPARTURE A23 (only for models WITHOUT a binary head, i.e. the five BASELINE.json configs whose
  single 9-class head is all there is): class 0 then stands for "no particle" and element i yields
  a candidate iff type != 0 and PID != 0.  This is not the paper's rule; it is a stop-gap.
* Output: candidates in element order (stable), grouped per event by integer offsets.

Floating point in fp64; the integer outputs (offsets, element index, PID) are exact given the
fp32 logits handed in.  Pins: tests/test_oracle_pins.py (Eq. 2 round trip, atan2 quadrants,
loop restatement, offset invariants).  Shares no code with the CUDA path.
"""
from __future__ import annotations

import numpy as np


def build_candidates(X, offsets, logits, regress, binary=None):
    """X [N,F] fp32 element features; offsets [E+1]; logits [N,C]; regress [N,5] = (pT', eta, sin phi,
    cos phi, E'); binary [N] = the binary head's logit or None (departure A23).  Returns dict(cand_offsets int32 [E+1], cand_elem int32 [M] (global row of the
    element), cand_pid int32 [M], cand_p4 float64 [M,4] = (pT, eta, phi, E))."""
    offsets = np.asarray(offsets, dtype=np.int64)
    E = len(offsets) - 1
    N = int(offsets[-1])
    X = np.asarray(X)[:N]
    logits = np.asarray(logits)[:N]
    regress = np.asarray(regress, dtype=np.float64)[:N]
    etype = np.clip(X[:, 0].astype(np.int64), 0, 4)       # reading A1: feature 0 is the type id, clamped to 0..4 as in the forward pass
    pid = np.argmax(logits, axis=1) if N else np.zeros(0, np.int64)   # first maximum wins
    if binary is None:
        keep = (etype != 0) & (pid != 0)                   # departure A23: no binary head
    else:
        b = np.asarray(binary, dtype=np.float64)[:N]
        # L156: binary score above 0.5.  The score is sigmoid(b); sigmoid is strictly increasing with sigmoid(0) = 1/2, so
        # "score > 0.5" is exactly "b > 0" (evaluating 1 / (1 + exp(-b)) in floating point would round tiny b > 0 to 0.5)
        keep = (etype != 0) & (b > 0.0)
    cand_elem = np.nonzero(keep)[0].astype(np.int32)
    cand_offsets = np.zeros(E + 1, np.int32)
    for e in range(E):
        cand_offsets[e + 1] = cand_offsets[e] + int(keep[offsets[e]:offsets[e + 1]].sum())
    r = regress[cand_elem]
    x = X[cand_elem].astype(np.float64)
    p4 = np.empty((len(cand_elem), 4), np.float64)
    p4[:, 0] = x[:, 1] * np.exp(r[:, 0])                   # Eq. 2 inverted, L137-L139
    p4[:, 1] = r[:, 1]
    p4[:, 2] = np.arctan2(r[:, 2], r[:, 3])                # L126
    p4[:, 3] = x[:, 4] * np.exp(r[:, 4])
    return dict(cand_offsets=cand_offsets, cand_elem=cand_elem, cand_pid=pid[cand_elem].astype(np.int32),
                cand_p4=p4)
