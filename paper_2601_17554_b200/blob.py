"""Flat weight blob writer (include/mlpf.h 'weight blob'): argument marshalling only, no arithmetic."""
from __future__ import annotations
import struct
import numpy as np

MAGIC = b"MLPFBLOB"
VERSION = 2
HEADER_BYTES = 256


def pack_blob(W: dict, m) -> bytes:
    """W: name -> float32 array (synth.weight_names order/shapes); m: model config with n_layers,
    d_model, n_heads, d_ff, n_feat, n_types, n_classes, reg_dims, activation, final_ln, ln_eps."""
    reg = list(m.reg_dims) + [0] * (4 - len(m.reg_dims))
    n_stacks, binary = int(getattr(m, "n_stacks", 1)), 1 if getattr(m, "binary_head", False) else 0
    hdr = struct.pack("<8s9I4I2If2I", MAGIC, VERSION, m.n_layers, m.d_model, m.n_heads, m.d_ff, m.n_feat,
                      m.n_types, m.n_classes, len(m.reg_dims), *reg,
                      0 if m.activation == "relu" else 1, 1 if m.final_ln else 0, float(m.ln_eps), n_stacks, binary)
    hdr = hdr + b"\0" * (HEADER_BYTES - len(hdr))
    d, F, dff = m.d_model, m.n_feat, m.d_ff
    names = []
    for t in range(1, m.n_types + 1):
        names += [f"emb.{t}.W1", f"emb.{t}.b1", f"emb.{t}.W2", f"emb.{t}.b2"]
    pre = lambda s: "" if n_stacks == 1 else f"enc{s}."
    for s in range(n_stacks):
        for l in range(m.n_layers):
            p = f"{pre(s)}layer.{l}."
            names += [p + k for k in ("ln1.g", "ln1.b", "Wqkv", "bqkv", "Wo", "bo", "ln2.g", "ln2.b", "W1", "b1", "W2", "b2")]
    for s in range(n_stacks):
        names += [pre(s) + "lnf.g", pre(s) + "lnf.b"]
    if binary:
        names += ["bin.W1", "bin.b1", "bin.W2", "bin.b2"]
    names += ["cls.W1", "cls.b1", "cls.W2", "cls.b2"]
    for k in range(len(m.reg_dims)):
        names += [f"reg.{k}.W1", f"reg.{k}.b1", f"reg.{k}.W2", f"reg.{k}.b2"]
    parts = [hdr]
    for n in names:
        parts.append(np.ascontiguousarray(W[n], dtype="<f4").tobytes())
    return b"".join(parts)
