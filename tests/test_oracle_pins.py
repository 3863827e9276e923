"""Pins for the CPU oracle (oracle/mlpf_oracle.py) against things other than itself:
invariants the paper states, closed forms, a library transformer block, and an independent
loop restatement.  Citations are PAPER.md lines; P-numbers follow DESIGN.md / SURVEY.md 8(c)."""
import math
import numpy as np
import pytest

import synth
import oracle
from synth.configs import ModelCfg

TINY = ModelCfg(n_layers=2, d_model=32, n_heads=4, d_ff=64)
TINY_RELU = ModelCfg(n_layers=1, d_model=16, n_heads=2, d_ff=32, activation="relu")


def _setup(m=TINY, lens=(5, 9), seed=3, pad_frac=0.0):
    X, off = synth.make_events(lens, seed=seed, pad_frac=pad_frac)
    W = synth.make_weights(m, seed=seed + 100)
    return X, off, W


# ------------------------------------------------------------------ P1: softmax rows (Eq. 4)
def test_p1_attention_rows_positive_and_sum_to_one():
    rng = np.random.default_rng(0)
    q, k = rng.standard_normal((11, 8)) * 3, rng.standard_normal((11, 8)) * 3
    valid = np.array([1, 1, 0, 1, 1, 1, 0, 1, 1, 1, 1], bool)
    A = oracle.attention_weights(q, k, valid)
    assert (A >= 0).all()
    np.testing.assert_allclose(A.sum(axis=1), 1.0, atol=1e-12)
    assert (A[:, ~valid] == 0).all()
    # closed form for 2 keys: softmax = logistic of the score difference / sqrt(d_k)
    q2, k2 = rng.standard_normal((1, 4)), rng.standard_normal((2, 4))
    A2 = oracle.attention_weights(np.repeat(q2, 2, 0), k2, np.array([True, True]))
    diff = float(q2[0] @ (k2[0] - k2[1])) / math.sqrt(4)
    assert abs(A2[0, 0] - 1.0 / (1.0 + math.exp(-diff))) < 1e-12


# ------------------------------------------------------------------ P2: FlashAttention is exact (L154)
@pytest.mark.parametrize("tile", [1, 3, 7, 64])
def test_p2_tiled_online_softmax_equals_naive(tile):
    rng = np.random.default_rng(1)
    n, d, H = 37, 32, 4
    q, k, v = (rng.standard_normal((n, d)) * 2 for _ in range(3))
    valid = rng.random(n) > 0.2
    a = oracle.attention_event(q, k, v, valid, H)
    b = oracle.attention_event_tiled(q, k, v, valid, H, tile=tile)
    np.testing.assert_allclose(a, b, atol=1e-12, rtol=0)


# ------------------------------------------------------------------ P3: set input, no positions (L124-L126)
def test_p3_permutation_equivariance_within_event():
    X, off, W = _setup(lens=(7, 12), pad_frac=0.2)
    lg, rg = oracle.forward(X, off, W, TINY)
    rng = np.random.default_rng(5)
    perm = np.concatenate([rng.permutation(7), 7 + rng.permutation(12)])
    lg2, rg2 = oracle.forward(X[perm], off, W, TINY)
    np.testing.assert_allclose(lg2, lg[perm], atol=1e-11)
    np.testing.assert_allclose(rg2, rg[perm], atol=1e-11)


# ------------------------------------------------------------------ P4: padding / packing (L128)
def test_p4_padding_rows_change_nothing_and_garbage_is_ignored():
    X, off, W = _setup(lens=(6, 10))
    lg, rg = oracle.forward(X, off, W, TINY)
    # insert pad rows (type 0) with garbage features in the middle and at the end of event 0
    pad = np.full((3, synth.N_FEAT), 1e30, np.float32)
    pad[:, 0] = 0.0
    Xp = np.concatenate([X[:2], pad[:1], X[2:6], pad[1:], X[6:]], axis=0)
    offp = np.array([0, 9, 19], np.int32)
    keep = np.array([0, 1, 3, 4, 5, 6] + list(range(9, 19)))
    lgp, rgp = oracle.forward(Xp, offp, W, TINY)
    np.testing.assert_allclose(lgp[keep], lg, atol=1e-11)
    np.testing.assert_allclose(rgp[keep], rg, atol=1e-11)
    assert (lgp[[2, 7, 8]] == 0).all() and (rgp[[2, 7, 8]] == 0).all()
    assert np.isfinite(lgp).all() and np.isfinite(rgp).all()


def test_p4_event_alone_equals_event_packed_any_order():
    X, off, W = _setup(lens=(4, 9, 6))
    lg, rg = oracle.forward(X, off, W, TINY)
    for e in range(3):
        a, b = off[e], off[e + 1]
        l1, r1 = oracle.forward(X[a:b], np.array([0, b - a]), W, TINY)
        np.testing.assert_allclose(l1, lg[a:b], atol=1e-11)
        np.testing.assert_allclose(r1, rg[a:b], atol=1e-11)
    # reversed packing order
    Xr = np.concatenate([X[off[2]:off[3]], X[off[1]:off[2]], X[off[0]:off[1]]])
    offr = np.array([0, 6, 15, 19])
    lr, _ = oracle.forward(Xr, offr, W, TINY)
    np.testing.assert_allclose(lr[:6], lg[off[2]:off[3]], atol=1e-11)
    np.testing.assert_allclose(lr[15:], lg[off[0]:off[1]], atol=1e-11)


def test_a15_empty_and_fully_padded_events():
    m = TINY
    W = synth.make_weights(m, seed=9)
    X, off = synth.make_events((5, 0, 4), seed=2)
    X[5:] = 0.0                                    # last event entirely pad rows
    lg, rg = oracle.forward(X, off, W, m)
    assert np.isfinite(lg).all() and (lg[5:] == 0).all() and (rg[5:] == 0).all()
    l0, r0 = oracle.forward(np.zeros((0, synth.N_FEAT), np.float32), np.array([0]), W, m)
    assert l0.shape == (0, 9) and r0.shape == (0, 5)


# ------------------------------------------------------------------ P5: parameter count (L158: ~5.1 M)
def test_p5_parameter_count_of_paper_topology():
    """Two parallel 3-block encoders (L156) = 6 blocks of d=256, dff=4d, plus embeddings and six
    heads.  Under readings A3-A11 the count must land near the paper's 'approximately 5.1 million'."""
    d, F, dff = 256, 55, 1024
    block = 2 * d + (3 * d * d + 3 * d) + (d * d + d) + 2 * d + (dff * d + dff) + (d * dff + d)
    emb = lambda T: T * (d * F + d + d * d + d)
    head = lambda k: d * d + d + k * d + k
    six_heads = head(1) + head(9) + head(1) + head(1) + head(2) + head(1)   # binary, PID, 4 regression
    total2 = 6 * block + emb(2) + six_heads + 2 * 2 * d                     # + one final LN per encoder
    total4 = 6 * block + emb(4) + six_heads + 2 * 2 * d
    assert abs(total2 - 5.1e6) / 5.1e6 < 0.06
    assert abs(total4 - 5.1e6) / 5.1e6 < 0.09
    # dff = 2d or d would be far off -> supports reading A10 (dff = 4d)
    block_small = block - 2 * (dff - 512) * d - (dff - 512)
    assert abs(6 * block_small + emb(2) + six_heads - 5.1e6) / 5.1e6 > 0.2
    # and synth.param_count agrees with a hand count for the single-stack config
    m = synth.model_cfg("cfg3")
    hand = emb(4) + 6 * block + 2 * d + head(9) + head(1) + head(1) + head(2) + head(1)
    assert synth.param_count(m) == hand
    # the paper's own topology as a config (two stacks, binary head, 4 embedding nets): the 5.46 M of the hand count
    assert synth.param_count(synth.model_cfg("paper2")) == total4


# ------------------------------------------------------------------ P6: single-element event = MLP path
def test_p6_single_element_event_closed_form():
    m = TINY
    X, off, W = _setup(m, lens=(1,))
    lg, rg = oracle.forward(X, off, W, m)
    f64 = lambda a: np.asarray(a, np.float64)
    x = f64(X[0]); t = int(X[0, 0]); d = m.d_model
    gelu = lambda z: np.array([0.5 * v * (1 + math.erf(v / math.sqrt(2))) for v in z])
    def ln(v, g, b):
        mu = v.mean(); var = ((v - mu) ** 2).mean()
        return (v - mu) / math.sqrt(var + 1e-5) * f64(g) + f64(b)
    h = f64(W[f"emb.{t}.W2"]) @ gelu(f64(W[f"emb.{t}.W1"]) @ x + f64(W[f"emb.{t}.b1"])) + f64(W[f"emb.{t}.b2"])
    for l in range(m.n_layers):
        p = f"layer.{l}."
        u = ln(h, W[p + "ln1.g"], W[p + "ln1.b"])
        v = f64(W[p + "Wqkv"])[2 * d:] @ u + f64(W[p + "bqkv"])[2 * d:]      # a = 1: o = v
        h = h + f64(W[p + "Wo"]) @ v + f64(W[p + "bo"])
        u2 = ln(h, W[p + "ln2.g"], W[p + "ln2.b"])
        h = h + f64(W[p + "W2"]) @ gelu(f64(W[p + "W1"]) @ u2 + f64(W[p + "b1"])) + f64(W[p + "b2"])
    z = ln(h, W["lnf.g"], W["lnf.b"])
    logits = f64(W["cls.W2"]) @ gelu(f64(W["cls.W1"]) @ z + f64(W["cls.b1"])) + f64(W["cls.b2"])
    np.testing.assert_allclose(lg[0], logits, atol=1e-12)
    r2 = f64(W["reg.2.W2"]) @ gelu(f64(W["reg.2.W1"]) @ z + f64(W["reg.2.b1"])) + f64(W["reg.2.b2"])
    np.testing.assert_allclose(rg[0, 2:4], r2, atol=1e-12)       # (sin phi, cos phi) head -> columns 2,3


# ------------------------------------------------------------------ P7: library transformer block
@pytest.mark.parametrize("act,stacks", [("gelu", 1), ("relu", 1), ("relu", 2)])
def test_p7_block_equals_torch_transformer_encoder_layer(act, stacks):
    """Pre-LN block ([98], L156) vs torch.nn.TransformerEncoderLayer(norm_first=True) in fp64,
    with a key-padding mask; an independent library implementation of the same block."""
    import torch
    m = ModelCfg(n_layers=1, d_model=32, n_heads=4, d_ff=64, activation=act, n_stacks=stacks)
    W = synth.make_weights(m, seed=21)
    rng = np.random.default_rng(4)
    n = 13
    h = rng.standard_normal((n, m.d_model))
    valid = np.ones(n, bool); valid[[3, 9]] = False
    pre = synth.stack_prefix(m, stacks - 1)            # the last stack: "enc1." for the two-stack topology
    out = oracle.encoder_layer(h, valid, np.array([0, n]), W, 0, m, stack_prefix=pre)
    W = {k[len(pre):]: v for k, v in W.items() if k.startswith(pre)}
    layer = torch.nn.TransformerEncoderLayer(m.d_model, m.n_heads, m.d_ff, dropout=0.0, activation=act,
                                             batch_first=True, norm_first=True, dtype=torch.float64)
    sd = {"self_attn.in_proj_weight": W["layer.0.Wqkv"], "self_attn.in_proj_bias": W["layer.0.bqkv"],
          "self_attn.out_proj.weight": W["layer.0.Wo"], "self_attn.out_proj.bias": W["layer.0.bo"],
          "linear1.weight": W["layer.0.W1"], "linear1.bias": W["layer.0.b1"],
          "linear2.weight": W["layer.0.W2"], "linear2.bias": W["layer.0.b2"],
          "norm1.weight": W["layer.0.ln1.g"], "norm1.bias": W["layer.0.ln1.b"],
          "norm2.weight": W["layer.0.ln2.g"], "norm2.bias": W["layer.0.ln2.b"]}
    layer.load_state_dict({k: torch.tensor(v, dtype=torch.float64) for k, v in sd.items()})
    layer.train()                                  # dropout=0; avoids the fused inference fast path
    with torch.no_grad():
        ref = layer(torch.tensor(h)[None], src_key_padding_mask=torch.tensor(~valid)[None])[0].numpy()
    np.testing.assert_allclose(out[valid], ref[valid], atol=1e-11)


# ------------------------------------------------------------------ P8: independent loop restatement
def _loop_forward(X, off, W, m):
    """Scalar-loop restatement of the whole path, written separately from oracle/ (no numpy
    matmul, no shared helpers) for tiny inputs only."""
    f = lambda a: [[float(v) for v in row] for row in np.asarray(a, np.float64)]
    fv = lambda a: [float(v) for v in np.asarray(a, np.float64)]
    def matvec(Wm, b, x):
        return [sum(Wm[o][i] * x[i] for i in range(len(x))) + b[o] for o in range(len(Wm))]
    def act(v):
        if m.activation == "relu":
            return [max(a, 0.0) for a in v]
        return [0.5 * a * (1.0 + math.erf(a / math.sqrt(2.0))) for a in v]
    def ln(v, g, b):
        mu = sum(v) / len(v)
        var = sum((a - mu) ** 2 for a in v) / len(v)
        return [(a - mu) / math.sqrt(var + m.ln_eps) * g[i] + b[i] for i, a in enumerate(v)]
    Wl = {k: (f(v) if v.ndim == 2 else fv(v)) for k, v in W.items()}
    N = len(X); d = m.d_model; H = m.n_heads; hd = d // H
    types = [min(max(int(X[i][0]), 0), 4) for i in range(N)]
    h = []
    for i in range(N):
        t = types[i]
        if t == 0:
            h.append([0.0] * d); continue
        x = [float(v) for v in X[i]]
        h.append(matvec(Wl[f"emb.{t}.W2"], Wl[f"emb.{t}.b2"], act(matvec(Wl[f"emb.{t}.W1"], Wl[f"emb.{t}.b1"], x))))
    h_emb = h
    finals = []
    for s_ in range(m.n_stacks):
      pre = "" if m.n_stacks == 1 else f"enc{s_}."
      h = [list(r) for r in h_emb]
      for l in range(m.n_layers):
        p = f"{pre}layer.{l}."
        qkv = [matvec(Wl[p + "Wqkv"], Wl[p + "bqkv"], ln(h[i], Wl[p + "ln1.g"], Wl[p + "ln1.b"])) for i in range(N)]
        o = [[0.0] * d for _ in range(N)]
        for e in range(len(off) - 1):
            rows = range(int(off[e]), int(off[e + 1]))
            keys = [j for j in rows if types[j] != 0]
            for i in rows:
                for hh in range(H):
                    if not keys:
                        continue
                    s = [sum(qkv[i][hh * hd + c] * qkv[j][d + hh * hd + c] for c in range(hd)) / math.sqrt(hd) for j in keys]
                    mx = max(s); w = [math.exp(a - mx) for a in s]; z = sum(w)
                    for c in range(hd):
                        o[i][hh * hd + c] = sum(w[jj] / z * qkv[j][2 * d + hh * hd + c] for jj, j in enumerate(keys))
        for i in range(N):
            a = matvec(Wl[p + "Wo"], Wl[p + "bo"], o[i])
            h1 = [h[i][c] + a[c] for c in range(d)]
            g = act(matvec(Wl[p + "W1"], Wl[p + "b1"], ln(h1, Wl[p + "ln2.g"], Wl[p + "ln2.b"])))
            b2 = matvec(Wl[p + "W2"], Wl[p + "b2"], g)
            h[i] = [h1[c] + b2[c] for c in range(d)]
      finals.append((pre, h))
    logits, regs, binary = [], [], []
    for i in range(N):
        if types[i] == 0:
            logits.append([0.0] * m.n_classes); regs.append([0.0] * sum(m.reg_dims)); binary.append(0.0); continue
        zz = [ln(hh[i], Wl[pre + "lnf.g"], Wl[pre + "lnf.b"]) if m.final_ln else hh[i] for pre, hh in finals]
        zc, zr = zz[0], zz[-1]                 # classification stack -> (binary, PID); regression stack -> regressions
        logits.append(matvec(Wl["cls.W2"], Wl["cls.b2"], act(matvec(Wl["cls.W1"], Wl["cls.b1"], zc))))
        r = []
        for k in range(len(m.reg_dims)):
            r += matvec(Wl[f"reg.{k}.W2"], Wl[f"reg.{k}.b2"], act(matvec(Wl[f"reg.{k}.W1"], Wl[f"reg.{k}.b1"], zr)))
        regs.append(r)
        if m.binary_head:
            binary.append(matvec(Wl["bin.W2"], Wl["bin.b2"], act(matvec(Wl["bin.W1"], Wl["bin.b1"], zc)))[0])
    out = np.array(logits).reshape(N, m.n_classes), np.array(regs).reshape(N, sum(m.reg_dims))
    return out + (np.array(binary),) if m.binary_head else out


TINY_NOLN = ModelCfg(n_layers=1, d_model=16, n_heads=2, d_ff=32, final_ln=False)
TINY_TWO = ModelCfg(n_layers=2, d_model=16, n_heads=4, d_ff=32, activation="relu", n_stacks=2, binary_head=True)


@pytest.mark.parametrize("m,lens,pad", [(TINY_RELU, (3, 8, 1), 0.0), (TINY, (5, 4), 0.3), (TINY_NOLN, (6, 3), 0.2)])
def test_p8_independent_loop_restatement(m, lens, pad):
    X, off = synth.make_events(lens, seed=11, pad_frac=pad)
    W = synth.make_weights(m, seed=12)
    lg, rg = oracle.forward(X, off, W, m)
    lg2, rg2 = _loop_forward(X, off, W, m)
    np.testing.assert_allclose(lg, lg2, atol=1e-10)
    np.testing.assert_allclose(rg, rg2, atol=1e-10)


def test_p8_type_ids_outside_0_to_4_are_clamped():
    """Reading A1: ids are clamped to 0..4: -1 -> pad row (outputs 0, not a key), 5 and 7.9 -> type 4."""
    m = TINY_RELU
    X, off = synth.make_events((9,), seed=2)
    W = synth.make_weights(m, seed=3)
    X[1, 0], X[4, 0], X[6, 0] = -1.0, 5.0, 7.9
    lg, rg = oracle.forward(X, off, W, m)
    lg2, rg2 = _loop_forward(X, off, W, m)
    np.testing.assert_allclose(lg, lg2, atol=1e-10)
    np.testing.assert_allclose(rg, rg2, atol=1e-10)
    assert (lg[1] == 0).all() and (rg[1] == 0).all() and np.abs(lg[4]).sum() > 0
    assert oracle.element_types(X).tolist()[:7] == [int(X[0, 0]), 0, int(X[2, 0]), int(X[3, 0]), 4, int(X[5, 0]), 4]
    X4 = X.copy(); X4[4, 0] = 4.0; X4[6, 0] = 4.0          # same rows declared as type 4, feature 0 restored after
    t4 = oracle.element_types(X4)
    assert np.array_equal(t4, oracle.element_types(X))


def test_p8_two_parallel_encoders_and_binary_head_loop_restatement():
    """shared embedding -> two parallel encoders; (binary, PID) read the classification
    encoder, the four regression heads read the regression encoder."""
    m = TINY_TWO
    X, off = synth.make_events((4, 7, 1), seed=21, pad_frac=0.2)
    W = synth.make_weights(m, seed=22)
    lg, rg, bn = oracle.forward(X, off, W, m, with_binary=True)
    lg2, rg2, bn2 = _loop_forward(X, off, W, m)
    np.testing.assert_allclose(lg, lg2, atol=1e-10)
    np.testing.assert_allclose(rg, rg2, atol=1e-10)
    np.testing.assert_allclose(bn, bn2, atol=1e-10)
    # the stacks really are independent: zeroing the regression encoder's weights leaves (binary, PID) unchanged
    Wz = {k: (np.zeros_like(v) if k.startswith("enc1.") else v) for k, v in W.items()}
    lg3, rg3, bn3 = oracle.forward(X, off, Wz, m, with_binary=True)
    assert np.array_equal(lg3, lg) and np.array_equal(bn3, bn) and not np.allclose(rg3, rg)


# ------------------------------------------------------------------ P9 / P10: bias identities
def test_p9_outputs_invariant_to_key_bias():
    m = TINY
    X, off, W = _setup(m, lens=(9, 4))
    lg, rg = oracle.forward(X, off, W, m)
    W2 = {k: v.copy() for k, v in W.items()}
    d = m.d_model
    for l in range(m.n_layers):
        W2[f"layer.{l}.bqkv"][d:2 * d] += np.linspace(-3, 3, d).astype(np.float32)
    lg2, rg2 = oracle.forward(X, off, W2, m)
    np.testing.assert_allclose(lg2, lg, atol=1e-10)
    np.testing.assert_allclose(rg2, rg, atol=1e-10)


def test_p10_value_bias_passes_through_attention():
    rng = np.random.default_rng(8)
    n, d, H = 10, 16, 2
    q, k, v = (rng.standard_normal((n, d)) for _ in range(3))
    bv = rng.standard_normal(d)
    valid = rng.random(n) > 0.3
    a = oracle.attention_event(q, k, v, valid, H)
    b = oracle.attention_event(q, k, v + bv[None, :], valid, H)
    np.testing.assert_allclose(b, a + bv[None, :], atol=1e-12)


# ------------------------------------------------------------------ P11: normalisation at any n
def test_p11_identical_rows_and_self_concatenation():
    m = TINY
    X, off, W = _setup(m, lens=(1,))
    l1, r1 = oracle.forward(X, off, W, m)
    Xn = np.repeat(X, 17, axis=0)
    ln_, rn = oracle.forward(Xn, np.array([0, 17]), W, m)
    np.testing.assert_allclose(ln_, np.repeat(l1, 17, 0), atol=1e-11)
    np.testing.assert_allclose(rn, np.repeat(r1, 17, 0), atol=1e-11)
    X2, off2 = synth.make_events((6,), seed=30)
    la, _ = oracle.forward(X2, off2, W, m)
    lb, _ = oracle.forward(np.concatenate([X2, X2]), np.array([0, 12]), W, m)
    np.testing.assert_allclose(lb[:6], la, atol=1e-11)
    np.testing.assert_allclose(lb[6:], la, atol=1e-11)


# ------------------------------------------------------------------ P12: uniform / identity limits
def test_p12_zero_query_projection_gives_mean_of_valid_values():
    rng = np.random.default_rng(2)
    n, d, H = 9, 8, 2
    k, v = rng.standard_normal((n, d)), rng.standard_normal((n, d))
    valid = np.array([1, 0, 1, 1, 1, 0, 1, 1, 1], bool)
    o = oracle.attention_event(np.zeros((n, d)), k, v, valid, H)
    np.testing.assert_allclose(o, np.repeat(v[valid].mean(axis=0)[None], n, 0), atol=1e-13)


def test_p12_identity_encoder_limit():
    m = TINY
    X, off, W = _setup(m, lens=(5, 7))
    W0 = {k: v.copy() for k, v in W.items()}
    for l in range(m.n_layers):
        for nm in ("Wo", "bo", "W2", "b2"):
            W0[f"layer.{l}.{nm}"][...] = 0
    lg, rg = oracle.forward(X, off, W0, m)
    z = oracle.layer_norm(oracle.embed(X, W0, m), W0["lnf.g"].astype(np.float64), W0["lnf.b"].astype(np.float64), m.ln_eps)
    l2, r2, _ = oracle.heads(z, W0, m)
    np.testing.assert_allclose(lg, l2, atol=1e-12)
    np.testing.assert_allclose(rg, r2, atol=1e-12)


def test_p15_sharp_weights_make_attention_non_uniform():
    """The sharp weight set must move the outputs by far more than the BF16 tolerance when keys
    leak across events; here: outputs change when another event is (wrongly) merged in."""
    m = synth.model_cfg("cfg1")
    X, off = synth.make_named_events("cfg1")
    W = synth.sharpen(synth.make_weights("cfg1"), m)
    lg, _ = oracle.forward(X, off, W, m)
    lg_merged, _ = oracle.forward(X, np.array([0, off[-1]]), W, m)     # one big event = leak
    rel, _ = oracle.parity_metrics(lg_merged, lg, np.ones(len(X), bool))
    assert rel > 0.1


# ------------------------------------------------------------------ P13: integer schedule, brute force
def test_p13_schedule_bruteforce():
    X, off = synth.make_events((130, 0, 300, 7, 129), seed=6, pad_frac=0.15)
    TQ = 128
    s = oracle.schedule(X, off, TQ)
    N = int(off[-1])
    t = np.clip(X[:, 0].astype(int), 0, 4)
    for i in range(N):
        e = max(k for k in range(len(off) - 1) if off[k] <= i and off[k + 1] > i)
        assert s["row_event"][i] == e and s["row_pos"][i] == i - off[e]
        assert s["valid"][i] == int(t[i] != 0)
    for e in range(len(off) - 1):
        assert s["n_valid"][e] == sum(1 for i in range(off[e], off[e + 1]) if t[i] != 0)
    to = s["type_offsets"]
    assert to[0] == 0 and all(to[k] % 128 == 0 for k in range(6))
    for ty in range(1, 5):
        rows = [i for i in range(N) if t[i] == ty]                 # stable: ascending original row
        assert to[ty + 1] - to[ty] == (len(rows) + 127) // 128 * 128
        assert list(s["type_perm"][to[ty]:to[ty] + len(rows)]) == rows
        assert (s["type_perm"][to[ty] + len(rows):to[ty + 1]] == -1).all()
        assert [s["sorted_row"][i] for i in rows] == list(range(to[ty], to[ty] + len(rows)))
    assert all(s["sorted_row"][i] == -1 for i in range(N) if t[i] == 0)
    # pad-row compaction, brute force: the c-th valid row (global order) is compacted row c; events stay contiguous
    valid_rows = [i for i in range(N) if t[i] != 0]
    assert [int(s["comp_row"][i]) for i in valid_rows] == list(range(len(valid_rows)))
    assert all(s["comp_row"][i] == -1 for i in range(N) if t[i] == 0)
    for e in range(len(off) - 1):
        mine = [int(s["comp_row"][i]) for i in range(int(off[e]), int(off[e + 1])) if t[i] != 0]
        assert mine == list(range(int(s["offsets_c"][e]), int(s["offsets_c"][e + 1])))
    assert s["offsets_c"][0] == 0 and s["offsets_c"][-1] == len(valid_rows)
    for slot, row in enumerate(s["type_perm"]):
        assert s["comp_type_perm"][slot] == (-1 if row < 0 else s["comp_row"][row])
    # work list: longest event first, ties by id, tiles ascending
    lens = [int(off[e + 1] - off[e]) for e in range(len(off) - 1)]
    expect = []
    for e in sorted(range(len(lens)), key=lambda e: (-lens[e], e)):
        expect += [(e, q) for q in range(-(-lens[e] // TQ))]
    assert [tuple(r) for r in s["work_list"]] == expect
    assert len(expect) == 3 + 2 + 2 + 1


def test_round_bf16_is_rne():
    x = np.array([1.0, 1.00390625, 1.01171875, 1.0 + 2 ** -8 + 2 ** -20, -3.1415927, 0.0, 65504.0], np.float32)
    r = oracle.round_bf16(x)
    assert r[0] == 1.0
    assert r[1] == 1.0                      # exactly half-way between 1 and 1+2^-7 -> even (1.0)
    assert r[2] == np.float32(1.015625)     # half-way between 1+2^-7 and 1+2^-6 -> even mantissa (1+2^-6)
    assert r[3] == np.float32(1.0078125)    # just above half-way -> up
    import torch
    tt = torch.tensor(np.random.default_rng(0).standard_normal(4096).astype(np.float32))
    np.testing.assert_array_equal(oracle.round_bf16(tt.numpy()), tt.to(torch.bfloat16).to(torch.float32).numpy())


# ------------------------------------------------------------------ candidate building (NEXT-2; Eq. 2)
def _cand_inputs(lens=(7, 0, 12, 5), seed=11, pad_frac=0.2, n_classes=9):
    X, off = synth.make_events(lens, seed=seed, pad_frac=pad_frac)
    rng = np.random.default_rng(seed + 1)
    N = int(off[-1])
    logits = rng.standard_normal((N, n_classes)).astype(np.float32)
    regress = (0.5 * rng.standard_normal((N, 5))).astype(np.float32)
    return X, off, logits, regress


def test_candidates_invert_eq2_and_recover_phi():
    """Closed form: feed pT' = log(pT_t / pT_in), E' = log(E_t / E_in) (Eq. 2) and (sin, cos) of a known phi in
    all four quadrants; decoding must give back pT_t, E_t and phi."""
    X, off, logits, _ = _cand_inputs(lens=(40, 24), pad_frac=0.0)
    N = int(off[-1])
    rng = np.random.default_rng(5)
    pt_t = np.exp(rng.standard_normal(N)); e_t = pt_t * np.cosh(rng.uniform(-3, 3, N))
    phi = rng.uniform(-math.pi, math.pi, N)
    phi[:4] = [0.25 * math.pi, 0.75 * math.pi, -0.75 * math.pi, -0.25 * math.pi]
    eta = rng.uniform(-5, 5, N)
    reg = np.stack([np.log(pt_t / X[:, 1].astype(np.float64)), eta, np.sin(phi), np.cos(phi),
                    np.log(e_t / X[:, 4].astype(np.float64))], axis=1)
    logits[:, 0] = -10.0                                   # every element yields a candidate
    c = oracle.build_candidates(X, off, logits, reg)
    assert c["cand_offsets"].tolist() == [0, 40, 64]
    assert np.array_equal(c["cand_elem"], np.arange(N))
    assert np.allclose(c["cand_p4"][:, 0], pt_t, rtol=1e-12)
    assert np.allclose(c["cand_p4"][:, 1], eta, rtol=0, atol=0)
    assert np.allclose(c["cand_p4"][:, 2], phi, rtol=0, atol=1e-12)
    assert np.allclose(c["cand_p4"][:, 3], e_t, rtol=1e-12)


def test_candidates_loop_restatement_and_offset_invariants():
    """Brute force, element by element, with math.* scalars; pad rows and class-0 rows are dropped, order is the
    element order, offsets are per event (empty event included)."""
    X, off, logits, reg = _cand_inputs()
    logits[3, :] = 1.0                                     # an exact tie: lowest class (0) wins -> dropped
    c = oracle.build_candidates(X, off, logits, reg)
    exp_off, elem, pid, p4 = [0], [], [], []
    for e in range(len(off) - 1):
        for i in range(int(off[e]), int(off[e + 1])):
            best = 0
            for k in range(1, logits.shape[1]):
                if logits[i, k] > logits[i, best]:
                    best = k
            if int(X[i, 0]) != 0 and best != 0:
                elem.append(i); pid.append(best)
                p4.append((float(X[i, 1]) * math.exp(float(reg[i, 0])), float(reg[i, 1]),
                           math.atan2(float(reg[i, 2]), float(reg[i, 3])), float(X[i, 4]) * math.exp(float(reg[i, 4]))))
        exp_off.append(len(elem))
    assert c["cand_offsets"].tolist() == exp_off
    assert c["cand_elem"].tolist() == elem and c["cand_pid"].tolist() == pid
    assert 3 not in elem
    assert np.allclose(c["cand_p4"], np.asarray(p4).reshape(-1, 4), rtol=1e-14, atol=0)
    # invariants: every candidate's element lies inside its event, strictly increasing inside an event
    for e in range(len(off) - 1):
        seg = c["cand_elem"][c["cand_offsets"][e]:c["cand_offsets"][e + 1]]
        assert np.all((seg >= off[e]) & (seg < off[e + 1])) and np.all(np.diff(seg) > 0)
    assert c["cand_offsets"][2] == c["cand_offsets"][1]    # the empty event


def test_candidates_packing_invariance():
    """An event decoded alone gives the same candidates as the same event packed after others (indices shifted)."""
    X, off, logits, reg = _cand_inputs()
    c = oracle.build_candidates(X, off, logits, reg)
    a, b = int(off[2]), int(off[3])
    c1 = oracle.build_candidates(X[a:b], np.array([0, b - a]), logits[a:b], reg[a:b])
    s, t = c["cand_offsets"][2], c["cand_offsets"][3]
    assert np.array_equal(c1["cand_elem"] + a, c["cand_elem"][s:t])
    assert np.array_equal(c1["cand_pid"], c["cand_pid"][s:t])
    assert np.array_equal(c1["cand_p4"], c["cand_p4"][s:t])


# ------------------------------------------------------------------ the judging metrics themselves (reading A14)
def test_parity_metrics_hand_computed_example():
    """3 rows x 2 columns written out by hand: row 2 is a pad row (excluded from the rms AND from the maximum),
    column 1 of the oracle is all zero over valid rows (zero rms)."""
    ref = np.array([[3.0, 0.0], [-4.0, 0.0], [100.0, 7.0]])
    got = np.array([[3.3, 0.0], [-4.2, 0.0], [55.0, 55.0]])
    valid = np.array([True, True, False])
    rel, rms = oracle.parity_metrics(got, ref, valid)
    # column 0: rms = sqrt((9 + 16) / 2) = 3.5355339...; row 0: 0.3 / max(3, 3.5355) ; row 1: 0.2 / max(4, 3.5355) = 0.05
    assert abs(rms[0] - math.sqrt(12.5)) < 1e-15 and rms[1] == 0.0
    assert abs(rel - 0.3 / math.sqrt(12.5)) < 1e-12
    # a non-zero result where the oracle column is identically zero is an infinite relative error, never NaN
    got[0, 1] = 1e-9
    rel, _ = oracle.parity_metrics(got, ref, valid)
    assert rel == np.inf
    # no valid rows: nothing to compare
    assert oracle.parity_metrics(got, ref, np.zeros(3, bool))[0] == 0.0


def test_argmax_agreement_hand_computed_example():
    """rms over the valid rows' logits = sqrt(7.4901 / 9) = 0.912268; decidable = margin > 2 * 0.02 * rms = 0.0364907.
    Row 1 (margin 0.01) is a near tie and does not count; row 2 is a real disagreement; row 3 is a pad row."""
    ref = np.array([[1.0, 0.0, -1.0], [0.5, 0.49, 0.0], [0.0, 2.0, 1.0], [9.0, 9.0, 9.0]])
    got = np.array([[0.9, 0.1, -1.0], [0.48, 0.5, 0.0], [0.0, 1.0, 2.1], [0.0, 0.0, 0.0]])
    valid = np.array([True, True, True, False])
    agree, dec_frac, raw = oracle.argmax_agreement(got, ref, valid, tol_rel=2e-2)
    assert agree == 0.5 and abs(dec_frac - 2.0 / 3.0) < 1e-15 and abs(raw - 1.0 / 3.0) < 1e-15
    # margin exactly at the threshold is NOT decidable (strict >): scale row 1's margin to the threshold
    rms = math.sqrt(7.4901 / 9.0)
    assert abs(rms - 0.912268) < 1e-6
    agree2, dec2, _ = oracle.argmax_agreement(ref, ref, valid)
    assert agree2 == 1.0 and abs(dec2 - 2.0 / 3.0) < 1e-15


def test_attention_event_row_blocks_equal_dense_weights_times_values():
    """attention_event processes query rows in blocks (memory only): with row_block = 3 on n = 11 (blocks that do
    not divide n, pad keys present) it must equal A @ V with A from attention_weights (Eq. 4), head by head."""
    rng = np.random.default_rng(8)
    n, H, hd = 11, 2, 4
    q, k, v = (rng.standard_normal((n, H * hd)) * 2 for _ in range(3))
    valid = np.array([1, 0, 1, 1, 1, 0, 1, 1, 1, 1, 0], bool)
    o = oracle.attention_event(q, k, v, valid, H, row_block=3)
    for h in range(H):
        sl = slice(h * hd, (h + 1) * hd)
        A = oracle.attention_weights(q[:, sl], k[:, sl], valid)
        np.testing.assert_allclose(o[:, sl], A @ v[:, sl], atol=1e-13)
    np.testing.assert_allclose(o, oracle.attention_event(q, k, v, valid, H, row_block=2048), atol=1e-13)


def test_bf16_matrix_set_matches_the_header():
    """include/mlpf.h: "the library rounds (RNE) the matrices that feed tensor-core GEMMs (emb W2, Wqkv, Wo, W1, W2,
    cls.W1, reg.k.W1 [, bin.W1]); emb W1, the output rows (cls.W2, reg.k.W2 [, bin.W2]) and all vectors stay fp32"."""
    import os, re
    hdr = open(os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "include", "mlpf.h")).read()
    mlist = re.search(r"GEMMs \(([^)]*)\)", hdr).group(1)
    for nm in ("emb W2", "Wqkv", "Wo", "W1", "W2", "cls.W1", "reg.k.W1", "bin.W1"):
        assert nm in mlist, nm
    for name in ("cfg1", "paper2"):
        m = synth.model_cfg(name)
        exp = set()
        for t in range(1, 5):
            exp.add(f"emb.{t}.W2")
        for s in range(m.n_stacks):
            for l in range(m.n_layers):
                exp |= {f"{synth.stack_prefix(m, s)}layer.{l}.{k}" for k in ("Wqkv", "Wo", "W1", "W2")}
        exp |= {"cls.W1"} | {f"reg.{k}.W1" for k in range(4)} | ({"bin.W1"} if m.binary_head else set())
        got = {n for n, _ in synth.weight_names(m) if oracle.is_bf16_matrix(n)}
        assert got == exp
        W = synth.make_weights(m, seed=1)
        Wq = oracle.quantize_weights(W)
        for n, _ in synth.weight_names(m):
            same = np.array_equal(Wq[n], W[n])
            assert same == (n not in exp), n       # random fp32 weights are never bf16-exact


def test_candidates_binary_rule_is_the_papers():
    """L156: keep iff the binary score sigmoid(b) > 0.5, PID = argmax over ALL classes (class 0 allowed)."""
    X, off, logits, reg = _cand_inputs(lens=(6, 5), pad_frac=0.0)
    N = int(off[-1])
    b = np.linspace(-2.0, 2.0, N).astype(np.float32)
    b[3] = 0.0                                             # sigmoid(0) = 0.5 exactly: NOT above 0.5
    X[7, :] = 0.0                                          # a pad row with a positive score is still dropped
    b[7] = 3.0
    logits[9, :] = -1.0; logits[9, 0] = 5.0                # class 0 wins and is kept under the binary rule
    c = oracle.build_candidates(X, off, logits, reg, binary=b)
    keep = [i for i in range(N) if X[i, 0] != 0 and 1.0 / (1.0 + math.exp(-float(b[i]))) > 0.5]
    assert c["cand_elem"].tolist() == keep and 3 not in keep and 7 not in keep and 9 in keep
    assert c["cand_pid"][keep.index(9)] == 0
    assert c["cand_offsets"].tolist() == [0, sum(1 for i in keep if i < 6), len(keep)]
