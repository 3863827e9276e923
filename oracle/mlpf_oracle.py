"""CPU oracle for the MLPF encoder forward pass -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Plain, slow, fp64 numpy restatement of what the hot path computes, written from
/root/reference/PAPER.md (CMS-PFT-25-001, arxiv 2601.17554) and the readings A1-A19
listed in DESIGN.md.  Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s
cpu_baseline / `--impl reference` legs may import this package.  It shares no code
with `paper_2601_17554_b200/` (the CUDA path) and never calls it.

The forward pass is a *definition* (FlashAttention "preserv[es] exact
attention values", L154), so the oracle is that definition written out: dense per-event
attention with the n x n weight matrix materialised (the paper's own "naive attention
formulation via matrix multiplication" CPU fallback, L154/L220), no tiling of the softmax,
no fusion, no reduced precision.  numpy matmul / scipy erf are the only library steps.

Pins (tests/test_oracle_pins.py): P1 softmax rows sum to 1; P2 tiled online-softmax == naive;
P3 permutation equivariance; P4 padding / packing invariance; P5 parameter count vs the
paper's 5.1 M; P6 single-element closed form; P7 torch.nn.TransformerEncoderLayer (fp64);
P8 independent loop restatement on tiny events; P9/P10 K-/V-bias identities; P11 n identical
rows; P12 W_q = 0 (mean of values) and identity-encoder limits; P13 brute-force schedule.
Trained-weight (physics) behaviour is "parity unpinned": no weights or data exist here.

Weight dict keys and shapes: synth.configs.weight_names (== blob order, include/mlpf.h).
Every matrix is [out, in]; y = x W^T + b.
"""
from __future__ import annotations

import numpy as np
from scipy.special import erf as _erf

# matrices the CUDA BF16 path feeds to tensor-core GEMMs; the oracle
# rounds exactly these (RNE) when asked, so weight quantisation is not counted as error.
_BF16_LEAVES = ("Wqkv", "Wo", "W1", "W2")


def round_bf16(a):
    """Round-to-nearest-even of float32 values to bfloat16 precision (returned as float32)."""
    a = np.ascontiguousarray(a, dtype=np.float32)
    u = a.view(np.uint32).astype(np.uint64)
    lsb = (u >> 16) & 1
    u = (u + 0x7FFF + lsb) & 0xFFFF0000
    return u.astype(np.uint32).view(np.float32).reshape(a.shape)


def is_bf16_matrix(name: str) -> bool:
    """True for the weight matrices the BF16 path stores in bf16.  fp32 exceptions: the first
    embedding layer emb.t.W1 (raw features span 1e-2..1e4) and the 14 output rows cls.W2 /
    reg.k.W2 (applied in an fp32 epilogue)."""
    leaf = name.split(".")[-1]
    if leaf not in _BF16_LEAVES:
        return False
    if name.startswith("emb.") and leaf == "W1":
        return False
    if (name.startswith("cls.") or name.startswith("reg.") or name.startswith("bin.")) and leaf == "W2":
        return False
    return True


def quantize_weights(W: dict) -> dict:
    """W-bf16 mode: the bf16-stored matrices rounded (RNE), everything else untouched."""
    return {k: (round_bf16(v) if is_bf16_matrix(k) else v) for k, v in W.items()}


# ----------------------------------------------------------------------------- pointwise pieces
def activation(x, kind: str):
    """ReLU or exact-erf GELU (BASELINE.json configs; reading A6)."""
    if kind == "relu":
        return np.maximum(x, 0.0)
    if kind == "gelu":
        return 0.5 * x * (1.0 + _erf(x / np.sqrt(2.0)))
    raise ValueError(kind)


def layer_norm(x, g, b, eps):
    """Per-row LayerNorm, biased variance, affine (reading A8; 'layer normalization', L156)."""
    mu = x.mean(axis=-1, keepdims=True)
    var = ((x - mu) ** 2).mean(axis=-1, keepdims=True)
    return (x - mu) / np.sqrt(var + eps) * g + b


def linear(x, Wm, b):
    return x @ np.asarray(Wm, dtype=np.float64).T + np.asarray(b, dtype=np.float64)


def element_types(X):
    """Reading A1/A2: feature 0 holds the type id; clamp to 0..4; 0 = pad row."""
    t = np.asarray(X)[:, 0].astype(np.int64) if len(X) else np.zeros(0, np.int64)
    return np.clip(t, 0, 4)


# ----------------------------------------------------------------------------- steps a1..a8
def embed(X, W, m):
    """a1: per-type two-layer FFN (L156 'tracks and clusters are each embedded ... using simple
    FFNs'); readings A3-A5: one net per type, Linear(55->d) act Linear(d->d); pad rows -> 0."""
    X64 = np.asarray(X, dtype=np.float64)
    t = element_types(X)
    h = np.zeros((X64.shape[0], m.d_model), dtype=np.float64)
    for ty in range(1, m.n_types + 1):
        rows = np.nonzero(t == ty)[0]
        if rows.size == 0:
            continue
        a = activation(linear(X64[rows], W[f"emb.{ty}.W1"], W[f"emb.{ty}.b1"]), m.activation)
        h[rows] = linear(a, W[f"emb.{ty}.W2"], W[f"emb.{ty}.b2"])
    return h


def attention_weights(q, k, valid):
    """Eq. 4 (L150): A = softmax(Q K^T / sqrt(d_k)) for ONE head of ONE event, keys restricted
    to valid rows (reading A2).  Returns the dense [n, n] matrix (zero columns for pad keys)."""
    n, hd = q.shape
    A = np.zeros((n, n), dtype=np.float64)
    kv = np.nonzero(valid)[0]
    if kv.size == 0:
        return A                                   # reading A15: empty key set -> no weights
    s = (q @ k[kv].T) / np.sqrt(float(hd))
    s = s - s.max(axis=1, keepdims=True)
    e = np.exp(s)
    A[:, kv] = e / e.sum(axis=1, keepdims=True)
    return A


def attention_event(q, k, v, valid, n_heads, row_block=2048):
    """Multi-head SDPA for one event: o_i = sum_j A_ij v_j per head, heads concatenated [94].
    Query rows are independent, so they are processed in blocks only to bound memory; each
    block's rows of A are fully materialised (no online softmax)."""
    n, d = q.shape
    hd = d // n_heads
    o = np.zeros((n, d), dtype=np.float64)
    for h in range(n_heads):
        sl = slice(h * hd, (h + 1) * hd)
        for r0 in range(0, n, row_block):
            r1 = min(n, r0 + row_block)
            kv = np.nonzero(valid)[0]
            if kv.size == 0:
                continue
            s = (q[r0:r1, sl] @ k[kv, sl].T) / np.sqrt(float(hd))
            s -= s.max(axis=1, keepdims=True)
            e = np.exp(s)
            a = e / e.sum(axis=1, keepdims=True)
            o[r0:r1, sl] = a @ v[kv, sl]
    return o


def attention_event_tiled(q, k, v, valid, n_heads, tile=7):
    """Pin P2 only: the FlashAttention recurrence (running max, running sum, rescaled
    accumulator over key tiles), to show it equals `attention_event` (L154 'exact')."""
    n, d = q.shape
    hd = d // n_heads
    kv = np.nonzero(valid)[0]
    o = np.zeros((n, d), dtype=np.float64)
    if kv.size == 0:
        return o
    for h in range(n_heads):
        sl = slice(h * hd, (h + 1) * hd)
        mrun = np.full((n, 1), -np.inf)
        lrun = np.zeros((n, 1))
        acc = np.zeros((n, hd))
        for j0 in range(0, kv.size, tile):
            jj = kv[j0:j0 + tile]
            s = (q[:, sl] @ k[jj, sl].T) / np.sqrt(float(hd))
            mnew = np.maximum(mrun, s.max(axis=1, keepdims=True))
            p = np.exp(s - mnew)
            corr = np.exp(mrun - mnew)
            lrun = lrun * corr + p.sum(axis=1, keepdims=True)
            acc = acc * corr + p @ v[jj, sl]
            mrun = mnew
        o[:, sl] = acc / lrun
    return o


def encoder_layer(h, valid, offsets, W, l, m, dump=None, attn=attention_event, stack_prefix=""):
    """One pre-LN transformer block (L156 + [98]; readings A5-A10):
       h <- h + Wo.MHA(LN1(h)) + bo ;  h <- h + W2.act(W1.LN2(h) + b1) + b2.
    stack_prefix: "" for one stack, "enc0." / "enc1." for the paper's two parallel encoders (L156)."""
    p = f"{stack_prefix}layer.{l}."
    d = m.d_model
    u = layer_norm(h, W[p + "ln1.g"].astype(np.float64), W[p + "ln1.b"].astype(np.float64), m.ln_eps)
    qkv = linear(u, W[p + "Wqkv"], W[p + "bqkv"])
    q, k, v = qkv[:, :d], qkv[:, d:2 * d], qkv[:, 2 * d:]
    o = np.zeros_like(h)
    for e in range(len(offsets) - 1):
        a, b = int(offsets[e]), int(offsets[e + 1])
        if b > a:
            o[a:b] = attn(q[a:b], k[a:b], v[a:b], valid[a:b], m.n_heads)
    h1 = h + linear(o, W[p + "Wo"], W[p + "bo"])
    u2 = layer_norm(h1, W[p + "ln2.g"].astype(np.float64), W[p + "ln2.b"].astype(np.float64), m.ln_eps)
    g = activation(linear(u2, W[p + "W1"], W[p + "b1"]), m.activation)
    h2 = h1 + linear(g, W[p + "W2"], W[p + "b2"])
    if dump is not None:                                  # keys carry the stack prefix: "enc1.layer.0.o"
        dump[p + "u"] = u
        dump[p + "qkv"] = qkv
        dump[p + "o"] = o
        dump[p + "h_attn"] = h1
        dump[p + "u2"] = u2
        dump[p + "g"] = g
        dump[p + "h"] = h2
    return h2


def heads(z_cls, W, m, z_reg=None):
    """a8: two-layer FFN heads (L156 'six two-layer FFN heads'; reading A11): PID logits [N,9]
    and (pT', eta, sin phi, cos phi, E') [N,5] as raw head outputs (reading A12); with
    m.binary_head also the binary "valid" logit [N] (L156 'binary primary target particle
    classification', Fig. 2).  Binary and PID heads read z_cls (the classification encoder),
    the regression heads read z_reg (the regression encoder, L156); one stack: z_reg = z_cls."""
    if z_reg is None:
        z_reg = z_cls
    hc = activation(linear(z_cls, W["cls.W1"], W["cls.b1"]), m.activation)
    logits = linear(hc, W["cls.W2"], W["cls.b2"])
    regs = []
    for k in range(len(m.reg_dims)):
        hr = activation(linear(z_reg, W[f"reg.{k}.W1"], W[f"reg.{k}.b1"]), m.activation)
        regs.append(linear(hr, W[f"reg.{k}.W2"], W[f"reg.{k}.b2"]))
    binary = None
    if getattr(m, "binary_head", False):
        hb = activation(linear(z_cls, W["bin.W1"], W["bin.b1"]), m.activation)
        binary = linear(hb, W["bin.W2"], W["bin.b2"])[:, 0]
    return logits, np.concatenate(regs, axis=1), binary


def forward(X, offsets, W, m, dump=None, attn=attention_event, with_binary=False):
    """Whole path a1..a8 for packed events.  Returns (logits [N,9], regress [N,5]) float64, and with
    with_binary=True also the binary logit [N] (needs m.binary_head); pad rows (type 0) are exactly 0
    (reading A2).  m.n_stacks == 2 is the paper's topology (L156): the shared embedding feeds two
    parallel encoders, stack 0 -> (binary, PID), stack 1 -> the regression heads."""
    X = np.asarray(X, dtype=np.float32)
    offsets = np.asarray(offsets, dtype=np.int64)
    t = element_types(X)
    valid = t != 0
    h0 = embed(X, W, m)
    if dump is not None:
        dump["h0"] = h0
    n_stacks = getattr(m, "n_stacks", 1)
    zs = []
    for s in range(n_stacks):
        pre = "" if n_stacks == 1 else f"enc{s}."
        h = h0
        for l in range(m.n_layers):
            h = encoder_layer(h, valid, offsets, W, l, m, dump=dump, attn=attn, stack_prefix=pre)
        z = layer_norm(h, W[pre + "lnf.g"].astype(np.float64), W[pre + "lnf.b"].astype(np.float64), m.ln_eps) if m.final_ln else h
        if dump is not None:
            dump[pre + "z"] = z
        zs.append(z)
    logits, regress, binary = heads(zs[0], W, m, z_reg=zs[-1])
    logits[~valid] = 0.0
    regress[~valid] = 0.0
    if with_binary:
        if binary is None:
            raise ValueError("with_binary needs a model with binary_head")
        binary[~valid] = 0.0
        return logits, regress, binary
    return logits, regress


# ----------------------------------------------------------------------------- step a0 (integers)
def schedule(X, offsets, tile_q: int):
    """a0: the integer packing / schedule arrays, by the plain rules:
    row_event, row_pos, valid, n_valid per event, the stable by-type row order with each type
    segment padded to a multiple of 128 rows (type_offsets in padded 'sorted' space), and the
    attention work list (event, q_tile) ordered by descending n_e, then ascending event id,
    then ascending q_tile; events with n_e = 0 contribute no tiles.  Pad-row compaction: the valid rows keep
    their order and are numbered consecutively (comp_row, -1 for pad rows; comp_type_perm = type_perm through
    that numbering), so event e owns the compacted rows offsets_c[e] .. offsets_c[e+1]-1 (offsets_c =
    running sum of n_valid): pad rows take part in nothing (reading A2), the kernels skip them altogether."""
    offsets = np.asarray(offsets, dtype=np.int64)
    E = len(offsets) - 1
    N = int(offsets[-1])
    t = element_types(np.asarray(X)[:N])
    row_event = np.zeros(N, np.int32)
    row_pos = np.zeros(N, np.int32)
    n_valid = np.zeros(E, np.int32)
    for e in range(E):
        a, b = int(offsets[e]), int(offsets[e + 1])
        row_event[a:b] = e
        row_pos[a:b] = np.arange(b - a)
        n_valid[e] = int((t[a:b] != 0).sum())
    valid = (t != 0).astype(np.int32)
    # stable counting sort of the valid rows by type 1..4; each segment starts at a multiple of 128
    type_count = np.array([(t == ty).sum() for ty in range(5)], np.int64)
    type_offsets = np.zeros(6, np.int32)            # [0]=0 unused slot for type 0; [ty]..[ty+1] for ty>=1
    pos = 0
    seg_start = np.zeros(5, np.int64)
    for ty in range(1, 5):
        seg_start[ty] = pos
        type_offsets[ty] = pos
        pos += (int(type_count[ty]) + 127) // 128 * 128
    type_offsets[5] = pos
    sorted_row = np.full(N, -1, np.int32)           # original row -> slot in sorted space (-1: pad)
    fill = seg_start.copy()
    for i in range(N):
        ty = int(t[i])
        if ty != 0:
            sorted_row[i] = fill[ty]
            fill[ty] += 1
    type_perm = np.full(int(type_offsets[5]), -1, np.int32)   # sorted slot -> original row (-1: filler)
    for i in range(N):
        if sorted_row[i] >= 0:
            type_perm[sorted_row[i]] = i
    comp_row = np.full(N, -1, np.int32)
    nxt = 0
    for i in range(N):
        if t[i] != 0:
            comp_row[i] = nxt
            nxt += 1
    offsets_c = np.zeros(E + 1, np.int32)
    for e in range(E):
        offsets_c[e + 1] = offsets_c[e] + n_valid[e]
    comp_type_perm = np.where(type_perm >= 0, comp_row[np.maximum(type_perm, 0)], -1).astype(np.int32)
    lens = offsets[1:] - offsets[:-1]
    order = sorted(range(E), key=lambda e: (-int(lens[e]), e))
    work = []
    for e in order:
        for qt in range((int(lens[e]) + tile_q - 1) // tile_q):
            work.append((e, qt))
    work = np.asarray(work, np.int32).reshape(-1, 2)
    return dict(row_event=row_event, row_pos=row_pos, valid=valid, n_valid=n_valid,
                type_offsets=type_offsets, sorted_row=sorted_row, type_perm=type_perm,
                comp_row=comp_row, offsets_c=offsets_c, comp_type_perm=comp_type_perm, work_list=work)


# ----------------------------------------------------------------------------- error metric (A14)
def parity_metrics(got, ref, valid):
    """Reading A14: rel_i = |g - o| / max(|o|, rms_c), rms_c = oracle RMS of that output column
    over valid rows.  Returns (max rel, per-column rms)."""
    got = np.asarray(got, np.float64)
    ref = np.asarray(ref, np.float64)
    v = np.asarray(valid, bool)
    if v.sum() == 0:
        return 0.0, np.zeros(ref.shape[1])
    rms = np.sqrt((ref[v] ** 2).mean(axis=0))
    den = np.maximum(np.abs(ref[v]), rms[None, :])
    err = np.abs(got[v] - ref[v])
    # an all-zero oracle column has den = 0: exact agreement counts as 0, anything else as infinite
    rel = np.where(den > 0, err / np.where(den > 0, den, 1.0), np.where(err == 0, 0.0, np.inf))
    return float(rel.max()), rms


def argmax_agreement(got_logits, ref_logits, valid, tol_rel=2e-2):
    """Reading A14: agreement over 'decidable' rows (oracle top-2 margin > 2*tol*rms of logits).
    Returns (agreement on decidable rows, decidable fraction, raw agreement)."""
    v = np.asarray(valid, bool)
    g = np.asarray(got_logits, np.float64)[v]
    r = np.asarray(ref_logits, np.float64)[v]
    if len(r) == 0:
        return 1.0, 1.0, 1.0
    rms = np.sqrt((r ** 2).mean())
    srt = np.sort(r, axis=1)
    margin = srt[:, -1] - srt[:, -2]
    dec = margin > 2.0 * tol_rel * rms
    same = g.argmax(axis=1) == r.argmax(axis=1)
    agree_dec = float(same[dec].mean()) if dec.any() else 1.0
    return agree_dec, float(dec.mean()), float(same.mean())
