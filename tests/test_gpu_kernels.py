"""Kernel-level GPU parity: the tcgen05 GEMM and flash-attention kernels (through the C ABI) against the
oracle's plain definitions (oracle.linear = numpy fp64 matmul, oracle.attention_event = Eq. 4 written out)."""
import numpy as np
import pytest

import synth
import oracle

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

import paper_2601_17554_b200 as P


@pytest.fixture(scope="module", autouse=True)
def _need_gpu():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    assert P.lib() is not None


def _bf16(a):
    return torch.from_numpy(a).cuda().to(torch.bfloat16)


@pytest.mark.parametrize("M,N,K", [(1, 64, 64), (127, 128, 64), (128, 64, 256), (300, 768, 256), (1000, 256, 2048),
                                   (257, 192, 128), (4096, 1024, 256)])
@pytest.mark.parametrize("split", [False, True])
def test_tc_gemm_matches_fp64_matmul(M, N, K, split):
    rng = np.random.default_rng(M * 7 + N + K)
    A = rng.standard_normal((M, K)).astype(np.float32)
    W = (rng.standard_normal((N, K)) / np.sqrt(K)).astype(np.float32)
    Ad, Wd = _bf16(A), _bf16(W)
    Aq = Ad.float().cpu().numpy().astype(np.float64)
    Wq = Wd.float().cpu().numpy().astype(np.float64)
    Alo = None
    if split:
        Alo = _bf16(A - Ad.float().cpu().numpy())
        Aq = Aq + Alo.float().cpu().numpy().astype(np.float64)
    got = P.tc_gemm_bf16(Ad, Wd, Alo).cpu().numpy()
    torch.cuda.synchronize()
    ref = oracle.linear(Aq, Wq, np.zeros(N))
    err = np.abs(got - ref).max()
    assert err <= 2e-5 * max(1.0, np.abs(ref).max()), err


# impl: 1 = bound-based kernel (tc_attn2.cu; these inputs take its fast path), 2 = its exact two-sweep path forced,
# 0 = round 1's lazy-rescale kernel (kept selectable through MLPF_OPT_ATTN)
# 3 / 4 = 1 / 2 with the q columns already multiplied by log2(e) / sqrt(hd) before their bf16 rounding: the form the model
# path feeds the kernel (a3's epilogue folds the softmax scale into q; the fast path then subtracts nothing from S)
IMPLS = [1, 2, 0, 3, 4]


def _attn_inputs(qkv, d, hd, impl):
    """bf16 QKV for the kernel and the fp64 (q | k | v) the oracle sees: the bf16 values, q divided by the folded scale."""
    qkv = qkv.copy()
    c = np.log2(np.e) / np.sqrt(hd) if impl >= 3 else 1.0
    qkv[:, :d] *= np.float32(c)
    QKV = _bf16(qkv)
    q64 = QKV.float().cpu().numpy().astype(np.float64)
    q64[:, :d] /= c
    return QKV, q64


@pytest.mark.parametrize("impl", IMPLS)
@pytest.mark.parametrize("hd,H", [(32, 8), (16, 4), (64, 8)])
@pytest.mark.parametrize("lens,pad", [((128,), 0.0), ((256, 64), 0.0), ((1, 129, 700, 257), 0.0), ((300, 1000), 0.15),
                                      ((0, 40, 0), 0.5), ((33, 95, 160, 417), 0.0)])
def test_tc_attention_matches_dense_softmax(hd, H, lens, pad, impl):
    d = hd * H
    rng = np.random.default_rng(hd + sum(lens))
    N = sum(lens)
    off = np.zeros(len(lens) + 1, np.int32)
    off[1:] = np.cumsum(lens)
    qkv = rng.standard_normal((N, 3 * d)).astype(np.float32)
    qkv[:, :d] *= 2.0                                     # sharper than unit-variance scores
    valid = (rng.random(N) >= pad)
    QKV, qk64 = _attn_inputs(qkv, d, hd, impl)
    kv = torch.from_numpy(valid.astype(np.int32)).cuda()
    O = P.tc_attention_bf16(QKV, kv if pad > 0 else None, off, d, H, impl=impl).float().cpu().numpy()
    if pad == 0:
        valid[:] = True
    v64 = qk64[:, 2 * d:]
    for e in range(len(lens)):
        a, b = off[e], off[e + 1]
        if b == a:
            continue
        ref = oracle.attention_event(qk64[a:b, :d], qk64[a:b, d:2 * d], v64[a:b], valid[a:b], H)
        err = np.abs(O[a:b] - ref)
        scale = np.sqrt((ref ** 2).mean()) + 1e-6
        assert (err / np.maximum(np.abs(ref), scale)).max() <= 2e-2, (e, err.max(), scale)


# ------------------------------------------------------------------------------------------- adversarial softmax inputs
def _attn_check(qkv, lens, valid, hd, H, tol=2e-2, impl=1):
    """tcgen05 attention vs oracle.attention_event (Eq. 4 written out) element by element; the scale of the floor is
    the rms of the oracle output of that event."""
    d = hd * H
    off = np.zeros(len(lens) + 1, np.int32)
    off[1:] = np.cumsum(lens)
    QKV, q64 = _attn_inputs(qkv, d, hd, impl)
    kv = None if valid is None else torch.from_numpy(valid.astype(np.int32)).cuda()
    O = P.tc_attention_bf16(QKV, kv, off, d, H, impl=impl).float().cpu().numpy()
    torch.cuda.synchronize()
    assert np.isfinite(O).all()
    vv = np.ones(len(qkv), bool) if valid is None else valid
    worst = 0.0
    for e in range(len(lens)):
        a, b = off[e], off[e + 1]
        if b == a:
            continue
        ref = oracle.attention_event(q64[a:b, :d], q64[a:b, d:2 * d], q64[a:b, 2 * d:], vv[a:b], H)
        scale = np.sqrt((ref ** 2).mean()) + 1e-6
        worst = max(worst, float((np.abs(O[a:b] - ref) / np.maximum(np.abs(ref), scale)).max()))
    assert worst <= tol, worst
    return O


@pytest.mark.parametrize("impl", IMPLS)
@pytest.mark.parametrize("hd,H", [(32, 4), (64, 2), (16, 4)])
def test_tc_attention_running_max_climbs_every_tile(hd, H, impl):
    """Keys ordered so that the row maximum rises by far more than 2^8 from one 64-key tile to the next (and, for the
    rows with a negative query coefficient, falls): the reference maximum of an online softmax has to move on every
    tile (or a one-shot bound has to be far from the first tiles' scores)."""
    rng = np.random.default_rng(hd)
    n, d = 1000, hd * H
    qkv = (0.3 * rng.standard_normal((n, 3 * d))).astype(np.float32)
    u = rng.standard_normal(d).astype(np.float32)
    u /= np.sqrt((u.reshape(H, hd) ** 2).sum(axis=1)).repeat(hd)           # unit vector per head
    ramp = np.linspace(0.0, 40.0, n, dtype=np.float32)                      # k.u rises by 0.04 per key ...
    sign = np.where(rng.random(n) < 0.5, 1.0, -1.0).astype(np.float32)
    qkv[:, :d] += 24.0 * sign[:, None] * u[None, :]                         # ... = 61 raw units per 64-key tile: 11 log2 units at hd = 64, 15 at hd = 32
    qkv[:, d:2 * d] += ramp[:, None] * u[None, :]
    _attn_check(qkv, (n,), None, hd, H, impl=impl)


@pytest.mark.parametrize("impl", IMPLS)
@pytest.mark.parametrize("hd,H", [(32, 4), (64, 2)])
def test_tc_attention_outlier_key_in_the_last_tile(hd, H, impl):
    """One key 40 sigma away from the others, in the last (ragged) tile: every row's weight ends up on it."""
    rng = np.random.default_rng(hd + 1)
    n, d = 777, hd * H
    qkv = rng.standard_normal((n, 3 * d)).astype(np.float32)
    qkv[n - 3, d:2 * d] = 40.0 * np.sign(rng.standard_normal(d))
    _attn_check(qkv, (n,), None, hd, H, impl=impl)


@pytest.mark.parametrize("impl", IMPLS)
@pytest.mark.parametrize("hd,H", [(32, 4), (64, 2)])
def test_tc_attention_only_the_last_key_is_valid(hd, H, impl):
    """Every key but the last one of each event is a pad row: O must equal that key's V row for all queries."""
    rng = np.random.default_rng(hd + 2)
    lens = (300, 131)
    n, d = sum(lens), hd * H
    qkv = rng.standard_normal((n, 3 * d)).astype(np.float32)
    valid = np.zeros(n, bool)
    valid[[299, 430]] = True
    O = _attn_check(qkv, lens, valid, hd, H, impl=impl)
    v = _bf16(qkv).float().cpu().numpy()[:, 2 * d:]
    assert np.abs(O[:300] - v[299]).max() <= 2e-2 * np.abs(v[299]).max()
    assert np.abs(O[300:] - v[430]).max() <= 2e-2 * np.abs(v[430]).max()


@pytest.mark.parametrize("impl", IMPLS)
@pytest.mark.parametrize("hd,H", [(32, 4), (64, 2)])
def test_tc_attention_sharp_scores_with_pad_rows(hd, H, impl):
    """10 % scattered pad rows together with Q x 8: a leaked pad key would carry real weight."""
    rng = np.random.default_rng(hd + 3)
    lens = (1500, 333, 900)
    n, d = sum(lens), hd * H
    qkv = rng.standard_normal((n, 3 * d)).astype(np.float32)
    qkv[:, :d] *= 8.0
    valid = rng.random(n) >= 0.10
    qkv[~valid, d:2 * d] *= 3.0                           # pad keys would win the softmax if they were not masked
    _attn_check(qkv, lens, valid, hd, H, impl=impl)


@pytest.mark.parametrize("impl", IMPLS)
@pytest.mark.parametrize("hd,H", [(32, 2), (64, 1)])
def test_tc_attention_16384_keys(hd, H, impl):
    """The longest event of BASELINE.json (config 5): 16384 elements, 10 % pad rows, scores sharper than unit variance."""
    rng = np.random.default_rng(hd + 4)
    n, d = 16384, hd * H
    qkv = rng.standard_normal((n, 3 * d)).astype(np.float32)
    qkv[:, :d] *= 3.0
    valid = rng.random(n) >= 0.10
    _attn_check(qkv, (n,), valid, hd, H, impl=impl)


@pytest.mark.parametrize("impl", IMPLS)
def test_tc_attention_huge_scores(impl):
    """Scores near +-1e3 (|q.k| / sqrt(hd) up to ~1200): exponent range, not precision, is what is exercised."""
    rng = np.random.default_rng(9)
    hd, H, n = 32, 2, 500
    d = hd * H
    qkv = rng.standard_normal((n, 3 * d)).astype(np.float32)
    qkv[:, :2 * d] *= 14.0
    _attn_check(qkv, (n,), None, hd, H, impl=impl)


# ------------------------------------------------------------------------------------------- fused post-attention block
@pytest.mark.parametrize("M,d,dff,act", [(128, 256, 1024, "gelu"), (300, 256, 1024, "relu"), (77, 64, 256, "gelu"),
                                         (1000, 128, 384, "gelu"), (20000, 256, 1024, "gelu"), (129, 256, 128, "relu")])
@pytest.mark.parametrize("next_ln", [True, False])
def test_tc_post_matches_the_block_written_out(M, d, dff, act, next_ln):
    """k_tc_post against the same steps composed from the oracle's pieces (oracle.linear / layer_norm / activation) in
    fp64 on the very bf16 operands the kernel reads: h2 to 2e-5 of its scale (fp32 accumulation), the LayerNorm outputs
    to a few bf16-pair ulps."""
    rng = np.random.default_rng(M + d + dff)
    o = rng.standard_normal((M, d)).astype(np.float32)
    h = (3.0 * rng.standard_normal((M, d)) + rng.standard_normal((M, 1))).astype(np.float32)
    mk = lambda *s: (rng.standard_normal(s) / np.sqrt(s[-1])).astype(np.float32)
    Wo, W1, W2 = mk(d, d), mk(dff, d), mk(d, dff)
    vec = lambda n, c=0.0: (c + 0.1 * rng.standard_normal(n)).astype(np.float32)
    bo, b1, b2, g2, b2ln, gn, bn = vec(d), vec(dff), vec(d), vec(d, 1.0), vec(d), vec(d, 1.0), vec(d)
    o_hi = _bf16(o)
    o_lo = _bf16(o - o_hi.float().cpu().numpy())
    Wod, W1d, W2d = _bf16(Wo), _bf16(W1), _bf16(W2)
    f64 = lambda t: t.float().cpu().numpy().astype(np.float64)
    cu = lambda a: torch.from_numpy(a).cuda()
    hd_ = cu(h.copy())
    u_hi, u_lo = P.tc_post_bf16(o_hi, o_lo, hd_, Wod, cu(bo), cu(g2), cu(b2ln), W1d, cu(b1), W2d, cu(b2),
                                cu(gn) if next_ln else None, cu(bn) if next_ln else None, 0 if act == "relu" else 1, 1e-5)
    torch.cuda.synchronize()
    # the block, step by step (readings A5-A8)
    h1 = h.astype(np.float64) + oracle.linear(f64(o_hi) + f64(o_lo), f64(Wod), bo)
    u2 = oracle.layer_norm(h1, g2.astype(np.float64), b2ln.astype(np.float64), 1e-5)
    g = oracle.activation(oracle.linear(u2, f64(W1d), b1), act)
    h2 = h1 + oracle.linear(g, f64(W2d), b2)
    un = oracle.layer_norm(h2, gn.astype(np.float64), bn.astype(np.float64), 1e-5) if next_ln else h2
    got_h = hd_.cpu().numpy().astype(np.float64)
    got_u = f64(u_hi) + f64(u_lo)
    assert np.isfinite(got_h).all() and np.isfinite(got_u).all()
    sc = np.sqrt((h2 ** 2).mean())
    assert np.abs(got_h - h2).max() <= 3e-4 * sc, np.abs(got_h - h2).max() / sc      # u2, g rounded to bf16 hi + lo (2^-17)
    su = np.sqrt((un ** 2).mean())
    assert np.abs(got_u - un).max() <= 3e-4 * su, np.abs(got_u - un).max() / su
    assert np.abs(f64(u_hi) - un).max() <= 6e-3 * max(su, np.abs(un).max())           # hi alone: one bf16 rounding


# ------------------------------------------------------------------------------------------- FP8 operands (NEXT-3)
@pytest.mark.parametrize("M,N,K", [(128, 128, 128), (300, 768, 256), (1000, 1536, 512), (4097, 256, 128)])
def test_tc_gemm_fp8_matches_fp64_matmul_of_the_e4m3_values(M, N, K):
    """kind::f8f6f4 multiplies e4m3 values exactly and accumulates in fp32: against numpy fp64 on the dequantised operands."""
    rng = np.random.default_rng(M + N + K)
    A = torch.from_numpy(rng.standard_normal((M, K)).astype(np.float32) * 4).cuda().to(torch.float8_e4m3fn)
    W = torch.from_numpy((rng.standard_normal((N, K)) * 30).astype(np.float32)).cuda().to(torch.float8_e4m3fn)
    got = P.tc_gemm_fp8(A, W, out_scale=0.125).cpu().numpy()
    torch.cuda.synchronize()
    ref = 0.125 * oracle.linear(A.float().cpu().numpy().astype(np.float64), W.float().cpu().numpy().astype(np.float64), np.zeros(N))
    assert np.abs(got - ref).max() <= 2e-5 * np.abs(ref).max()
