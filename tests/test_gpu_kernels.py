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


@pytest.mark.parametrize("hd,H", [(32, 8), (16, 4), (64, 8)])
@pytest.mark.parametrize("lens,pad", [((128,), 0.0), ((256, 64), 0.0), ((1, 129, 700, 257), 0.0), ((300, 1000), 0.15),
                                      ((0, 40, 0), 0.5)])
def test_tc_attention_matches_dense_softmax(hd, H, lens, pad):
    d = hd * H
    rng = np.random.default_rng(hd + sum(lens))
    N = sum(lens)
    off = np.zeros(len(lens) + 1, np.int32)
    off[1:] = np.cumsum(lens)
    qkv = rng.standard_normal((N, 3 * d)).astype(np.float32)
    qkv[:, :d] *= 2.0                                     # sharper than unit-variance scores
    valid = (rng.random(N) >= pad)
    QKV = _bf16(qkv)
    kv = torch.from_numpy(valid.astype(np.int32)).cuda()
    O = P.tc_attention_bf16(QKV, kv if pad > 0 else None, off, d, H).float().cpu().numpy()
    if pad == 0:
        valid[:] = True
    qk64 = QKV.float().cpu().numpy().astype(np.float64)
    v64 = qk64[:, 2 * d:]
    for e in range(len(lens)):
        a, b = off[e], off[e + 1]
        if b == a:
            continue
        ref = oracle.attention_event(qk64[a:b, :d], qk64[a:b, d:2 * d], v64[a:b], valid[a:b], H)
        err = np.abs(O[a:b] - ref)
        scale = np.sqrt((ref ** 2).mean()) + 1e-6
        assert (err / np.maximum(np.abs(ref), scale)).max() <= 2e-2, (e, err.max(), scale)
