"""GPU parity for candidate building (include/mlpf.h "candidate building") against
oracle/candidates.py on the same inputs.  Integer outputs (offsets, element index, PID) bit-exact; pT, E relative
1e-5 and phi absolute 1e-5 (fp32 expf / atan2f of the same fp32 regressions vs fp64: a few ulp = 4e-7)."""
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


def _compare(X, off, logits, regress, binary=None):
    c = P.build_candidates(torch.from_numpy(X).cuda(), off, torch.from_numpy(logits).cuda(), torch.from_numpy(regress).cuda(),
                           binary=None if binary is None else torch.from_numpy(binary).cuda())
    torch.cuda.synchronize()
    ref = oracle.build_candidates(X, off, logits, regress, binary=binary)
    got_off = c["cand_offsets"].cpu().numpy()
    assert np.array_equal(got_off, ref["cand_offsets"])
    M = int(got_off[-1]) if len(got_off) else 0
    assert np.array_equal(c["cand_elem"].cpu().numpy()[:M], ref["cand_elem"])
    assert np.array_equal(c["cand_pid"].cpu().numpy()[:M], ref["cand_pid"])
    p4 = c["cand_p4"].cpu().numpy()[:M].astype(np.float64)
    r = ref["cand_p4"]
    if M:
        assert np.max(np.abs(p4[:, 0] - r[:, 0]) / np.abs(r[:, 0])) <= 1e-5
        assert np.max(np.abs(p4[:, 3] - r[:, 3]) / np.abs(r[:, 3])) <= 1e-5
        assert np.array_equal(p4[:, 1], r[:, 1])
        dphi = np.abs(p4[:, 2] - r[:, 2])
        assert np.max(np.minimum(dphi, 2 * np.pi - dphi)) <= 1e-5
    return M


def _random_outputs(N, seed, C=9):
    rng = np.random.default_rng(seed)
    logits = rng.standard_normal((N, C)).astype(np.float32)
    logits[:, 0] += 1.0                                    # ~ a third of the elements are "no particle"
    regress = (0.5 * rng.standard_normal((N, 5))).astype(np.float32)
    return logits, regress


@pytest.mark.parametrize("lens,pad", [
    ((64, 192), 0.0),                                      # cfg1 shape
    ((5, 0, 0, 300, 1, 0), 0.2),                           # empty events (also trailing), ragged, pad rows
    ((256,), 0.0),                                         # N a multiple of the block: offsets[E] in the virtual block
    ((0, 0), 0.0),                                         # N = 0
    ((1000, 1500, 777, 2049), 0.1),                        # several blocks, ragged tail
])
def test_candidates_match_oracle(lens, pad):
    X, off = synth.make_events(lens, seed=21, pad_frac=pad)
    logits, regress = _random_outputs(int(off[-1]), 22)
    if len(logits) > 3:
        logits[3, :] = 0.5                                 # exact tie -> class 0 -> dropped
    _compare(X, off, logits, regress)


def test_candidates_all_kept_and_none_kept():
    X, off = synth.make_events((700, 300), seed=5)
    logits, regress = _random_outputs(1000, 6)
    logits[:, 0] = -50.0
    assert _compare(X, off, logits, regress) == 1000
    logits[:, 0] = 50.0
    assert _compare(X, off, logits, regress) == 0


def test_candidates_from_the_forward_pass_cfg1():
    """End to end on cfg1: mlpf_infer's own device outputs feed mlpf_build_candidates; the oracle decodes the same
    fp32 logits (the argmax decision is taken on identical numbers on both sides)."""
    m = synth.model_cfg("cfg1")
    W = synth.make_weights("cfg1")
    X, off = synth.make_named_events("cfg1")
    mod = P.Mlpf(W, m)
    Xd = torch.from_numpy(X).cuda()
    lg, rg = mod.infer(Xd, off)
    c = P.build_candidates(Xd, off, lg, rg)
    torch.cuda.synchronize()
    ref = oracle.build_candidates(X, off, lg.cpu().numpy(), rg.cpu().numpy())
    assert np.array_equal(c["cand_offsets"].cpu().numpy(), ref["cand_offsets"])
    M = int(ref["cand_offsets"][-1])
    assert M > 0
    assert np.array_equal(c["cand_elem"].cpu().numpy()[:M], ref["cand_elem"])
    assert np.array_equal(c["cand_pid"].cpu().numpy()[:M], ref["cand_pid"])
    assert np.allclose(c["cand_p4"].cpu().numpy()[:M], ref["cand_p4"], rtol=1e-5, atol=1e-5)


def test_candidates_full_size_cfg5b_shape():
    """BASELINE.json's largest row count (262144 elements, 32 events, 10 % pad rows), element by element."""
    X, off = synth.make_named_events("cfg5b")
    logits, regress = _random_outputs(int(off[-1]), 31)
    M = _compare(X, off, logits, regress)
    assert 0 < M < int(off[-1])


def test_candidates_deterministic_and_scratch_reuse():
    X, off = synth.make_events((3000, 1234), seed=8, pad_frac=0.05)
    logits, regress = _random_outputs(int(off[-1]), 9)
    Xd, lg, rg = (torch.from_numpy(a).cuda() for a in (X, logits, regress))
    scratch = torch.empty(int(P.lib().mlpf_candidates_scratch_bytes(int(off[-1]), 2)), dtype=torch.uint8, device="cuda")
    a = P.build_candidates(Xd, off, lg, rg, scratch=scratch)
    b = P.build_candidates(Xd, off, lg, rg, scratch=scratch)
    torch.cuda.synchronize()
    M = int(a["cand_offsets"][-1])
    for k in a:
        n = M if k != "cand_offsets" else 3
        assert torch.equal(a[k][:n], b[k][:n])


@pytest.mark.parametrize("lens,pad", [((64, 192), 0.0), ((5, 0, 0, 300, 1, 0), 0.2), ((1000, 1500, 777, 2049), 0.1)])
def test_candidates_binary_rule_matches_oracle(lens, pad):
    """The paper's selection (L156): binary score > 0.5; PID = argmax over all classes (class 0 can be kept); a type id
    outside 0..4 is clamped as in the forward pass (-1 -> pad row, 7 -> a real element)."""
    X, off = synth.make_events(lens, seed=41, pad_frac=pad)
    N = int(off[-1])
    logits, regress = _random_outputs(N, 42)
    rng = np.random.default_rng(43)
    binary = rng.standard_normal(N).astype(np.float32)
    binary[::7] = 0.0                                      # sigmoid(0) = 0.5: not above
    binary[1::11] = 1e-30                                  # tiny positive logit: above
    if N > 20:
        X[3, 0], X[5, 0] = -1.0, 7.0
        binary[3] = binary[5] = 2.0
    M = _compare(X, off, logits, regress, binary=binary)
    assert M > 0
