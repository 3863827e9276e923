"""mlpf_build_candidates_static (include/mlpf.h): candidate building for callers that cannot allocate.  The kernels' scratch
is a file-scope device array inside libmlpf.so, so the entry point takes no scratch and allocates nothing.  Checked here
against the existing caller-scratch path (mlpf_build_candidates_ex) on the same inputs: integer outputs bit-exact, the
four-momenta bit-exact too (same kernels, same inputs), on two calls in a row with DIFFERENT inputs, so that the second
call runs on a scratch array that still holds the first call's contents.  The file sorts last on purpose (the suite runs
with pytest -x) and passes alone in a fresh process as well as after the other tests."""
import ctypes as C

import numpy as np
import pytest

import synth

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

import paper_2601_17554_b200 as P


@pytest.fixture(scope="module", autouse=True)
def _need_gpu():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    assert P.lib() is not None


def _inputs(lens, seed, pad, with_binary):
    X, off = synth.make_events(lens, seed=seed, pad_frac=pad)
    N = X.shape[0]
    rng = np.random.default_rng(seed + 100)
    logits = rng.standard_normal((N, 9)).astype(np.float32)
    logits[:, 0] += 1.0
    regress = (0.5 * rng.standard_normal((N, 5))).astype(np.float32)
    binary = rng.standard_normal(N).astype(np.float32) if with_binary else None
    return X, off, logits, regress, binary


def _outputs(N, E):
    # filled with a sentinel: entries beyond the candidate count must be left alone by both paths
    return dict(cand_offsets=torch.full((E + 1,), -7, dtype=torch.int32, device="cuda"),
                cand_elem=torch.full((N,), -7, dtype=torch.int32, device="cuda"),
                cand_pid=torch.full((N,), -7, dtype=torch.int32, device="cuda"),
                cand_p4=torch.full((N, 4), -7.0, dtype=torch.float32, device="cuda"))


CASES = [((1000, 1500, 777, 2049), 21, 0.1, True),      # several blocks, ragged tail, pad rows, the paper's binary rule
         ((5, 0, 0, 300, 1, 0), 22, 0.2, False),        # fewer rows than the call before (stale scratch beyond N), empty events
         ((64, 192), 23, 0.0, True)]


def test_static_scratch_entry_matches_the_caller_scratch_path_on_calls_in_a_row():
    for lens, seed, pad, with_binary in CASES:
        X, off, logits, regress, binary = _inputs(lens, seed, pad, with_binary)
        N, E = X.shape[0], len(off) - 1
        Xd, lg, rg = torch.from_numpy(X).cuda(), torch.from_numpy(logits).cuda(), torch.from_numpy(regress).cuda()
        bd = None if binary is None else torch.from_numpy(binary).cuda()
        ref = P.build_candidates(Xd, off, lg, rg, binary=bd)                 # existing path: caller-owned scratch
        got = P.build_candidates_static(Xd, off, lg, rg, _outputs(N, E), binary=bd)
        torch.cuda.synchronize()
        ref_off = ref["cand_offsets"].cpu().numpy()
        assert np.array_equal(got["cand_offsets"].cpu().numpy(), ref_off)
        M = int(ref_off[-1])
        assert 0 < M < N
        for k in ("cand_elem", "cand_pid"):
            assert np.array_equal(got[k].cpu().numpy()[:M], ref[k].cpu().numpy()[:M]), k
            assert (got[k].cpu().numpy()[M:] == -7).all(), k
        # same kernels on the same inputs: the tolerance of tests/test_gpu_candidates.py (1e-5) is met with zero difference
        assert np.array_equal(got["cand_p4"].cpu().numpy()[:M], ref["cand_p4"].cpu().numpy()[:M])


def test_static_scratch_entry_repeats_itself():
    X, off, logits, regress, binary = _inputs(CASES[0][0], 31, 0.1, True)
    N, E = X.shape[0], len(off) - 1
    args = (torch.from_numpy(X).cuda(), off, torch.from_numpy(logits).cuda(), torch.from_numpy(regress).cuda())
    bd = torch.from_numpy(binary).cuda()
    a = P.build_candidates_static(*args, _outputs(N, E), binary=bd)
    b = P.build_candidates_static(*args, _outputs(N, E), binary=bd)
    torch.cuda.synchronize()
    for k in a:
        assert torch.equal(a[k], b[k]), k


def test_static_scratch_limits_are_stated_and_enforced():
    max_n, max_e, held = (P.candidates_static_limit(i) for i in range(3))
    assert (max_n, max_e) == (262144, 4096) and 0 < held <= 1 << 20
    L = P.lib()
    off = (C.c_int32 * 2)(0, max_n + 1)
    assert L.mlpf_build_candidates_static(None, 55, off, 1, None, 9, None, 5, None, None, None, None, None, None) == -6
    assert b"exceed" in L.mlpf_last_error()
    off = (C.c_int32 * (max_e + 2))(*([0] * (max_e + 2)))
    assert L.mlpf_build_candidates_static(None, 55, off, max_e + 1, None, 9, None, 5, None, None, None, None, None, None) == -6
    # the maximum itself runs (N = max_n rows in one event)
    rng = np.random.default_rng(5)
    X = np.zeros((max_n, 8), dtype=np.float32)
    X[:, 0] = rng.integers(0, 5, max_n); X[:, 1] = 1.0 + rng.random(max_n); X[:, 4] = 2.0 + rng.random(max_n)
    logits = rng.standard_normal((max_n, 9)).astype(np.float32)
    regress = (0.5 * rng.standard_normal((max_n, 5))).astype(np.float32)
    o = np.array([0, max_n], dtype=np.int32)
    Xd, lg, rg = torch.from_numpy(X).cuda(), torch.from_numpy(logits).cuda(), torch.from_numpy(regress).cuda()
    ref = P.build_candidates(Xd, o, lg, rg)
    got = P.build_candidates_static(Xd, o, lg, rg, _outputs(max_n, 1))
    torch.cuda.synchronize()
    M = int(ref["cand_offsets"][-1])
    assert torch.equal(got["cand_offsets"], ref["cand_offsets"])
    for k in ("cand_elem", "cand_pid", "cand_p4"):
        assert torch.equal(got[k][:M], ref[k][:M]), k
