"""GPU parity: libmlpf.so (through the C ABI) against the fp64 CPU oracle on the same seeded inputs.

Tolerances (BASELINE.json north_star; metric = DESIGN.md reading A14): max relative error <= 2e-2 on
logits and regressions in BF16, <= 1e-4 on the fp32 debug path, argmax agreement >= 99.9 % over
decidable rows, integer schedule arrays bit-exact."""
import os
import numpy as np
import pytest

import synth
import oracle
from synth.configs import ModelCfg

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

import paper_2601_17554_b200 as P

TOL_BF16 = 2e-2
TOL_FP32 = 1e-4
TINY_FOR_NAN = ModelCfg(n_layers=2, d_model=64, n_heads=2, d_ff=256)


@pytest.fixture(scope="module", autouse=True)
def _need_gpu():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    assert P.lib() is not None          # fail loudly if the extension is missing


def gpu_forward(W, m, X, off, precision=P.PREC_BF16, kernels=P.KERNELS_TC, tap=None):
    mod = P.Mlpf(W, m)
    mod.set_option(P.OPT_PRECISION, precision)
    mod.set_option(P.OPT_KERNELS, kernels)
    if tap is not None:
        mod.set_option(P.OPT_TAP_LAYER, tap)
    Xd = torch.from_numpy(X).cuda()
    lg, rg = mod.infer(Xd, off)
    torch.cuda.synchronize()
    return mod, lg.cpu().numpy(), rg.cpu().numpy()


def oracle_events(W, m, X, off, events, quantized):
    """Oracle outputs for a subset of events (events are independent: pin P4)."""
    Wq = oracle.quantize_weights(W) if quantized else W
    rows, lgs, rgs = [], [], []
    for e in events:
        a, b = int(off[e]), int(off[e + 1])
        lg, rg = oracle.forward(X[a:b], np.array([0, b - a]), Wq, m)
        rows.append(np.arange(a, b)); lgs.append(lg); rgs.append(rg)
    return np.concatenate(rows), np.concatenate(lgs), np.concatenate(rgs)


GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def oracle_cached(name, fp32=False):
    """Oracle outputs of the large configs written by tests/golden/make_oracle_cache.py (which imports only oracle/
    and synth/): rows = global row indices of the stored sample (documented event subset, every 4th row)."""
    z = np.load(os.path.join(GOLDEN, f"oracle_{name}.npz"))
    if fp32:
        return z["fp32_rows"], z["fp32_logits"].astype(np.float64), z["fp32_regress"].astype(np.float64)
    return z["rows"], z["logits"].astype(np.float64), z["regress"].astype(np.float64)


def check(lg_gpu, rg_gpu, rows, lg_ref, rg_ref, X, tol, argmax=True):
    valid = X[rows, 0] != 0
    e_lg, _ = oracle.parity_metrics(lg_gpu[rows], lg_ref, valid)
    e_rg, _ = oracle.parity_metrics(rg_gpu[rows], rg_ref, valid)
    assert np.isfinite(lg_gpu).all() and np.isfinite(rg_gpu).all()
    assert (lg_gpu[X[:, 0] == 0] == 0).all() and (rg_gpu[X[:, 0] == 0] == 0).all()    # pad rows exactly 0
    assert e_lg <= tol and e_rg <= tol, (e_lg, e_rg)
    if argmax:
        agree, dec_frac, raw = oracle.argmax_agreement(lg_gpu[rows], lg_ref, valid, tol_rel=tol)
        assert agree >= 0.999, (agree, dec_frac, raw)
    return e_lg, e_rg


# ------------------------------------------------------------------------------------------- a0 schedule
@pytest.mark.parametrize("lens,pad", [((64, 192), 0.0), ((0, 5, 0, 300, 129, 1, 0), 0.3), ((1,), 0.0),
                                      ((1500, 700, 1500, 2049), 0.1)])
@pytest.mark.parametrize("tile_q", [64, 128])
def test_schedule_bit_exact(lens, pad, tile_q):
    m = synth.model_cfg("cfg1")
    W = synth.make_weights("cfg1")
    X, off = synth.make_events(lens, seed=11, pad_frac=pad)
    mod = P.Mlpf(W, m)
    mod.set_option(P.OPT_TILE_Q, tile_q)
    mod.set_option(P.OPT_TAP_LAYER, -2)
    mod.infer(torch.from_numpy(X).cuda(), off)
    ref = oracle.schedule(X, off, tile_q)
    for k in ("row_event", "row_pos", "valid", "n_valid", "type_offsets", "sorted_row", "type_perm", "work_list",
              "comp_row", "offsets_c", "comp_type_perm"):
        got = mod.schedule(k)
        assert got.dtype == np.int32
        np.testing.assert_array_equal(got, ref[k], err_msg=k)


# ------------------------------------------------------------------------------------------- fp32 debug path
@pytest.mark.parametrize("name,events", [("cfg1", None), ("cfg2", [0, 5]), ("cfg3", [1, 6]), ("cfg5b", "cache")])
def test_fp32_debug_path(name, events):
    m = synth.model_cfg(name)
    W = synth.make_weights(name)
    X, off = synth.make_named_events(name)
    if events == "cache":                       # one 8192-row event of cfg5b (W-fp32 oracle output from tests/golden/)
        rows, lr, rr = oracle_cached(name, fp32=True)
        e = int(np.searchsorted(off, rows[0], side="right") - 1)
        a, b = int(off[e]), int(off[e + 1])
        _, lg1, rg1 = gpu_forward(W, m, X[a:b], np.array([0, b - a], np.int32), precision=P.PREC_FP32_DEBUG)
        lg = np.zeros((X.shape[0], lg1.shape[1]), np.float32); rg = np.zeros((X.shape[0], rg1.shape[1]), np.float32)
        lg[a:b], rg[a:b] = lg1, rg1
    else:
        _, lg, rg = gpu_forward(W, m, X, off, precision=P.PREC_FP32_DEBUG)
        ev = range(len(off) - 1) if events is None else events
        rows, lr, rr = oracle_events(W, m, X, off, ev, quantized=False)
    check(lg, rg, rows, lr, rr, X, TOL_FP32)


# ------------------------------------------------------------------------------------------- bf16 path
# "paper" = the paper's own block shape: d_model 256, 16 heads x 16, ReLU, 3 blocks
# cfg1-3: every event against the oracle run here; cfg4 / cfg5a / cfg5b: against tests/golden/oracle_<cfg>.npz (cfg5a whole;
# cfg4 / cfg5b: first, last, longest, shortest + 25 % random events, every 4th row of each: make_oracle_cache.py)
BF16_CASES = [("cfg1", None), ("cfg2", None), ("cfg3", None), ("cfg4", "cache"), ("cfg5a", "cache"), ("cfg5b", "cache"),
              ("paper", [1])]


@pytest.mark.parametrize("kernels", [P.KERNELS_TC, P.KERNELS_SIMPLE])
@pytest.mark.parametrize("name,events", BF16_CASES)
def test_bf16_parity(name, events, kernels):
    if kernels == P.KERNELS_SIMPLE and name not in ("cfg1", "cfg2"):
        pytest.skip("CUDA-core debugging kernels are only exercised on the small configs")
    m = synth.model_cfg(name)
    W = synth.make_weights(name)
    X, off = synth.make_named_events(name)
    mod, lg, rg = gpu_forward(W, m, X, off, kernels=kernels)
    if events == "cache":
        rows, lr, rr = oracle_cached(name)
    else:
        ev = range(len(off) - 1) if events is None else events
        rows, lr, rr = oracle_events(W, m, X, off, ev, quantized=True)
    e = check(lg, rg, rows, lr, rr, X, TOL_BF16)
    print(name, "max rel err (logits, regress) =", e, "launches", mod.query(P.Q_LAUNCHES))


def test_bf16_parity_sharp_attention():
    """Pin P15's weight set: W_q x4 makes attention far from uniform so masking/leak bugs show."""
    name = "cfg2"
    m = synth.model_cfg(name)
    W = synth.sharpen(synth.make_weights(name), m, 4.0)
    X, off = synth.make_named_events(name, max_events=4)
    _, lg, rg = gpu_forward(W, m, X, off)
    rows, lr, rr = oracle_events(W, m, X, off, range(len(off) - 1), quantized=True)
    check(lg, rg, rows, lr, rr, X, TOL_BF16)


# ------------------------------------------------------------------------------------------- per-step parity
def _rel(got, ref, valid):
    ref = ref[valid]; got = got[valid]
    rms = np.sqrt((ref ** 2).mean())
    return float((np.abs(got - ref) / np.maximum(np.abs(ref), rms)).max())


@pytest.mark.parametrize("precision,tol", [(P.PREC_FP32_DEBUG, 1e-4), (P.PREC_BF16, 2e-2)])
@pytest.mark.parametrize("name,max_events", [("cfg1", None), ("cfg2", 3), ("cfg3", 1)])
def test_per_step_intermediates(name, max_events, precision, tol):
    m = synth.model_cfg(name)
    W = synth.make_weights(name)
    X, off = synth.make_named_events(name, max_events=max_events)
    N, d = X.shape[0], m.d_model
    valid = X[:, 0] != 0
    dump = {}
    Wq = oracle.quantize_weights(W) if precision == P.PREC_BF16 else W
    oracle.forward(X, off, Wq, m, dump=dump)
    # after the embedding
    mod, _, _ = gpu_forward(W, m, X, off, precision=precision, tap=-2)
    assert _rel(mod.tensor("H", (N, d)), dump["h0"], valid) <= tol
    for l in (0, m.n_layers - 1):
        mod, _, _ = gpu_forward(W, m, X, off, precision=precision, tap=l)
        p = f"layer.{l}."
        qkv = dump[p + "qkv"]
        assert _rel(mod.tensor("QK", (N, 2 * d)), qkv[:, :2 * d], valid) <= tol, "qk"
        assert _rel(mod.tensor("V", (N, d)), qkv[:, 2 * d:], valid) <= tol, "v"
        assert _rel(mod.tensor("O", (N, d)), dump[p + "o"], valid) <= tol, "o"
        assert _rel(mod.tensor("U", (N, d)), dump[p + "u2"], valid) <= tol, "u2"
        assert _rel(mod.tensor("G", (N, m.d_ff)), dump[p + "g"], valid) <= tol, "g"
        assert _rel(mod.tensor("H", (N, d)), dump[p + "h"], valid) <= tol, "h"


@pytest.mark.parametrize("name,max_events", [("cfg1", None), ("cfg2", 3), ("paper", 1)])
def test_tensor_pipe_embedding_matches_the_oracle_as_well_as_the_fp32_first_layer(name, max_events):
    """MLPF_OPT_TC_EMBED: the first embedding layer (fp32 weights, reading A3) as one K = 192 bf16 GEMM over hi + lo terms
    of features and weights.  Features span orders of magnitude (energies, angles, flags), so the check is against the
    fp64 oracle's embedding output with FP32 first-layer weights (what the CUDA-core kernel computes) at a tolerance far
    below the step's 2e-2: both first layers must sit at the level of the bf16 hi + lo rounding of the hidden layer."""
    m = synth.model_cfg(name)
    W = synth.make_weights(name)
    X, off = synth.make_named_events(name, max_events=max_events)
    X = X.copy()
    X[X[:, 0] != 0, 4] *= 37.0                     # energies up to a few 1e3: the hi + lo split has to carry them
    N, d = X.shape[0], m.d_model
    valid = X[:, 0] != 0
    dump = {}
    oracle.forward(X, off, oracle.quantize_weights(W), m, dump=dump)
    errs = {}
    for tc_embed in (0, 1):
        mod = P.Mlpf(W, m)
        mod.set_option(P.OPT_TC_EMBED, tc_embed)
        mod.set_option(P.OPT_TAP_LAYER, -2)
        mod.infer(torch.from_numpy(X).cuda(), off)
        torch.cuda.synchronize()
        errs[tc_embed] = _rel(mod.tensor("H", (N, d)), dump["h0"], valid)
    # measured (paper config): 1.4e-4 with the fp32 first layer (the hidden layer's own bf16 hi + lo rounding, 2^-17, through
    # the second layer's dot products), 2.4e-4 on the tensor pipe (the hi + lo terms of x and W1 add 2^-17 each)
    assert errs[0] <= 5e-4 and errs[1] <= 5e-4, errs


@pytest.mark.parametrize("name,max_events", [("cfg2", None), ("cfg3", 2)])
def test_programmatic_dependent_launch_changes_nothing(name, max_events):
    """MLPF_OPT_PDL: the tensor-core kernels start while their predecessor's last wave drains and order every access with
    griddepcontrol.wait: outputs bit-identical to plain stream order, call after call."""
    m = synth.model_cfg(name)
    W = synth.make_weights(name)
    X, off = synth.make_named_events(name, max_events=max_events)
    Xd = torch.from_numpy(X).cuda()
    out = {}
    for pdl in (0, 1):
        mod = P.Mlpf(W, m)
        mod.set_option(P.OPT_PDL, pdl)
        runs = []
        for _ in range(3):
            lg, rg = mod.infer(Xd, off)
            torch.cuda.synchronize()
            runs.append((lg.clone(), rg.clone()))
        for lg, rg in runs[1:]:
            assert torch.equal(lg, runs[0][0]) and torch.equal(rg, runs[0][1])
        out[pdl] = runs[0]
    assert torch.equal(out[0][0], out[1][0]) and torch.equal(out[0][1], out[1][1])


def test_quadratic_softmax_polynomial_is_an_option_within_tolerance():
    """MLPF_OPT_ATTN_POLY_DEG = 2 (off by default): half of the softmax weights from a quadratic 2^f (relative error 1.8e-3,
    the size of the weight's own bf16 rounding) instead of the cubic (1e-4).  Still far inside the 2e-2 tolerance; the
    measured cost in accuracy and gain in time are in profiles/r02_README.md."""
    m = synth.model_cfg("cfg2")
    W = synth.make_weights("cfg2")
    X, off = synth.make_named_events("cfg2")
    rows, lr, rr = oracle_events(W, m, X, off, range(len(off) - 1), quantized=True)
    try:
        mod = P.Mlpf(W, m)
        mod.set_option(P.OPT_ATTN_POLY_DEG, 2)
        lg, rg = mod.infer(torch.from_numpy(X).cuda(), off)
        torch.cuda.synchronize()
        check(lg.cpu().numpy(), rg.cpu().numpy(), rows, lr, rr, X, TOL_BF16)
    finally:
        mod.set_option(P.OPT_ATTN_POLY_DEG, 3)       # process-wide knob


def test_non_finite_features_stay_inside_their_event():
    """include/mlpf.h: NaN / Inf features give undefined outputs for THAT event only.  The 128-row K / V tile at the end of
    event A runs into event B's first rows: their keys get weight exactly 0, and the v values are made finite by a3's
    epilogue so that 0 x v cannot poison A's accumulators."""
    m = TINY_FOR_NAN
    W = synth.make_weights(m, seed=11)
    X, off = synth.make_events((300, 257, 190), seed=12)
    X = X.copy()
    b0 = int(off[1])
    X[b0, 3] = np.nan                         # first rows of event B: NaN, +Inf, -Inf features (types stay valid)
    X[b0 + 1, 5] = np.inf
    X[b0 + 2, 7] = -np.inf
    for precision, tol, Wo in ((P.PREC_BF16, TOL_BF16, oracle.quantize_weights(W)), (P.PREC_FP32_DEBUG, TOL_FP32, W)):
        mod = P.Mlpf(W, m)
        mod.set_option(P.OPT_PRECISION, precision)
        lg, rg = mod.infer(torch.from_numpy(X).cuda(), off)
        torch.cuda.synchronize()
        lg = lg.cpu().numpy(); rg = rg.cpu().numpy()
        for e in (0, 2):                      # the events before and after the poisoned one
            a, b = int(off[e]), int(off[e + 1])
            lr, rr = oracle.forward(X[a:b], np.array([0, b - a], np.int32), Wo, m)
            valid = X[a:b, 0] != 0
            assert np.isfinite(lg[a:b]).all() and np.isfinite(rg[a:b]).all(), (precision, e)
            e_lg, _ = oracle.parity_metrics(lg[a:b], lr, valid)
            e_rg, _ = oracle.parity_metrics(rg[a:b], rr, valid)
            assert e_lg <= tol and e_rg <= tol, (precision, e, e_lg, e_rg)


def test_concurrent_calls_from_host_threads_on_their_own_streams():
    """include/mlpf.h: concurrent mlpf_infer calls on DIFFERENT streams of one handle are safe (one workspace per stream, the
    enqueue serialised by the handle's mutex).  Four host threads, one stream each, ragged batches of different sizes; every
    result bit-identical to the same batch run alone afterwards."""
    import threading
    m = synth.model_cfg("cfg2")
    W = synth.make_weights("cfg2")
    mod = P.Mlpf(W, m)
    rng = np.random.default_rng(3)
    batches = []
    for i in range(16):
        lens = [int(x) for x in rng.integers(0, 700, int(rng.integers(1, 10)))]
        X, off = synth.make_events(lens, seed=100 + i, pad_frac=float(rng.choice([0.0, 0.1])))
        if X.shape[0]:
            batches.append((torch.from_numpy(X).cuda(), off))
    results, errors = {}, []

    def worker(tid):
        try:
            st = torch.cuda.Stream()
            for rep in range(4):
                for bi in range(tid, len(batches), 4):
                    Xd, off = batches[bi]
                    lg, rg = mod.infer(Xd, off, stream=st)
                    st.synchronize()
                    results[(bi, rep)] = (lg.clone(), rg.clone())
        except Exception as e:                      # surfaced in the main thread below
            errors.append(e)

    threads = [threading.Thread(target=worker, args=(t,)) for t in range(4)]
    for t in threads:
        t.start()
    for t in threads:
        t.join()
    assert not errors, errors
    for bi, (Xd, off) in enumerate(batches):
        lg, rg = mod.infer(Xd, off)
        torch.cuda.synchronize()
        for rep in range(4):
            a, b = results[(bi, rep)]
            assert torch.equal(a, lg) and torch.equal(b, rg), (bi, rep)


# ------------------------------------------------------------------------------------------- random shapes
@pytest.mark.parametrize("seed", [101, 102, 103, 104])
def test_random_models_and_ragged_batches_against_the_oracle(seed):
    """Seeded random draws of everything the blob header can express at d_model <= 256 (1-3 layers, head widths 16 / 32 /
    64, d_ff 128..1024, GELU / ReLU, with and without the final LayerNorm, one or two stacks, binary head) on ragged batches
    (empty events, lengths around the 64 / 128 tile edges, pad rows): the tensor-core path within 2e-2 and the fp32 debug
    path within 1e-4 of the oracle (reading A14), pad rows exactly 0.  A sweep of 150 such cases measured <= 9.2e-3 / 2.1e-5."""
    rng = np.random.default_rng(seed)
    for case in range(6):
        d, H = [(64, 4), (128, 8), (256, 8), (256, 16), (128, 2), (64, 1), (256, 4)][rng.integers(0, 7)]
        stacks = int(rng.integers(1, 3))
        m = ModelCfg(n_layers=int(rng.integers(1, 4)), d_model=d, n_heads=H, d_ff=int(rng.choice([128, 256, 512, 1024])),
                     activation=str(rng.choice(["gelu", "relu"])), final_ln=bool(rng.integers(0, 2)), n_stacks=stacks,
                     binary_head=bool(stacks == 2 and rng.integers(0, 2)))
        E = int(rng.integers(1, 20))
        kind = rng.integers(0, 3)
        if kind == 0:
            lens = rng.integers(0, 40, E)
        elif kind == 1:
            lens = np.where(rng.random(E) < 0.3, 0, rng.integers(1, 400, E))
        else:
            lens = rng.choice([1, 63, 64, 65, 127, 128, 129, 255, 256, 257, 383, 384, 385], E)
        W = synth.make_weights(m, seed=int(rng.integers(1, 1 << 30)))
        X, off = synth.make_events([int(x) for x in lens], seed=int(rng.integers(1, 1 << 30)), pad_frac=float(rng.choice([0.0, 0.1, 0.5])))
        valid = X[:, 0] != 0
        if valid.sum() < 2:
            continue
        Xd = torch.from_numpy(X).cuda()
        for precision, tol, Wo in ((P.PREC_BF16, TOL_BF16, oracle.quantize_weights(W)), (P.PREC_FP32_DEBUG, TOL_FP32, W)):
            mod = P.Mlpf(W, m)
            mod.set_option(P.OPT_PRECISION, precision)
            got = mod.infer(Xd, off, with_binary=True) if m.binary_head else mod.infer(Xd, off)
            torch.cuda.synchronize()
            ref = oracle.forward(X, off, Wo, m, with_binary=True) if m.binary_head else oracle.forward(X, off, Wo, m)
            for g, r in zip(got, ref):
                g = g.cpu().numpy().reshape(X.shape[0], -1)
                r = np.asarray(r).reshape(X.shape[0], -1)
                assert np.isfinite(g).all() and (g[~valid] == 0).all(), (seed, case)
                err, _ = oracle.parity_metrics(g, r, valid)
                assert err <= tol, (seed, case, precision, err, m, [int(x) for x in lens])


# ------------------------------------------------------------------------------------------- edge cases
TINY = ModelCfg(n_layers=2, d_model=64, n_heads=4, d_ff=256)


@pytest.mark.parametrize("lens,pad", [((1,), 0.0), ((0, 7, 0), 0.0), ((129, 1, 257, 128), 0.0), ((40, 300), 0.5),
                                      ((5, 6), 1.0)])
@pytest.mark.parametrize("precision,tol", [(P.PREC_FP32_DEBUG, TOL_FP32), (P.PREC_BF16, TOL_BF16)])
def test_edge_cases(lens, pad, precision, tol):
    W = synth.make_weights(TINY, seed=5)
    X, off = synth.make_events(lens, seed=9, pad_frac=pad)
    if pad == 0.5:
        X[X[:, 0] == 0, 1:] = 1e30            # garbage in pad rows must be ignored (P4 iii)
    _, lg, rg = gpu_forward(W, TINY, X, off, precision=precision)
    Wq = oracle.quantize_weights(W) if precision == P.PREC_BF16 else W
    lr, rr = oracle.forward(X, off, Wq, TINY)
    # with a handful of rows the per-column rms of A14 degenerates (one row: rms = |value|), so the floor is
    # the rms over all valid outputs of the case
    valid = X[:, 0] != 0
    assert np.isfinite(lg).all() and np.isfinite(rg).all()
    assert (lg[~valid] == 0).all() and (rg[~valid] == 0).all()
    for got, ref in ((lg, lr), (rg, rr)):
        if valid.any():
            floor = np.sqrt((ref[valid] ** 2).mean())
            rel = np.abs(got[valid] - ref[valid]) / np.maximum(np.abs(ref[valid]), floor)
            assert rel.max() <= tol, rel.max()


def test_empty_calls_and_bad_offsets():
    W = synth.make_weights(TINY, seed=5)
    mod = P.Mlpf(W, TINY)
    X = torch.zeros((4, 55), device="cuda")
    lg, rg = mod.infer(X[:0], np.array([0], np.int32))                 # zero events
    lg, rg = mod.infer(X[:0], np.array([0, 0, 0], np.int32))           # zero rows
    with pytest.raises(P.MlpfError, match="-3"):
        mod.infer(X, np.array([1, 4], np.int32))
    with pytest.raises(P.MlpfError, match="-3"):
        mod.infer(X, np.array([0, 3, 2, 4], np.int32))


def test_determinism_and_packing_invariance():
    """L232: the same event gives identical outputs; per-event tile schedule -> also when packed."""
    name = "cfg2"
    m = synth.model_cfg(name)
    W = synth.make_weights(name)
    X, off = synth.make_named_events(name, max_events=5)
    mod = P.Mlpf(W, m)
    Xd = torch.from_numpy(X).cuda()
    a = [t.clone() for t in mod.infer(Xd, off)]
    b = [t.clone() for t in mod.infer(Xd, off)]
    torch.cuda.synchronize()
    assert torch.equal(a[0], b[0]) and torch.equal(a[1], b[1])
    s0, s1 = int(off[2]), int(off[3])
    c = mod.infer(Xd[s0:s1].contiguous(), np.array([0, s1 - s0], np.int32))
    torch.cuda.synchronize()
    assert torch.equal(c[0], a[0][s0:s1]) and torch.equal(c[1], a[1][s0:s1])


def test_concurrent_streams_match_single_stream():
    name = "cfg2"
    m = synth.model_cfg(name)
    W = synth.make_weights(name)
    X, off = synth.make_named_events(name)
    mod = P.Mlpf(W, m)
    Xd = torch.from_numpy(X).cuda()
    ref = [t.clone() for t in mod.infer(Xd, off)]
    torch.cuda.synchronize()
    E = len(off) - 1
    streams = [torch.cuda.Stream() for _ in range(4)]
    outs = []
    for i, s in enumerate(streams):
        e0, e1 = i * E // 4, (i + 1) * E // 4
        r0, r1 = int(off[e0]), int(off[e1])
        s.wait_stream(torch.cuda.current_stream())
        with torch.cuda.stream(s):
            outs.append((r0, r1, mod.infer(Xd[r0:r1], off[e0:e1 + 1] - off[e0], stream=s)))
    torch.cuda.synchronize()
    for r0, r1, (lg, rg) in outs:
        assert torch.equal(lg, ref[0][r0:r1]) and torch.equal(rg, ref[1][r0:r1])
    assert mod.query(P.Q_WORKSPACE_BYTES) > 0


def test_host_entry_point_matches_device_entry_point():
    m = synth.model_cfg("cfg1")
    W = synth.make_weights("cfg1")
    X, off = synth.make_named_events("cfg1")
    mod = P.Mlpf(W, m)
    lg, rg = mod.infer(torch.from_numpy(X).cuda(), off)
    xh = torch.from_numpy(X).pin_memory()
    lh = torch.empty((X.shape[0], 9)).pin_memory()
    rh = torch.empty((X.shape[0], 5)).pin_memory()
    mod.infer_host(xh, off, lh, rh)
    assert torch.equal(lh, lg.cpu()) and torch.equal(rh, rg.cpu())


def test_largest_event_properties():
    """cfg5a (one event of 16384 elements, 10 % pad rows, hd = 64): the oracle needs minutes for it, so the full-size
    run is checked through properties that hold at any size: pad rows exactly 0, finite outputs, permutation
    equivariance (no positional encoding: a row permutation permutes the outputs; tiles then hold
    different keys, so agreement is within the BF16 tolerance, not bitwise), and packing invariance (bitwise)."""
    name = "cfg5a"
    m = synth.model_cfg(name)
    W = synth.make_weights(name)
    X, off = synth.make_named_events(name)
    N = X.shape[0]
    mod = P.Mlpf(W, m)
    lg, rg = [t.cpu().numpy() for t in mod.infer(torch.from_numpy(X).cuda(), off)]
    valid = X[:, 0] != 0
    assert np.isfinite(lg).all() and np.isfinite(rg).all()
    assert (lg[~valid] == 0).all() and (rg[~valid] == 0).all() and valid.sum() > 0.85 * N
    perm = np.random.default_rng(3).permutation(N)
    lg2, rg2 = [t.cpu().numpy() for t in mod.infer(torch.from_numpy(np.ascontiguousarray(X[perm])).cuda(), off)]
    for a, b in ((lg, lg2), (rg, rg2)):
        ref, got = a[perm][valid[perm]], b[valid[perm]]
        rms = np.sqrt((ref ** 2).mean(axis=0, keepdims=True))
        assert (np.abs(got - ref) / np.maximum(np.abs(ref), rms)).max() <= TOL_BF16
    # the same event packed behind a short one: identical tiles -> identical bits
    Xs, offs = synth.make_events((77,), seed=1)
    Xp = np.concatenate([Xs, X])
    lg3, rg3 = [t.cpu().numpy() for t in mod.infer(torch.from_numpy(Xp).cuda(), np.array([0, 77, 77 + N], np.int32))]
    assert np.array_equal(lg3[77:], lg) and np.array_equal(rg3[77:], rg)


@pytest.mark.parametrize("precision,tol", [(P.PREC_FP32_DEBUG, TOL_FP32), (P.PREC_BF16, TOL_BF16)])
def test_without_final_layernorm(precision, tol):
    """Header flag final_ln = 0 (reading A7): the heads read the residual stream itself."""
    from dataclasses import replace
    m = replace(synth.model_cfg("cfg1"), final_ln=False)
    W = synth.make_weights(m, seed=7)
    X, off = synth.make_events((70, 130, 9), seed=4, pad_frac=0.1)
    _, lg, rg = gpu_forward(W, m, X, off, precision=precision)
    Wq = oracle.quantize_weights(W) if precision == P.PREC_BF16 else W
    lr, rr = oracle.forward(X, off, Wq, m)
    check(lg, rg, np.arange(X.shape[0]), lr, rr, X, tol, argmax=False)


# ------------------------------------------------------------------------------------------- the paper's topology (NEXT-1)
def _two_stack_check(W, m, X, off, precision, tol, fuse=1):
    mod = P.Mlpf(W, m)
    mod.set_option(P.OPT_PRECISION, precision)
    mod.set_option(P.OPT_FUSE, fuse)
    lg, rg, bn = [t.cpu().numpy() for t in mod.infer(torch.from_numpy(X).cuda(), off, with_binary=True)]
    torch.cuda.synchronize()
    Wq = oracle.quantize_weights(W) if precision == P.PREC_BF16 else W
    lr, rr, br = oracle.forward(X, off, Wq, m, with_binary=True)
    valid = X[:, 0] != 0
    check(lg, rg, np.arange(X.shape[0]), lr, rr, X, tol, argmax=X.shape[0] > 1000)
    e_b, _ = oracle.parity_metrics(bn[:, None], br[:, None], valid)
    assert (bn[~valid] == 0).all() and e_b <= tol, e_b
    return mod, lg, rg, bn


TWO_TINY = ModelCfg(n_layers=2, d_model=64, n_heads=4, d_ff=256, activation="relu", n_stacks=2, binary_head=True)


@pytest.mark.parametrize("precision,tol", [(P.PREC_FP32_DEBUG, TOL_FP32), (P.PREC_BF16, TOL_BF16)])
@pytest.mark.parametrize("fuse", [1, 0])
@pytest.mark.parametrize("lens,pad", [((70, 130, 9), 0.1), ((1,), 0.0), ((0, 300, 0, 129), 0.3), ((128, 256), 0.0)])
def test_two_stack_small(lens, pad, fuse, precision, tol):
    """Two parallel encoders + binary head on ragged / padded / empty events; N both a multiple of 128
    (no gap between the stacks' row blocks) and not."""
    W = synth.make_weights(TWO_TINY, seed=31)
    X, off = synth.make_events(lens, seed=32, pad_frac=pad)
    _two_stack_check(W, TWO_TINY, X, off, precision, tol, fuse)


def test_two_stack_paper_topology_bf16_and_candidates():
    """config `paper2` = the paper's network (two 3-block encoders, d 256, 16 x 16, ReLU, six heads): all 4 events against the
    oracle, then the paper's decode (binary score > 0.5, L156) of the GPU's own outputs, integers bit-exact."""
    name = "paper2"
    m = synth.model_cfg(name)
    W = synth.make_weights(name)
    X, off = synth.make_named_events(name)
    mod, lg, rg, bn = _two_stack_check(W, m, X, off, P.PREC_BF16, TOL_BF16)
    print("paper2 launches per step:", mod.query(P.Q_LAUNCHES))
    Xd = torch.from_numpy(X).cuda()
    c = P.build_candidates(Xd, off, torch.from_numpy(lg).cuda(), torch.from_numpy(rg).cuda(), binary=torch.from_numpy(bn).cuda())
    torch.cuda.synchronize()
    ref = oracle.build_candidates(X, off, lg, rg, binary=bn)
    Mc = int(ref["cand_offsets"][-1])
    assert 0 < Mc < X.shape[0]
    assert np.array_equal(c["cand_offsets"].cpu().numpy(), ref["cand_offsets"])
    assert np.array_equal(c["cand_elem"].cpu().numpy()[:Mc], ref["cand_elem"])
    assert np.array_equal(c["cand_pid"].cpu().numpy()[:Mc], ref["cand_pid"])
    assert np.allclose(c["cand_p4"].cpu().numpy()[:Mc], ref["cand_p4"], rtol=1e-5, atol=1e-5)


def test_two_stack_fp32_debug_one_event():
    name = "paper2"
    m = synth.model_cfg(name)
    X, off = synth.make_named_events(name, max_events=1)
    _two_stack_check(synth.make_weights(name), m, X, off, P.PREC_FP32_DEBUG, TOL_FP32)


# ------------------------------------------------------------------------------------------- NEXT-4: latency / pipelined entries
def test_graph_replay_is_bitwise_identical():
    """MLPF_OPT_GRAPH: the second call with the same key is captured, later ones replayed; other events in between get
    graphs of their own; results are bitwise those of plain launches."""
    name = "cfg2"
    m = synth.model_cfg(name)
    W = synth.make_weights(name)
    X, off = synth.make_named_events(name, max_events=4)
    mod = P.Mlpf(W, m)
    Xd = torch.from_numpy(X).cuda()
    st = torch.cuda.Stream()
    N = X.shape[0]
    lg = torch.empty((N, 9), device="cuda"); rg = torch.empty((N, 5), device="cuda")
    ref = [t.clone() for t in mod.infer(Xd, off)]
    torch.cuda.synchronize()
    mod.set_option(P.OPT_GRAPH, 1)
    with torch.cuda.stream(st):
        for rep in range(4):                               # eager, capture, replay, replay -- per event
            for e in range(4):
                a, b = int(off[e]), int(off[e + 1])
                lg[a:b].zero_(); rg[a:b].zero_()
                mod.infer(Xd[a:b], np.array([0, b - a], np.int32), lg[a:b], rg[a:b], stream=st)
            st.synchronize()
            assert torch.equal(lg, ref[0]) and torch.equal(rg, ref[1]), rep
    assert mod.query(P.Q_LAUNCHES) > 0


def test_pipelined_host_entry_matches_synchronous_calls():
    name = "cfg2"
    m = synth.model_cfg(name)
    W = synth.make_weights(name)
    mod = P.Mlpf(W, m)
    st = torch.cuda.Stream()
    batches = []
    for k in range(5):
        X, off = synth.make_events((300 + 50 * k, 517, 64 * k + 1), seed=50 + k, pad_frac=0.1)
        xh = torch.from_numpy(X).pin_memory()
        N = X.shape[0]
        batches.append((xh, off, torch.empty((N, 9)).pin_memory(), torch.empty((N, 5)).pin_memory(), X))
    for xh, off, lh, rh, X in batches:                     # all five in flight, one synchronisation at the end
        mod.infer_host_async(xh, off, lh, rh, stream=st)
    mod.host_sync(stream=st)
    for xh, off, lh, rh, X in batches:
        lg, rg = mod.infer(torch.from_numpy(X).cuda(), off)
        torch.cuda.synchronize()
        assert torch.equal(lh, lg.cpu()) and torch.equal(rh, rg.cpu())


# ------------------------------------------------------------------------------------------- NEXT-3: FP8 operands
@pytest.mark.parametrize("name,max_events", [("cfg2", 4), ("cfg3", 2), ("paper2", 1)])
def test_fp8_qkv_projection_drift(name, max_events):
    """MLPF_OPT_FP8 = 1: the QKV projection with e4m3 operands.  Not a parity claim: the drift against the (unchanged)
    fp64 / W-bf16 oracle is MEASURED, printed, and only bounded loosely (it is recorded in DESIGN.md; BF16 stays the default)."""
    m = synth.model_cfg(name)
    W = synth.make_weights(name)
    X, off = synth.make_named_events(name, max_events=max_events)
    mod = P.Mlpf(W, m)
    Xd = torch.from_numpy(X).cuda()
    lg0, rg0 = [t.cpu().numpy() for t in mod.infer(Xd, off)]
    mod.set_option(P.OPT_FP8, 1)
    lg8, rg8 = [t.cpu().numpy() for t in mod.infer(Xd, off)]
    torch.cuda.synchronize()
    assert np.isfinite(lg8).all() and np.isfinite(rg8).all() and not np.array_equal(lg8, lg0)
    lr, rr = oracle.forward(X, off, oracle.quantize_weights(W), m)
    valid = X[:, 0] != 0
    e_bf16 = max(oracle.parity_metrics(lg0, lr, valid)[0], oracle.parity_metrics(rg0, rr, valid)[0])
    e_fp8 = max(oracle.parity_metrics(lg8, lr, valid)[0], oracle.parity_metrics(rg8, rr, valid)[0])
    agree = oracle.argmax_agreement(lg8, lr, valid)
    print(f"FP8 drift {name}: max rel err bf16 {e_bf16:.2e} -> fp8-qkv {e_fp8:.2e}; argmax agreement (decidable, frac, raw) {agree}")
    assert e_bf16 <= TOL_BF16 and e_fp8 <= 0.25
