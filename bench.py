#!/usr/bin/env python
"""bench.py -- MLPF encoder forward (steps a0..a8) on synthetic CMS-like events.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg3] [--streams S] [--impl ours|reference]

One "step" = one mlpf_infer call over one batch of the workload (default: BASELINE.json configs[2],
the CMS-scale config the metric is quoted on: 8 events, ~5000 PF elements each, L=6, d=256, H=8).
Prints ONE JSON line (rank 0).  `value` = events/s with inputs resident in HBM; `e2e` = the same through
mlpf_infer_host (pinned host buffers, H2D + D2H inside the timed region); `roofline` = the attention
kernel (a4, the dominant kernel) against the measured dense-bf16 peak; `cpu_baseline` = the fp64 numpy
oracle timed on this box's host cores on a bounded sample.  N > 1: events are independent, so every rank
runs its own batch (weak scaling, no data-path collective); time = max over ranks.
"""
from __future__ import annotations
import argparse
import json
import os
import sys
import threading
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, HERE)

import synth  # noqa: E402

METRIC = "events_per_s"
UNIT = "events/s"
L2_FLUSH_BYTES = 256 << 20          # > 126 MB L2


def load_peaks():
    p = os.path.join(HERE, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        return dict(hbm_gbs=d["hbm_gbs"], tflops_burst=d["bf16_tflops"],
                    tflops_sustained=d.get("bf16_tflops_sustained", d["bf16_tflops"]), source="measured")
    return dict(hbm_gbs=6650.0, tflops_burst=1590.0, tflops_sustained=1400.0, source="fallback")


def workload(name, rank=0):
    """Seeded synthetic batch; rank r > 0 draws its own batch of the same recipe."""
    seed = None if rank == 0 else synth.BASE_SEED + 100 * rank + synth.configs.CFG_INDEX[name]
    X, off = synth.make_named_events(name, seed=seed)
    return X, off


def flop_model(m, off, X=None):
    """Algorithmic FLOPs of one forward pass (linear 2*M*N*K, attention 4*d*sum n_e^2 per layer).  With X the
    row counts are those of the VALID rows: pad rows (type 0) take part in nothing (reading A2) and are dropped after a0."""
    n = np.diff(off).astype(np.float64)
    if X is not None:
        v = np.concatenate([[0], np.cumsum(X[:, 0] != 0)])
        n = (v[off[1:]] - v[off[:-1]]).astype(np.float64)
    N, s2 = n.sum(), (n * n).sum()
    d, dff, L, F = m.d_model, m.d_ff, m.n_layers, m.n_feat
    attn_layer = 4.0 * d * s2
    lin_layer = 2.0 * N * (3 * d * d + d * d + 2 * d * dff)
    emb = 2.0 * N * (F * d + d * d)
    heads = 2.0 * N * ((1 + len(m.reg_dims)) * d * d + (m.n_classes + sum(m.reg_dims)) * d)
    S = getattr(m, "n_stacks", 1)
    heads += 2.0 * N * (m.d_model * m.d_model + m.d_model) * (1 if getattr(m, "binary_head", False) else 0)
    return dict(attn_per_launch=S * attn_layer, total=S * L * (attn_layer + lin_layer) + emb + heads,
                gemm_per_layer=S * lin_layer)


class ClockSampler(threading.Thread):
    """Samples SM clock + throttle reasons through NVML while the timed region runs."""

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.stop_flag, self.sm, self.reasons, self.sm_max, self.ok = index, False, [], set(), None, False
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.sm_max = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
            self.ok = True
        except Exception:
            self.ok = False

    def run(self):
        if not self.ok:
            return
        nv = self.nv
        names = {0x8: "hw_slowdown", 0x40: "hw_thermal_slowdown", 0x20: "sw_thermal_slowdown", 0x4: "sw_power_cap",
                 0x80: "hw_power_brake", 0x2: "applications_clocks_setting", 0x100: "display_clock_setting"}
        while not self.stop_flag:
            try:
                self.sm.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for bit, nm in names.items():
                    if r & bit:
                        self.reasons.add(nm)
            except Exception:
                pass
            time.sleep(0.02)

    def result(self):
        if not self.ok or not self.sm:
            return {"sm_mhz": None, "sm_max_mhz": self.sm_max, "reasons": ["nvml_unavailable"]}
        return {"sm_mhz": float(np.median(self.sm)), "sm_max_mhz": self.sm_max, "reasons": sorted(self.reasons)}


# ------------------------------------------------------------------------------------------------ CPU oracle leg
def oracle_sample(name, X, off, m, budget_s):
    """Bounded sample of the workload for the oracle: the shortest event, or a prefix of it when even that
    would not fit `budget_s` (the oracle runs at roughly 10 GFLOP/s per host core in fp64 numpy)."""
    n = np.diff(off)
    e = int(np.argmin(np.where(n > 0, n, n.max() + 1)))
    a, b = int(off[e]), int(off[e + 1])
    cores = os.cpu_count() or 1
    est_rate = 1.2e10 * min(cores, 8) / 8 * 1.0          # FLOP/s, calibrated on 8 cores: 21 s for a 5048-row cfg3 event
    ns = b - a
    while ns > 256:
        f = flop_model(m, np.array([0, ns]))["total"]
        if f / est_rate <= budget_s:
            break
        ns = int(ns * 0.85)
    whole = ns == b - a
    desc = (f"{name} event {e} ({'whole, ' if whole else 'first '}{ns} of {b - a} elements), fp64 numpy oracle; "
            f"events/s = (model FLOPs of the sample / seconds) / (model FLOPs per mean event of the batch)")
    return X[a:a + ns], np.array([0, ns], np.int32), desc


def time_oracle(Xs, offs, W, m, flops_per_event):
    import oracle
    t0 = time.perf_counter()
    oracle.forward(Xs, offs, W, m)
    dt = time.perf_counter() - t0
    return flop_model(m, offs)["total"] / dt / flops_per_event, dt


def numpy_threads():
    try:
        from threadpoolctl import threadpool_info
        ns = [p.get("num_threads", 1) for p in threadpool_info()]
        return max(ns) if ns else 1
    except Exception:
        return os.cpu_count() or 1


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    name = args.workload
    m = synth.model_cfg(name)
    W = synth.make_weights(name)
    X, off = workload(name)
    E = len(off) - 1
    fl = flop_model(m, off)
    per_step_budget = max(2.0, min(25.0, 240.0 / (args.steps + args.warmup)))
    Xs, offs, desc = oracle_sample(name, X, off, m, per_step_budget)
    for _ in range(args.warmup):
        time_oracle(Xs, offs, W, m, fl["total"] / E)
    times = []
    for _ in range(args.steps):
        _, dt = time_oracle(Xs, offs, W, m, fl["total"] / E)
        times.append(dt)
    tot = float(np.sum(times))
    sample_events = flop_model(m, offs)["total"] / (fl["total"] / E)      # the sample, in mean-event units
    value = sample_events * args.steps / tot
    cores = numpy_threads()
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * tot / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": name, "events": E, "elements": int(off[-1]), "n_layers": m.n_layers,
                       "d_model": m.d_model, "n_heads": m.n_heads, "d_ff": m.d_ff, "step": "one oracle pass over the sample"},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def max_over_ranks(x, dist, device):
    """Time of a multi-rank region = the slowest rank's (no-op without a process group)."""
    if dist is None:
        return x
    import torch
    t = torch.tensor([x], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


# ------------------------------------------------------------------------------------------------ GPU arm
def run_ours(args):
    import torch
    import paper_2601_17554_b200 as P

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (libmlpf has no CPU fallback)")
    torch.cuda.set_device(local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    name = args.workload
    m = synth.model_cfg(name)
    W = synth.make_weights(name)
    X, off = workload(name, rank)
    E, N = len(off) - 1, int(off[-1])
    fl = flop_model(m, off, X)
    peaks = load_peaks()

    mod = P.Mlpf(W, m)
    for key, val in (args.opt or []):
        mod.set_option(int(key), int(val))
    st = torch.cuda.Stream()
    Xd = torch.from_numpy(X).cuda()
    lg = torch.empty((N, mod.n_classes), dtype=torch.float32, device="cuda")
    rg = torch.empty((N, mod.n_regress), dtype=torch.float32, device="cuda")
    flush = torch.empty(L2_FLUSH_BYTES, dtype=torch.uint8, device="cuda")
    torch.cuda.synchronize()

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    def timed_steps(k, profile):
        """k steps; L2 flushed (untimed) before each; returns per-step ms (CUDA events on `st`) and per-class ms."""
        mod.set_option(P.OPT_PROFILE, 1 if profile else 0)
        ms, cls = [], {c: [0.0, 0] for c in P.KERNEL_CLASSES}
        with torch.cuda.stream(st):
            for _ in range(k):
                flush.zero_()
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(st)
                mod.infer(Xd, off, lg, rg, stream=st)
                e1.record(st)
                e1.synchronize()
                ms.append(e0.elapsed_time(e1))
                if profile:
                    for c, (t, n) in mod.profile(stream=st).items():
                        cls[c][0] += t
                        cls[c][1] += n
        mod.set_option(P.OPT_PROFILE, 0)
        return np.array(ms), cls

    timed_steps(args.warmup, False)
    barrier()
    sampler = ClockSampler(local_rank)
    sampler.start()
    t_wall0 = time.perf_counter()
    ms, _ = timed_steps(args.steps, False)
    barrier()
    t_wall = time.perf_counter() - t_wall0
    # the same K steps again with a CUDA-event pair around every kernel class (roofline numerator)
    ms_prof, cls = timed_steps(args.steps, True)
    sampler.stop_flag = True
    sampler.join()
    launches_per_step = int(mod.query(P.Q_LAUNCHES))
    total_ms = max_over_ranks(float(ms.sum()), dist, "cuda")
    value = world * E * args.steps / (total_ms * 1e-3)

    # ---- end to end: pinned host buffers in, host buffers out, every step's H2D and D2H inside the timed region.
    # `e2e.value`: K steps issued back to back through mlpf_infer_host_async (the copies of one step overlap the kernels of
    # its neighbours: two staging slots, the library's own copy streams) and ONE mlpf_host_sync at the end, wall clock;
    # `e2e.sync_ms_per_step`: the synchronous mlpf_infer_host, one step at a time (H2D, kernels, D2H strictly in sequence).
    xh = [torch.from_numpy(X).pin_memory() for _ in range(2)]
    lh = [torch.empty((N, mod.n_classes), dtype=torch.float32).pin_memory() for _ in range(2)]
    rh = [torch.empty((N, mod.n_regress), dtype=torch.float32).pin_memory() for _ in range(2)]
    for _ in range(max(3, args.warmup // 2)):
        mod.infer_host(xh[0], off, lh[0], rh[0], stream=st)
    barrier()
    sync_ms = []
    for _ in range(min(args.steps, 20)):
        with torch.cuda.stream(st):
            flush.zero_()
        st.synchronize()
        t0 = time.perf_counter()
        mod.infer_host(xh[0], off, lh[0], rh[0], stream=st)            # synchronises before returning
        sync_ms.append(1e3 * (time.perf_counter() - t0))
    barrier()
    t0 = time.perf_counter()
    for i in range(args.steps):
        mod.infer_host_async(xh[i & 1], off, lh[i & 1], rh[i & 1], stream=st)
    mod.host_sync(stream=st)
    e2e_wall = 1e3 * (time.perf_counter() - t0)
    e2e_total = max_over_ranks(float(e2e_wall), dist, "cuda")
    e2e_value = world * E * args.steps / (e2e_total * 1e-3)
    result_check = float(lh[0].abs().sum() + rh[0].abs().sum() + lh[1].abs().sum())     # the device->host results are read

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    # ---- single-event latency (one event per call, as the paper deploys it, L224): p50 / p90 over events x repeats,
    # (i) device-timed plain launches, (ii) device-timed with MLPF_OPT_GRAPH (one CUDA-graph launch per call once a key
    # repeats), (iii) end to end through the synchronous mlpf_infer_host (H2D + kernels + D2H, wall clock)
    reps = max(4, min(10, args.steps // 2))

    def one_event_sweeps(graph):
        mod.set_option(P.OPT_GRAPH, 1 if graph else 0)
        out = []
        with torch.cuda.stream(st):
            for rep in range(reps + 2):
                for e in range(E):
                    a, b = int(off[e]), int(off[e + 1])
                    if b == a:
                        continue
                    o1 = np.array([0, b - a], np.int32)
                    flush.zero_()
                    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    e0.record(st)
                    mod.infer(Xd[a:b], o1, lg[a:b], rg[a:b], stream=st)
                    e1.record(st)
                    e1.synchronize()
                    if rep >= 2:                                      # sweeps 0, 1: warm-up / graph capture
                        out.append(e0.elapsed_time(e1))
        mod.set_option(P.OPT_GRAPH, 0)
        return np.array(out)

    lat = one_event_sweeps(False)
    lat_graph = one_event_sweeps(True)
    lat_e2e = []
    for rep in range(reps + 1):
        for e in range(E):
            a, b = int(off[e]), int(off[e + 1])
            if b == a:
                continue
            o1 = np.array([0, b - a], np.int32)
            t0 = time.perf_counter()
            mod.infer_host(xh[0][a:b], o1, lh[0][a:b], rh[0][a:b], stream=st)
            if rep >= 1:
                lat_e2e.append(1e3 * (time.perf_counter() - t0))
    lat_e2e = np.array(lat_e2e)

    # ---- candidate building (the step after the forward pass): mlpf_build_candidates on this batch's
    # own outputs, L2 flushed before each call; HBM / launch-latency bound, reported against the copy peak
    cand_ms = []
    scratch = torch.empty(int(P.lib().mlpf_candidates_scratch_bytes(N, E)), dtype=torch.uint8, device="cuda")
    with torch.cuda.stream(st):
        mod.infer(Xd, off, lg, rg, stream=st)
        for i in range(13):
            flush.zero_()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(st)
            cand = P.build_candidates(Xd, off, lg, rg, scratch=scratch, stream=st)
            e1.record(st)
            e1.synchronize()
            if i >= 3:
                cand_ms.append(e0.elapsed_time(e1))
    n_cand = int(cand["cand_offsets"][-1])
    cand_bytes = N * (4 * mod.n_classes + 4 + 20 + 8 + 2) + n_cand * 24     # logits, type, regress, pT/E in, code; outputs
    candidates = {"ms_p50": float(np.percentile(cand_ms, 50)), "launches": 2, "candidates": n_cand, "elements": N,
                  "algorithmic_bytes": int(cand_bytes), "gbs": cand_bytes / (np.percentile(cand_ms, 50) * 1e-3) / 1e9,
                  "hbm_peak_gbs": peaks["hbm_gbs"]}

    # ---- several concurrent streams (north_star: "also with several concurrent streams"): the batch is split into
    # S contiguous event groups, one CUDA stream each, enqueued round-robin from this thread (mlpf_infer only enqueues)
    multi = None
    if args.streams > 1:
        S = min(args.streams, E)
        bounds = [i * E // S for i in range(S + 1)]
        streams = [torch.cuda.Stream() for _ in range(S)]
        fork = torch.cuda.Stream()

        def one_round():
            with torch.cuda.stream(fork):
                flush.zero_()
                t0 = torch.cuda.Event(enable_timing=True)
                t0.record(fork)
            ends = []
            for i, sx in enumerate(streams):
                e0_, e1_ = bounds[i], bounds[i + 1]
                r0, r1 = int(off[e0_]), int(off[e1_])
                sx.wait_event(t0)
                mod.infer(Xd[r0:r1], off[e0_:e1_ + 1] - off[e0_], lg[r0:r1], rg[r0:r1], stream=sx)
                ev = torch.cuda.Event(enable_timing=True)
                ev.record(sx)
                ends.append(ev)
            torch.cuda.synchronize()
            return max(t0.elapsed_time(ev) for ev in ends)

        for _ in range(max(3, args.warmup)):
            one_round()
        mt = np.array([one_round() for _ in range(args.steps)])
        multi = {"n": S, "events_per_s": E / (mt.mean() * 1e-3), "ms_per_step": float(mt.mean()),
                 "ms_p50": float(np.percentile(mt, 50)), "ms_p90": float(np.percentile(mt, 90)),
                 "workspace_bytes_all_streams": int(mod.query(P.Q_WORKSPACE_BYTES))}

    # ---- roofline of the dominant kernel (a4 attention): algorithmic FLOPs per launch / mean launch duration.
    # The class time includes the norms pre-pass (one small launch per layer); launches = layers.
    at_ms, at_n = cls["attention"]
    n_att = m.n_layers * args.steps                                      # attention launches (grouped over the stacks)
    per_launch_s = at_ms * 1e-3 / max(n_att, 1)
    achieved = fl["attn_per_launch"] / per_launch_s / 1e12 if at_ms else None
    peak = peaks["tflops_sustained"]
    share = {c: round(t / max(sum(v[0] for v in cls.values()), 1e-9), 4) for c, (t, n) in cls.items()}
    gemm_ms = sum(cls[c][0] for c in ("qkv", "outproj", "ffn1", "ffn2", "post"))
    gemm_tflops = fl["gemm_per_layer"] * m.n_layers * args.steps / (gemm_ms * 1e-3) / 1e12 if gemm_ms else None
    traffic, traffic_note = None, None                # DRAM bytes per launch from the committed ncu --set full capture
    tpath = os.path.join(HERE, "profiles", "attn_traffic.json")
    if os.path.exists(tpath):
        with open(tpath) as f:
            tj = json.load(f)
        if tj.get("workload") == name and tj.get("kernel") == "k_tc_attn2":
            traffic, traffic_note = tj["dram_bytes_per_launch"], tj.get("source")
    # The binding unit of this kernel is not the tensor pipe but the softmax exponentials (one per score = per 4 hd tensor
    # FLOPs): MUFU ex2 plus the share moved to the FMA pipe.  ALU ceiling = measured MUFU results / clk / SM (micro-benchmark
    # in the library, run here) x SMs x the SM clock seen during the run / the share of exponentials left on the MUFU, in
    # tensor-FLOP equivalents (x 4 hd).
    S_ = getattr(m, "n_stacks", 1)
    mufu_rate = P.microbench(0, 4096, stream=st)
    poly_rate = P.microbench(2, 2048, stream=st)
    bf16x2_rate = P.microbench(1, 4096, stream=st)
    clk = (sampler.result()["sm_mhz"] or sampler.result()["sm_max_mhz"] or 1965.0) * 1e6
    nsm = torch.cuda.get_device_properties(0).multi_processor_count
    # the library's default (include/mlpf.h MLPF_OPT_ATTN_POLY): 8 of 16 pairs with the prescaled scores of the model path;
    # 7 (hd <= 32) / 0 (hd = 64) with MLPF_OPT_EPI_NORMS = 0; an explicit --opt 9 n wins
    opts = {int(k): int(v) for k, v in (args.opt or [])}
    pe = opts.get(9, -1)
    if pe < 0:
        pe = 8 if opts.get(14, 1) == 1 else (7 if m.head_dim <= 32 else 0)
    poly_share = pe / 16.0
    mufu_only = mufu_rate * nsm * clk * 4 * m.head_dim / 1e12            # every exponential on the MUFU
    alu_peak = mufu_only / max(1.0 - poly_share, 1e-9)                   # with the kernel's share on the FMA pipe
    nvalid_rows = int((X[:, 0] != 0).sum())
    roofline = {"bound": "alu", "kernel": "k_tc_attn2 (a4)", "achieved": achieved, "peak": peak, "unit": "TFLOP/s",
                "frac": (achieved / peak) if achieved else None, "traffic": traffic, "traffic_source": traffic_note,
                "peak_source": f"{peaks['source']} bf16_tflops_sustained (dense bf16 tensor peak; the kernel is a contraction)",
                "alu": {"binding_pipe": "issue slots of the softmax warps: exponentials on XU (MUFU ex2) + FMA pipes, one per 4*hd tensor FLOPs; packed and 16-lane instructions take two issue cycles",
                        "mufu_ex2_per_clk_per_sm_measured": mufu_rate, "mufu_ex2_bf16x2_per_clk_per_sm_measured": bf16x2_rate,
                        "fma_poly_exp_per_clk_per_sm_measured": poly_rate,
                        "sm_clock_hz": clk, "poly_share": poly_share,
                        "mufu_only_ceiling_tflops": mufu_only, "alu_ceiling_tflops": alu_peak,
                        "frac_of_alu_ceiling": (achieved / alu_peak) if achieved else None,
                        "mufu_only_ceiling_frac_of_tensor_peak": mufu_only / peak},
                "algorithmic_bytes_per_launch": float(S_ * nvalid_rows) * m.d_model * 2 * (3 + 2),   # read q,k,v; write o hi + lo
                "flops_per_launch": fl["attn_per_launch"], "ms_per_launch": per_launch_s * 1e3,
                "class_time_share": share,
                "class_ms_per_step": {c: round(t / args.steps, 4) for c, (t, n) in cls.items()},
                "gemm_tflops": gemm_tflops, "gemm_frac": (gemm_tflops / peak) if gemm_tflops else None,
                "whole_step_tflops": fl["total"] * args.steps / (total_ms * 1e-3) / 1e12}
    # per-class fractions of the GEMM-shaped steps (tensor peak) and of the HBM-bound glue kernels (copy peak)
    Nv, d_, dff_, L_ = float(nvalid_rows), m.d_model, m.d_ff, m.n_layers

    def tfl(flops_per_step, c):
        t = cls[c][0] / args.steps * 1e-3
        return None if t <= 0 else {"tflops": flops_per_step / t / 1e12, "frac_tensor": flops_per_step / t / 1e12 / peak,
                                    "ms_per_step": t * 1e3}
    roofline["per_class"] = {
        "qkv (a3)": tfl(S_ * L_ * 2 * Nv * 3 * d_ * d_, "qkv"),
        "post (a5+a6+a7 fused)": tfl(S_ * L_ * 2 * Nv * (d_ * d_ + 2 * d_ * dff_), "post"),
        "outproj (a5)": tfl(S_ * L_ * 2 * Nv * d_ * d_, "outproj"),
        "ffn1 (a6)": tfl(S_ * L_ * 2 * Nv * d_ * dff_, "ffn1"),
        "ffn2 (a7)": tfl(S_ * L_ * 2 * Nv * d_ * dff_, "ffn2"),
        "heads_l1 (a8)": tfl(2 * Nv * (1 + len(m.reg_dims) + (1 if getattr(m, "binary_head", False) else 0)) * d_ * d_, "heads_l1"),
        "embed_l2 (a1)": tfl(2 * Nv * d_ * d_, "embed_l2")}
    n_ln = cls["layernorm"][1] / max(args.steps, 1)
    roofline["glue_gbs"] = {"hbm_peak": peaks["hbm_gbs"],
                            "layernorm": (N * d_ * (4 + 2) * n_ln) * args.steps / max(cls["layernorm"][0], 1e-9) / 1e6,
                            "embed_l1": N * (m.n_feat * 4 + d_ * 4) * args.steps / max(cls["embed_l1"][0], 1e-9) / 1e6,
                            # null when the output rows are part of k_tc_heads (d <= 256): no separate launch to time
                            "heads_l2": (Nv * ((1 + len(m.reg_dims)) * d_ * 4 + 56) * args.steps / cls["heads_l2"][0] / 1e6
                                         if cls["heads_l2"][0] > 0 else None)}

    # ---- CPU oracle on a bounded sample (rank 0, N = 1 only)
    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        Xs, offs, desc = oracle_sample(name, X, off, m, 25.0)
        v, dt = time_oracle(Xs, offs, W, m, fl["total"] / E)
        cpu = {"value": v, "unit": UNIT, "cores": numpy_threads(), "kind": "oracle", "sample": desc, "seconds": dt}

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": total_ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "bf16", "data": "synthetic",
            "config": {"workload": name, "events": E, "elements": N, "max_event": int(np.diff(off).max()),
                       "n_layers": m.n_layers, "d_model": m.d_model, "n_heads": m.n_heads, "d_ff": m.d_ff,
                       "activation": m.activation, "parallelism": f"events sharded over {world} GPU(s), no collective",
                       "l2": "flushed (256 MB memset) before every timed step", "split_activations": 1},
            "ms_per_event": total_ms / args.steps / E,
            "step_ms_p50": float(np.percentile(ms, 50)), "step_ms_p90": float(np.percentile(ms, 90)),
            "ms_per_step_with_class_events": float(ms_prof.mean()),
            "single_event_ms_p50": float(np.percentile(lat, 50)), "single_event_ms_p90": float(np.percentile(lat, 90)),
            "single_event_graph_ms_p50": float(np.percentile(lat_graph, 50)), "single_event_graph_ms_p90": float(np.percentile(lat_graph, 90)),
            "single_event_e2e_ms_p50": float(np.percentile(lat_e2e, 50)), "single_event_e2e_ms_p90": float(np.percentile(lat_e2e, 90)),
            "wall_s_timed_region": t_wall,
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": int(N * mod.n_feat * 4),
                    "d2h_bytes_per_step": int(N * (mod.n_classes + mod.n_regress) * 4),
                    "ms_per_step": e2e_total / args.steps, "sync_ms_per_step": float(np.mean(sync_ms)),
                    "how": "K steps through mlpf_infer_host_async + one mlpf_host_sync (copies overlap neighbouring steps' kernels)",
                    "result_checksum": result_check},
            "gpu_launches": launches_per_step * args.steps, "launches_per_step": launches_per_step,
            "peak_bytes": {"weights": int(mod.query(P.Q_WEIGHT_BYTES)), "workspace": int(mod.query(P.Q_WORKSPACE_BYTES)),
                           "torch_max_allocated": int(torch.cuda.max_memory_allocated())},
            "streams": multi, "candidates": candidates, "clocks": sampler.result(), "roofline": roofline, "cpu_baseline": cpu}
    print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--workload", default="cfg3", choices=["cfg1", "cfg2", "cfg3", "cfg4", "cfg5a", "cfg5b", "paper", "paper2"])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--opt", nargs=2, action="append", metavar=("KEY", "VALUE"),
                    help="mlpf_set_option(KEY, VALUE) before the run (tuning experiments; include/mlpf.h MLPF_OPT_*)")
    ap.add_argument("--streams", type=int, default=1, help="also time the batch split over this many concurrent CUDA streams")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
