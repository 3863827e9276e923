"""N > 1 host logic of bench.py on CPU (gloo, world_size 2): per-rank batches differ and keep the recipe,
the step time is the max over ranks, and under torchrun only rank 0 prints the reference-arm line."""
import json
import os
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
import bench  # noqa: E402


def test_rank_batches_differ_but_follow_the_recipe():
    X0, o0 = bench.workload("cfg2", 0)
    X1, o1 = bench.workload("cfg2", 1)
    assert len(o0) == len(o1) == 17 and o0[0] == o1[0] == 0
    assert not np.array_equal(np.diff(o0), np.diff(o1))
    for o in (o0, o1):
        n = np.diff(o)
        assert n.min() >= 500 and n.max() <= 2000
    assert X0.shape[1] == X1.shape[1] == 55 and set(np.unique(X1[:, 0])) <= {1.0, 2.0, 3.0, 4.0}


def _worker(rank, port, out):
    import torch.distributed as dist
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=2)
    v = bench.max_over_ranks(10.0 + 5.0 * rank, dist, "cpu")
    dist.barrier()
    dist.destroy_process_group()
    out[rank] = v


def test_max_over_ranks_gloo():
    import torch.multiprocessing as mp
    with mp.Manager() as mgr:
        out = mgr.dict()
        mp.spawn(_worker, args=(29731, out), nprocs=2, join=True)
        assert out[0] == out[1] == 15.0


@pytest.mark.timeout(300)
def test_reference_arm_under_torchrun_prints_one_line():
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr",
           "127.0.0.1", "--master-port", "29733", os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
           "--workload", "cfg1", "--steps", "1", "--warmup", "0"]
    r = subprocess.run(cmd, capture_output=True, text=True, cwd=ROOT, timeout=280)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["cpu_baseline"]["kind"] == "oracle"
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["value"] > 0
