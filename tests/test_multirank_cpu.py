"""The N > 1 path on CPU (world_size 2, gloo).  The hot path does not shard across GPUs in this build
(replicas only -- BASELINE.json says one GPU; the paper's own parallelism is an
ensemble of independent quenches), so what there is to cover is bench.py's rank logic: every
rank quenches its own seed, timings are reduced with MAX over ranks, the whole-job value counts every
rank's pair-terms, rank 0 alone prints, and the reference arm runs on rank 0 only."""
import json
import os
import socket
import subprocess
import sys
from pathlib import Path

import numpy as np
import pytest

ROOT = Path(__file__).resolve().parent.parent


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    import torch.distributed as dist
    sys.path.insert(0, str(ROOT))
    import bench
    from paper_2304_09139_b200 import inputs
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    ms = bench.max_over_ranks([10.0 + 5.0 * rank, 3.0 - rank], "cpu")
    hi, _ = inputs.uniform_positions(inputs.CONFIGS["cfg1"], rank)      # replica r quenches seed r
    digest = float(hi[:4].sum())
    gathered = [None] * world
    dist.all_gather_object(gathered, digest)
    if rank == 0:
        with open(out, "w") as f:
            json.dump({"ms": ms, "digests": gathered,
                       "value": bench.whole_job_value(1000, 4, world, ms[0])}, f)
    dist.barrier()
    dist.destroy_process_group()


def test_max_over_ranks_and_replica_seeds(tmp_path):
    import torch.multiprocessing as mp
    out = tmp_path / "r.json"
    mp.spawn(_worker, args=(2, _free_port(), str(out)), nprocs=2, join=True)
    r = json.loads(out.read_text())
    assert r["ms"] == [15.0, 3.0]                      # MAX over ranks, element-wise
    assert r["digests"][0] != r["digests"][1]          # different seeds on different ranks
    assert r["value"] == pytest.approx(2 * 1000 * 4 / 15e-3)


def test_identity_without_process_group():
    sys.path.insert(0, str(ROOT))
    import bench
    assert bench.max_over_ranks([1.5, 2.5], "cpu") == [1.5, 2.5]
    assert bench.whole_job_value(9e9, 10, 1, 222.0) == pytest.approx(9e9 * 10 / 0.222)


def test_reference_arm_under_torchrun_world2():
    """`bench.py --impl reference` launched exactly as the driver launches N = 2: rank 0 alone runs the
    oracle and prints ONE JSON line, rank 1 exits 0 without work."""
    env = dict(os.environ, OMP_NUM_THREADS="4")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
           "--master-addr", "127.0.0.1", "--master-port", str(_free_port()), str(ROOT / "bench.py"),
           "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0", "--config", "cfg1"]
    p = subprocess.run(cmd, capture_output=True, text=True, timeout=600, env=env, cwd=str(ROOT))
    assert p.returncode == 0, p.stderr[-2000:]
    lines = [ln for ln in p.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1, p.stdout
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["value"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["e2e"]["h2d_bytes_per_step"] == 0
