"""The N > 1 paths on CPU (world_size 2, gloo): bench.py's rank logic (replica mode) and, at the end of the file, the
host-side plumbing of particle shards.  Replica mode (the paper's own parallelism is an
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


# ---------------------------------------------------------------------------------------------------------------
# Particle shards: the host-side plumbing of bench.py --gpus N / paper_2304_09139_b200.sharding,
# world_size 2 on gloo.  The partial sums are opaque bytes added by the library's kernel in rank order; what is
# checked here is that the ranges deal out every particle exactly once, that the 128 communicator bytes reach every
# rank, and that the all-gather lays the ranks' partials out rank 0 first -- with the oracle standing in for the
# kernels: rank r's partial rho over its own particles, gathered, added in rank order, must be the oracle's full rho.
def _shard_worker(rank, world, port, out):
    import torch
    import torch.distributed as dist
    sys.path.insert(0, str(ROOT))
    from paper_2304_09139_b200 import inputs, sharding
    from oracle import shd_oracle as O
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    cfg = inputs.CONFIGS["cfg1"]
    hi, lo = inputs.uniform_positions(cfg, 0)
    a, b = sharding.shard_range(cfg.N, rank, world)
    hl, ll = sharding.local_positions(hi, lo, cfg.d, cfg.N, rank, world)
    uid = bytes(range(128)) if rank == 0 else None
    got_uid = sharding.broadcast_bytes(uid, 128, 0, "cpu")
    n = O.enumerate_Q(cfg.d, cfg.m_star)
    re, im = O.rho(cfg.d, b - a, cfg.L, hl, ll, n)                 # this rank's particles only
    mine = np.concatenate([np.stack(O.to_dd(re)).reshape(-1), np.stack(O.to_dd(im)).reshape(-1)])
    gathered = sharding.gather_partials(torch.from_numpy(mine.view(np.uint8).copy()))
    parts = gathered.numpy().view(np.float64).reshape(world, 2, 2, len(n))      # [rank][re/im][hi/lo][k]
    if rank == 0:
        with open(out, "w") as f:
            json.dump({"range": [a, b], "uid_ok": got_uid == bytes(range(128)),
                       "parts": parts.tolist()}, f)
    else:
        assert got_uid == bytes(range(128))
    dist.barrier()
    dist.destroy_process_group()


def test_shard_plumbing_world2(tmp_path):
    import torch.multiprocessing as mp
    sys.path.insert(0, str(ROOT))
    from paper_2304_09139_b200 import inputs, sharding
    from oracle import shd_oracle as O
    # ranges: every particle exactly once, contiguous, sizes differ by at most one
    for N, G in ((128, 2), (100000, 8), (10, 3), (7, 7)):
        r = [sharding.shard_range(N, k, G) for k in range(G)]
        assert r[0][0] == 0 and r[-1][1] == N and all(r[k][1] == r[k + 1][0] for k in range(G - 1))
        sizes = [b - a for a, b in r]
        assert max(sizes) - min(sizes) <= 1
    out = tmp_path / "s.json"
    mp.spawn(_shard_worker, args=(2, _free_port(), str(out)), nprocs=2, join=True)
    res = json.loads(out.read_text())
    assert res["uid_ok"] and res["range"] == [0, 64]
    cfg = inputs.CONFIGS["cfg1"]
    hi, lo = inputs.uniform_positions(cfg, 0)
    n = O.enumerate_Q(cfg.d, cfg.m_star)
    re, im = O.rho(cfg.d, cfg.N, cfg.L, hi, lo, n)
    parts = np.array(res["parts"])                                  # [rank][re/im][hi/lo][k]
    # fixed rank order: rank 0 first; (hi + lo) of rank 0 plus (hi + lo) of rank 1 against the oracle's full sum
    a_, b_ = parts[0, :, 0], parts[1, :, 0]
    tot_hi = a_ + b_
    bb = tot_hi - a_
    tot_lo = parts[0, :, 1] + parts[1, :, 1] + ((a_ - (tot_hi - bb)) + (b_ - bb))        # TwoSum error term
    err = O.cabsdiff_dd(re, im, tot_hi[0], tot_lo[0], tot_hi[1], tot_lo[1])
    assert err.max() < 1e-28 * cfg.N
    # and the order matters for what is checked: rank 0's partial is the sum over particles 0..63
    r0, i0 = O.rho(cfg.d, 64, cfg.L, *sharding.local_positions(hi, lo, cfg.d, cfg.N, 0, 2), n)
    assert O.cabsdiff_dd(r0, i0, parts[0, 0, 0], parts[0, 0, 1], parts[0, 1, 0], parts[0, 1, 1]).max() < 1e-30   # (dd carries 106 of binary128's 113 bits)
