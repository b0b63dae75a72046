#!/usr/bin/env python
"""bench.py -- one JSON line for the hot path of arXiv:2304.09139 on B200 (contract: task prompt, (4)).

A "step" is one pass of the whole evaluation hot path (phasor tables,
rho pass, Phi / S_max reduction, gradient pass) through the C-ABI of include/shd.h on one batch of
synthetic positions.  Workload at N=1: BASELINE.json configs[3] (d=2, N=1e5, chi=0.45, |Q|=9e4), the
configuration the metric "ms/eval at N=1e5" is quoted on.  Metric: energy+gradient pair-terms per
second (N*M per evaluation, "2 calculations, each with M N terms").

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config cfg4] [--impl reference]

N > 1 (torchrun, one rank per GPU): the particles are SHARDED over the ranks: every rank builds
the tables of its own particles, one all-gather of the partial sums of rho per evaluation (NCCL, bytes, added in fixed
rank order by the library's kernel), local gradient pass; total work fixed: "scaling": "strong".  `--replicas` runs
the paper's own ensemble parallelism instead (independent systems; no collective; "weak").
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent
sys.path.insert(0, str(ROOT))

from paper_2304_09139_b200 import inputs  # noqa: E402  (pure numpy workload recipes)

METRIC = "dd energy+grad pair-terms/s"
UNIT = "pair-terms/s"
# FP64 FMAs the formulation itself needs per particle-wavevector pair:
# rho pass 24 per (p,q) cell = 2 wavevectors -> 12; gradient pass 48 per cell -> 24 (issued as
# DMMA.8x8x4, 256 FMAs per warp instruction).
ALG_DFMA_RHO, ALG_DFMA_GRAD = 12.0, 24.0


def ncu_traffic(kernel, workload):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of `kernel`, read from the NEWEST committed ncu summary
    under profiles/ that states it for this workload, in the line format
        `traffic` (<workload>, dram read + write per launch): `k_a` 1.23 GB, `k_b` 4.56 GB
    Returns (bytes, file name) or (None, None): nothing is hard-coded here."""
    import re
    best = (None, None)
    for f in sorted((ROOT / "profiles").glob("r*_summary.md")):
        for ln in f.read_text().splitlines():
            if not ln.startswith("`traffic` (") or workload not in ln.split(")")[0]:
                continue
            m = re.search(r"`%s`\s+([0-9.]+)\s*GB" % re.escape(kernel), ln)
            if m:
                best = (float(m.group(1)) * 1e9, "profiles/" + f.name)
    return best

# INT8 tensor-core engines (k_rho8.cu, k_grad8.cu): 91 digit pairs per real product; 4 real products per (p,q)
# cell = 2 wavevectors in the rho pass, 8 in the gradient pass; 2 operations per multiply-accumulate
ALG_MAC_RHO8, ALG_MAC_GRAD8 = 182.0, 364.0


def dist_env():
    return int(os.environ.get("RANK", 0)), int(os.environ.get("LOCAL_RANK", 0)), int(os.environ.get("WORLD_SIZE", 1))


def max_over_ranks(values, device):
    """Element-wise MAX over all ranks of a short list of floats (timings): the contract's "time on the
    device, max over ranks".  Works on whatever backend the process group has (nccl on the GPU box,
    gloo in the CPU tests); with no process group it is the identity."""
    import torch
    import torch.distributed as dist
    t = torch.tensor(list(values), dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(x) for x in t.cpu()]


def whole_job_value(pairs_per_rank, steps, world, total_ms):
    """Whole-job throughput of N independent replicas (replicas only, weak
    scaling): every rank processes pairs_per_rank * steps pair-terms in the max-over-ranks time."""
    return world * float(pairs_per_rank) * steps / (total_ms * 1e-3)


# ------------------------------------------------------------------------------ oracle legs
def oracle_sample(cfg, hi, lo, budget_pairs, rho_dd=None, jrange=None):
    """Time the binary128 oracle (direct mode, as it stands) on a bounded sample of the workload:
    a strided set of wavevectors x all particles (rho) and a strided set of particles x all
    wavevectors (gradient).  Returns timing, the sample description and the oracle values."""
    from oracle import shd_oracle as O
    n = O.enumerate_Q(cfg.d, cfg.m_star)
    M = len(n)
    nk = int(max(1, min(M, budget_pairs // cfg.N)))
    nj = int(max(1, min(cfg.N, budget_pairs // M)))
    ks = np.unique(np.linspace(0, M - 1, nk).astype(np.int64))
    j0, j1 = jrange if jrange else (0, cfg.N)       # (sharded bench: the gradient sample lies in rank 0's particles)
    js = np.unique(np.linspace(j0, j1 - 1, min(nj, j1 - j0)).astype(np.int64))
    t0 = time.perf_counter()
    re, im = O.rho(cfg.d, cfg.N, cfg.L, hi, lo, n[ks])
    t1 = time.perf_counter()
    if rho_dd is None:          # timing only: the cost of the gradient sum does not depend on rho
        fr, fi = O.qzeros(M), O.qzeros(M)
    else:
        fr, fi = O.from_dd(rho_dd[0], rho_dd[1]), O.from_dd(rho_dd[2], rho_dd[3])
    t2 = time.perf_counter()
    g = O.grad(cfg.d, cfg.N, cfg.L, hi, lo, n, fr, fi, jlist=js)
    t3 = time.perf_counter()
    p_rho, p_grad = len(ks) * cfg.N, len(js) * M
    s_per_pair = (t1 - t0) / p_rho + (t3 - t2) / p_grad      # energy+gradient = both sums
    return dict(value=1.0 / s_per_pair, seconds=(t1 - t0) + (t3 - t2), cores=O.num_threads(),
                sample=f"direct mode: {len(ks)} strided k x {cfg.N} particles (rho) + "
                       f"{len(js)} strided particles x {M} k (gradient)",
                ks=ks, js=js, re=re, im=im, grad=g, n=n, pairs=0.5 * (p_rho + p_grad))


def run_reference(args, cfg):
    """--impl reference: the oracle, as it stands, on the host cores (rank 0 only)."""
    rank, _, world = dist_env()
    if rank != 0:
        return
    from oracle import shd_oracle as O
    O.build()
    hi, lo = inputs.uniform_positions(cfg, 0)
    cores = O.num_threads()
    total = args.steps + args.warmup
    budget = int(max(2e5, min(2.5e6 * cores, 1.2e8 * cores / 8 / total * 0.5)))
    times, values, last = [], [], None
    for i in range(total):
        last = oracle_sample(cfg, hi, lo, budget)
        if i >= args.warmup:
            times.append(last["seconds"])
            values.append(last["value"])
    # pair-terms/s of energy+gradient (both sums), harmonic mean over the timed steps
    value = len(values) / sum(1.0 / v for v in values)
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * float(np.mean(times)),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "binary128",
        "data": "synthetic", "config": workload_config(cfg, world),
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": last["sample"]},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def workload_config(cfg, world, replicas=True):
    src = f"BASELINE.json configs[{int(cfg.name[3:]) - 1}]" if cfg.name.startswith("cfg") else \
        "the paper's system size (P:33, P:89; not a BASELINE.json config)"
    return {"workload": f"{src}: d={cfg.d}, N={cfg.N}, unit density, "
                        f"chi={cfg.chi} (m*={cfg.m_star}, |Q|={cfg.M}), v=1, uniform seeded positions",
            "d": cfg.d, "N": cfg.N, "M": cfg.M, "pair_terms_per_eval": cfg.pairs,
            "parallelism": "single GPU" if world == 1 else (f"{world} independent replicas (seed = rank)" if replicas else
                            f"{world} particle shards, one all-gather of partial rho per evaluation (NCCL)"),
            "l2": "256 MB memset between timed steps (> 126 MB L2); table_bytes = the phasor tables an evaluation streams"}


# ------------------------------------------------------------------------------ clocks
class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        try:
            self.p = subprocess.Popen(["nvidia-smi", f"--id={index}", f"--query-gpu={self.Q}",
                                       "--format=csv,noheader,nounits", "-lms", "100"],
                                      stdout=self.f, stderr=subprocess.DEVNULL)
        except OSError:
            self.p = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.p is None:
            return out
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.p.kill()
        self.f.flush()
        self.f.seek(0)
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.f.read().splitlines():
            parts = [x.strip() for x in ln.split(",")]
            if len(parts) < 7:
                continue
            try:
                sm.append(float(parts[0])); mx.append(float(parts[1])); pw.append(float(parts[2]))
            except ValueError:
                continue
            for nm, val in zip(names, parts[3:7]):
                if val.lower().startswith("active"):
                    reasons.add(nm)
        self.f.close()
        os.unlink(self.f.name)
        if sm:
            out.update(sm_mhz=float(np.median(sm)), sm_max_mhz=float(max(mx)), reasons=sorted(reasons),
                       samples=len(sm), power_w_max=float(max(pw)))
        return out


# ------------------------------------------------------------------------------ the CUDA arm
def run_gpu(args, cfg):
    import torch
    rank, local_rank, world = dist_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (libshd has no CPU fallback)")
    torch.cuda.set_device(local_rank)
    if world > 1 or args.force_shard:
        import torch.distributed as dist
        if args.force_shard and world == 1 and "MASTER_ADDR" not in os.environ:
            os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT="29517", RANK="0", WORLD_SIZE="1")
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    from paper_2304_09139_b200 import shd

    sharded = (world > 1 and not args.replicas) or args.force_shard
    from paper_2304_09139_b200 import sharding
    if sharded:
        hi, lo = inputs.uniform_positions(cfg, 0)           # one system, its particles dealt out in contiguous ranges
        j_begin, j_end = sharding.shard_range(cfg.N, rank, world)
        hi_l, lo_l = sharding.local_positions(hi, lo, cfg.d, cfg.N, rank, world)
    else:
        hi, lo = inputs.uniform_positions(cfg, rank)        # replica r quenches seed r
        j_begin, j_end = 0, cfg.N
        hi_l, lo_l = hi, lo
    n_local = j_end - j_begin
    h = shd.Shd(cfg.d, n_local, cfg.L, m_star=cfg.m_star)
    assert h.M == cfg.M
    stream = torch.cuda.current_stream()
    h.set_stream(stream)
    if args.engine != "auto":
        h.set_engine(int(args.engine))      # else: the engine the library chose for this workload (shd_set_engine -1)
    engine = h.engine
    if sharded:
        h.set_shard(cfg.N, rank, world)
        sharding.init_comm(h)
    pos_hi, pos_lo = shd.from_host(hi_l, lo_l)
    grad_hi, grad_lo = torch.empty_like(pos_hi), torch.empty_like(pos_hi)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def timed_steps(steps, warmup, sample_clocks):
        """`steps` evaluations timed with CUDA events on the handle's stream (L2 flushed before each)."""
        h.set_timing(True)
        for _ in range(warmup):
            h.energy_grad(pos_hi, pos_lo, grad_hi, grad_lo)
        barrier()
        clocks = ClockSampler(local_rank) if (rank == 0 and sample_clocks) else None
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
        kms = {k: 0.0 for k in ("tables", "rho", "finish", "ctable", "grad")}
        launches, phi = 0, None
        for i in range(steps):
            flush.zero_()
            ev[i][0].record(stream)
            phi, _, _ = h.energy_grad(pos_hi, pos_lo, grad_hi, grad_lo)
            ev[i][1].record(stream)
            for k, v in h.kernel_ms().items():
                kms[k] += v
            launches += int(h.stat(1))
        barrier()
        clk = clocks.stop() if clocks else None
        h.set_timing(False)
        return float(sum(a.elapsed_time(b) for a, b in ev)), kms, launches, phi, clk

    # ---- device-resident leg (value)
    h.set_precision(args.precision)      # 3 (default) = the headline; 2 / 1 = the truncated evaluations of the precision ladder
    total_ms, kms, launches, phi, clk = timed_steps(args.steps, args.warmup, True)

    # ---- end-to-end leg: host (pinned) buffers through shd_energy_grad_host
    ph = torch.from_numpy(hi_l).pin_memory(); pl = torch.from_numpy(lo_l).pin_memory()
    gh = torch.empty(cfg.d * n_local, dtype=torch.float64).pin_memory(); gl = torch.empty_like(gh).pin_memory()
    for _ in range(max(1, min(args.warmup, 2))):
        h.energy_grad_host(ph.numpy(), pl.numpy(), gh.numpy(), gl.numpy())
    barrier()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        h.energy_grad_host(ph.numpy(), pl.numpy(), gh.numpy(), gl.numpy())
    torch.cuda.synchronize()
    e2e_s = time.perf_counter() - t0
    barrier()

    # ---- the same evaluation at a mid-quench state (non-zero lo words; dd paths with lo = 0 can be
    # accidentally cheaper): positions after --midquench-evals L-BFGS evaluations from the seeded start
    mid = None
    if args.midquench_evals > 0 and args.precision == 3:
        start = (pos_hi.clone(), pos_lo.clone())
        rep_ = h.minimize(pos_hi, pos_lo, smax_tol=0.0, max_evals=args.midquench_evals, poll_every=16)
        nz = float((pos_lo != 0).double().mean().item())
        nmid = max(3, min(args.steps, 10))
        mid_ms, _, _, _, _ = timed_steps(nmid, 3, False)
        mid = {"ms": mid_ms, "steps": nmid, "evals_before": rep_["evals"], "smax": rep_["smax"][0], "lo_nonzero_fraction": nz}
        pos_hi.copy_(start[0]); pos_lo.copy_(start[1])
        h.energy_grad(pos_hi, pos_lo, grad_hi, grad_lo)     # rho() / last_smax() below belong to the seeded start

    total_ms, e2e_ms, mid_ms = max_over_ranks([total_ms, e2e_s * 1e3, mid["ms"] if mid else 0.0], "cuda")
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return
    pairs = float(cfg.pairs)
    jobs = 1 if sharded else world          # sharded: ONE system's pair-terms over all ranks; replicas: one system per rank
    value = whole_job_value(pairs, args.steps, jobs, total_ms)
    e2e_value = whole_job_value(pairs, args.steps, jobs, e2e_ms)
    nbytes = 2 * cfg.d * n_local * 8
    pairs_rank = pairs * n_local / cfg.N    # pair-terms this rank's O(N M) kernels process per evaluation

    # ---- rooflines of the dominant kernel
    dfma_best, dfma_sus = shd.fp64_peak(0, 0.5)
    dadd_best, dadd_sus = shd.fp64_peak(1, 0.5)
    dmma_best, dmma_sus = shd.fp64_peak(2, 1.0)      # the instruction k_rho / k_grad issue (same FP64 pipe)
    pipe_sus = max(dfma_sus, dmma_sus)

    def fp64_roofline(kms_, total_ms_, steps_):
        """FP64 limb engine: ALU-bound on the FP64 pipe, peak measured live."""
        grad_ms, rho_ms = kms_["grad"] / steps_, kms_["rho"] / steps_
        dom = "k_grad" if grad_ms >= rho_ms else "k_rho"
        dom_ms = max(grad_ms, rho_ms)
        alg = ALG_DFMA_GRAD if dom == "k_grad" else ALG_DFMA_RHO
        achieved = pairs_rank * alg * 2.0 / (dom_ms * 1e-3) / 1e12     # TFLOP/s, DFMA = 2 FLOP
        peak = pipe_sus * 2.0 / 1e12
        launched = h.stat(12) if dom == "k_grad" else h.stat(0)
        return {
            "bound": "alu", "kernel": dom, "achieved": achieved, "peak": peak, "unit": "TFLOP/s",
            "frac": achieved / peak, "traffic": ncu_traffic(dom, cfg.name)[0] if world == 1 else None,
            "traffic_source": ncu_traffic(dom, cfg.name)[1] if world == 1 else None,
            "peak_source": "measured live: shd_fp64_peak, max of dependent-DFMA chains and DMMA.8x8x4 chains "
                           "(one FP64 pipe), sustained over 1 s (of measured)",
            "peak_burst": max(dfma_best, dmma_best) * 2.0 / 1e12, "dfma_peak_tfma": dfma_sus / 1e12,
            "dmma_peak_tfma": dmma_sus / 1e12, "dadd_peak_tinstr": dadd_sus / 1e12,
            "nominal_peak": 148 * 64 * 2 * 1.965e9 / 1e12,
            "kernel_ms": dom_ms, "algorithmic_dfma_per_pair": alg,
            "launched_dfma_per_pair": launched / pairs_rank,
            "issue_frac_launched": launched / (dom_ms * 1e-3) / pipe_sus,
            "whole_eval_frac": pairs_rank * (ALG_DFMA_RHO + ALG_DFMA_GRAD) / (total_ms_ / steps_ * 1e-3) / pipe_sus,
            "kernel_ms_all": {k: v / steps_ for k, v in kms_.items()},
        }

    fp64_engine = None
    if engine == 0:
        roofline = fp64_roofline(kms, total_ms, args.steps)
    else:
        # INT8 tensor-core engines: bound by the tensor pipe; peak = the issue rate of tcgen05.mma.kind::i8
        # measured live by shd_i8_probe (which also re-checks that the integer products are exact)
        i8_tops, i8_bad = shd.i8_probe()
        grad_ms, rho_ms = kms["grad"] / args.steps, kms["rho"] / args.steps
        grad8 = engine == 2
        dom = "k_grad8" if (grad8 and grad_ms >= rho_ms) else ("k_rho8" if rho_ms >= grad_ms or not grad8 else "k_grad8")
        if not grad8 and grad_ms >= rho_ms:
            roofline = fp64_roofline(kms, total_ms, args.steps)         # FP64 gradient pass still dominates
        else:
            dom_ms = grad_ms if dom == "k_grad8" else rho_ms
            mac = ALG_MAC_GRAD8 if dom == "k_grad8" else ALG_MAC_RHO8
            achieved = pairs_rank * mac * 2.0 / (dom_ms * 1e-3) / 1e12  # TOP/s, 2 per multiply-accumulate
            mp = json.load(open(ROOT / "MEASURED_PEAKS.json")) if (ROOT / "MEASURED_PEAKS.json").exists() else {}
            roofline = {
                "bound": "tensor", "kernel": dom, "achieved": achieved, "peak": i8_tops, "unit": "TFLOP/s",
                "frac": achieved / i8_tops, "traffic": ncu_traffic(dom, cfg.name)[0] if world == 1 else None,
                "traffic_source": ncu_traffic(dom, cfg.name)[1] if world == 1 else None,
                # the guide's rule for a contraction in another dtype: measured bf16 peak x nominal int8 : bf16 = 2
                "frac_of_measured_bf16_x2_burst": achieved / (2.0 * mp["bf16_tflops"]) if "bf16_tflops" in mp else None,
                "frac_of_measured_bf16_x2_sustained": achieved / (2.0 * mp["bf16_tflops_sustained"]) if "bf16_tflops_sustained" in mp else None,
                # SM clock at which one tcgen05.mma.kind::i8 of N = 256 takes its 128 cycles and gives this peak; the hot
                # kernels themselves run at ~1.66 GHz (clock64 against globaltimer inside k_rho8, profiles/r2a_summary.md)
                "peak_implied_sm_mhz": i8_tops * 1e12 / (148 * 8192 * 2.0) / 1e6,
                # the SM clock INSIDE the timed tensor kernels (clock64 against globaltimer, last evaluation) and the
                # roofline at that clock: 148 SMs x 8192 MAC per cycle x 2
                "sm_mhz_in_kernel": {"k_rho8": h.stat(28), "k_grad8": h.stat(29)},
                "frac_at_kernel_clock": achieved * 1e12 / (148 * 8192 * 2.0 * 1e6 * (h.stat(29) if dom == "k_grad8" else h.stat(28)))
                                        if (h.stat(29) if dom == "k_grad8" else h.stat(28)) > 0 else None,
                "dtype": "s8 x s8 -> s32 (exact digit-sliced contraction; counted in integer operations)",
                "peak_source": "measured live: shd_i8_probe, tcgen05.mma.kind::i8 M=128 N=256 K=32 issued back to "
                               "back on all SMs; MEASURED_PEAKS.json bf16 x 2 (nominal int8 : bf16) for comparison",
                "peak_from_measured_bf16_x2": 2.0 * float(mp["bf16_tflops"]) if "bf16_tflops" in mp else None,
                "i8_products_exact": i8_bad == 0,
                # why k_grad8's epilogue is integer arithmetic: FP64 beside a tcgen05.mma.kind::i8 stream (shd_mix_probe)
                "alu_beside_mma": shd.mix_probe(),
                "kernel_ms": dom_ms, "algorithmic_mac_per_pair": mac,
                "whole_eval_frac": pairs_rank * (ALG_MAC_RHO8 + ALG_MAC_GRAD8) * 2.0 / (total_ms / args.steps * 1e-3) / 1e12 / i8_tops,
                "kernel_ms_all": {k: v / args.steps for k, v in kms.items()},
            }
        # the FP64 limb engine (the reference engine of this library) on the same inputs, for comparison
        # (single GPU only: a sharded evaluation is a collective and the other ranks have left)
        n64 = max(3, min(args.steps, 5))
        if sharded or args.no_fp64_compare:
            fp64_engine = {"skipped": "sharded run" if sharded else "--no-fp64-compare"}
        else:
          h.set_engine(0)
          try:
            t64, k64, _, _, _ = timed_steps(n64, 3, False)
            fp64_engine = {"ms_per_step": t64 / n64, "value": pairs_rank * n64 / (t64 * 1e-3),
                           "roofline": fp64_roofline(k64, t64, n64)}
          except shd.ShdError as e:        # at the paper's N the FP64 engine's tables do not fit
            if e.code != shd.SHD_ENOMEM:
                raise
            fp64_engine = {"unavailable": "the FP64 engine's limb tables do not fit"}
          h.set_engine(engine)
          h.energy_grad(pos_hi, pos_lo, grad_hi, grad_lo)               # rho() below belongs to the timed engine

    # ---- oracle on the host cores, same run, bounded sample; doubles as a live parity sample
    from oracle import shd_oracle as O
    O.build()
    cores = O.num_threads()
    rho_dd = [x.cpu().numpy() for x in h.rho()]
    g_hi, g_lo = gh.numpy(), gl.numpy()
    s = oracle_sample(cfg, hi, lo, int(2.5e6 * cores), rho_dd, jrange=(j_begin, j_end))
    e_rho = O.cabsdiff_dd(s["re"], s["im"], *[x[s["ks"]] for x in rho_dd])
    sel = np.concatenate([a * n_local + (s["js"] - j_begin) for a in range(cfg.d)])
    e_g = O.absdiff_dd(s["grad"], g_hi[sel], g_lo[sel])
    tol_rho, tol_g = 1e-28 * cfg.N, 1e-27 * cfg.N * cfg.M * cfg.K
    smax, arg = h.last_smax()
    line = {
        "metric": METRIC if args.precision == 3 else f"{METRIC} [shd_set_precision {args.precision}: truncated evaluation, not the headline]",
        "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": total_ms / args.steps, "higher_is_better": True,
        "scaling": "strong" if sharded else "weak", "vs_baseline": None,
        "dtype": {0: "f64 (exact 22-bit limb products on the FP64 matrix instruction -> double-double)",
                  1: "rho pass: s8 digit slices of 102-bit fixed point -> s32 exact -> double-double; gradient pass: f64 limbs",
                  2: "s8 digit slices of 102-bit fixed point -> s32 exact (tensor memory) -> exact integer contraction -> "
                     "double-double in and out"}[engine],
        "data": "synthetic",
        "config": workload_config(cfg, world, replicas=not sharded),
        "clocks": clk,
        "e2e": {"value": e2e_value, "unit": UNIT, "ms_per_step": e2e_ms / args.steps,
                "h2d_bytes_per_step": nbytes, "d2h_bytes_per_step": nbytes + 64},
        "gpu_launches": launches,
        "chunks_per_evaluation": int(h.stat(19)), "table_bytes": h.stat(26),
        "value_midquench": (whole_job_value(pairs, mid["steps"], jobs, mid_ms) if mid else None),
        "midquench": ({k: v for k, v in mid.items() if k != "ms"} | {"ms_per_step": mid_ms / mid["steps"]}) if mid else None,
        "engine_selected_by": "library (shd_set_engine -1)" if args.engine == "auto" else "--engine",
        "engine": {0: "fp64 limbs on DMMA.8x8x4", 1: "rho pass on INT8 tensor cores (tcgen05), gradient pass on FP64 limbs",
                   2: "both O(N M) passes on INT8 tensor cores (tcgen05.mma.kind::i8, exact digit slices)"}[engine],
        "precision_limbs": args.precision,
        "roofline": roofline,
        "fp64_engine": fp64_engine,
        "cpu_baseline": {"value": s["value"], "unit": UNIT, "cores": s["cores"], "kind": "oracle",
                         "sample": s["sample"], "seconds": s["seconds"]},
        "parity_sample": {"rho_max_abs_err": float(e_rho.max()), "rho_tol": tol_rho,
                          "grad_max_abs_err": float(e_g.max()), "grad_tol": tol_g,
                          "ok": bool(e_rho.max() <= tol_rho and e_g.max() <= tol_g)},
        "phi": phi[0], "smax": smax[0],
    }
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=40)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", default="cfg4", choices=sorted(inputs.CONFIGS))
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--engine", default="auto", choices=["auto", "0", "1", "2"],
                    help="engine of the two O(N M) passes: 0 FP64 limbs (DMMA), 1 rho on INT8 tensor cores, 2 both")
    ap.add_argument("--no-fp64-compare", action="store_true", help="do not time the FP64 limb engine beside the INT8 one")
    ap.add_argument("--force-shard", action="store_true",
                    help="N = 1: run the sharded code path anyway (one shard, a library-owned NCCL communicator of one rank)")
    ap.add_argument("--replicas", action="store_true",
                    help="N > 1: independent replicas (weak scaling, no collective) instead of particle shards (strong scaling)")
    ap.add_argument("--midquench-evals", type=int, default=300,
                    help="also time the evaluation at the state this many L-BFGS evaluations into the quench (0 = skip)")
    ap.add_argument("--precision", type=int, default=3, choices=[1, 2, 3],
                    help="shd_set_precision: 3 = full double-double (the headline); 2 / 1 time the truncated evaluations of "
                         "the precision ladder (their line fails the parity sample by design and is not a bench value)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "cuda" else args.warmup
    cfg = inputs.CONFIGS[args.config]
    if args.impl == "reference":
        run_reference(args, cfg)
    else:
        run_gpu(args, cfg)


if __name__ == "__main__":
    main()
