"""Quench one BASELINE.json configuration from its seeded random start to S_max < tol.

    python -m paper_2304_09139_b200.quench --config cfg4 [--seed 0] [--tol 1e-30] [--max-evals 20000]
                                           [--kind 0|1] [--weight one|n2] [--history 10] [--ladder1 1e-6 --ladder 1e-24]
                                           [--out file.json]

ONE shd_minimize call: the whole iteration runs on the device, the precision ladder (--ladder1 / --ladder) switches
rungs inside the library, the device writes a trace record per evaluation (shd_get_trace), and the poll callback of the
call logs progress and writes periodic checkpoints (shd_minimize_snapshot).  One JSON line at the end.  ``--save prefix``
writes the final positions as ``prefix_hi.npy`` / ``prefix_lo.npy`` (axis-major, x[a*N + j]); with
``--checkpoint-every K`` also every K polls while running.
"""
from __future__ import annotations

import argparse
import json
import sys
import time

import numpy as np

from . import inputs


def main(argv=None):
    ap = argparse.ArgumentParser(description=__doc__.split("\n")[0])
    ap.add_argument("--config", default="cfg4", choices=sorted(inputs.CONFIGS))
    ap.add_argument("--seed", type=int, default=0)
    ap.add_argument("--tol", type=float, default=1e-30)
    ap.add_argument("--max-evals", type=int, default=20000)
    ap.add_argument("--kind", type=int, default=0, help="0 = L-BFGS, 1 = FIRE")
    ap.add_argument("--history", type=int, default=10)
    ap.add_argument("--poll-every", type=int, default=16)
    ap.add_argument("--weight", default="one", choices=["one", "n2"],
                    help="v(k): 'one' = the step potential of BASELINE.json's configs; 'n2' = 1/|n|^2 "
                         "(P:50: any positive v has the same ground states; S_max does not depend on v; "
                         "SURVEY.md 8(f) NEXT-1: it removes the k^2 ill-conditioning, decisive in d = 1)")
    ap.add_argument("--fire-dt0", type=float, default=0.0)
    ap.add_argument("--engine", type=int, default=-1, choices=[-1, 0, 1, 2],
                    help="engine of the O(N M) passes (shd_set_engine): -1 the library's choice, 0 FP64 limbs, 1 rho on the "
                         "INT8 tensor cores, 2 both")
    ap.add_argument("--workspace-gb", type=float, default=0.0, help="cap on the phasor tables (shd_set_workspace); 0 = what fits")
    ap.add_argument("--log-every", type=int, default=32, help="progress line every this many polls (0 = none)")
    ap.add_argument("--checkpoint-every", type=int, default=0,
                    help="with --save: write the minimizer's current best point every this many polls")
    ap.add_argument("--ladder", type=float, default=0.0,
                    help="precision ladder (P:77 'tunable precision'; SURVEY.md 8(f) NEXT-1): evaluate with two "
                         "limbs (shd_set_precision 2) until S_max < this value, e.g. 1e-18, then with three")
    ap.add_argument("--ladder1", type=float, default=0.0,
                    help="optional first rung below that: ONE limb (22-bit operands) until S_max < this value, "
                         "e.g. 1e-8")
    ap.add_argument("--start", default=None,
                    help="continue from positions saved by --save (PREFIX_hi.npy, PREFIX_lo.npy) instead of the seeded start")
    ap.add_argument("--out", default=None)
    ap.add_argument("--save", default=None)
    args = ap.parse_args(argv)

    import torch
    from . import shd

    cfg = inputs.CONFIGS[args.config]
    hi, lo = inputs.uniform_positions(cfg, args.seed)
    if args.start:
        hi, lo = np.load(args.start + "_hi.npy").reshape(-1), np.load(args.start + "_lo.npy").reshape(-1)
        if hi.size != cfg.d * cfg.N or lo.size != hi.size:
            raise SystemExit(f"--start: {args.start}_hi/_lo.npy do not hold d*N = {cfg.d * cfg.N} doubles each")
    v = None
    h = shd.Shd(cfg.d, cfg.N, cfg.L, m_star=cfg.m_star)
    if args.weight == "n2":
        n = h.k().astype(np.float64)
        h.close()
        v = 1.0 / (n * n).sum(axis=1)
        h = shd.Shd(cfg.d, cfg.N, cfg.L, m_star=cfg.m_star, v=v)
    if args.engine >= 0:
        h.set_engine(args.engine)          # default: the library's own choice
    if args.workspace_gb > 0:
        h.set_workspace(int(args.workspace_gb * 2 ** 30))
    pos_hi, pos_lo = shd.from_host(hi, lo)
    phi0, _, _ = h.energy_grad(pos_hi, pos_lo, want_grad=False)
    smax0, _ = h.last_smax()
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    polls = [0]

    def on_poll(rep):
        """host side of a poll: a progress line every --log-every polls, a checkpoint every --checkpoint-every polls"""
        polls[0] += 1
        if args.log_every > 0 and polls[0] % args.log_every == 0:
            print(f"[quench {cfg.name}] evals={rep['evals']} iters={rep['iters']} Phi={rep['phi'][0]:.6e} "
                  f"S_max={rep['smax'][0]:.6e} t={time.perf_counter() - t0:.1f}s", file=sys.stderr, flush=True)
        if args.save and args.checkpoint_every > 0 and polls[0] % args.checkpoint_every == 0:
            sh, sl = h.minimize_snapshot()
            np.save(args.save + "_hi.npy", sh.cpu().numpy())
            np.save(args.save + "_lo.npy", sl.cpu().numpy())
        return False

    rep = h.minimize(pos_hi, pos_lo, kind=args.kind, history=args.history, smax_tol=args.tol,
                     max_evals=args.max_evals, poll_every=args.poll_every, fire_dt0=args.fire_dt0,
                     ladder=(args.ladder1, args.ladder), on_poll=on_poll)
    torch.cuda.synchronize()
    seconds = time.perf_counter() - t0
    status, evals, iters = rep["status"], rep["evals"], rep["iters"]
    tr = h.trace()
    # the trace the device wrote (one record per evaluation), thinned to <= 400 points for the JSON line
    keep = np.unique(np.concatenate([np.linspace(0, len(tr) - 1, min(len(tr), 400)).astype(np.int64),
                                     np.nonzero(np.diff(tr["limbs"]))[0] + 1])) if len(tr) else []
    trace = [{"evals": int(tr["evals"][i]), "iters": int(tr["iters"][i]), "phi": float(tr["phi"][i]),
              "smax": float(tr["smax"][i]), "gnorm": float(tr["gnorm"][i]), "step": float(tr["step"][i]),
              "limbs": int(tr["limbs"][i])} for i in keep]
    by_limbs = {int(l): int((tr["limbs"] == l).sum()) for l in np.unique(tr["limbs"])} if len(tr) else {}
    smax, arg = h.smax(pos_hi, pos_lo)
    n = h.k()
    line = {"config": cfg.name, "d": cfg.d, "N": cfg.N, "M": cfg.M, "chi_realised": cfg.M / (cfg.d * (cfg.N - 1)),
            "seed": args.seed, "start": args.start, "kind": "lbfgs" if args.kind == 0 else "fire", "weight": args.weight, "engine": h.engine,
            "chunks": int(h.stat(19)), "history": args.history,
            "tol": args.tol, "ladder": args.ladder, "ladder1": args.ladder1, "status": status, "evals": evals, "iters": iters,
            "evals_by_limbs": by_limbs, "seconds": seconds,
            "ms_per_eval": 1e3 * seconds / max(evals, 1), "phi_start": phi0[0], "smax_start": smax0[0],
            "phi_final": rep["phi"][0], "smax_final": smax[0], "argmax_n": n[arg].tolist(), "trace": trace}
    if args.save:
        np.save(args.save + "_hi.npy", pos_hi.cpu().numpy())
        np.save(args.save + "_lo.npy", pos_lo.cpu().numpy())
    s = json.dumps(line)
    if args.out:
        with open(args.out, "w") as f:
            f.write(s + "\n")
    print(s, flush=True)
    h.close()
    return 0 if status == shd.SHD_OK else 1


if __name__ == "__main__":
    sys.exit(main())
