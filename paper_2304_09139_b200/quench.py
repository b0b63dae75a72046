"""Quench one BASELINE.json configuration from its seeded random start to S_max < tol.

    python -m paper_2304_09139_b200.quench --config cfg4 [--seed 0] [--tol 1e-30] [--max-evals 20000]
                                           [--kind 0|1] [--weight one|n2] [--history 10] [--chunk 500]
                                           [--out file.json]

The whole iteration runs on the device (shd_minimize); this script only calls it in chunks of
``--chunk`` evaluations (shd_minimize is re-entrant) to log the S_max / Phi trajectory, and
prints one JSON line at the end.  ``--save prefix`` writes the final positions as
``prefix_hi.npy`` / ``prefix_lo.npy`` (axis-major, x[a*N + j]).
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
    ap.add_argument("--chunk", type=int, default=500)
    ap.add_argument("--poll-every", type=int, default=16)
    ap.add_argument("--weight", default="one", choices=["one", "n2"],
                    help="v(k): 'one' = the step potential of BASELINE.json's configs; 'n2' = 1/|n|^2 "
                         "(P:50: any positive v has the same ground states; S_max does not depend on v; "
                         "SURVEY.md 8(f) NEXT-1: it removes the k^2 ill-conditioning, decisive in d = 1)")
    ap.add_argument("--fire-dt0", type=float, default=0.0)
    ap.add_argument("--engine", type=int, default=0, choices=[0, 1, 2],
                    help="engine of the O(N M) passes (shd_set_engine): 0 FP64 limbs, 1 rho on the INT8 tensor cores, 2 both")
    ap.add_argument("--ladder", type=float, default=0.0,
                    help="precision ladder (P:77 'tunable precision'; SURVEY.md 8(f) NEXT-1): evaluate with two "
                         "limbs (shd_set_precision 2) until S_max < this value, e.g. 1e-18, then with three")
    ap.add_argument("--ladder1", type=float, default=0.0,
                    help="optional first rung below that: ONE limb (22-bit operands) until S_max < this value, "
                         "e.g. 1e-8")
    ap.add_argument("--out", default=None)
    ap.add_argument("--save", default=None)
    args = ap.parse_args(argv)

    import torch
    from . import shd

    cfg = inputs.CONFIGS[args.config]
    hi, lo = inputs.uniform_positions(cfg, args.seed)
    h = shd.Shd(cfg.d, cfg.N, cfg.L, m_star=cfg.m_star)
    if args.weight == "n2":
        n = h.k().astype(np.float64)
        h.close()
        h = shd.Shd(cfg.d, cfg.N, cfg.L, m_star=cfg.m_star, v=1.0 / (n * n).sum(axis=1))
    h.set_engine(args.engine)
    pos_hi, pos_lo = shd.from_host(hi, lo)
    phi0, _, _ = h.energy_grad(pos_hi, pos_lo, want_grad=False)
    smax0, _ = h.last_smax()
    trace = [{"evals": 0, "iters": 0, "phi": phi0[0], "smax": smax0[0], "seconds": 0.0}]
    evals = iters = 0
    status = shd.SHD_EMAXEVAL
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    # rungs: (limbs, stop below this S_max); the last rung is always 3 limbs down to --tol
    # (on the INT8 engines the rungs are digit counts: 4, 7 and 13 base-256 digits)
    rungs = [(1, args.ladder1)] if args.ladder1 > max(args.ladder, args.tol) else []
    if args.ladder > args.tol:
        rungs.append((2, args.ladder))
    rungs.append((3, args.tol))
    rung = 0
    h.set_precision(rungs[0][0])
    while evals < args.max_evals:
        fast = rung < len(rungs) - 1
        rep = h.minimize(pos_hi, pos_lo, kind=args.kind, history=args.history,
                         smax_tol=rungs[rung][1],
                         max_evals=min(args.chunk, args.max_evals - evals), poll_every=args.poll_every,
                         resume=evals > 0, fire_dt0=args.fire_dt0)
        evals += rep["evals"]
        iters += rep["iters"]
        status = rep["status"]
        trace.append({"evals": evals, "iters": iters, "phi": rep["phi"][0], "smax": rep["smax"][0],
                      "seconds": time.perf_counter() - t0})
        print(f"[quench {cfg.name}] evals={evals} iters={iters} Phi={rep['phi'][0]:.6e} "
              f"S_max={rep['smax'][0]:.6e} t={trace[-1]['seconds']:.1f}s", file=sys.stderr, flush=True)
        if fast and status in (shd.SHD_OK, shd.SHD_ESTALL):
            rung += 1                         # next rung: more limbs from here on
            h.set_precision(rungs[rung][0])
            trace[-1]["switched_to_limbs"] = rungs[rung][0]
            status = shd.SHD_EMAXEVAL
            continue
        if status != shd.SHD_EMAXEVAL:
            break
    seconds = time.perf_counter() - t0
    smax, arg = h.smax(pos_hi, pos_lo)
    n = h.k()
    line = {"config": cfg.name, "d": cfg.d, "N": cfg.N, "M": cfg.M, "chi_realised": cfg.M / (cfg.d * (cfg.N - 1)),
            "seed": args.seed, "kind": "lbfgs" if args.kind == 0 else "fire", "weight": args.weight, "engine": args.engine, "history": args.history,
            "tol": args.tol, "ladder": args.ladder, "ladder1": args.ladder1, "status": status, "evals": evals, "iters": iters, "seconds": seconds,
            "ms_per_eval": 1e3 * seconds / max(evals, 1), "phi_start": phi0[0], "smax_start": smax0[0],
            "phi_final": trace[-1]["phi"], "smax_final": smax[0], "argmax_n": n[arg].tolist(), "trace": trace}
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
