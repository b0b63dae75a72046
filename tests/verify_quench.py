"""Oracle verdict on a quenched configuration (R16: only the ORACLE's S_max on the device's final positions
counts).  Test infrastructure: reads the positions that `python -m paper_2304_09139_b200.quench --save PREFIX` wrote
(PREFIX_hi.npy / PREFIX_lo.npy) and evaluates S(k) with the binary128 oracle, in direct mode (the definition), on

  * every wavevector of the lowest shells (with the step potential the maximum sits at k_min), and
  * a strided sample of all of Q,

or on all of Q in factored mode with --full.  Prints one JSON line.

    python tests/verify_quench.py --config paper01 --prefix gpurun_out/paper01 [--lowest 300] [--strided 300] [--full]
"""
import argparse
import json
import sys
import time
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent.parent
sys.path.insert(0, str(ROOT))

from oracle import shd_oracle as O                 # noqa: E402
from paper_2304_09139_b200 import inputs           # noqa: E402


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", required=True, choices=sorted(inputs.CONFIGS))
    ap.add_argument("--prefix", required=True)
    ap.add_argument("--lowest", type=int, default=300, help="wavevectors of the lowest shells, all of them up to this count")
    ap.add_argument("--strided", type=int, default=300, help="evenly strided wavevectors over all of Q")
    ap.add_argument("--full", action="store_true", help="all of Q in factored mode instead of the samples")
    args = ap.parse_args()
    cfg = inputs.CONFIGS[args.config]
    hi, lo = np.load(args.prefix + "_hi.npy"), np.load(args.prefix + "_lo.npy")
    assert hi.size == cfg.d * cfg.N
    n = O.enumerate_Q(cfg.d, cfg.m_star)
    nn = (n.astype(np.int64) ** 2).sum(axis=1)
    t0 = time.perf_counter()
    if args.full:
        ks = np.arange(len(n))
        re, im = O.rho(cfg.d, cfg.N, cfg.L, hi, lo, n, mode="factored")
    else:
        low = np.argsort(nn, kind="stable")[:args.lowest]
        ks = np.unique(np.concatenate([low, np.linspace(0, len(n) - 1, args.strided).astype(np.int64)]))
        re, im = O.rho(cfg.d, cfg.N, cfg.L, hi, lo, n[ks], mode="direct")
    phi, smax, arg, s2 = O.energy(cfg.N, re, im)
    S = O.to_float(s2) / cfg.N
    line = {"config": cfg.name, "N": cfg.N, "M": cfg.M, "mode": "factored, all of Q" if args.full else "direct, sampled",
            "wavevectors_checked": int(len(ks)), "lowest_shells_up_to_nn": int(nn[ks].min()) if args.full else int(np.sort(nn)[min(args.lowest, len(nn)) - 1]),
            "oracle_smax": float(O.to_float(smax)[0]), "oracle_smax_at_n": n[ks[arg]].tolist(),
            "oracle_S_median": float(np.median(S)), "oracle_phi_over_checked": float(O.to_float(phi)[0]),
            "oracle_seconds": round(time.perf_counter() - t0, 1), "cores": O.num_threads()}
    print(json.dumps(line))


if __name__ == "__main__":
    main()
