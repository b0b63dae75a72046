"""Writes tests/golden/*.txt.  Calls ONLY oracle/ (plus the shared seeded input recipes).

Run:  python tests/golden/make_golden.py
The paper prints no worked example, so these are regression values of the pinned
oracle (direct mode, binary128, 34 significant digits), used (a) to notice any later change in
the oracle's arithmetic and (b) as ready-made expected values for the GPU parity tests of cfg1.
"""
import sys
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parents[2]
sys.path.insert(0, str(ROOT))
from oracle import shd_oracle as o  # noqa: E402
from paper_2304_09139_b200 import inputs  # noqa: E402


def dump(path, header, rows):
    with open(path, "w") as f:
        f.write(header)
        for key, val in rows:
            f.write(f"{key} {val}\n")


def main():
    here = Path(__file__).resolve().parent
    # example B: d=2, L=4, four particles, m*=2
    hi = np.array([0.5, 3.0, 2.25, 1.0, 1.25, 0.75, 2.0, 3.5])
    n = o.enumerate_Q(2, 2)
    r = o.energy_grad(2, 4, 4.0, hi, np.zeros(8), n)
    rows = []
    for k in range(len(n)):
        rows.append((f"rho_re[{n[k,0]},{n[k,1]}]", o.fmt(r["rho_re"], k, 34)))
        rows.append((f"rho_im[{n[k,0]},{n[k,1]}]", o.fmt(r["rho_im"], k, 34)))
    rows.append(("phi", o.fmt(r["phi"], 0, 34)))
    rows.append(("smax", o.fmt(r["smax"], 0, 34)))
    for i in range(8):
        rows.append((f"grad[{i}]", o.fmt(r["grad"], i, 34)))
    dump(here / "example_B.txt",
         "# d=2 L=4 r=((0.5,1.25),(3.0,0.75),(2.25,2.0),(1.0,3.5)) m*=2; oracle direct mode;\n"
         "# definitions: Eq.4 P:47 (conjugated), Eq.2 P:39, Eq.1 P:27, Eq.6 P:72; grad axis-major\n", rows)

    cfg = inputs.CONFIGS["cfg1"]
    hi, lo = inputs.uniform_positions(cfg, 0)
    n = o.enumerate_Q(cfg.d, cfg.m_star)
    r = o.energy_grad(cfg.d, cfg.N, cfg.L, hi, lo, n)
    rows = [("pos_hex[0]", float(hi[0]).hex()), ("pos_hex[128]", float(hi[128]).hex()),
            ("pos_hex[127]", float(hi[127]).hex()), ("pos_hex[255]", float(hi[255]).hex())]
    for k in range(len(n)):
        rows.append((f"rho_re[{n[k,0]},{n[k,1]}]", o.fmt(r["rho_re"], k, 34)))
        rows.append((f"rho_im[{n[k,0]},{n[k,1]}]", o.fmt(r["rho_im"], k, 34)))
    rows.append(("phi", o.fmt(r["phi"], 0, 34)))
    rows.append(("smax", o.fmt(r["smax"], 0, 34)))
    rows.append(("argmax", f"{n[r['argmax'],0]},{n[r['argmax'],1]}"))
    for i in range(2 * cfg.N):
        rows.append((f"grad[{i}]", o.fmt(r["grad"], i, 34)))
    dump(here / "cfg1_seed0.txt",
         "# BASELINE.json configs[0]: d=2 N=128 L=sqrt(128) m*=49 |Q|=74, default_rng(0).random((128,2))*L,\n"
         "# lo=0; oracle direct mode; grad axis-major grad[a*N+j]\n", rows)


if __name__ == "__main__":
    main()
