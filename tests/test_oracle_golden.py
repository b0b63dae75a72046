"""Regression of the oracle against tests/golden/*.txt (written by tests/golden/make_golden.py,
which calls only oracle/) and of the seeded input recipe (SURVEY.md 8c generator check)."""
from pathlib import Path

import numpy as np

from paper_2304_09139_b200 import inputs

GOLD = Path(__file__).resolve().parent / "golden"


def read_golden(name):
    out = {}
    for line in (GOLD / name).read_text().splitlines():
        if line.startswith("#") or not line.strip():
            continue
        k, v = line.split(" ", 1)
        out[k] = v.strip()
    return out


def test_seeded_generator_bits():
    """numpy PCG64 stream: the exact FP64 bit patterns of cfg1's first/last particle."""
    g = read_golden("cfg1_seed0.txt")
    hi, lo = inputs.uniform_positions(inputs.CONFIGS["cfg1"], 0)
    assert float(hi[0]).hex() == g["pos_hex[0]"] == "0x1.cd35a38b71816p+2"
    assert float(hi[128]).hex() == g["pos_hex[128]"] == "0x1.86b16184b3c09p+1"
    assert float(hi[127]).hex() == g["pos_hex[127]"]
    assert float(hi[255]).hex() == g["pos_hex[255]"]
    assert not lo.any()
    for cfg in inputs.CONFIGS.values():
        assert abs(cfg.L ** cfg.d - cfg.N) < 4e-16 * cfg.N * cfg.d  # unit density


def test_oracle_matches_golden_cfg1(oracle):
    g = read_golden("cfg1_seed0.txt")
    cfg = inputs.CONFIGS["cfg1"]
    hi, lo = inputs.uniform_positions(cfg, 0)
    n = oracle.enumerate_Q(cfg.d, cfg.m_star)
    r = oracle.energy_grad(cfg.d, cfg.N, cfg.L, hi, lo, n)
    want_re = oracle.parse([g[f"rho_re[{a},{b}]"] for a, b in n])
    want_im = oracle.parse([g[f"rho_im[{a},{b}]"] for a, b in n])
    h, l = oracle.to_dd(r["rho_re"])
    assert oracle.absdiff_dd(want_re, h, l).max() < 1e-31
    h, l = oracle.to_dd(r["rho_im"])
    assert oracle.absdiff_dd(want_im, h, l).max() < 1e-31
    h, l = oracle.to_dd(r["phi"])
    assert oracle.absdiff_dd(oracle.parse(g["phi"]), h, l).max() < 1e-28
    assert f"{n[r['argmax'],0]},{n[r['argmax'],1]}" == g["argmax"] == "2,3"
    want_g = oracle.parse([g[f"grad[{i}]"] for i in range(2 * cfg.N)])
    h, l = oracle.to_dd(r["grad"])
    assert oracle.absdiff_dd(want_g, h, l).max() < 1e-29


def test_oracle_matches_golden_example_B(oracle):
    g = read_golden("example_B.txt")
    hi = np.array([0.5, 3.0, 2.25, 1.0, 1.25, 0.75, 2.0, 3.5])
    n = oracle.enumerate_Q(2, 2)
    r = oracle.energy_grad(2, 4, 4.0, hi, np.zeros(8), n)
    want = oracle.parse([g[f"grad[{i}]"] for i in range(8)])
    h, l = oracle.to_dd(r["grad"])
    assert oracle.absdiff_dd(want, h, l).max() < 1e-30
    h, l = oracle.to_dd(r["phi"])
    assert oracle.absdiff_dd(oracle.parse(g["phi"]), h, l).max() < 1e-30
