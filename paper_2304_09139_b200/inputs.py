"""Seeded synthetic inputs shared by the oracle tests and the CUDA path (and nothing else).

This module holds NONE of the method's arithmetic: no wavevector enumeration, no phases, no
sums.  It only states the workloads of BASELINE.json (``configs``) and produces positions.

The paper measures on no public data set (its 20 configurations were never uploaded);
these inputs stand in for its "random initial conditions defined by a Poisson point process"
 at fixed N (reading R9): i.i.d. uniform in [0,L)^d,
``numpy.random.default_rng(seed).random((N, d)) * L`` in FP64, lo word 0.

Layout everywhere: SoA axis-major, ``x[a*N + j]`` = coordinate a of particle j.
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np


@dataclass(frozen=True)
class Config:
    name: str
    d: int
    N: int
    L: float      # box edge, correctly rounded N**(1/d) (unit density, BASELINE.json)
    chi: float    # requested chi = M / (d (N-1)), Eq. 5
    m_star: int   # integer shell cutoff n.n <= m_star (complete shells, R6)
    M: int        # realised |Q| (checked against both enumerators in tests)

    @property
    def pairs(self) -> int:
        """pair-terms of one energy+gradient evaluation (M N terms per sum)."""
        return self.N * self.M

    @property
    def K(self) -> float:
        """cutoff passed to shd_create: K = (2 pi / L) sqrt(m_star + 1/2) (R8)."""
        return 2.0 * np.pi / self.L * np.sqrt(self.m_star + 0.5)


# BASELINE.json configs[0..4]; m_star = complete shell whose half-space count is nearest to
# round(chi d (N-1)).
CONFIGS = {
    "cfg1": Config("cfg1", 2, 128, float.fromhex("0x1.6a09e667f3bcdp+3"), 0.30, 49, 74),
    "cfg2": Config("cfg2", 2, 10_000, 100.0, 0.40, 5090, 8002),
    "cfg3": Config("cfg3", 3, 10_000, float.fromhex("0x1.58b5a51868c62p+4"), 0.40, 321, 12055),
    "cfg4": Config("cfg4", 2, 100_000, float.fromhex("0x1.3c3a4edfa9759p+8"), 0.45, 57290, 90000),
    "cfg5": Config("cfg5", 1, 200_000, 200000.0, 0.30, 60000 * 60000, 60000),
    # the paper's own system size (d = 2, N = 2 x 10^6) at its smallest chi; context, not a
    # BASELINE.json config: one evaluation is 8 x 10^11 pair-terms and needs ~150 GB of phasor tables
    "paper01": Config("paper01", 2, 2_000_000, float.fromhex("0x1.618dab0184066p+10"), 0.10, 254626, 399996),
    # the paper's other three chi: their phasor tables (up to 225 GB) are built chunk by chunk (shd_set_workspace)
    "paper02": Config("paper02", 2, 2_000_000, float.fromhex("0x1.618dab0184066p+10"), 0.20, 509290, 800002),
    "paper03": Config("paper03", 2, 2_000_000, float.fromhex("0x1.618dab0184066p+10"), 0.30, 763940, 1200000),
    "paper04": Config("paper04", 2, 2_000_000, float.fromhex("0x1.618dab0184066p+10"), 0.40, 1018580, 1599996),
}


def uniform_positions(cfg: Config, seed: int = 0):
    """(pos_hi, pos_lo), each of length d*N, axis-major; lo == 0 (BASELINE.json configs)."""
    r = np.random.default_rng(seed).random((cfg.N, cfg.d)) * cfg.L
    hi = np.ascontiguousarray(r.T).reshape(-1).copy()
    return hi, np.zeros_like(hi)


def uniform_positions_raw(d: int, N: int, L: float, seed: int = 0):
    r = np.random.default_rng(seed).random((N, d)) * L
    hi = np.ascontiguousarray(r.T).reshape(-1).copy()
    return hi, np.zeros_like(hi)


def jitter_lo(pos_hi, seed: int = 1):
    """Non-zero lo words (|lo| <= ulp(hi)/2) so that dd code paths with lo != 0 are exercised
    (timing and parity must also be taken with non-zero lo)."""
    rng = np.random.default_rng(seed)
    ulp = np.spacing(np.abs(pos_hi))
    return (rng.random(pos_hi.shape) - 0.5) * ulp * 0.999


def single_site(d: int, N: int, r0):
    """All particles at r0 (closed form: rho(k) = N exp(i k.r0), |rho|^2 = N^2)."""
    hi = np.repeat(np.asarray(r0, dtype=np.float64)[:d], N)
    return hi.copy(), np.zeros_like(hi)


def lattice(shape, L: float, offset=None):
    """Perfect lattice with shape[a] sites along axis a in a box of edge L."""
    d = len(shape)
    axes = [np.arange(s, dtype=np.float64) * (L / s) for s in shape]
    grids = np.meshgrid(*axes, indexing="ij")
    cols = [g.reshape(-1) for g in grids]
    if offset is not None:
        cols = [c + float(offset[a]) for a, c in enumerate(cols)]
    hi = np.concatenate(cols)
    assert hi.size == d * int(np.prod(shape))
    return hi, np.zeros_like(hi)


def quarter_grid(d: int, N: int, L: float, seed: int = 0):
    """Every coordinate a multiple of L/4 (L a power of two): every term of rho is in
    {1, i, -1, -i}.  Returns positions and the integer quarter indices g[j, a]."""
    g = np.random.default_rng(seed).integers(0, 4, size=(N, d))
    hi = np.ascontiguousarray((g * (L / 4.0)).T).reshape(-1).astype(np.float64)
    return hi, np.zeros_like(hi), g
