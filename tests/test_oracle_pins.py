"""Pins for oracle/shd_oracle.c against things OTHER than itself (CPU only).

Each test states the mathematics / paper passage that fixes the expected value:
closed forms, integer arithmetic, an independent real-space formula, brute force in mpmath at
50+ digits on tiny inputs, finite differences, symmetries.  A dropped term, wrong sign, wrong
index or transposed operand in the oracle fails at least one of them.
"""
import itertools
import math

import mpmath as mp
import numpy as np
import pytest

from paper_2304_09139_b200 import inputs

mp.mp.dps = 50


def q2mp(o, q):
    """binary128 array -> list of mpmath numbers (through 40-digit decimal strings)."""
    return [mp.mpf(o.fmt(q, i, 40)) for i in range(q.size)]


def mp_rho(d, L, pos, nvec):
    """The definition, straight in mpmath: rho = sum_j exp(+2 pi i n.r_j / L)."""
    N = len(pos) // d
    L = mp.mpf(L)
    tot = mp.mpc(0)
    for j in range(N):
        t = sum(int(nvec[a]) * mp.mpf(float(pos[a * N + j])) for a in range(d)) / L
        tot += mp.expjpi(2 * t)
    return tot


# --------------------------------------------------------------------------- a0: Q
@pytest.mark.parametrize("d,m_star", [(1, 49), (2, 2), (2, 49), (2, 5090), (3, 27), (3, 321), (4, 3), (4, 10)])
def test_enumeration_count_order_halfspace(oracle, d, m_star):
    """of the 2M non-zero lattice vectors with n.n <= m*, M are independent."""
    n = oracle.enumerate_Q(d, m_star)
    R = math.isqrt(m_star)
    full = sum(1 for t in itertools.product(range(-R, R + 1), repeat=d)
               if 0 < sum(c * c for c in t) <= m_star)
    assert full % 2 == 0 and len(n) == full // 2
    tup = [tuple(int(c) for c in row) for row in n]
    assert tup == sorted(tup), "canonical order is lexicographic, component 0 slowest"
    s = set(tup)
    assert len(s) == len(tup)
    for t in tup:
        assert tuple(-c for c in t) not in s
        first = next(c for c in t if c != 0)
        assert first > 0
        assert 0 < sum(c * c for c in t) <= m_star


def test_enumeration_matches_baseline_configs(oracle):
    """realised |Q| of the five BASELINE.json configs."""
    for cfg in inputs.CONFIGS.values():
        assert oracle.enumerate_Q(cfg.d, cfg.m_star).shape == (cfg.M, cfg.d)
        target = round(cfg.chi * cfg.d * (cfg.N - 1))
        assert abs(cfg.M - target) <= 0.005 * target + 2  # complete shells, nearest count


# --------------------------------------------------------------- closed-form examples
def test_example_A_closed_form(oracle):
    """d=1, L=3, r=(1/4, 1, 5/2), Q={1,2}: angles pi/6, 2pi/3, 5pi/3 (and doubles) give
    rho(1)=sqrt(3)/2 + i/2, rho(2) = -1/2 - i sqrt(3)/2, Phi=2, S_max=1/3,
    grad = (0, -4pi/3, +4pi/3)."""
    hi = np.array([0.25, 1.0, 2.5])
    n = oracle.enumerate_Q(1, 4)
    assert n.tolist() == [[1], [2]]
    r = oracle.energy_grad(1, 3, 3.0, hi, np.zeros(3), n)
    re, im = q2mp(oracle, r["rho_re"]), q2mp(oracle, r["rho_im"])
    s3 = mp.sqrt(3) / 2
    for got, want in [(re[0], s3), (im[0], mp.mpf(0.5)), (re[1], mp.mpf(-0.5)), (im[1], -s3)]:
        assert abs(got - want) < mp.mpf(10) ** -32
    assert abs(q2mp(oracle, r["phi"])[0] - 2) < mp.mpf(10) ** -32
    assert abs(q2mp(oracle, r["smax"])[0] - mp.mpf(1) / 3) < mp.mpf(10) ** -32
    g = q2mp(oracle, r["grad"])
    want = [0, -4 * mp.pi / 3, 4 * mp.pi / 3]
    for a, b in zip(g, want):
        assert abs(a - b) < mp.mpf(10) ** -31


@pytest.mark.parametrize("d", [1, 2, 3])
def test_single_site_pattern(oracle, d):
    """BASELINE.json: r_j = r0 for all j => rho(k) = N exp(i k.r0), |rho|^2 = N^2,
    Phi = N^2 |Q|, S_max = N, gradient = 0."""
    N, L = 37, 7.5
    r0 = [1.3125, 4.75, 6.0625][:d]
    hi, lo = inputs.single_site(d, N, r0)
    n = oracle.enumerate_Q(d, 11)
    r = oracle.energy_grad(d, N, L, hi, lo, n)
    s2 = q2mp(oracle, r["s2"])
    assert max(abs(s - N * N) for s in s2) < mp.mpf(10) ** -28
    assert abs(q2mp(oracle, r["phi"])[0] - N * N * len(n)) < mp.mpf(10) ** -26
    assert abs(q2mp(oracle, r["smax"])[0] - N) < mp.mpf(10) ** -30
    assert max(abs(g) for g in q2mp(oracle, r["grad"])) < mp.mpf(10) ** -28
    re, im = q2mp(oracle, r["rho_re"]), q2mp(oracle, r["rho_im"])
    for k in range(0, len(n), 3):
        t = sum(int(n[k, a]) * mp.mpf(r0[a]) for a in range(d)) / mp.mpf(L)
        want = N * mp.expjpi(2 * t)
        assert abs(mp.mpc(re[k], im[k]) - want) < mp.mpf(10) ** -29


def test_single_particle(oracle):
    """N = 1: |rho| = 1 for every k, Phi = |Q|, S_max = 1, gradient = 0."""
    n = oracle.enumerate_Q(2, 25)
    r = oracle.energy_grad(2, 1, 3.0, np.array([0.7, 2.9]), np.zeros(2), n)
    assert max(abs(s - 1) for s in q2mp(oracle, r["s2"])) < mp.mpf(10) ** -32
    assert abs(q2mp(oracle, r["phi"])[0] - len(n)) < mp.mpf(10) ** -30
    assert max(abs(g) for g in q2mp(oracle, r["grad"])) < mp.mpf(10) ** -30


@pytest.mark.parametrize("shape,L,m_star", [((16, 8), inputs.CONFIGS["cfg1"].L, 49),
                                            ((5, 4, 6), 5.0, 15), ((64,), 64.0, 63 * 63)])
def test_perfect_lattice_is_stealthy(oracle, shape, L, m_star):
    """BASELINE.json: a perfect lattice whose first reciprocal shell lies beyond K has rho = 0
    on all of Q (geometric sum over each axis).  cfg1: 16 x 8 sites, first hit |n| = 8 > 7."""
    d = len(shape)
    hi, lo = inputs.lattice(shape, L, offset=[0.1, 0.2, 0.3][:d])
    N = int(np.prod(shape))
    n = oracle.enumerate_Q(d, m_star)
    assert all(any(int(c) % s for c, s in zip(row, shape)) for row in n)
    r = oracle.energy_grad(d, N, L, hi, lo, n)
    # lattice sites j L / s are not exact doubles: |rho| <~ N 2 pi |n| 2^-53 relative to exact
    # sites -- so compare with the mpmath value at the SAME double inputs instead of with 0,
    # and check smallness separately.
    assert oracle.to_float(r["smax"])[0] < 1e-25
    for k in (0, len(n) // 2, len(n) - 1):
        want = mp_rho(d, L, hi, n[k])
        got = mp.mpc(q2mp(oracle, r["rho_re"][k:k + 1])[0], q2mp(oracle, r["rho_im"][k:k + 1])[0])
        assert abs(got - want) < mp.mpf(10) ** -30


@pytest.mark.parametrize("d,N,L", [(1, 64, 8.0), (2, 256, 16.0), (3, 100, 4.0)])
def test_quarter_grid_gaussian_integers(oracle, d, N, L):
    """all coordinates multiples of L/4 (L a power of two) => every term is a power
    of i and rho(n) = sum_j i^{(n.g_j) mod 4}, computable in pure integer arithmetic."""
    hi, lo, g = inputs.quarter_grid(d, N, L, seed=3)
    n = oracle.enumerate_Q(d, 30)
    r = oracle.energy_grad(d, N, L, hi, lo, n)
    e = (n.astype(np.int64) @ g.T.astype(np.int64)) % 4          # (M, N)
    want_re = (e == 0).sum(1) - (e == 2).sum(1)
    want_im = (e == 1).sum(1) - (e == 3).sum(1)
    re, im = q2mp(oracle, r["rho_re"]), q2mp(oracle, r["rho_im"])
    assert max(abs(a - int(b)) for a, b in zip(re, want_re)) < mp.mpf(10) ** -30
    assert max(abs(a - int(b)) for a, b in zip(im, want_im)) < mp.mpf(10) ** -30
    want_phi = int((want_re ** 2 + want_im ** 2).sum())
    assert abs(q2mp(oracle, r["phi"])[0] - want_phi) < mp.mpf(10) ** -27


# ------------------------------------------------------ independent formulas for Phi
def test_phi_dirichlet_kernel_d1(oracle):
    """d=1, v=1: Phi = N M + 2 sum_{l<m} sum_{n=1..M} cos(n x_lm), x = 2 pi (r_l - r_m)/L, and
    sum_{n=1..M} cos(n x) = sin(M x/2) cos((M+1) x/2) / sin(x/2): a real-space evaluation that
    shares nothing with the k-space sum."""
    N, L, M = 23, 23.0, 40
    hi, lo = inputs.uniform_positions_raw(1, N, L, seed=5)
    n = oracle.enumerate_Q(1, M * M)
    assert len(n) == M
    r = oracle.energy_grad(1, N, L, hi, lo, n, want_grad=False)
    tot = mp.mpf(N * M)
    for l in range(N):
        for m in range(l + 1, N):
            x = 2 * mp.pi * (mp.mpf(float(hi[l])) - mp.mpf(float(hi[m]))) / mp.mpf(L)
            tot += 2 * mp.sin(M * x / 2) * mp.cos((M + 1) * x / 2) / mp.sin(x / 2)
    assert abs(q2mp(oracle, r["phi"])[0] - tot) < mp.mpf(10) ** -28


@pytest.mark.parametrize("d,N,L,m_star", [(2, 8, 3.0, 10), (3, 6, 2.5, 6), (1, 7, 4.0, 25)])
def test_phi_brute_force_pair_sum(oracle, d, N, L, m_star):
    """BASELINE.json: brute-force Phi on N <= 8 from the double sum
    Phi = sum_k v_k sum_{l,m} cos(k.(r_l - r_m)) (weights v included)."""
    hi, lo = inputs.uniform_positions_raw(d, N, L, seed=11)
    n = oracle.enumerate_Q(d, m_star)
    v = 0.5 + np.random.default_rng(2).random(len(n))
    r = oracle.energy_grad(d, N, L, hi, lo, n, v=v, want_grad=False)
    tot = mp.mpf(0)
    for k in range(len(n)):
        for l in range(N):
            for m in range(N):
                arg = sum(int(n[k, a]) * (mp.mpf(float(hi[a * N + l])) - mp.mpf(float(hi[a * N + m])))
                          for a in range(d)) * 2 * mp.pi / mp.mpf(L)
                tot += mp.mpf(float(v[k])) * mp.cos(arg)
    assert abs(q2mp(oracle, r["phi"])[0] - tot) < mp.mpf(10) ** -29


def test_rho_mpmath_spot_checks_incl_large_n(oracle):
    """The definition at 50 digits on sampled k, including d=1 with n = 60000 and r ~ 2e5 where a
    naive theta = k.r would lose ~1e-28 (S8c: argument reduced exactly before sincos)."""
    cfg = inputs.CONFIGS["cfg1"]
    hi, lo = inputs.uniform_positions(cfg, 0)
    lo = inputs.jitter_lo(hi, 7)
    n = oracle.enumerate_Q(cfg.d, cfg.m_star)
    re, im = oracle.rho(cfg.d, cfg.N, cfg.L, hi, lo, n)
    for k in (0, 6, 33, 73):
        L = mp.mpf(cfg.L)
        tot = mp.mpc(0)
        for j in range(cfg.N):
            t = sum(int(n[k, a]) * (mp.mpf(float(hi[a * cfg.N + j])) + mp.mpf(float(lo[a * cfg.N + j])))
                    for a in range(cfg.d)) / L
            tot += mp.expjpi(2 * t)
        got = mp.mpc(q2mp(oracle, re[k:k + 1])[0], q2mp(oracle, im[k:k + 1])[0])
        assert abs(got - tot) < mp.mpf(10) ** -30
    # d = 1, huge n
    N, L = 50, 200000.0
    hi, lo = inputs.uniform_positions_raw(1, N, L, seed=4)
    nn = np.array([[60000], [59999], [31337]], dtype=np.int32)
    for mode in ("direct", "factored"):
        re, im = oracle.rho(1, N, L, hi, lo, nn, mode=mode)
        for k in range(3):
            want = mp_rho(1, L, hi, nn[k])
            got = mp.mpc(q2mp(oracle, re[k:k + 1])[0], q2mp(oracle, im[k:k + 1])[0])
            assert abs(got - want) < mp.mpf(10) ** -30


# ---------------------------------------------------------------------------- gradient
@pytest.mark.parametrize("d,N,L,m_star", [(1, 5, 3.0, 9), (2, 6, 4.0, 5), (3, 4, 2.0, 3)])
def test_gradient_vs_mpmath_derivative(oracle, d, N, L, m_star):
    """Gradient sign and scale (D:R2): mpmath.diff of the brute-force Phi at 50 digits."""
    hi, lo = inputs.uniform_positions_raw(d, N, L, seed=21)
    n = oracle.enumerate_Q(d, m_star)
    v = 0.5 + np.random.default_rng(8).random(len(n))
    r = oracle.energy_grad(d, N, L, hi, lo, n, v=v)
    g = q2mp(oracle, r["grad"])

    def phi_of(idx, x):
        pos = [mp.mpf(float(t)) for t in hi]
        pos[idx] = x
        tot = mp.mpf(0)
        for k in range(len(n)):
            z = mp.mpc(0)
            for j in range(N):
                t = sum(int(n[k, a]) * pos[a * N + j] for a in range(d)) / mp.mpf(L)
                z += mp.expjpi(2 * t)
            tot += mp.mpf(float(v[k])) * (z.real ** 2 + z.imag ** 2)
        return tot

    for idx in range(d * N):
        want = mp.diff(lambda x: phi_of(idx, x), mp.mpf(float(hi[idx])))
        assert abs(g[idx] - want) < mp.mpf(10) ** -24 * (1 + abs(want))


def test_gradient_finite_differences_cfg1(oracle):
    """BASELINE.json: central finite differences of the oracle's own Phi in binary128
    (h = 2^-36; O(h^2) error ~1e-19 relative) at the seeded cfg1 start."""
    cfg = inputs.CONFIGS["cfg1"]
    hi, lo = inputs.uniform_positions(cfg, 0)
    n = oracle.enumerate_Q(cfg.d, cfg.m_star)
    r = oracle.energy_grad(cfg.d, cfg.N, cfg.L, hi, lo, n)
    g = q2mp(oracle, r["grad"])
    h = 2.0 ** -36
    for idx in (0, 5, 127, 128, 200, 255):
        lp, lm = lo.copy(), lo.copy()
        lp[idx] += h
        lm[idx] -= h
        pp = oracle.eval_q(cfg.d, cfg.N, cfg.L, oracle.from_dd(hi, lp), n)[0]
        pm = oracle.eval_q(cfg.d, cfg.N, cfg.L, oracle.from_dd(hi, lm), n)[0]
        fd = (q2mp(oracle, pp)[0] - q2mp(oracle, pm)[0]) / (2 * mp.mpf(h))
        assert abs(fd - g[idx]) < mp.mpf(10) ** -15 * (1 + abs(g[idx]))


def test_symmetries_translation_periodicity_inversion(oracle):
    """BASELINE.json / SURVEY 8c: sum_j dPhi/dr_j = 0 per axis; a rigid shift leaves |rho|, Phi,
    S_max unchanged and rotates rho by exp(i k.c); moving one particle by L changes nothing;
    evaluating on -Q gives conj(rho) and the same Phi and gradient (P:52 inversion symmetry)."""
    d, N, L = 2, 40, 6.0
    hi, lo = inputs.uniform_positions_raw(d, N, L, seed=9)
    hi = np.round(hi * 2.0 ** 30) / 2.0 ** 30      # coarse grid: the shifts below are exact
    n = oracle.enumerate_Q(d, 20)
    v = 0.5 + np.random.default_rng(1).random(len(n))
    r = oracle.energy_grad(d, N, L, hi, lo, n, v=v)
    g = q2mp(oracle, r["grad"])
    for a in range(d):
        assert abs(sum(g[a * N:(a + 1) * N])) < mp.mpf(10) ** -28
    # rigid shift by c (exactly representable so inputs stay exact)
    c = [0.375, 1.625]
    hs = hi + np.repeat(c, N)
    assert np.all((hs - np.repeat(c, N)) == hi)
    r2 = oracle.energy_grad(d, N, L, hs, lo, n, v=v)
    assert abs(q2mp(oracle, r2["phi"])[0] - q2mp(oracle, r["phi"])[0]) < mp.mpf(10) ** -27
    for k in (0, 7, len(n) - 1):
        rot = mp.expjpi(2 * sum(int(n[k, a]) * mp.mpf(c[a]) for a in range(d)) / mp.mpf(L))
        z = mp.mpc(q2mp(oracle, r["rho_re"][k:k + 1])[0], q2mp(oracle, r["rho_im"][k:k + 1])[0])
        z2 = mp.mpc(q2mp(oracle, r2["rho_re"][k:k + 1])[0], q2mp(oracle, r2["rho_im"][k:k + 1])[0])
        assert abs(z2 - z * rot) < mp.mpf(10) ** -29
    g2 = q2mp(oracle, r2["grad"])
    assert max(abs(x - y) for x, y in zip(g, g2)) < mp.mpf(10) ** -27
    # one particle moved by +L along axis 1 (L = 6 exact)
    hp = hi.copy()
    hp[1 * N + 3] += L
    lp = lo.copy()
    lp[1 * N + 3] = (hi[1 * N + 3] - (hp[1 * N + 3] - L))   # restore bits lost by the rounding
    r3 = oracle.energy_grad(d, N, L, hp, lp, n, v=v)
    assert abs(q2mp(oracle, r3["phi"])[0] - q2mp(oracle, r["phi"])[0]) < mp.mpf(10) ** -27
    assert max(abs(x - y) for x, y in zip(g, q2mp(oracle, r3["grad"]))) < mp.mpf(10) ** -27
    # inversion
    r4 = oracle.energy_grad(d, N, L, hi, lo, -n, v=v)
    assert abs(q2mp(oracle, r4["phi"])[0] - q2mp(oracle, r["phi"])[0]) < mp.mpf(10) ** -28
    for a, b in zip(q2mp(oracle, r4["rho_im"]), q2mp(oracle, r["rho_im"])):
        assert abs(a + b) < mp.mpf(10) ** -30
    for a, b in zip(q2mp(oracle, r4["rho_re"]), q2mp(oracle, r["rho_re"])):
        assert abs(a - b) < mp.mpf(10) ** -30
    assert max(abs(x - y) for x, y in zip(g, q2mp(oracle, r4["grad"]))) < mp.mpf(10) ** -27


def test_uniform_random_is_ideal_gas(oracle):
    """a Poisson pattern is uncorrelated, <S(k)> = 1, so Phi / (N |Q|) ~ 1."""
    cfg = inputs.CONFIGS["cfg1"]
    vals = []
    for seed in range(6):
        hi, lo = inputs.uniform_positions(cfg, seed)
        n = oracle.enumerate_Q(cfg.d, cfg.m_star)
        r = oracle.energy_grad(cfg.d, cfg.N, cfg.L, hi, lo, n, want_grad=False)
        vals.append(oracle.to_float(r["phi"])[0] / (cfg.N * cfg.M))
    assert 0.8 < np.mean(vals) < 1.2


# ------------------------------------------------------------- factored mode == direct
@pytest.mark.parametrize("name", ["cfg1"])
def test_factored_equals_direct(oracle, name):
    cfg = inputs.CONFIGS[name]
    hi, lo = inputs.uniform_positions(cfg, 0)
    lo = inputs.jitter_lo(hi, 3)
    n = oracle.enumerate_Q(cfg.d, cfg.m_star)
    a = oracle.energy_grad(cfg.d, cfg.N, cfg.L, hi, lo, n, mode="direct")
    b = oracle.energy_grad(cfg.d, cfg.N, cfg.L, hi, lo, n, mode="factored")
    for key in ("rho_re", "rho_im", "grad"):
        x, y = q2mp(oracle, a[key]), q2mp(oracle, b[key])
        assert max(abs(p - q) for p, q in zip(x, y)) < mp.mpf(10) ** -28, key


@pytest.mark.parametrize("d,N,L,m_star", [(3, 50, 3.7, 30), (1, 40, 40.0, 700 * 700)])
def test_factored_equals_direct_small(oracle, d, N, L, m_star):
    hi, lo = inputs.uniform_positions_raw(d, N, L, seed=2)
    n = oracle.enumerate_Q(d, m_star)
    a = oracle.energy_grad(d, N, L, hi, lo, n, mode="direct")
    b = oracle.energy_grad(d, N, L, hi, lo, n, mode="factored")
    for key in ("rho_re", "rho_im", "grad"):
        diff = np.abs(oracle.to_float(a[key]) - oracle.to_float(b[key]))
        hi_a, lo_a = oracle.to_dd(a[key])
        assert oracle.absdiff_dd(b[key], hi_a, lo_a).max() < 1e-27 * len(n), key
        assert diff.max() < 1e-12


# --------------------------------------------------------------------------- minimizer
def test_lbfgs_oracle_reaches_ground_state_cfg1(oracle):
    """for chi < 1/2 every quench from a random start reaches a ground state.
    Outcome only (degenerate manifold): direct-mode S_max at the final positions < 1e-30."""
    cfg = inputs.CONFIGS["cfg1"]
    hi, lo = inputs.uniform_positions(cfg, 0)
    n = oracle.enumerate_Q(cfg.d, cfg.m_star)
    out = oracle.minimize_lbfgs(cfg.d, cfg.N, cfg.L, hi, lo, n, smax_tol=1e-30, max_evals=3000)
    assert out["status"] == 0, out
    r = oracle.energy_grad(cfg.d, cfg.N, cfg.L, out["pos_hi"], out["pos_lo"], n, want_grad=False)
    assert oracle.to_float(r["smax"])[0] < 1e-30
    assert oracle.to_float(r["phi"])[0] >= 0
    assert out["evals"] < 1.2 * out["iters"] + 20


# --------------------------------------------------------------------------- FIRE (ref.[37])
def test_fire_oracle_first_steps_closed_form(oracle):
    """From rest the first FIRE evaluation has P = F.v = 0, so the step is: v <- 0, dt <- dt0 / 2,
    v <- -dt g, x <- x - dt^2 g (closed form, using the gradient pinned by finite differences above).
    One further evaluation has P > 0 and 'since' = 0 (no dt growth):
    v <- (1-a) v + a |v| F/|F| with v parallel to F is v itself, then v <- v + dt F2, x <- x + dt v."""
    d, N, L, m_star = 2, 12, 4.0, 5
    hi, lo = inputs.uniform_positions_raw(d, N, L, 5)
    n = oracle.enumerate_Q(d, m_star)
    dt0 = 1e-3
    g1 = oracle.to_float(oracle.energy_grad(d, N, L, hi, lo, n)["grad"])
    out = oracle.minimize_fire(d, N, L, hi, lo, n, dt0=dt0, smax_tol=0.0, max_evals=2)
    assert out["status"] == 1 and out["steps"] == 1 and out["evals"] == 2
    dt = dt0 / 2
    x1 = hi - dt * dt * g1
    assert np.abs(out["pos_hi"] - x1).max() < 1e-15
    # the second move: v1 = -dt g1 is parallel to F1 but F2 != F1, so the mixing changes v slightly:
    # v' = (1-a) v1 + a |v1| F2/|F2|, then v'' = v' - dt g2, x2 = x1 + dt v''
    out2 = oracle.minimize_fire(d, N, L, hi, lo, n, dt0=dt0, smax_tol=0.0, max_evals=3)
    g2 = oracle.to_float(oracle.energy_grad(d, N, L, out["pos_hi"], out["pos_lo"], n)["grad"])
    v1 = -dt * g1
    assert np.dot(-g2, v1) > 0
    vm = 0.9 * v1 - 0.1 * np.linalg.norm(v1) * g2 / np.linalg.norm(g2)
    x2 = out["pos_hi"] + dt * (vm - dt * g2)
    assert np.abs(out2["pos_hi"] - x2).max() < 1e-14


@pytest.mark.parametrize("d,N,L,m_star", [(2, 32, 32 ** 0.5, 12), (1, 40, 40.0, 36), (3, 27, 3.0, 3)])
def test_fire_oracle_reaches_ground_state(oracle, d, N, L, m_star):
    """every quench below the chi threshold reaches a ground state -- with the paper's own
    minimizer.  Outcome only: direct-mode S_max at the final positions < 1e-30, Phi -> 0."""
    hi, lo = inputs.uniform_positions_raw(d, N, L, 1)
    n = oracle.enumerate_Q(d, m_star)
    chi = len(n) / (d * (N - 1))
    assert chi < (1 / 3 if d == 1 else 1 / 2)
    out = oracle.minimize_fire(d, N, L, hi, lo, n, mode="factored", smax_tol=1e-30, max_evals=40000)
    assert out["status"] == 0, out
    r = oracle.energy_grad(d, N, L, out["pos_hi"], out["pos_lo"], n, want_grad=False)
    assert oracle.to_float(r["smax"])[0] < 1e-30
    r0 = oracle.energy_grad(d, N, L, hi, lo, n, want_grad=False)
    assert oracle.to_float(r["phi"])[0] < 1e-25 * oracle.to_float(r0["phi"])[0]


# --------------------------------------------------------------------------- S(k), tau (Eq. 3, Eq. 7)
def test_structure_factor_closed_forms(oracle):
    """S(k) = |rho|^2 / N and sum_k (S-1)^2: single site => S = N for every k, sum = M (N-1)^2;
    perfect lattice with its first reciprocal shell beyond the cutoff => S = 0 on Q, sum = M
    (a stealthy state contributes exactly 2M K^d V / N^2 to tau from inside the exclusion region);
    ideal gas (tau = 0 in the thermodynamic limit) => S(k) is exponentially distributed with
    mean 1 at finite N, so the sample mean of (S-1)^2 is 1 within statistics."""
    d, N, L, m_star = 2, 128, 128 ** 0.5, 49
    n = oracle.enumerate_Q(d, m_star)
    M = len(n)
    hi, lo = inputs.single_site(d, N, [1.234, 5.678])
    re, im = oracle.rho(d, N, L, hi, lo, n)
    S, dev2 = oracle.structure_factor(N, re, im)
    assert np.abs(oracle.to_float(S) - N).max() < 1e-10
    assert abs(oracle.to_float(dev2)[0] - M * (N - 1) ** 2) < 1e-6
    hi, lo = inputs.lattice((16, 8), L)
    re, im = oracle.rho(d, N, L, hi, lo, n)
    S, dev2 = oracle.structure_factor(N, re, im)
    assert np.abs(oracle.to_float(S)).max() < 1e-25      # lattice sites are rounded to double (lo = 0)
    assert abs(oracle.to_float(dev2)[0] - M) < 1e-20
    K = 2 * np.pi / L * np.sqrt(m_star + 0.5)
    assert oracle.tau(d, N, L, K, dev2) == pytest.approx(2 * M * K ** d * L ** d / N ** 2, rel=1e-14)
    vals = []
    for seed in range(8):
        hi, lo = inputs.uniform_positions_raw(d, N, L, 100 + seed)
        re, im = oracle.rho(d, N, L, hi, lo, n, mode="factored")
        S, dev2 = oracle.structure_factor(N, re, im)
        vals.append(oracle.to_float(dev2)[0] / M)
    assert 0.8 < np.mean(vals) < 1.2, vals


def test_four_dimensions_direct_mode(oracle):
    """d = 4 ("dimensions d = 1-4"): the direct-mode oracle is dimension-generic; pin it with the
    single-site closed form, translation invariance of the gradient, a central finite difference of Phi
    and the brute-force pair sum Phi = sum_k sum_{l,m} cos(k.(r_l - r_m))."""
    d, N, L, m_star = 4, 6, 2.5, 3
    n = oracle.enumerate_Q(d, m_star)
    assert len(n) == 32                                   # (65 - 1) / 2 lattice points of the 4-ball
    hi, lo = inputs.single_site(d, N, [0.3, 1.1, 2.2, 0.7])
    r = oracle.energy_grad(d, N, L, hi, lo, n)
    assert abs(oracle.to_float(r["phi"])[0] - N * N * len(n)) < 1e-9
    assert np.abs(oracle.to_float(r["grad"])).max() < 1e-25
    hi, lo = inputs.uniform_positions_raw(d, N, L, 9)
    r = oracle.energy_grad(d, N, L, hi, lo, n)
    g = oracle.to_float(r["grad"]).reshape(d, N)
    assert np.abs(g.sum(axis=1)).max() < 1e-12
    x = hi.reshape(d, N)
    brute = 0.0
    for k in n:
        ph = 2 * np.pi * (k[:, None] * x).sum(axis=0) / L
        brute += np.cos(ph[:, None] - ph[None, :]).sum()
    assert abs(oracle.to_float(r["phi"])[0] - brute) < 1e-9 * brute
    h = 1e-6
    for (a, j) in ((0, 0), (3, 4), (2, 5)):
        xp, xm = hi.copy(), hi.copy()
        xp[a * N + j] += h; xm[a * N + j] -= h
        fp = oracle.to_float(oracle.energy_grad(d, N, L, xp, lo, n, want_grad=False)["phi"])[0]
        fm = oracle.to_float(oracle.energy_grad(d, N, L, xm, lo, n, want_grad=False)["phi"])[0]
        assert abs((fp - fm) / (2 * h) - g[a, j]) < 1e-5 * (1 + abs(g[a, j]))


def test_structure_factor_shells_pins(oracle):
    """Radial average of S(k) (Fig. 2a, Fig. S1a), bins = ranges of the integer n.n.
    Counts: a shell n.n = m of the square lattice holds r2(m) vectors, half of them in the half space (brute-force
    count over the square here); the bins partition Q.  Values: single site => every mean is N exactly; perfect
    lattice with its first reciprocal shell beyond the cutoff => every mean is 0; a bin that holds one wavevector
    returns that wavevector's S(k); the count-weighted mean of the means is the plain mean of S over Q."""
    d, N, L, m_star = 2, 128, inputs.CONFIGS["cfg1"].L, 49
    n = oracle.enumerate_Q(d, m_star)
    nn = (n.astype(np.int64) ** 2).sum(axis=1)
    shells = np.unique(nn)
    edges = np.concatenate([shells, [m_star + 1]])
    hi, lo = inputs.uniform_positions(inputs.CONFIGS["cfg1"], 0)
    re, im = oracle.rho(d, N, L, hi, lo, n)
    count, Sm = oracle.structure_factor_shells(d, N, n, re, im, edges)
    # brute-force r2(m) / 2
    R = 8
    g = np.arange(-R, R + 1)
    a, b = np.meshgrid(g, g, indexing="ij")
    allnn = (a * a + b * b).reshape(-1)
    for m, c in zip(shells, count):
        assert 2 * c == int((allnn == m).sum())
    assert count.sum() == len(n)
    S, _ = oracle.structure_factor(N, re, im)
    Sf, Smf = oracle.to_float(S), oracle.to_float(Sm)
    for m, c, v in zip(shells, count, Smf):
        assert abs(v - Sf[nn == m].mean()) <= 1e-14 * max(1.0, v)
    assert abs((count * Smf).sum() / count.sum() - Sf.mean()) <= 1e-13
    # coarser bins: [1, 10), [10, 30), [30, 50) and an empty one [50, 60)
    c2, S2 = oracle.structure_factor_shells(d, N, n, re, im, [1, 10, 30, 50, 60])
    assert c2.tolist() == [int(((nn >= lo_) & (nn < hi_)).sum()) for lo_, hi_ in ((1, 10), (10, 30), (30, 50), (50, 60))]
    assert c2[3] == 0 and oracle.to_float(S2)[3] == 0.0
    assert abs(oracle.to_float(S2)[1] - Sf[(nn >= 10) & (nn < 30)].mean()) <= 1e-14
    # single site: S(k) = N for every k
    shi, slo = inputs.single_site(d, N, (1.2345, 7.0))
    re, im = oracle.rho(d, N, L, shi, slo, n)
    _, Sm = oracle.structure_factor_shells(d, N, n, re, im, edges)
    assert oracle.absdiff_dd(Sm, np.full(len(shells), float(N)), np.zeros(len(shells))).max() <= 1e-28 * N
    # perfect 16 x 8 lattice: rho = 0 on all of Q
    lhi, llo = inputs.lattice((16, 8), L)
    re, im = oracle.rho(d, N, L, lhi, llo, n)
    _, Sm = oracle.structure_factor_shells(d, N, n, re, im, edges)
    assert np.abs(oracle.to_float(Sm)).max() <= 1e-26      # (the lattice sites k L / 16 are rounded to doubles: |rho| ~ 1e-13)
