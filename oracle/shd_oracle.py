"""ctypes harness around oracle/shd_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this module.  It shares nothing with paper_2304_09139_b200 (the CUDA path) and neither
imports the other.  binary128 arrays are carried as numpy ``V16`` buffers; they are turned
into double-double pairs, decimal strings or |difference| doubles by C helpers, never by
Python float arithmetic.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "shd_oracle.c"
_LIB = _HERE / "libshd_oracle.so"
Q = np.dtype("V16")  # one binary128


def build(force: bool = False) -> Path:
    """Compile the oracle with gcc (C, libquadmath, OpenMP)."""
    if force or not _LIB.exists() or _LIB.stat().st_mtime < _SRC.stat().st_mtime:
        tmp = _LIB.with_suffix(f".so.tmp{os.getpid()}")
        cmd = ["gcc", "-O2", "-std=gnu11", "-fopenmp", "-fPIC", "-shared", "-Wall", "-Wextra",
               "-o", str(tmp), str(_SRC), "-lquadmath", "-lm"]
        subprocess.run(cmd, check=True)
        os.replace(tmp, _LIB)
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(str(_LIB))
        vp, dp, ip, lp = C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_int), C.POINTER(C.c_long)
        L.shdo_num_threads.restype = C.c_int
        L.shdo_set_threads.argtypes = [C.c_int]
        L.shdo_from_dd.argtypes = [C.c_long, dp, dp, vp]
        L.shdo_to_dd.argtypes = [C.c_long, vp, dp, dp]
        L.shdo_absdiff_dd.argtypes = [C.c_long, vp, dp, dp, dp]
        L.shdo_cabsdiff_dd.argtypes = [C.c_long, vp, vp, dp, dp, dp, dp, dp]
        L.shdo_format.argtypes = [vp, C.c_int, C.c_char_p, C.c_int]
        L.shdo_parse.argtypes = [C.c_char_p, vp]
        L.shdo_enumerate.argtypes = [C.c_int, C.c_long, ip]
        L.shdo_enumerate.restype = C.c_long
        L.shdo_rho_direct.argtypes = [C.c_int, C.c_long, C.c_double, dp, dp, C.c_long, ip, vp, vp]
        L.shdo_rho_factored.argtypes = L.shdo_rho_direct.argtypes
        L.shdo_energy.argtypes = [C.c_long, C.c_long, vp, vp, dp, vp, vp, lp, vp]
        L.shdo_grad_direct.argtypes = [C.c_int, C.c_long, C.c_double, dp, dp, C.c_long, ip, dp,
                                       vp, vp, C.c_long, lp, vp]
        L.shdo_grad_factored.argtypes = L.shdo_grad_direct.argtypes
        L.shdo_eval_q.argtypes = [C.c_int, C.c_long, C.c_double, vp, C.c_long, ip, dp, C.c_int,
                                  vp, vp, lp, vp]
        L.shdo_minimize_lbfgs.argtypes = [C.c_int, C.c_long, C.c_double, vp, C.c_long, ip, dp,
                                          C.c_int, C.c_int, C.c_double, C.c_long, lp, vp, vp]
        L.shdo_minimize_lbfgs.restype = C.c_int
        L.shdo_minimize_fire.argtypes = [C.c_int, C.c_long, C.c_double, vp, C.c_long, ip, dp,
                                         C.c_int, C.c_double, C.c_double, C.c_long, lp, vp, vp]
        L.shdo_minimize_fire.restype = C.c_int
        L.shdo_structure_factor.argtypes = [C.c_long, C.c_long, vp, vp, vp, vp]
        L.shdo_structure_factor_shells.argtypes = [C.c_int, C.c_long, C.c_long, ip, vp, vp, C.c_long, lp, lp, vp]
        _lib = L
    return _lib


# ----------------------------------------------------------------- marshalling helpers
def _d(a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a, a.ctypes.data_as(C.POINTER(C.c_double))


def _i(a):
    a = np.ascontiguousarray(a, dtype=np.int32)
    return a, a.ctypes.data_as(C.POINTER(C.c_int))


def _q(a):
    assert a.dtype == Q and a.flags.c_contiguous
    return C.c_void_p(a.ctypes.data)


def qzeros(n) -> np.ndarray:
    return np.zeros(int(n), dtype=Q)


def num_threads() -> int:
    return int(lib().shdo_num_threads())


def set_threads(n: int) -> None:
    lib().shdo_set_threads(int(n))


def from_dd(hi, lo) -> np.ndarray:
    hi, php = _d(hi)
    lo, plp = _d(lo)
    out = qzeros(hi.size)
    lib().shdo_from_dd(hi.size, php, plp, _q(out))
    return out


def to_dd(q):
    hi = np.empty(q.size)
    lo = np.empty(q.size)
    lib().shdo_to_dd(q.size, _q(q), hi.ctypes.data_as(C.POINTER(C.c_double)),
                     lo.ctypes.data_as(C.POINTER(C.c_double)))
    return hi, lo


def to_float(q) -> np.ndarray:
    return to_dd(q)[0]


def absdiff_dd(ref_q, hi, lo) -> np.ndarray:
    """|(hi+lo) - ref| evaluated in binary128, returned as doubles."""
    hi, php = _d(hi)
    lo, plp = _d(lo)
    assert ref_q.size == hi.size == lo.size
    out = np.empty(hi.size)
    lib().shdo_absdiff_dd(hi.size, _q(ref_q), php, plp, out.ctypes.data_as(C.POINTER(C.c_double)))
    return out


def cabsdiff_dd(ref_re, ref_im, re_hi, re_lo, im_hi, im_lo) -> np.ndarray:
    a, pa = _d(re_hi)
    b, pb = _d(re_lo)
    c, pc = _d(im_hi)
    e, pe = _d(im_lo)
    out = np.empty(a.size)
    lib().shdo_cabsdiff_dd(a.size, _q(ref_re), _q(ref_im), pa, pb, pc, pe,
                           out.ctypes.data_as(C.POINTER(C.c_double)))
    return out


def fmt(q, i=0, digits=36) -> str:
    buf = C.create_string_buffer(96)
    one = np.ascontiguousarray(q[i:i + 1])
    lib().shdo_format(_q(one), digits, buf, 96)
    return buf.value.decode()


def parse(strings) -> np.ndarray:
    if isinstance(strings, str):
        strings = [strings]
    out = qzeros(len(strings))
    for i, s in enumerate(strings):
        one = qzeros(1)
        lib().shdo_parse(s.encode(), _q(one))
        out[i] = one[0]
    return out


# ----------------------------------------------------------------------- the oracle API
def enumerate_Q(d: int, m_star: int) -> np.ndarray:
    """Canonical half-space set Q as an (M, d) int32 array."""
    M = lib().shdo_enumerate(d, m_star, None)
    if M < 0:
        raise ValueError("bad d or m_star")
    n = np.zeros((M, d), dtype=np.int32)
    got = lib().shdo_enumerate(d, m_star, n.ctypes.data_as(C.POINTER(C.c_int)))
    assert got == M
    return n


def rho(d, N, L, pos_hi, pos_lo, n, mode="direct"):
    """rho(n) = sum_j exp(+i k.r_j) (Eq. 4 P:47 conjugated).  Returns (re, im) binary128."""
    ph, pph = _d(pos_hi)
    pl, ppl = _d(pos_lo)
    assert ph.size == pl.size == N * d
    n, pn = _i(n)
    M = n.size // d
    re, im = qzeros(M), qzeros(M)
    f = lib().shdo_rho_direct if mode == "direct" else lib().shdo_rho_factored
    f(d, N, float(L), pph, ppl, M, pn, _q(re), _q(im))
    return re, im


def energy(N, rho_re, rho_im, v=None):
    """(Phi, S_max, argmax, |rho|^2 array): Eq. 2 P:39 / Eq. 1 P:27 / Eq. 3 P:43."""
    M = rho_re.size
    phi, smax, s2 = qzeros(1), qzeros(1), qzeros(M)
    arg = C.c_long(-1)
    pv = None
    if v is not None:
        v, pv = _d(v)
        assert v.size == M
    lib().shdo_energy(N, M, _q(rho_re), _q(rho_im), pv, _q(phi), _q(smax), C.byref(arg), _q(s2))
    return phi, smax, int(arg.value), s2


def grad(d, N, L, pos_hi, pos_lo, n, rho_re, rho_im, v=None, jlist=None, mode="direct"):
    """dPhi/dr_{j,a} (Eq. 6, sign D:R2); axis-major over the evaluated subset."""
    ph, pph = _d(pos_hi)
    pl, ppl = _d(pos_lo)
    n, pn = _i(n)
    M = n.size // d
    pv = None
    if v is not None:
        v, pv = _d(v)
    if jlist is None:
        nj, pj = N, None
    else:
        jl = np.ascontiguousarray(jlist, dtype=np.int64)
        nj, pj = jl.size, jl.ctypes.data_as(C.POINTER(C.c_long))
    out = qzeros(nj * d)
    f = lib().shdo_grad_direct if mode == "direct" else lib().shdo_grad_factored
    f(d, N, float(L), pph, ppl, M, pn, pv, _q(rho_re), _q(rho_im), nj, pj, _q(out))
    return out


def energy_grad(d, N, L, pos_hi, pos_lo, n, v=None, mode="direct", want_grad=True):
    re, im = rho(d, N, L, pos_hi, pos_lo, n, mode)
    phi, smax, arg, s2 = energy(N, re, im, v)
    g = grad(d, N, L, pos_hi, pos_lo, n, re, im, v, None, mode) if want_grad else None
    return dict(rho_re=re, rho_im=im, phi=phi, smax=smax, argmax=arg, s2=s2, grad=g)


def eval_q(d, N, L, xq, n, v=None, mode="direct", want_grad=False):
    """Phi, S_max (and grad) at binary128 positions xq (used by finite-difference pins)."""
    n, pn = _i(n)
    M = n.size // d
    pv = None
    if v is not None:
        v, pv = _d(v)
    phi, smax = qzeros(1), qzeros(1)
    arg = C.c_long(-1)
    g = qzeros(N * d) if want_grad else None
    lib().shdo_eval_q(d, N, float(L), _q(xq), M, pn, pv, 0 if mode == "direct" else 1,
                      _q(phi), _q(smax), C.byref(arg), _q(g) if want_grad else None)
    return phi, smax, int(arg.value), g


def minimize_lbfgs(d, N, L, pos_hi, pos_lo, n, v=None, mode="direct", history=10,
                   smax_tol=1e-30, max_evals=5000):
    """Textbook binary128 L-BFGS (S8c).  Returns dict with final dd positions and report."""
    n, pn = _i(n)
    M = n.size // d
    pv = None
    if v is not None:
        v, pv = _d(v)
    x = from_dd(pos_hi, pos_lo)
    rep = (C.c_long * 2)()
    phi, smax = qzeros(1), qzeros(1)
    st = lib().shdo_minimize_lbfgs(d, N, float(L), _q(x), M, pn, pv, 0 if mode == "direct" else 1,
                                   history, float(smax_tol), int(max_evals), rep, _q(phi), _q(smax))
    hi, lo = to_dd(x)
    return dict(status=st, iters=int(rep[0]), evals=int(rep[1]), phi=phi, smax=smax,
                pos_hi=hi, pos_lo=lo)


def fire_dt0(d, N, L, n) -> float:
    """Default FIRE time step: the stiffest collective mode of Phi = sum |rho|^2 has
    curvature ~ 2 N k_max^2 (unit masses), so explicit integration is stable for dt < 2 / (k_max sqrt(2N));
    dt_max = 10 dt0 is put at half of that bound."""
    n = np.asarray(n).reshape(-1, d)
    kmax = 2.0 * np.pi * np.sqrt(float((n.astype(np.int64) ** 2).sum(axis=1).max())) / float(L)
    return 0.1 / (kmax * np.sqrt(2.0 * N))


def minimize_fire(d, N, L, pos_hi, pos_lo, n, v=None, mode="direct", dt0=None,
                  smax_tol=1e-30, max_evals=20000):
    """Binary128 FIRE (ref.[37]).  Returns dict with final dd positions and report."""
    if dt0 is None:
        dt0 = fire_dt0(d, N, L, n)
    n, pn = _i(n)
    M = n.size // d
    pv = None
    if v is not None:
        v, pv = _d(v)
    x = from_dd(pos_hi, pos_lo)
    rep = (C.c_long * 2)()
    phi, smax = qzeros(1), qzeros(1)
    st = lib().shdo_minimize_fire(d, N, float(L), _q(x), M, pn, pv, 0 if mode == "direct" else 1,
                                  float(dt0), float(smax_tol), int(max_evals), rep, _q(phi), _q(smax))
    hi, lo = to_dd(x)
    return dict(status=st, steps=int(rep[0]), evals=int(rep[1]), phi=phi, smax=smax,
                pos_hi=hi, pos_lo=lo, dt0=float(dt0))


def structure_factor(N, rho_re, rho_im):
    """S(k) = |rho|^2 / N (binary128 array) and sum_k (S - 1)^2 (Eq. 3, Eq. 7)."""
    M = len(rho_re)
    S, dev2 = qzeros(M), qzeros(1)
    lib().shdo_structure_factor(int(N), M, _q(rho_re), _q(rho_im), _q(S), _q(dev2))
    return S, dev2


def structure_factor_shells(d, N, n, rho_re, rho_im, edges):
    """Radial average of S(k) (Fig. 2a, Fig. S1a): bin b = wavevectors with edges[b] <= n.n < edges[b+1].
    Returns (count int64 array, S_mean binary128 array)."""
    n, pn = _i(n)
    M = n.size // d
    e = np.ascontiguousarray(edges, dtype=np.int64)
    nb = e.size - 1
    count = np.zeros(nb, dtype=np.int64)
    S = qzeros(nb)
    lib().shdo_structure_factor_shells(d, int(N), M, pn, _q(rho_re), _q(rho_im), nb,
                                       e.ctypes.data_as(C.POINTER(C.c_long)), count.ctypes.data_as(C.POINTER(C.c_long)), _q(S))
    return count, S


def tau(d, N, L, K, dev2) -> float:
    """tau = K^d V / N^2 * 2 * sum_{k in half space} (S(k) - 1)^2   (Eq. 7, D = 1/K)."""
    return float(K) ** d * float(L) ** d / float(N) ** 2 * 2.0 * float(to_float(dev2)[0])
