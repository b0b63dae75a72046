"""Thin ctypes binding over libshd.so (include/shd.h).  Argument marshalling only: every step of the
hot path runs inside the library's CUDA kernels.  PyTorch is used for device buffers and streams.

There is NO CPU fallback: importing this module without a built ``libshd.so`` raises, and every
compute call needs a CUDA device.
"""
from __future__ import annotations

import ctypes as C
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
LIB_PATH = _HERE / "libshd.so"

SHD_OK, SHD_EINVAL, SHD_ENOMEM, SHD_ECUDA, SHD_ENAN, SHD_ESTALL, SHD_EMAXEVAL, SHD_ESTOPPED = 0, -1, -2, -3, -4, -5, -6, -7
SHD_NOALLOC_MAX_Q = 4194304          # shd.h: the most wavevectors shd_structure_factor_noalloc accepts
EXPORTS = ["shd_create", "shd_create_shell", "shd_create_table", "shd_destroy", "shd_set_stream", "shd_num_k", "shd_get_k",
           "shd_energy_grad", "shd_energy_grad_host", "shd_set_timing", "shd_smax", "shd_last_smax", "shd_get_rho", "shd_minimize",
           "shd_last_error", "shd_stat", "shd_fp64_peak", "shd_structure_factor", "shd_set_precision", "shd_i8_probe", "shd_set_engine",
           "shd_set_workspace", "shd_set_shard", "shd_comm_unique_id", "shd_comm_init", "shd_partial_bytes", "shd_rho_partial", "shd_rho_finish",
           "shd_grad_local", "shd_structure_factor_shells", "shd_tau", "shd_get_trace", "shd_minimize_snapshot", "shd_mix_probe", "shd_num_shells", "shd_get_shells",
           "shd_structure_factor_noalloc"]


class ShdError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"libshd error {code}: {msg}")
        self.code = code


class shd_min_report(C.Structure):
    _fields_ = [("iters", C.c_long), ("evals", C.c_long), ("phi", C.c_double * 2),
                ("smax", C.c_double * 2), ("status", C.c_int)]


shd_poll_fn = C.CFUNCTYPE(C.c_int, C.POINTER(shd_min_report), C.c_void_p)


class shd_min_opts(C.Structure):
    _fields_ = [("kind", C.c_int), ("history", C.c_int), ("smax_tol", C.c_double),
                ("max_evals", C.c_long), ("poll_every", C.c_int), ("fire_dt0", C.c_double),
                ("resume", C.c_int), ("ladder_tol", C.c_double * 2), ("on_poll", shd_poll_fn),
                ("on_poll_user", C.c_void_p)]


class shd_trace_rec(C.Structure):
    _fields_ = [("iters", C.c_long), ("evals", C.c_long), ("phi", C.c_double), ("smax", C.c_double),
                ("gnorm", C.c_double), ("step", C.c_double), ("limbs", C.c_int), ("accepted", C.c_int)]


def _load():
    if not LIB_PATH.exists():
        raise ImportError(f"{LIB_PATH} is missing: run `python -m paper_2304_09139_b200.build` "
                          "(libshd has no CPU fallback)")
    lib = C.CDLL(str(LIB_PATH))
    vp, dp = C.c_void_p, C.POINTER(C.c_double)
    lib.shd_create.argtypes = [C.c_int, C.c_long, C.c_double, C.c_double, dp, C.POINTER(vp)]
    lib.shd_create_shell.argtypes = [C.c_int, C.c_long, C.c_double, C.c_long, dp, C.POINTER(vp)]
    lib.shd_create_table.argtypes = [C.c_int, C.c_long, C.c_double, C.c_long, C.POINTER(C.c_int), dp, C.POINTER(vp)]
    lib.shd_destroy.argtypes = [vp]
    lib.shd_destroy.restype = None
    lib.shd_set_stream.argtypes = [vp, vp]
    lib.shd_num_k.argtypes = [vp]
    lib.shd_num_k.restype = C.c_long
    lib.shd_get_k.argtypes = [vp, C.POINTER(C.c_int)]
    lib.shd_energy_grad.argtypes = [vp, vp, vp, dp, vp, vp]
    lib.shd_energy_grad_host.argtypes = [vp, dp, dp, dp, dp, dp]
    lib.shd_set_timing.argtypes = [vp, C.c_int]
    lib.shd_smax.argtypes = [vp, vp, vp, dp, C.POINTER(C.c_long)]
    lib.shd_last_smax.argtypes = [vp, dp, C.POINTER(C.c_long)]
    lib.shd_get_rho.argtypes = [vp, vp, vp, vp, vp]
    lib.shd_minimize.argtypes = [vp, vp, vp, C.POINTER(shd_min_opts), C.POINTER(shd_min_report)]
    lib.shd_last_error.argtypes = [vp]
    lib.shd_last_error.restype = C.c_char_p
    lib.shd_stat.argtypes = [vp, C.c_int]
    lib.shd_stat.restype = C.c_double
    lib.shd_fp64_peak.argtypes = [C.c_int, C.c_double, dp]
    lib.shd_structure_factor.argtypes = [vp, vp, dp]
    lib.shd_structure_factor_noalloc.argtypes = [vp, vp, vp, C.c_int]
    lib.shd_set_precision.argtypes = [vp, C.c_int]
    lib.shd_i8_probe.argtypes = [dp, C.POINTER(C.c_long)]
    lib.shd_set_engine.argtypes = [vp, C.c_int]
    lib.shd_set_workspace.argtypes = [vp, C.c_ulong]
    lib.shd_set_shard.argtypes = [vp, C.c_long, C.c_int, C.c_int]
    lib.shd_comm_unique_id.argtypes = [vp]
    lib.shd_comm_init.argtypes = [vp, vp]
    lib.shd_partial_bytes.argtypes = [vp]
    lib.shd_partial_bytes.restype = C.c_ulong
    lib.shd_rho_partial.argtypes = [vp, vp, vp, vp]
    lib.shd_rho_finish.argtypes = [vp, vp, C.c_int, dp]
    lib.shd_grad_local.argtypes = [vp, vp, vp, vp, vp]
    lib.shd_structure_factor_shells.argtypes = [vp, C.c_long, C.POINTER(C.c_long), C.POINTER(C.c_long), dp, dp]
    lib.shd_tau.argtypes = [vp, C.c_double, dp]
    lib.shd_get_trace.argtypes = [vp, C.c_long, C.c_long, C.POINTER(shd_trace_rec)]
    lib.shd_get_trace.restype = C.c_long
    lib.shd_minimize_snapshot.argtypes = [vp, vp, vp]
    lib.shd_mix_probe.argtypes = [dp]
    lib.shd_num_shells.argtypes = [vp]
    lib.shd_num_shells.restype = C.c_long
    lib.shd_get_shells.argtypes = [vp, C.POINTER(C.c_long)]
    return lib


lib = _load()


def _torch():
    import torch
    if not torch.cuda.is_available():
        raise RuntimeError("libshd needs a CUDA device (no CPU fallback)")
    return torch


class Shd:
    """One handle (shd_ctx).  Tensors are CUDA float64, axis-major ``x[a*N + j]``."""

    def __init__(self, d, N, L, K=None, v=None, m_star=None, table=None):
        self.d, self.N, self.L = int(d), int(N), float(L)
        self._h = C.c_void_p()
        pv = None
        if v is not None:
            self._v = np.ascontiguousarray(v, dtype=np.float64)
            pv = self._v.ctypes.data_as(C.POINTER(C.c_double))
        if table is not None:
            self._table = np.ascontiguousarray(table, dtype=np.int32).reshape(-1, self.d)
            rc = lib.shd_create_table(self.d, self.N, self.L, len(self._table),
                                      self._table.ctypes.data_as(C.POINTER(C.c_int)), pv, C.byref(self._h))
        elif m_star is not None:
            rc = lib.shd_create_shell(self.d, self.N, self.L, int(m_star), pv, C.byref(self._h))
        else:
            rc = lib.shd_create(self.d, self.N, self.L, float(K), pv, C.byref(self._h))
        if rc != SHD_OK:
            msg = lib.shd_last_error(self._h).decode() if self._h else "invalid argument"
            if self._h:
                lib.shd_destroy(self._h)
                self._h = C.c_void_p()
            raise ShdError(rc, msg)
        self.M = int(lib.shd_num_k(self._h))

    def close(self):
        if getattr(self, "_h", None):
            lib.shd_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, rc, ok=(SHD_OK,)):
        if rc not in ok:
            raise ShdError(rc, lib.shd_last_error(self._h).decode())
        return rc

    def set_stream(self, stream):
        """stream: a torch.cuda.Stream (or None for the legacy default stream)."""
        self._check(lib.shd_set_stream(self._h, C.c_void_p(stream.cuda_stream if stream is not None else 0)))

    def k(self) -> np.ndarray:
        n = np.zeros((self.M, self.d), dtype=np.int32)
        self._check(lib.shd_get_k(self._h, n.ctypes.data_as(C.POINTER(C.c_int))))
        return n

    def _pos(self, pos_hi, pos_lo):
        torch = _torch()
        for t in (pos_hi, pos_lo):
            assert t.is_cuda and t.dtype == torch.float64 and t.is_contiguous() and t.numel() == self.d * self.N
        return C.c_void_p(pos_hi.data_ptr()), C.c_void_p(pos_lo.data_ptr())

    def energy_grad(self, pos_hi, pos_lo, grad_hi=None, grad_lo=None, want_grad=True):
        """shd_energy_grad: returns (phi_hi, phi_lo), grad_hi, grad_lo (device tensors or None)."""
        torch = _torch()
        ph, pl = self._pos(pos_hi, pos_lo)
        if want_grad and grad_hi is None:
            grad_hi = torch.empty_like(pos_hi)
            grad_lo = torch.empty_like(pos_hi)
        phi = (C.c_double * 2)()
        gh = C.c_void_p(grad_hi.data_ptr()) if want_grad else None
        gl = C.c_void_p(grad_lo.data_ptr()) if want_grad else None
        self._check(lib.shd_energy_grad(self._h, ph, pl, phi, gh, gl))
        return (phi[0], phi[1]), (grad_hi if want_grad else None), (grad_lo if want_grad else None)

    def energy_grad_host(self, pos_hi, pos_lo, grad_hi=None, grad_lo=None):
        """shd_energy_grad_host: numpy float64 arrays in HOST memory (e.g. views of pinned tensors);
        grad arrays are filled in place.  Returns (phi_hi, phi_lo)."""
        dp = C.POINTER(C.c_double)
        for a in (pos_hi, pos_lo, grad_hi, grad_lo):
            assert a is None or (a.dtype == np.float64 and a.flags.c_contiguous and a.size == self.d * self.N)
        phi = (C.c_double * 2)()
        g = [a.ctypes.data_as(dp) if a is not None else None for a in (grad_hi, grad_lo)]
        self._check(lib.shd_energy_grad_host(self._h, pos_hi.ctypes.data_as(dp), pos_lo.ctypes.data_as(dp),
                                             phi, g[0], g[1]))
        return phi[0], phi[1]

    def set_timing(self, on: bool):
        self._check(lib.shd_set_timing(self._h, 1 if on else 0))

    def kernel_ms(self):
        """milliseconds of the last call's launch groups (after set_timing(True))."""
        names = ["tables", "rho", "finish", "ctable", "grad"]
        return {n: self.stat(20 + i) for i, n in enumerate(names)}

    def smax(self, pos_hi, pos_lo):
        ph, pl = self._pos(pos_hi, pos_lo)
        s = (C.c_double * 2)()
        arg = C.c_long(-1)
        self._check(lib.shd_smax(self._h, ph, pl, s, C.byref(arg)))
        return (s[0], s[1]), int(arg.value)

    def last_smax(self):
        s = (C.c_double * 2)()
        arg = C.c_long(-1)
        self._check(lib.shd_last_smax(self._h, s, C.byref(arg)))
        return (s[0], s[1]), int(arg.value)

    def rho(self):
        """rho(k) of the last evaluation: (re_hi, re_lo, im_hi, im_lo) device tensors."""
        torch = _torch()
        out = [torch.empty(self.M, dtype=torch.float64, device="cuda") for _ in range(4)]
        self._check(lib.shd_get_rho(self._h, *[C.c_void_p(t.data_ptr()) for t in out]))
        return tuple(out)

    def set_precision(self, limbs: int):
        """shd_set_precision: 3 = double-double products (default), 2 = 44-bit operands, 1 = 22-bit operands."""
        self._check(lib.shd_set_precision(self._h, int(limbs)))

    def set_engine(self, rho_engine: int):
        """shd_set_engine: 2 = both passes on the INT8 tensor cores (tcgen05), 1 = rho pass only, 0 = FP64 limbs (DMMA),
        -1 = the library's own choice (what a fresh handle starts with)."""
        self._check(lib.shd_set_engine(self._h, int(rho_engine)))

    @property
    def engine(self) -> int:
        return int(self.stat(16))

    def set_workspace(self, nbytes: int):
        """shd_set_workspace: cap on the per-particle tables; the evaluation then runs chunk by chunk (bit-identical)."""
        self._check(lib.shd_set_workspace(self._h, int(nbytes)))

    def set_shard(self, N_total: int, rank: int, world: int):
        """shd_set_shard: this handle's N particles are shard `rank` of `world` of a system of N_total."""
        self._check(lib.shd_set_shard(self._h, int(N_total), int(rank), int(world)))

    def comm_init(self, id128: bytes):
        """shd_comm_init (collective): the 128 bytes of comm_unique_id() from one rank."""
        buf = C.create_string_buffer(bytes(id128), 128)
        self._check(lib.shd_comm_init(self._h, C.cast(buf, C.c_void_p)))

    def rho_partial(self, pos_hi, pos_lo, out=None):
        """shd_rho_partial: this shard's running sums as a CUDA uint8 tensor of shd_partial_bytes bytes."""
        torch = _torch()
        ph, pl = self._pos(pos_hi, pos_lo)
        if out is None:
            out = torch.empty(int(lib.shd_partial_bytes(self._h)), dtype=torch.uint8, device="cuda")
        self._check(lib.shd_rho_partial(self._h, ph, pl, C.c_void_p(out.data_ptr())))
        return out

    def rho_finish(self, gathered, nparts: int):
        """shd_rho_finish: gathered = CUDA uint8 tensor holding nparts partials in rank order.  Returns (phi_hi, phi_lo)."""
        phi = (C.c_double * 2)()
        self._check(lib.shd_rho_finish(self._h, C.c_void_p(gathered.data_ptr()), int(nparts), phi))
        return phi[0], phi[1]

    def grad_local(self, pos_hi, pos_lo, grad_hi=None, grad_lo=None):
        torch = _torch()
        ph, pl = self._pos(pos_hi, pos_lo)
        if grad_hi is None:
            grad_hi, grad_lo = torch.empty_like(pos_hi), torch.empty_like(pos_hi)
        self._check(lib.shd_grad_local(self._h, ph, pl, C.c_void_p(grad_hi.data_ptr()), C.c_void_p(grad_lo.data_ptr())))
        return grad_hi, grad_lo

    def structure_factor(self, want_S=True):
        """shd_structure_factor on the last evaluation: (S device tensor or None, (hi, lo) of
        sum_{k in Q} (S(k) - 1)^2)."""
        torch = _torch()
        S = torch.empty(self.M, dtype=torch.float64, device="cuda") if want_S else None
        dev2 = (C.c_double * 2)()
        self._check(lib.shd_structure_factor(self._h, C.c_void_p(S.data_ptr()) if want_S else None, dev2))
        return S, (dev2[0], dev2[1])

    def structure_factor_noalloc(self, dev2, S=None, wait=True):
        """shd_structure_factor_noalloc on the last evaluation: the caller passes the outputs (dev2: CUDA float64 tensor
        of 2 elements; S: CUDA float64 tensor of |Q| elements or None); nothing is allocated by the call."""
        for t, n in ((dev2, 2), (S, self.M)):
            if t is not None and not (t.is_cuda and t.dtype == _torch().float64 and t.is_contiguous() and t.numel() == n):
                raise ValueError("structure_factor_noalloc: outputs must be contiguous CUDA float64 tensors of 2 and |Q| elements")
        self._check(lib.shd_structure_factor_noalloc(self._h, C.c_void_p(S.data_ptr()) if S is not None else None,
                                                     C.c_void_p(dev2.data_ptr()), 1 if wait else 0))

    def tau(self, K):
        """shd_tau: order metric tau of Eq. 7 from the last evaluation on this handle, D = 1/K (hi + lo)."""
        t = (C.c_double * 2)()
        self._check(lib.shd_tau(self._h, float(K), t))
        return t[0] + t[1]

    def structure_factor_shells(self, edges=None):
        """shd_structure_factor_shells on the last evaluation.  edges: ascending integer n.n bin edges (default: one bin
        per distinct shell of this handle's Q).  Returns (edges, count, S_mean_hi, S_mean_lo) as numpy arrays."""
        if edges is None:
            sh = np.zeros(int(lib.shd_num_shells(self._h)), dtype=np.int64)
            self._check(lib.shd_get_shells(self._h, sh.ctypes.data_as(C.POINTER(C.c_long))))
            edges = np.concatenate([sh, [sh[-1] + 1]])
        e = np.ascontiguousarray(edges, dtype=np.int64)
        nb = e.size - 1
        count = np.zeros(nb, dtype=np.int64)
        hi, lo = np.zeros(nb), np.zeros(nb)
        lp, dp = C.POINTER(C.c_long), C.POINTER(C.c_double)
        self._check(lib.shd_structure_factor_shells(self._h, nb, e.ctypes.data_as(lp), count.ctypes.data_as(lp),
                                                    hi.ctypes.data_as(dp), lo.ctypes.data_as(dp)))
        return e, count, hi, lo

    def minimize(self, pos_hi, pos_lo, kind=0, history=10, smax_tol=1e-30, max_evals=10000, poll_every=8,
                 fire_dt0=0.0, resume=False, ladder=(0.0, 0.0), on_poll=None):
        """shd_minimize: kind 0 = L-BFGS, 1 = FIRE (fire_dt0 = 0: the library's default time step).
        ladder = (S_max below which one limb / 4 digits is left, S_max below which two limbs / 7 digits are left);
        on_poll(report dict) -> truthy to stop: host callback after every poll (trace / snapshot may be read in it)."""
        ph, pl = self._pos(pos_hi, pos_lo)
        cb = shd_poll_fn()
        if on_poll is not None:
            def _cb(rep, _user):
                r = rep.contents
                return 1 if on_poll(dict(iters=int(r.iters), evals=int(r.evals), phi=(r.phi[0], r.phi[1]),
                                         smax=(r.smax[0], r.smax[1]), status=int(r.status))) else 0
            cb = shd_poll_fn(_cb)
        opts = shd_min_opts(kind, history, smax_tol, max_evals, poll_every, fire_dt0, 1 if resume else 0,
                            (C.c_double * 2)(float(ladder[0]), float(ladder[1])), cb, None)
        rep = shd_min_report()
        rc = lib.shd_minimize(self._h, ph, pl, C.byref(opts), C.byref(rep))
        self._check(rc, ok=(SHD_OK, SHD_ESTALL, SHD_EMAXEVAL, SHD_ESTOPPED))
        return dict(status=rc, iters=int(rep.iters), evals=int(rep.evals),
                    phi=(rep.phi[0], rep.phi[1]), smax=(rep.smax[0], rep.smax[1]))

    def trace(self, first=0, max_records=1 << 22):
        """shd_get_trace: records of the last minimize call as a numpy structured array."""
        dt = np.dtype([("iters", "i8"), ("evals", "i8"), ("phi", "f8"), ("smax", "f8"), ("gnorm", "f8"), ("step", "f8"),
                       ("limbs", "i4"), ("accepted", "i4")])
        assert dt.itemsize == C.sizeof(shd_trace_rec)
        out, got = [], 0
        while got < max_records:
            buf = np.zeros(min(65536, max_records - got), dtype=dt)
            k = int(lib.shd_get_trace(self._h, first + got, len(buf), buf.ctypes.data_as(C.POINTER(shd_trace_rec))))
            out.append(buf[:k])
            got += k
            if k < len(buf):
                break
        return np.concatenate(out) if out else np.zeros(0, dtype=dt)

    def minimize_snapshot(self, pos_hi=None, pos_lo=None):
        """shd_minimize_snapshot: the minimizer's current best point (device tensors), e.g. from on_poll for a checkpoint."""
        torch = _torch()
        if pos_hi is None:
            pos_hi = torch.empty(self.d * self.N, dtype=torch.float64, device="cuda")
            pos_lo = torch.empty_like(pos_hi)
        self._check(lib.shd_minimize_snapshot(self._h, C.c_void_p(pos_hi.data_ptr()), C.c_void_p(pos_lo.data_ptr())))
        return pos_hi, pos_lo

    def stat(self, what: int) -> float:
        return float(lib.shd_stat(self._h, int(what)))


def fp64_peak(kind: int = 0, seconds: float = 1.0):
    """shd_fp64_peak: (best, sustained) thread-level FP64 instructions per second."""
    _torch()
    out = (C.c_double * 2)()
    rc = lib.shd_fp64_peak(int(kind), float(seconds), out)
    if rc != SHD_OK:
        raise ShdError(rc, "shd_fp64_peak failed")
    return out[0], out[1]


def i8_probe():
    """shd_i8_probe: (measured INT8 tensor-core TOPS, number of wrong entries of the exactness check)."""
    _torch()
    tops, bad = C.c_double(0.0), C.c_long(-1)
    rc = lib.shd_i8_probe(C.byref(tops), C.byref(bad))
    if rc != SHD_OK:
        raise ShdError(rc, "shd_i8_probe failed")
    return tops.value, bad.value


def mix_probe():
    """shd_mix_probe: FP64 / integer ALU chains beside a tcgen05.mma.kind::i8 stream (see include/shd_bench.h)."""
    _torch()
    out = (C.c_double * 8)()
    rc = lib.shd_mix_probe(out)
    if rc != SHD_OK:
        raise ShdError(rc, "shd_mix_probe failed")
    keys = ["dadd_cycles_alone", "dadd_cycles_beside_mma", "imad_cycles_alone", "imad_cycles_beside_mma",
            "mma_n256_cycles_alone", "mma_n256_cycles_beside_dadd", "mma_n256_cycles_beside_imad", "sm_mhz_under_mma"]
    return dict(zip(keys, [float(x) for x in out]))


def comm_unique_id() -> bytes:
    """shd_comm_unique_id: 128 bytes naming a new NCCL communicator (call on one rank, broadcast to all)."""
    buf = C.create_string_buffer(128)
    rc = lib.shd_comm_unique_id(C.cast(buf, C.c_void_p))
    if rc != SHD_OK:
        raise ShdError(rc, "shd_comm_unique_id failed (NCCL not loadable?)")
    return buf.raw


def from_host(hi: np.ndarray, lo: np.ndarray):
    """numpy (hi, lo) -> CUDA tensors."""
    torch = _torch()
    return (torch.from_numpy(np.ascontiguousarray(hi)).cuda(), torch.from_numpy(np.ascontiguousarray(lo)).cuda())
