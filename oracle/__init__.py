"""fp64 CPU oracle of the coupled LLG + cavity-mode RK45 step — TEST INFRASTRUCTURE.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` leg may import this package.  It never imports the CUDA package.
The arithmetic lives in ``cavmag_oracle.cpp`` (plain loops, fp64); this file only
marshals numpy arrays through ctypes.
"""
from __future__ import annotations

import ctypes as C
import dataclasses
from typing import Optional

import numpy as np

from . import build as _build

_dp = C.POINTER(C.c_double)


class _Problem(C.Structure):
    _fields_ = [("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int),
                ("dx", C.c_double), ("dy", C.c_double), ("dz", C.c_double),
                ("Ms", C.c_double), ("Aex", C.c_double), ("Ku", C.c_double),
                ("axis", C.c_double * 3), ("alpha", C.c_double), ("gamma", C.c_double),
                ("B0", C.c_double * 3), ("n_sub", C.c_int), ("B_exch_inter", C.c_double),
                ("renormalize", C.c_int), ("norm_sum_u", C.c_int), ("N", C.c_int),
                ("u", _dp), ("omega", _dp), ("kappa", _dp), ("g", _dp), ("Gamma", _dp), ("Phi", _dp),
                ("eta_amp", _dp), ("eta_t0", _dp), ("eta_sigma", _dp), ("eta_wd", _dp),
                ("g_b", _dp), ("Gamma_b", _dp), ("Phi_b", _dp), ("pol", _dp), ("quad", _dp), ("demag_N", _dp)]


class _Stats(C.Structure):
    _fields_ = [("accepted", C.c_longlong), ("rejected", C.c_longlong), ("rhs_evals", C.c_longlong),
                ("dt_min", C.c_double), ("dt_max", C.c_double), ("dt_next", C.c_double), ("t", C.c_double),
                ("status", C.c_int)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build.build())
        _lib.orc_rhs.argtypes = [C.POINTER(_Problem), C.c_double, _dp, _dp, _dp, _dp, _dp]
        _lib.orc_rhs.restype = None
        _lib.orc_run.argtypes = [C.POINTER(_Problem), _dp, _dp, _dp, C.c_double, C.c_double, C.c_double, _dp,
                                 C.c_longlong, C.c_double, _dp, C.c_int, C.POINTER(C.c_int), C.POINTER(_Stats)]
        _lib.orc_run.restype = C.c_int
        _lib.orc_run_split.argtypes = [C.POINTER(_Problem), _dp, _dp, _dp, C.c_double, C.c_longlong, C.c_int,
                                       C.c_longlong, _dp, C.c_int, C.POINTER(C.c_int)]
        _lib.orc_run_split.restype = C.c_int
        _lib.orc_dft.argtypes = [_dp, _dp, C.c_int, _dp, C.c_int, _dp]
        _lib.orc_dft.restype = None
        _lib.orc_demag_tensor.argtypes = [C.c_int, C.c_int, C.c_int, C.c_double, C.c_double, C.c_double, _dp]
        _lib.orc_demag_tensor.restype = None
        _lib.orc_tableau.argtypes = [_dp, _dp, _dp, _dp]
        _lib.orc_set_threads.argtypes = [C.c_int]
        _lib.orc_get_threads.restype = C.c_int
    return _lib


def _p(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data_as(_dp)


def _c64(x) -> np.ndarray:
    return np.ascontiguousarray(np.asarray(x, dtype=np.float64))


@dataclasses.dataclass
class RunResult:
    m: np.ndarray           # [n_sub][3][nz][ny][nx]
    a: np.ndarray           # [N] complex
    t: float
    dt: float
    accepted: int
    rejected: int
    rhs_evals: int
    dt_min: float
    dt_max: float
    status: int
    trace: Optional[np.ndarray]   # rows [t, a(re,im)xN, S(re,im)xN, <m_s> x n_sub]


class Oracle:
    """One problem instance (grid + material + modes), built from a cavmag_workloads.Workload
    or from keyword arguments with the same names."""

    def __init__(self, w=None, renormalize: bool = True, norm_sum_u: bool = False, drive: Optional[dict] = None,
                 backward: Optional[dict] = None, pol=None, quad=None, demag: bool = False, **kw):
        """drive = dict(amp [N] complex, t0 [N], sigma [N], omega_d [N] or None): the Gaussian-pulse drive
        eta_n(t) = amp_n exp(-(t-t0_n)^2/(2 sigma_n^2)) exp(-i omega_d,n (t-t0_n)) of Eq. 1 / Eq. 12."""
        get = (lambda k: kw[k] if k in kw else getattr(w, k))
        self.nx, self.ny, self.nz = int(get("nx")), int(get("ny")), int(get("nz"))
        self.n_sub = int(get("n_sub"))
        self.u = _c64(get("u")).reshape(-1, self.nz, self.ny, self.nx)
        self.N = self.u.shape[0] if self.u.size else 0
        self.omega, self.kappa, self.g = _c64(get("omega")), _c64(get("kappa")), _c64(get("g"))
        self.Gamma, self.Phi = _c64(get("Gamma")), _c64(get("Phi"))
        ax = np.asarray(get("ku_axis"), dtype=np.float64)
        ax = ax / np.linalg.norm(ax)
        P = _Problem()
        P.nx, P.ny, P.nz = self.nx, self.ny, self.nz
        P.dx, P.dy, P.dz = float(get("dx")), float(get("dy")), float(get("dz"))
        P.Ms, P.Aex, P.Ku = float(get("Ms")), float(get("Aex")), float(get("Ku"))
        P.axis = (C.c_double * 3)(*ax)
        P.alpha, P.gamma = float(get("alpha")), float(get("gamma"))
        P.B0 = (C.c_double * 3)(*[float(b) for b in get("B0")])
        P.n_sub, P.B_exch_inter = self.n_sub, float(get("B_exch_inter"))
        P.renormalize, P.norm_sum_u, P.N = int(renormalize), int(norm_sum_u), self.N
        P.u, P.omega, P.kappa, P.g = _p(self.u), _p(self.omega), _p(self.kappa), _p(self.g)
        P.Gamma, P.Phi = _p(self.Gamma), _p(self.Phi)
        if drive is not None and self.N:
            self.eta_amp = _c64(np.asarray(drive["amp"], dtype=np.complex128).reshape(self.N).view(np.float64))
            self.eta_t0 = _c64(np.broadcast_to(np.asarray(drive["t0"], dtype=np.float64), (self.N,)))
            self.eta_sigma = _c64(np.broadcast_to(np.asarray(drive["sigma"], dtype=np.float64), (self.N,)))
            wd = drive.get("omega_d")
            self.eta_wd = None if wd is None else _c64(np.broadcast_to(np.asarray(wd, dtype=np.float64), (self.N,)))
            P.eta_amp, P.eta_t0, P.eta_sigma, P.eta_wd = _p(self.eta_amp), _p(self.eta_t0), _p(self.eta_sigma), _p(self.eta_wd)
        if backward is not None and self.N:
            # non-reciprocal coupling: backward = dict(g [N], Gamma [N] or None, Phi [N] or None)
            self.g_b = _c64(np.broadcast_to(np.asarray(backward["g"], dtype=np.float64), (self.N,)))
            Gb, Pb = backward.get("Gamma"), backward.get("Phi")
            self.Gamma_b = None if Gb is None else _c64(np.broadcast_to(np.asarray(Gb, dtype=np.float64), (self.N,)))
            self.Phi_b = None if Pb is None else _c64(np.broadcast_to(np.asarray(Pb, dtype=np.float64), (self.N,)))
            P.g_b, P.Gamma_b, P.Phi_b = _p(self.g_b), _p(self.Gamma_b), _p(self.Phi_b)
        if pol is not None and self.N:
            # per-mode polarisation p_n [N][3] (unit vectors) and optional quadrature axes q_n (default z^ x p_n)
            self.pol = _c64(np.asarray(pol, dtype=np.float64).reshape(self.N, 3))
            self.quad = None if quad is None else _c64(np.asarray(quad, dtype=np.float64).reshape(self.N, 3))
            P.pol, P.quad = _p(self.pol), _p(self.quad)
        if demag:
            # dipolar field (reading G34; off in the paper): tensor table for every cell offset
            self.demag_N = demag_tensor(self.nx, self.ny, self.nz, P.dx, P.dy, P.dz)
            P.demag_N = _p(self.demag_N)
        self.P = P
        self.nc = self.nx * self.ny * self.nz
        self.gamma = P.gamma

    # -- f(m, a) --------------------------------------------------------------------
    def rhs(self, m: np.ndarray, a: np.ndarray, t: float = 0.0):
        """Returns (dm [n_sub,3,nz,ny,nx], da [N] complex, S [N] complex) at time t."""
        m = _c64(m).reshape(self.n_sub, 3, self.nz, self.ny, self.nx)
        a2 = _c64(np.asarray(a, dtype=np.complex128).view(np.float64))
        dm = np.empty_like(m)
        da = np.zeros(max(2 * self.N, 1))
        S = np.zeros(max(2 * self.N, 1))
        lib().orc_rhs(C.byref(self.P), float(t), _p(m), _p(a2), _p(dm), _p(da), _p(S))
        return dm, da[:2 * self.N].view(np.complex128).copy(), S[:2 * self.N].view(np.complex128).copy()

    # -- time integration -----------------------------------------------------------
    def run(self, m, a, t0: float = 0.0, t_end: float = np.inf, tol: float = 0.0, fixed_dt: float = 0.0,
            dt_init: float = 0.0, max_steps: int = 0, sample_dt: float = 0.0, trace_cap: int = 0) -> RunResult:
        m = _c64(m).reshape(self.n_sub, 3, self.nz, self.ny, self.nx).copy()
        a2 = np.zeros(max(2 * self.N, 1))
        a2[:2 * self.N] = np.asarray(a, dtype=np.complex128).reshape(self.N).view(np.float64)
        t = C.c_double(t0)
        dt = C.c_double(dt_init)
        rowlen = 1 + 4 * self.N + 3 * self.n_sub
        trace = np.zeros((max(trace_cap, 1), rowlen)) if (sample_dt > 0 and trace_cap > 0) else None
        ntr = C.c_int(0)
        st = _Stats()
        lib().orc_run(C.byref(self.P), _p(m), _p(a2), C.byref(t), float(t_end), float(tol), float(fixed_dt),
                      C.byref(dt), int(max_steps), float(sample_dt), _p(trace), int(trace_cap), C.byref(ntr),
                      C.byref(st))
        return RunResult(m=m, a=a2[:2 * self.N].view(np.complex128).copy(), t=t.value, dt=dt.value,
                         accepted=st.accepted, rejected=st.rejected, rhs_evals=st.rhs_evals,
                         dt_min=st.dt_min, dt_max=st.dt_max, status=st.status,
                         trace=None if trace is None else trace[:ntr.value].copy())


    # -- the paper's tier-2 operator-split loop (comparison integrator) ------------------
    def run_split(self, m, a, dt: float, n_steps: int, n_llg: int = 1, t0: float = 0.0, sample_every: int = 0,
                  trace_cap: int = 0) -> RunResult:
        m = _c64(m).reshape(self.n_sub, 3, self.nz, self.ny, self.nx).copy()
        a2 = np.zeros(max(2 * self.N, 1))
        a2[:2 * self.N] = np.asarray(a, dtype=np.complex128).reshape(self.N).view(np.float64)
        t = C.c_double(t0)
        rowlen = 1 + 4 * self.N + 3 * self.n_sub
        trace = np.zeros((max(trace_cap, 1), rowlen)) if (sample_every > 0 and trace_cap > 0) else None
        ntr = C.c_int(0)
        status = lib().orc_run_split(C.byref(self.P), _p(m), _p(a2), C.byref(t), float(dt), int(n_steps), int(n_llg),
                                     int(sample_every), _p(trace), int(trace_cap), C.byref(ntr))
        return RunResult(m=m, a=a2[:2 * self.N].view(np.complex128).copy(), t=t.value, dt=dt, accepted=int(n_steps),
                         rejected=0, rhs_evals=6 * int(n_steps) * int(n_llg), dt_min=dt, dt_max=dt, status=status,
                         trace=None if trace is None else trace[:ntr.value].copy())


def demag_tensor(nx: int, ny: int, nz: int, dx: float, dy: float, dz: float) -> np.ndarray:
    """[2nz-1][2ny-1][2nx-1][6] demagnetising tensor (xx, yy, zz, xy, xz, yz) between two cells at every offset."""
    out = np.zeros((2 * nz - 1, 2 * ny - 1, 2 * nx - 1, 6))
    lib().orc_demag_tensor(int(nx), int(ny), int(nz), float(dx), float(dy), float(dz), _p(out))
    return out


def dft(t, x, w) -> np.ndarray:
    """Plain Fourier sum X(w_k) = sum_j x_j exp(+i w_k t_j) of a sampled complex trace (orc_dft)."""
    t = _c64(t)
    xx = _c64(np.asarray(x, dtype=np.complex128).reshape(-1).view(np.float64))
    w = _c64(np.atleast_1d(w))
    out = np.zeros(2 * w.size)
    lib().orc_dft(_p(t), _p(xx), int(t.size), _p(w), int(w.size), _p(out))
    return out.view(np.complex128).copy()


def tableau():
    a = np.zeros((7, 7)); b = np.zeros(7); bh = np.zeros(7); c = np.zeros(7)
    lib().orc_tableau(_p(a), _p(b), _p(bh), _p(c))
    return a, b, bh, c


def set_threads(n: int) -> None:
    lib().orc_set_threads(int(n))


def get_threads() -> int:
    return int(lib().orc_get_threads())
