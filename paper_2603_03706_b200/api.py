"""Thin Python binding of include/cavmag.h (argument marshalling only).

Same names as the C ABI: ``cav_create``, ``cav_set_modes``, ``cav_set_m``, ``cav_run`` ...
Every step of the hot path runs inside ``libcavmag.so``'s CUDA kernels; this module holds no
arithmetic and has NO CPU fallback: if the library is missing or cannot be loaded, importing
this module raises.  PyTorch is used by callers only for device memory and streams — torch
tensors are passed as raw ``data_ptr()`` addresses.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
# CAVMAG_LIB selects another build of the same library (same ABI); there is no fallback.
LIB_PATH = os.environ.get("CAVMAG_LIB") or os.path.join(_HERE, "libcavmag.so")

CAV_OK = 0
CAV_E_ARG, CAV_E_STATE, CAV_E_CUDA, CAV_E_NOMEM = -1, -2, -3, -4
CAV_E_NONFINITE, CAV_E_DT_UNDERFLOW, CAV_E_SINGULAR_NORM, CAV_E_UNSUPPORTED = -5, -6, -7, -8
CAV_F32, CAV_F64 = 0, 1
CAV_NORM_NCELLS, CAV_NORM_SUM_U = 0, 1
CAV_LAUNCH_GRAPH, CAV_LAUNCH_STREAM = 0, 1
CAV_PATH_AUTO, CAV_PATH_GENERIC, CAV_PATH_TMA, CAV_PATH_BLOCK, CAV_PATH_COOP = 0, 1, 2, 3, 4
CAV_INTEGRATOR_UNIFIED, CAV_INTEGRATOR_SPLIT = 0, 1
CAV_MAX_MODES = 32


class cav_grid(C.Structure):
    _fields_ = [("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int),
                ("dx", C.c_double), ("dy", C.c_double), ("dz", C.c_double)]


class cav_params(C.Structure):
    _fields_ = [("Ms", C.c_double), ("Aex", C.c_double), ("Ku", C.c_double), ("ku_axis", C.c_double * 3),
                ("alpha", C.c_double), ("gamma", C.c_double), ("B0", C.c_double * 3), ("n_sub", C.c_int),
                ("B_exch_inter", C.c_double), ("precision", C.c_int), ("renormalize", C.c_int),
                ("overlap_norm", C.c_int)]


class cav_stats(C.Structure):
    _fields_ = [("accepted", C.c_longlong), ("rejected", C.c_longlong), ("rhs_evals", C.c_longlong),
                ("dt_min", C.c_double), ("dt_max", C.c_double), ("dt_next", C.c_double), ("t", C.c_double),
                ("last_err", C.c_double)]


class CavError(RuntimeError):
    def __init__(self, status: int, where: str, detail: str = ""):
        self.status = status
        super().__init__(f"{where}: {cav_strerror(status)} ({status}) {detail}".strip())


if not os.path.exists(LIB_PATH):
    raise ImportError(f"{LIB_PATH} not found: build it with `python -m paper_2603_03706_b200.build` "
                      "(there is no CPU fallback)")
_lib = C.CDLL(LIB_PATH)

_vp, _dp, _i, _d, _ll = C.c_void_p, C.POINTER(C.c_double), C.c_int, C.c_double, C.c_longlong
_SIGS = {
    "cav_create": ([C.POINTER(cav_grid), C.POINTER(cav_params), C.POINTER(_vp)], _i),
    "cav_destroy": ([_vp], _i),
    "cav_set_stream": ([_vp, _vp], _i),
    "cav_set_launch_mode": ([_vp, _i], _i),
    "cav_set_modes": ([_vp, _i, _vp, _i, _dp, _dp, _dp, _dp, _dp], _i),
    "cav_set_drive": ([_vp, _dp, _dp, _dp, _dp], _i),
    "cav_set_backaction": ([_vp, _dp, _dp, _dp], _i),
    "cav_batch_set_backaction": ([_vp, _dp, _dp, _dp], _i),
    "cav_set_polarisation": ([_vp, _dp, _dp], _i),
    "cav_set_integrator": ([_vp, _i, _i], _i),
    "cav_set_demag": ([_vp, _i], _i),
    "cav_set_spectrum": ([_vp, _i, _d, _d], _i),
    "cav_get_spectrum": ([_vp, _dp, C.POINTER(_ll)], _i),
    "cav_batch_set_polarisation": ([_vp, _dp, _dp], _i),
    "cav_batch_set_integrator": ([_vp, _i, _i], _i),
    "cav_batch_set_spectrum": ([_vp, _i, _d, _d], _i),
    "cav_batch_get_spectrum": ([_vp, _dp, C.POINTER(_ll)], _i),
    "cav_set_m": ([_vp, _vp, _i], _i),
    "cav_get_m": ([_vp, _vp, _i], _i),
    "cav_set_a": ([_vp, _dp], _i),
    "cav_get_a": ([_vp, _dp], _i),
    "cav_get_overlaps": ([_vp, _dp], _i),
    "cav_get_dmdt": ([_vp, _vp, _i], _i),
    "cav_get_dadt": ([_vp, _dp], _i),
    "cav_set_sweep_order": ([_vp, _i], _i),
    "cav_set_kernel_path": ([_vp, _i], _i),
    "cav_get_kernel_path": ([_vp, C.POINTER(_i)], _i),
    "cav_set_stage_overlap": ([_vp, _i], _i),
    "cav_get_stage_overlap": ([_vp, C.POINTER(_i)], _i),
    "cav_run": ([_vp, _d, _d, _d, _d], _i),
    "cav_run_steps": ([_vp, _d, _d, _d, _d, _ll], _i),
    "cav_sync": ([_vp], _i),
    "cav_get_time": ([_vp, _dp, _dp], _i),
    "cav_set_time": ([_vp, _d], _i),
    "cav_get_stats": ([_vp, C.POINTER(cav_stats)], _i),
    "cav_set_trace": ([_vp, _d, _i], _i),
    "cav_trace_row_len": ([_vp, C.POINTER(_i)], _i),
    "cav_get_trace": ([_vp, _dp, C.POINTER(_i)], _i),
    "cav_set_block_cells": ([_vp, _i], _i),
    "cav_get_launch_count": ([_vp, C.POINTER(_ll)], _i),
    "cav_strerror": ([_i], C.c_char_p),
    "cav_last_cuda_error": ([_vp], C.c_char_p),
    "cav_version": ([], C.c_char_p),
    "cav_sweep_create": ([C.POINTER(_vp), _i, C.POINTER(_vp)], _i),
    "cav_sweep_destroy": ([_vp], _i),
    "cav_sweep_run": ([_vp, _d, _d, _d, _d, _ll], _i),
    "cav_batch_create": ([C.POINTER(cav_grid), C.POINTER(cav_params), _i, C.POINTER(_vp)], _i),
    "cav_batch_destroy": ([_vp], _i),
    "cav_batch_set_stream": ([_vp, _vp], _i),
    "cav_batch_set_field": ([_vp, _dp], _i),
    "cav_batch_set_modes": ([_vp, _i, _vp, _dp, _dp, _dp, _dp, _dp, _i], _i),
    "cav_batch_set_drive": ([_vp, _dp, _dp, _dp, _dp], _i),
    "cav_batch_set_m": ([_vp, _vp, _i], _i),
    "cav_batch_set_a": ([_vp, _dp, _i], _i),
    "cav_batch_set_trace": ([_vp, _d, _i], _i),
    "cav_batch_trace_row_len": ([_vp, C.POINTER(_i)], _i),
    "cav_batch_run": ([_vp, _d, _d, _d, _d, _ll], _i),
    "cav_batch_get_m": ([_vp, _vp], _i),
    "cav_batch_get_a": ([_vp, _dp], _i),
    "cav_batch_get_stats": ([_vp, C.POINTER(cav_stats)], _i),
    "cav_batch_get_trace": ([_vp, _dp, C.POINTER(_i)], _i),
    "cav_overlaps_noalloc": ([_vp, _vp, _i, _i, _i, _i, _i, _i, _vp, _vp], _i),
    "cav_noalloc_last_error": ([], C.c_char_p),
}
for _name, (_args, _res) in _SIGS.items():
    _f = getattr(_lib, _name)
    _f.argtypes, _f.restype = _args, _res

EXPORTS = tuple(_SIGS)


def cav_strerror(status: int) -> str:
    return _lib.cav_strerror(int(status)).decode()


def cav_version() -> str:
    return _lib.cav_version().decode()


def _check(st: int, where: str, sim=None):
    if st != CAV_OK:
        detail = _lib.cav_last_cuda_error(sim).decode() if (sim and st == CAV_E_CUDA) else ""
        raise CavError(st, where, detail)


def cav_noalloc_last_error() -> str:
    return _lib.cav_noalloc_last_error().decode()


def cav_overlaps_noalloc(m, u, S_out, grid, n_sub: int = 1, cuda_stream: int = 0) -> None:
    """S_n of the device tensors m [n_sub][3][nz][ny][nx] and u [N][nz][ny][nx] into the device tensor S_out [N][2]
    (float64); grid = (nx, ny, nz).  Allocates nothing (cavmag.h); asynchronous on cuda_stream."""
    nx, ny, nz = (int(v) for v in grid)
    N = int(u.shape[0]) if u.dim() == 4 else int(u.numel() // max(nx * ny * nz, 1))
    prec = {"torch.float32": CAV_F32, "torch.float64": CAV_F64}.get(str(m.dtype))
    if prec is None or u.dtype != m.dtype:
        raise ValueError("m and u must both be float32 or both float64")
    dt = np.float32 if prec == CAV_F32 else np.float64
    pm, dm, _ = _ptr(m, dt, 3 * int(n_sub) * nx * ny * nz, "m")
    pu, du, _ = _ptr(u, dt, N * nx * ny * nz, "u")
    ps, ds, _ = _ptr(S_out, np.float64, 2 * N, "S_out")
    if not (dm and du and ds):
        raise ValueError("cav_overlaps_noalloc takes device tensors")
    st = _lib.cav_overlaps_noalloc(pm, pu, prec, nx, ny, nz, int(n_sub), N, ps, cuda_stream)
    if st != CAV_OK:
        raise CavError(st, "cav_overlaps_noalloc", cav_noalloc_last_error())


# handle -> (numpy dtype of the cell fields, n_sub, cells, replicas): what a cell-field buffer handed to the
# library must look like.  The C ABI takes untyped pointers, so the binding is the place to refuse a float64
# array for an f32 simulation, or a wrongly sized one, before the library reads or writes out of bounds.
_HANDLES: dict = {}


def _ptr(x, dtype=None, count=None, what="buffer"):
    """(address, is_device, keepalive) of a numpy array or a torch tensor; with dtype / count given, the
    element type and the number of elements must match exactly (ValueError otherwise)."""
    if isinstance(x, np.ndarray):
        if not x.flags["C_CONTIGUOUS"]:
            raise ValueError("array must be C-contiguous")
        if dtype is not None and x.dtype != np.dtype(dtype):
            raise ValueError(f"{what}: dtype {x.dtype} does not match the simulation's precision ({np.dtype(dtype)})")
        if count is not None and x.size != count:
            raise ValueError(f"{what}: {x.size} elements, expected {count}")
        return x.ctypes.data, 0, x
    if hasattr(x, "data_ptr"):          # torch tensor (duck-typed; torch is not imported here)
        if not x.is_contiguous():
            raise ValueError("tensor must be contiguous")
        if dtype is not None and str(x.dtype) != "torch." + np.dtype(dtype).name:
            raise ValueError(f"{what}: dtype {x.dtype} does not match the simulation's precision ({np.dtype(dtype)})")
        if count is not None and x.numel() != count:
            raise ValueError(f"{what}: {x.numel()} elements, expected {count}")
        return x.data_ptr(), (1 if x.is_cuda else 0), x
    raise TypeError(f"unsupported buffer type {type(x)}")


def _field_spec(h, n_fields=None, per_replica=True):
    """(dtype, element count) of a cell-field buffer of handle h: n_fields components per cell (default: the
    magnetisation, 3 n_sub), times the replicas of a batch when per_replica."""
    dt, n_sub, nc, n_rep = _HANDLES[h]
    nf = 3 * n_sub if n_fields is None else n_fields
    return dt, nf * nc * (n_rep if per_replica else 1)


def _darr(x, n):
    if x is None:
        return None, None
    a = np.ascontiguousarray(np.asarray(x, dtype=np.float64).reshape(n))
    return a.ctypes.data_as(_dp), a


def _grid_params(grid, params):
    g = cav_grid(int(grid[0]), int(grid[1]), int(grid[2]), float(grid[3]), float(grid[4]), float(grid[5]))
    p = cav_params()
    p.Ms, p.Aex, p.Ku = float(params["Ms"]), float(params["Aex"]), float(params.get("Ku", 0.0))
    p.ku_axis = (C.c_double * 3)(*[float(v) for v in params.get("ku_axis", (0, 0, 1))])
    p.alpha, p.gamma = float(params["alpha"]), float(params["gamma"])
    p.B0 = (C.c_double * 3)(*[float(v) for v in params["B0"]])
    p.n_sub = int(params.get("n_sub", 1))
    p.B_exch_inter = float(params.get("B_exch_inter", 0.0))
    p.precision = int(params.get("precision", CAV_F32))
    p.renormalize = int(params.get("renormalize", 1))
    p.overlap_norm = int(params.get("overlap_norm", CAV_NORM_NCELLS))
    return g, p


def cav_create(grid, params) -> int:
    """grid = (nx, ny, nz, dx, dy, dz); params = dict with the cav_params fields. Returns the handle."""
    g, p = _grid_params(grid, params)
    h = _vp()
    _check(_lib.cav_create(C.byref(g), C.byref(p), C.byref(h)), "cav_create")
    _HANDLES[h.value] = (np.float32 if p.precision == CAV_F32 else np.float64, p.n_sub, g.nx * g.ny * g.nz, 1)
    return h.value


def cav_destroy(sim) -> None:
    _HANDLES.pop(sim, None)
    _check(_lib.cav_destroy(sim), "cav_destroy")


def cav_set_stream(sim, cuda_stream: int) -> None:
    _check(_lib.cav_set_stream(sim, _vp(cuda_stream)), "cav_set_stream", sim)


def cav_set_launch_mode(sim, mode: int) -> None:
    _check(_lib.cav_set_launch_mode(sim, int(mode)), "cav_set_launch_mode", sim)


def cav_set_block_cells(sim, cells: int) -> None:
    _check(_lib.cav_set_block_cells(sim, int(cells)), "cav_set_block_cells", sim)


def cav_set_modes(sim, u, omega, kappa, g, Gamma=None, Phi=None) -> None:
    """u: [N, nz, ny, nx] numpy array or torch tensor in the simulation's precision (None for N = 0)."""
    N = 0 if omega is None else int(np.asarray(omega).size)
    if N == 0:
        _check(_lib.cav_set_modes(sim, 0, None, 0, None, None, None, None, None), "cav_set_modes", sim)
        return
    addr, dev, keep = _ptr(u, *_field_spec(sim, N), what="u")
    po, ko = _darr(omega, N)
    pk, kk = _darr(kappa, N)
    pg, kg = _darr(g, N)
    pG, kG = _darr(Gamma, N)
    pP, kP = _darr(Phi, N)
    _check(_lib.cav_set_modes(sim, N, _vp(addr), dev, po, pk, pg, pG, pP), "cav_set_modes", sim)


def cav_set_m(sim, m) -> None:
    addr, dev, keep = _ptr(m, *_field_spec(sim), what="m")
    _check(_lib.cav_set_m(sim, _vp(addr), dev), "cav_set_m", sim)


def cav_get_m(sim, out) -> None:
    addr, dev, keep = _ptr(out, *_field_spec(sim), what="m_out")
    _check(_lib.cav_get_m(sim, _vp(addr), dev), "cav_get_m", sim)


def cav_set_a(sim, a) -> None:
    a = np.ascontiguousarray(np.asarray(a, dtype=np.complex128)).view(np.float64)
    if a.size > 2 * CAV_MAX_MODES:
        raise ValueError("a: more than CAV_MAX_MODES amplitudes")
    _check(_lib.cav_set_a(sim, a.ctypes.data_as(_dp)), "cav_set_a", sim)


def cav_get_a(sim, N: int) -> np.ndarray:
    out = np.zeros(max(2 * N, 1))
    _check(_lib.cav_get_a(sim, out.ctypes.data_as(_dp)), "cav_get_a", sim)
    return out[:2 * N].view(np.complex128).copy()


def cav_get_overlaps(sim, N: int) -> np.ndarray:
    out = np.zeros(max(2 * N, 1))
    _check(_lib.cav_get_overlaps(sim, out.ctypes.data_as(_dp)), "cav_get_overlaps", sim)
    return out[:2 * N].view(np.complex128).copy()


def cav_get_dmdt(sim, out) -> None:
    addr, dev, keep = _ptr(out, *_field_spec(sim), what="dmdt_out")
    _check(_lib.cav_get_dmdt(sim, _vp(addr), dev), "cav_get_dmdt", sim)


def cav_get_dadt(sim, N: int) -> np.ndarray:
    out = np.zeros(max(2 * N, 1))
    _check(_lib.cav_get_dadt(sim, out.ctypes.data_as(_dp)), "cav_get_dadt", sim)
    return out[:2 * N].view(np.complex128).copy()


def cav_set_kernel_path(sim, path: int) -> None:
    _check(_lib.cav_set_kernel_path(sim, int(path)), "cav_set_kernel_path", sim)


def cav_get_kernel_path(sim) -> int:
    p = _i()
    _check(_lib.cav_get_kernel_path(sim, C.byref(p)), "cav_get_kernel_path", sim)
    return p.value


def cav_set_stage_overlap(sim, on: int) -> None:
    _check(_lib.cav_set_stage_overlap(sim, int(on)), "cav_set_stage_overlap", sim)


def cav_get_stage_overlap(sim) -> int:
    p = _i()
    _check(_lib.cav_get_stage_overlap(sim, C.byref(p)), "cav_get_stage_overlap", sim)
    return p.value


def cav_set_sweep_order(sim, serpentine: int) -> None:
    _check(_lib.cav_set_sweep_order(sim, int(serpentine)), "cav_set_sweep_order", sim)


def cav_run(sim, t_end: float, tol: float = 0.0, fixed_dt: float = 0.0, dt_init: float = 0.0) -> None:
    _check(_lib.cav_run(sim, float(t_end), float(tol), float(fixed_dt), float(dt_init)), "cav_run", sim)


def cav_run_steps(sim, t_end: float, tol: float = 0.0, fixed_dt: float = 0.0, dt_init: float = 0.0,
                  max_steps: int = 0) -> None:
    _check(_lib.cav_run_steps(sim, float(t_end), float(tol), float(fixed_dt), float(dt_init), int(max_steps)),
           "cav_run_steps", sim)


def cav_sync(sim) -> None:
    _check(_lib.cav_sync(sim), "cav_sync", sim)


def cav_get_time(sim):
    t, dt = _d(), _d()
    _check(_lib.cav_get_time(sim, C.byref(t), C.byref(dt)), "cav_get_time", sim)
    return t.value, dt.value


def cav_set_time(sim, t: float) -> None:
    _check(_lib.cav_set_time(sim, float(t)), "cav_set_time", sim)


def cav_get_stats(sim) -> dict:
    st = cav_stats()
    _check(_lib.cav_get_stats(sim, C.byref(st)), "cav_get_stats", sim)
    return {k: getattr(st, k) for k, _ in cav_stats._fields_}


def cav_set_trace(sim, sample_dt: float, capacity: int) -> None:
    _check(_lib.cav_set_trace(sim, float(sample_dt), int(capacity)), "cav_set_trace", sim)


def cav_trace_row_len(sim) -> int:
    row = _i()
    _check(_lib.cav_trace_row_len(sim, C.byref(row)), "cav_trace_row_len", sim)
    return row.value


def cav_last_cuda_error(sim) -> str:
    return _lib.cav_last_cuda_error(sim).decode()


def cav_get_trace(sim) -> np.ndarray:
    row = _i(cav_trace_row_len(sim))
    n = _i()
    _check(_lib.cav_get_trace(sim, None, C.byref(n)), "cav_get_trace", sim)
    out = np.zeros((max(n.value, 1), row.value))
    _check(_lib.cav_get_trace(sim, out.ctypes.data_as(_dp), C.byref(n)), "cav_get_trace", sim)
    return out[:n.value].copy()


def cav_get_launch_count(sim) -> int:
    n = _ll()
    _check(_lib.cav_get_launch_count(sim, C.byref(n)), "cav_get_launch_count", sim)
    return n.value


# ----------------------------------------------------------------------------------------
# convenience: build a simulation from a problem description (still marshalling only)
# ----------------------------------------------------------------------------------------
class Sim:
    """RAII wrapper around a cav_sim handle."""

    def __init__(self, w, precision: str = "f32", renormalize: bool = True, overlap_norm: int = CAV_NORM_NCELLS,
                 stream: int | None = None, path: int | None = None):
        self.np_dtype = np.float32 if precision == "f32" else np.float64
        self.N, self.n_sub = int(np.asarray(w.omega).size), int(w.n_sub)
        self.shape_m = (self.n_sub, 3, w.nz, w.ny, w.nx)
        self.h = cav_create((w.nx, w.ny, w.nz, w.dx, w.dy, w.dz),
                            dict(Ms=w.Ms, Aex=w.Aex, Ku=w.Ku, ku_axis=w.ku_axis, alpha=w.alpha, gamma=w.gamma,
                                 B0=w.B0, n_sub=w.n_sub, B_exch_inter=w.B_exch_inter,
                                 precision=CAV_F32 if precision == "f32" else CAV_F64,
                                 renormalize=int(renormalize), overlap_norm=overlap_norm))
        if stream is not None:
            cav_set_stream(self.h, stream)
        if self.N:
            cav_set_modes(self.h, np.ascontiguousarray(w.u, dtype=self.np_dtype), w.omega, w.kappa, w.g, w.Gamma, w.Phi)
        else:
            cav_set_modes(self.h, None, None, None, None)
        cav_set_m(self.h, np.ascontiguousarray(w.m0, dtype=self.np_dtype))
        if self.N:
            cav_set_a(self.h, w.a0)
        if path is not None:
            cav_set_kernel_path(self.h, path)

    def close(self):
        if self.h:
            cav_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def get_m(self) -> np.ndarray:
        out = np.empty(self.shape_m, dtype=self.np_dtype)
        cav_get_m(self.h, out)
        return out

    def get_a(self) -> np.ndarray:
        return cav_get_a(self.h, self.N)


# ---------------------------------------------------------------------------------------------------------
# Sweeps of mid-size grids: a joint launcher over ordinary handles
# ---------------------------------------------------------------------------------------------------------
def cav_sweep_create(sims) -> int:
    """sims: sequence of cav_sim handles (ints) or Sim objects."""
    hs = [getattr(x, "h", x) for x in sims]
    arr = (_vp * len(hs))(*hs)
    out = _vp()
    _check(_lib.cav_sweep_create(arr, len(hs), C.byref(out)), "cav_sweep_create")
    return out.value


def cav_sweep_destroy(sweep) -> None:
    _check(_lib.cav_sweep_destroy(sweep), "cav_sweep_destroy")


def cav_sweep_run(sweep, t_end: float, tol: float = 0.0, fixed_dt: float = 0.0, dt_init: float = 0.0, max_steps: int = 0) -> None:
    _check(_lib.cav_sweep_run(sweep, float(t_end), float(tol), float(fixed_dt), float(dt_init), int(max_steps)), "cav_sweep_run")


# ---------------------------------------------------------------------------------------------------------
# Batched sweeps of small grids (include/cavmag.h): same names, marshalling only
# ---------------------------------------------------------------------------------------------------------
def cav_batch_create(grid, params, n_rep: int) -> int:
    g, p = _grid_params(grid, params)
    h = _vp()
    _check(_lib.cav_batch_create(C.byref(g), C.byref(p), int(n_rep), C.byref(h)), "cav_batch_create")
    _HANDLES[h.value] = (np.float32 if p.precision == CAV_F32 else np.float64, p.n_sub, g.nx * g.ny * g.nz, int(n_rep))
    return h.value


def cav_batch_destroy(b) -> None:
    _HANDLES.pop(b, None)
    _check(_lib.cav_batch_destroy(b), "cav_batch_destroy")


def cav_batch_set_stream(b, cuda_stream: int) -> None:
    _check(_lib.cav_batch_set_stream(b, _vp(cuda_stream)), "cav_batch_set_stream")


def cav_batch_set_field(b, B0) -> None:
    a = np.ascontiguousarray(np.asarray(B0, dtype=np.float64))
    _check(_lib.cav_batch_set_field(b, a.ctypes.data_as(_dp)), "cav_batch_set_field")


def cav_batch_set_modes(b, u, omega, kappa, g, Gamma=None, Phi=None, per_replica: bool = False) -> None:
    """u: host array [N][nz][ny][nx] in the batch precision; parameters [N] or [n_rep][N]."""
    om = np.asarray(omega, dtype=np.float64) if omega is not None else np.zeros(0)
    N = 0 if om.size == 0 else int(om.shape[-1])
    if N == 0:
        _check(_lib.cav_batch_set_modes(b, 0, None, None, None, None, None, None, 0), "cav_batch_set_modes")
        return
    n = om.size
    addr, _, keep = _ptr(u, *_field_spec(b, N, per_replica=False), what="u")
    po, ko = _darr(omega, n)
    pk, kk = _darr(kappa, n)
    pg, kg = _darr(g, n)
    pG, kG = _darr(Gamma, n)
    pP, kP = _darr(Phi, n)
    _check(_lib.cav_batch_set_modes(b, N, _vp(addr), po, pk, pg, pG, pP, int(bool(per_replica))), "cav_batch_set_modes")


def _drive_args(amp, t0, sigma, omega_d):
    if amp is None:
        return (None, None, None, None), ()
    a = np.ascontiguousarray(np.asarray(amp, dtype=np.complex128).reshape(-1)).view(np.float64)
    n = a.size // 2
    pt, kt = _darr(np.broadcast_to(np.asarray(t0, dtype=np.float64), (n,)), n)
    ps, ks = _darr(np.broadcast_to(np.asarray(sigma, dtype=np.float64), (n,)), n)
    pw, kw = _darr(None if omega_d is None else np.broadcast_to(np.asarray(omega_d, dtype=np.float64), (n,)), n)
    return (a.ctypes.data_as(_dp), pt, ps, pw), (a, kt, ks, kw)


def _back_args(g_b, Gamma_b, Phi_b):
    if g_b is None:
        return (None, None, None), ()
    n = int(np.asarray(g_b).size)
    pg, kg = _darr(g_b, n)
    pG, kG = _darr(Gamma_b, n)
    pP, kP = _darr(Phi_b, n)
    return (pg, pG, pP), (kg, kG, kP)


def cav_set_backaction(sim, g_b, Gamma_b=None, Phi_b=None) -> None:
    """Backward coupling of the feedback field ([N] arrays; g_b None = reciprocal again)."""
    args, keep = _back_args(g_b, Gamma_b, Phi_b)
    _check(_lib.cav_set_backaction(sim, *args), "cav_set_backaction", sim)


def cav_batch_set_backaction(b, g_b, Gamma_b=None, Phi_b=None) -> None:
    args, keep = _back_args(g_b, Gamma_b, Phi_b)
    _check(_lib.cav_batch_set_backaction(b, *args), "cav_batch_set_backaction")


def _pol_args(pol, quad):
    if pol is None:
        return (None, None), ()
    p = np.ascontiguousarray(np.asarray(pol, dtype=np.float64).reshape(-1, 3))
    q = None if quad is None else np.ascontiguousarray(np.asarray(quad, dtype=np.float64).reshape(-1, 3))
    if q is not None and q.shape != p.shape:
        raise ValueError("quad must have the shape of pol")
    return (p.ctypes.data_as(_dp), None if q is None else q.ctypes.data_as(_dp)), (p, q)


def cav_set_polarisation(sim, pol, quad=None) -> None:
    """pol [N][3] (None: x^ again), quad [N][3] or None (z^ x p)."""
    args, keep = _pol_args(pol, quad)
    _check(_lib.cav_set_polarisation(sim, *args), "cav_set_polarisation", sim)


def cav_batch_set_polarisation(b, pol, quad=None) -> None:
    args, keep = _pol_args(pol, quad)
    _check(_lib.cav_batch_set_polarisation(b, *args), "cav_batch_set_polarisation")


def cav_set_integrator(sim, integrator: int, n_llg: int = 1) -> None:
    _check(_lib.cav_set_integrator(sim, int(integrator), int(n_llg)), "cav_set_integrator", sim)


def cav_batch_set_integrator(b, integrator: int, n_llg: int = 1) -> None:
    _check(_lib.cav_batch_set_integrator(b, int(integrator), int(n_llg)), "cav_batch_set_integrator")


def cav_set_demag(sim, on: int) -> None:
    _check(_lib.cav_set_demag(sim, int(on)), "cav_set_demag", sim)


def cav_set_spectrum(sim, n_bins: int, omega_lo: float = 0.0, omega_hi: float = 0.0) -> None:
    _check(_lib.cav_set_spectrum(sim, int(n_bins), float(omega_lo), float(omega_hi)), "cav_set_spectrum", sim)


def cav_get_spectrum(sim, n_bins: int, N: int):
    """Returns (X [n_bins][2N + n_sub] complex, n_samples): columns a_1..a_N, S_1..S_N, then <m_s,x> - i <m_s,y> per sublattice."""
    out = np.zeros((n_bins, 2 * N + _HANDLES[sim][1], 2))
    n = _ll()
    _check(_lib.cav_get_spectrum(sim, out.ctypes.data_as(_dp), C.byref(n)), "cav_get_spectrum", sim)
    return out[..., 0] + 1j * out[..., 1], n.value


def cav_batch_set_spectrum(b, n_bins: int, omega_lo: float = 0.0, omega_hi: float = 0.0) -> None:
    _check(_lib.cav_batch_set_spectrum(b, int(n_bins), float(omega_lo), float(omega_hi)), "cav_batch_set_spectrum")


def cav_batch_get_spectrum(b, n_rep: int, n_bins: int, N: int):
    """Returns (X [n_rep][n_bins][2N + n_sub] complex, n_samples [n_rep])."""
    out = np.zeros((n_rep, n_bins, 2 * N + _HANDLES[b][1], 2))
    ns = (_ll * n_rep)()
    _check(_lib.cav_batch_get_spectrum(b, out.ctypes.data_as(_dp), ns), "cav_batch_get_spectrum")
    return out[..., 0] + 1j * out[..., 1], np.array(list(ns))


def cav_set_drive(sim, amp, t0=None, sigma=None, omega_d=None) -> None:
    """amp [N] complex or None (off); t0, sigma [N] or scalars; omega_d [N], scalar or None."""
    args, keep = _drive_args(amp, t0, sigma, omega_d)
    _check(_lib.cav_set_drive(sim, *args), "cav_set_drive", sim)


def cav_batch_set_drive(b, amp, t0=None, sigma=None, omega_d=None) -> None:
    args, keep = _drive_args(amp, t0, sigma, omega_d)
    _check(_lib.cav_batch_set_drive(b, *args), "cav_batch_set_drive")


def cav_batch_set_m(b, m: np.ndarray, per_replica: bool = False) -> None:
    addr, _, keep = _ptr(m, *_field_spec(b, per_replica=bool(per_replica)), what="m")
    _check(_lib.cav_batch_set_m(b, _vp(addr), int(bool(per_replica))), "cav_batch_set_m")


def cav_batch_set_a(b, a, per_replica: bool = False) -> None:
    arr = np.ascontiguousarray(np.asarray(a, dtype=np.complex128)).view(np.float64)
    _check(_lib.cav_batch_set_a(b, arr.ctypes.data_as(_dp), int(bool(per_replica))), "cav_batch_set_a")


def cav_batch_set_trace(b, sample_dt: float, capacity: int) -> None:
    _check(_lib.cav_batch_set_trace(b, float(sample_dt), int(capacity)), "cav_batch_set_trace")


def cav_batch_trace_row_len(b) -> int:
    n = _i()
    _check(_lib.cav_batch_trace_row_len(b, C.byref(n)), "cav_batch_trace_row_len")
    return n.value


def cav_batch_run(b, t_end: float, tol: float = 0.0, fixed_dt: float = 0.0, dt_init: float = 0.0, max_steps: int = 0) -> None:
    _check(_lib.cav_batch_run(b, float(t_end), float(tol), float(fixed_dt), float(dt_init), int(max_steps)), "cav_batch_run")


def cav_batch_get_m(b, out: np.ndarray) -> None:
    addr, _, keep = _ptr(out, *_field_spec(b), what="m_out")
    _check(_lib.cav_batch_get_m(b, _vp(addr)), "cav_batch_get_m")


def cav_batch_get_a(b, n_rep: int, N: int) -> np.ndarray:
    out = np.zeros((n_rep, max(N, 0), 2), dtype=np.float64)
    _check(_lib.cav_batch_get_a(b, out.ctypes.data_as(_dp) if N else None), "cav_batch_get_a")
    return out[..., 0] + 1j * out[..., 1]


def cav_batch_get_stats(b, n_rep: int) -> list:
    arr = (cav_stats * n_rep)()
    _check(_lib.cav_batch_get_stats(b, arr), "cav_batch_get_stats")
    return [{k: getattr(st, k) for k, _ in cav_stats._fields_} for st in arr]


def cav_batch_get_trace(b, n_rep: int, capacity: int) -> list:
    """Per replica: array [n_samples][row_len]."""
    rl = cav_batch_trace_row_len(b)
    out = np.zeros((n_rep, max(capacity, 1), rl), dtype=np.float64)
    ns = (_i * n_rep)()
    _check(_lib.cav_batch_get_trace(b, out.ctypes.data_as(_dp) if capacity > 0 else None, ns), "cav_batch_get_trace")
    return [out[r, :ns[r]].copy() for r in range(n_rep)]


class Batch:
    """RAII wrapper around a cav_batch handle: n_rep replicas of workload w that differ in B0 (and optionally in the
    mode parameters)."""

    def __init__(self, w, n_rep: int, precision: str = "f64", B0=None, renormalize: bool = True,
                 overlap_norm: int = CAV_NORM_NCELLS, stream: int | None = None):
        self.np_dtype = np.float32 if precision == "f32" else np.float64
        self.n_rep, self.N, self.n_sub = int(n_rep), int(np.asarray(w.omega).size), int(w.n_sub)
        self.shape_m = (self.n_rep, self.n_sub, 3, w.nz, w.ny, w.nx)
        self.h = cav_batch_create((w.nx, w.ny, w.nz, w.dx, w.dy, w.dz),
                                  dict(Ms=w.Ms, Aex=w.Aex, Ku=w.Ku, ku_axis=w.ku_axis, alpha=w.alpha, gamma=w.gamma,
                                       B0=w.B0, n_sub=w.n_sub, B_exch_inter=w.B_exch_inter,
                                       precision=CAV_F32 if precision == "f32" else CAV_F64,
                                       renormalize=int(renormalize), overlap_norm=overlap_norm), n_rep)
        if stream is not None:
            cav_batch_set_stream(self.h, stream)
        if B0 is not None:
            cav_batch_set_field(self.h, B0)
        if self.N:
            cav_batch_set_modes(self.h, np.ascontiguousarray(w.u, dtype=self.np_dtype), w.omega, w.kappa, w.g, w.Gamma, w.Phi)
        cav_batch_set_m(self.h, np.ascontiguousarray(w.m0, dtype=self.np_dtype))
        if self.N:
            cav_batch_set_a(self.h, w.a0)

    def close(self):
        if self.h:
            cav_batch_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def run(self, t_end, tol=0.0, fixed_dt=0.0, dt_init=0.0, max_steps=0):
        cav_batch_run(self.h, t_end, tol, fixed_dt, dt_init, max_steps)

    def get_m(self) -> np.ndarray:
        out = np.empty(self.shape_m, dtype=self.np_dtype)
        cav_batch_get_m(self.h, out)
        return out

    def get_a(self) -> np.ndarray:
        return cav_batch_get_a(self.h, self.n_rep, self.N)

    def stats(self) -> list:
        return cav_batch_get_stats(self.h, self.n_rep)
