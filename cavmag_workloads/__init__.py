"""Seeded synthetic inputs for the cavity-magnonics hot path (inputs ONLY).

This module is the one thing the fp64 CPU oracle (``oracle/``) and the CUDA path
(``paper_2603_03706_b200/``) share.  It holds none of the method's arithmetic: no
effective field, no LLG torque, no overlap, no Runge-Kutta.  It only *describes*
problems (grid, material constants, mode tables) and *draws* the seeded arrays the
method consumes (initial magnetisation, mode profiles u_n(r), initial amplitudes).

The five workloads follow ``BASELINE.json`` ``configs[0..4]`` with the gaps filled as
SURVEY.md section 8(c) G20 / section 8(d) state (recipe restated in DESIGN.md):

    cfg1a / cfg1b  8x8x8, 5 nm, YIG, one uniform mode           (PAPER.md:217 material family)
    cfg2           64x64x16, 5 nm, two sin(n pi x/Lx) modes      (Eq. 11 profiles)
    cfg3           256x256x32, 4 nm, 8 random smooth modes, Ku   (the roofline target)
    cfg4           128x128x64, 2 nm, two-sublattice AFM
    cfg5           512x512x64, 5 nm, 32 modes, mixed coupling    (Eq. 19)

Random numbers come from one counter-based generator (SplitMix64 applied to
``seed, stream, index``), so any element can be regenerated independently and the
same values reach both implementations.  No public dataset is involved: the paper uses
none (all its inputs are analytic), so these synthetic inputs *are* the workload.
"""
from __future__ import annotations

import dataclasses
import math
from typing import Optional

import numpy as np

TWO_PI = 2.0 * math.pi
GAMMA = 1.76e11  # rad/(s T)

_M64 = (1 << 64) - 1


# ----------------------------------------------------------------------------------------
# counter-based RNG
# ----------------------------------------------------------------------------------------
def splitmix64(x: np.ndarray) -> np.ndarray:
    """SplitMix64 finaliser on uint64 counters (vectorised)."""
    x = np.asarray(x, dtype=np.uint64)
    with np.errstate(over="ignore"):
        x = x + np.uint64(0x9E3779B97F4A7C15)
        z = x
        z = (z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
        z = (z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
        z = z ^ (z >> np.uint64(31))
    return z


def uniform01(seed: int, stream: int, n: int, offset: int = 0) -> np.ndarray:
    """n doubles in [0,1): element i depends only on (seed, stream, offset+i)."""
    base = splitmix64(np.array([(seed * 0x100000001B3 + stream * 0x9E3779B1) & _M64], dtype=np.uint64))[0]
    idx = np.arange(offset, offset + n, dtype=np.uint64)
    with np.errstate(over="ignore"):
        bits = splitmix64(idx * np.uint64(0xD1342543DE82EF95) + base)
    return (bits >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)


# ----------------------------------------------------------------------------------------
# problem description
# ----------------------------------------------------------------------------------------
@dataclasses.dataclass
class Workload:
    """A fully specified problem instance.  Arrays are fp64 numpy, C-contiguous.

    Layouts (x fastest):  m0[n_sub][3][nz][ny][nx],  u[N][nz][ny][nx],  a0[N] complex.
    Rates are angular (rad/s), fields in tesla, lengths in metres.
    """
    name: str
    nx: int
    ny: int
    nz: int
    dx: float
    dy: float
    dz: float
    Ms: float
    Aex: float
    Ku: float
    ku_axis: tuple
    alpha: float
    gamma: float
    B0: tuple
    n_sub: int
    B_exch_inter: float
    omega: np.ndarray
    kappa: np.ndarray
    g: np.ndarray
    Gamma: np.ndarray
    Phi: np.ndarray
    u: np.ndarray
    m0: np.ndarray
    a0: np.ndarray
    t_end: float
    tol: float            # adaptive tolerance of the config (0 if the config is fixed-step)
    fixed_dt: float       # fixed step of the config (0 if adaptive only)
    precision: str        # "f32" | "f64": the precision the config is quoted in
    note: str = ""

    @property
    def n_cells(self) -> int:
        return self.nx * self.ny * self.nz

    @property
    def n_modes(self) -> int:
        return int(self.omega.shape[0])


def b0_for_ghz(f_ghz: float, gamma: float = GAMMA) -> float:
    """Static field (T) that puts the Kittel line gamma*B0/2pi at f_ghz (Eq. 9)."""
    return TWO_PI * f_ghz * 1e9 / gamma


# ----------------------------------------------------------------------------------------
# seeded arrays
# ----------------------------------------------------------------------------------------
def tilted_state(seed: int, stream: int, nx: int, ny: int, nz: int, max_tilt: float,
                 per_cell: bool = True, sign: float = 1.0) -> np.ndarray:
    """Unit vectors tilted away from sign*z by theta~U(0,max_tilt), phi~U(0,2pi).

    Returns [3][nz][ny][nx].  per_cell=False applies ONE draw to every cell (the state is
    then bit-uniform; SURVEY.md G24 case 1a).
    """
    n = nx * ny * nz
    if per_cell:
        th = uniform01(seed, stream, n) * max_tilt
        ph = uniform01(seed, stream + 1, n) * TWO_PI
    else:
        th = np.full(n, uniform01(seed, stream, 1)[0] * max_tilt)
        ph = np.full(n, uniform01(seed, stream + 1, 1)[0] * TWO_PI)
    m = np.empty((3, n), dtype=np.float64)
    m[0] = np.sin(th) * np.cos(ph)
    m[1] = np.sin(th) * np.sin(ph)
    m[2] = sign * np.cos(th)
    return m.reshape(3, nz, ny, nx)


def cell_centres(n: int) -> np.ndarray:
    """Cell-centre coordinate over the box length, (i+1/2)/n."""
    return (np.arange(n, dtype=np.float64) + 0.5) / n


def sine_profile_x(n_mode: int, nx: int, ny: int, nz: int) -> np.ndarray:
    """u(r) = sin(n pi x / Lx) on cell centres, constant in y,z (cfg2)."""
    s = np.sin(n_mode * math.pi * cell_centres(nx))
    return np.broadcast_to(s[None, None, :], (nz, ny, nx)).copy()


def cosine_profile(nmx: int, nmy: int, nmz: int, nx: int, ny: int, nz: int) -> np.ndarray:
    """Rectangular-cavity standing wave of PAPER.md:108 (Eq. 11) on cell centres."""
    cx = np.cos(nmx * math.pi * cell_centres(nx))
    cy = np.cos(nmy * math.pi * cell_centres(ny))
    cz = np.cos(nmz * math.pi * cell_centres(nz))
    return (cz[:, None, None] * cy[None, :, None] * cx[None, None, :]).copy()


def random_smooth_profiles(seed: int, n_modes: int, nx: int, ny: int, nz: int,
                           dtype=np.float64) -> np.ndarray:
    """n_modes profiles, each a seeded sum of 4 low-order 3-D sine harmonics, max|u| = 1.

    u_n = sum_{h=1..4} c_h sin(p_h pi x/Lx) sin(q_h pi y/Ly) sin(r_h pi z/Lz),
    p,q,r in {1,2,3}, c_h ~ U(-1,1)   (BASELINE.json configs[2], configs[4]).
    """
    sx = np.stack([np.sin(p * math.pi * cell_centres(nx)) for p in (1, 2, 3)])
    sy = np.stack([np.sin(p * math.pi * cell_centres(ny)) for p in (1, 2, 3)])
    sz = np.stack([np.sin(p * math.pi * cell_centres(nz)) for p in (1, 2, 3)])
    out = np.empty((n_modes, nz, ny, nx), dtype=dtype)
    for n in range(n_modes):
        r = uniform01(seed, 100 + n, 16)
        acc = np.zeros((nz, ny, nx), dtype=np.float64)
        for h in range(4):
            c = 2.0 * r[4 * h] - 1.0
            p = int(r[4 * h + 1] * 3.0)
            q = int(r[4 * h + 2] * 3.0)
            s = int(r[4 * h + 3] * 3.0)
            acc += c * (sz[s][:, None, None] * sy[q][None, :, None] * sx[p][None, None, :])
        acc /= np.max(np.abs(acc))
        out[n] = acc
    return out


# ----------------------------------------------------------------------------------------
# the five configurations
# ----------------------------------------------------------------------------------------
_YIG = dict(Ms=140e3, Aex=3.7e-12, gamma=GAMMA)


def _modes(f_ghz, g_mhz, kappa_mhz, Gamma_mhz=None, Phi=None):
    f = np.atleast_1d(np.asarray(f_ghz, dtype=np.float64))
    n = f.shape[0]
    g = np.broadcast_to(np.asarray(g_mhz, dtype=np.float64), (n,)).copy()
    k = np.broadcast_to(np.asarray(kappa_mhz, dtype=np.float64), (n,)).copy()
    G = np.zeros(n) if Gamma_mhz is None else np.broadcast_to(np.asarray(Gamma_mhz, dtype=np.float64), (n,)).copy()
    P = np.zeros(n) if Phi is None else np.broadcast_to(np.asarray(Phi, dtype=np.float64), (n,)).copy()
    return dict(omega=TWO_PI * f * 1e9, kappa=TWO_PI * k * 1e6, g=TWO_PI * g * 1e6,
                Gamma=TWO_PI * G * 1e6, Phi=P)


def cfg1(variant: str = "b", n: int = 8, seed: int = 1000) -> Workload:
    """Tiny ferromagnet (BASELINE.json configs[0]).  variant 'a': one tilt for all cells,
    fixed dt 0.5 ps; variant 'b': per-cell tilt, fixed dt 0.2 ps."""
    per_cell = variant == "b"
    m0 = tilted_state(seed, 1, n, n, n, 0.01, per_cell=per_cell)[None]
    md = _modes([10.0], 10.0, 1.0)
    return Workload(
        name=f"cfg1{variant}", nx=n, ny=n, nz=n, dx=5e-9, dy=5e-9, dz=5e-9,
        Ku=0.0, ku_axis=(0.0, 0.0, 1.0), alpha=1e-3, B0=(0.0, 0.0, b0_for_ghz(10.0)),
        n_sub=1, B_exch_inter=0.0, u=np.ones((1, n, n, n)), m0=m0, a0=np.zeros(1, dtype=np.complex128),
        t_end=20e-9, tol=1e-8, fixed_dt=(0.2e-12 if per_cell else 0.5e-12), precision="f64",
        note="cfg1a: uniform tilt, dt 0.5 ps; cfg1b: per-cell tilt, dt 0.2 ps", **_YIG, **md)


def cfg2(f_kittel_ghz: float = 10.0, nx: int = 64, ny: int = 64, nz: int = 16, seed: int = 2000) -> Workload:
    """YIG slab, two sine modes (BASELINE.json configs[1]); one point of the 41-field sweep."""
    m0 = tilted_state(seed, 1, nx, ny, nz, 0.01)[None]
    u = np.stack([sine_profile_x(1, nx, ny, nz), sine_profile_x(2, nx, ny, nz)])
    md = _modes([9.8, 10.2], 15.0, 2.0)
    return Workload(
        name="cfg2", nx=nx, ny=ny, nz=nz, dx=5e-9, dy=5e-9, dz=5e-9,
        Ku=0.0, ku_axis=(0.0, 0.0, 1.0), alpha=1e-4, B0=(0.0, 0.0, b0_for_ghz(f_kittel_ghz)),
        n_sub=1, B_exch_inter=0.0, u=u, m0=m0, a0=np.zeros(2, dtype=np.complex128),
        t_end=50e-9, tol=1e-6, fixed_dt=0.2e-12, precision="f32", **_YIG, **md)


def cfg2_sweep_ghz() -> np.ndarray:
    """The 41 Kittel frequencies of the cfg2 field sweep."""
    return np.linspace(9.6, 10.4, 41)


def _multimode(name, nx, ny, nz, cell, n_modes, seed, tilt, mixed, t_end, dtype=np.float64) -> Workload:
    m0 = tilted_state(seed, 1, nx, ny, nz, tilt)[None]
    u = random_smooth_profiles(seed, n_modes, nx, ny, nz, dtype=dtype)
    f = np.linspace(9.0, 11.0, n_modes)
    g = 5.0 + 15.0 * uniform01(seed, 50, n_modes)
    Gam = np.zeros(n_modes)
    Phi = np.zeros(n_modes)
    if mixed:  # odd n (1-based) coherent; even n: Gamma = g/2, Phi = pi/2
        even = (np.arange(1, n_modes + 1) % 2) == 0
        Gam[even] = 0.5 * g[even]
        Phi[even] = 0.5 * math.pi
    md = _modes(f, g, 1.0, Gam, Phi)
    return Workload(
        name=name, nx=nx, ny=ny, nz=nz, dx=cell, dy=cell, dz=cell,
        Ku=1e3, ku_axis=(1.0, 0.0, 0.0), alpha=1e-3 if not mixed else 1e-3,
        B0=(0.0, 0.0, b0_for_ghz(10.0)), n_sub=1, B_exch_inter=0.0, u=u, m0=m0,
        a0=np.zeros(n_modes, dtype=np.complex128), t_end=t_end, tol=1e-6, fixed_dt=0.0,
        precision="f32", **_YIG, **md)


def cfg3(nx: int = 256, ny: int = 256, nz: int = 32, seed: int = 3000, dtype=np.float64) -> Workload:
    """Multimode large film, 8 modes, Ku along x (BASELINE.json configs[2]): the roofline target."""
    return _multimode("cfg3", nx, ny, nz, 4e-9, 8, seed, 0.01, False, 10e-9, dtype)


def cfg5(nx: int = 512, ny: int = 512, nz: int = 64, seed: int = 5000, dtype=np.float32) -> Workload:
    """Throughput stress, 32 modes mixing coherent and dissipative coupling (configs[4])."""
    return _multimode("cfg5", nx, ny, nz, 5e-9, 32, seed, 0.05, True, 2e-9, dtype)


def afmr_omega(gamma: float, B_E: float, B_A: float) -> float:
    """Zero-field AFMR line of PAPER.md:134 (Eq. 15), used only to *tune the input* omega_c."""
    return gamma * math.sqrt(2.0 * B_E * B_A + B_A * B_A)


def cfg4(nx: int = 128, ny: int = 128, nz: int = 64, seed: int = 4000, dissipative: bool = False) -> Workload:
    """Two-sublattice antiferromagnet (BASELINE.json configs[3])."""
    Ms, Ku, B_E = 400e3, 50e3, 50.0
    m1 = tilted_state(seed, 1, nx, ny, nz, 0.01, sign=+1.0)
    m2 = tilted_state(seed, 3, nx, ny, nz, 0.01, sign=-1.0)
    wc = afmr_omega(GAMMA, B_E, 2.0 * Ku / Ms)
    md = _modes([wc / TWO_PI / 1e9], 1000.0, 500.0,
                [500.0] if dissipative else None, [0.5 * math.pi] if dissipative else None)
    return Workload(
        name="cfg4d" if dissipative else "cfg4", nx=nx, ny=ny, nz=nz, dx=2e-9, dy=2e-9, dz=2e-9,
        Ms=Ms, Aex=10e-12, Ku=Ku, ku_axis=(0.0, 0.0, 1.0), alpha=1e-3, gamma=GAMMA, B0=(0.0, 0.0, 0.0),
        n_sub=2, B_exch_inter=B_E, u=np.ones((1, nz, ny, nx)), m0=np.stack([m1, m2]),
        a0=np.zeros(1, dtype=np.complex128), t_end=2e-9, tol=1e-6, fixed_dt=0.0, precision="f32", **md)


def by_name(name: str, **kw) -> Workload:
    table = {"cfg1a": lambda **k: cfg1("a", **k), "cfg1b": lambda **k: cfg1("b", **k), "cfg2": cfg2,
             "cfg3": cfg3, "cfg4": cfg4, "cfg4d": lambda **k: cfg4(dissipative=True, **k), "cfg5": cfg5}
    return table[name](**kw)


def macrospin(f_kittel_ghz: float, f_c_ghz, g_mhz, kappa_mhz, alpha: float, a0=None,
              tilt: float = 0.0, Gamma_mhz=None, Phi=None, n: int = 2) -> Workload:
    """A bit-uniform n^3 ferromagnet with uniform modes: the lumped model of PAPER.md:43-65."""
    md = _modes(f_c_ghz, g_mhz, kappa_mhz, Gamma_mhz, Phi)
    N = md["omega"].shape[0]
    m0 = np.zeros((1, 3, n, n, n))
    m0[0, 0] = math.sin(tilt)
    m0[0, 2] = math.cos(tilt)
    a = np.zeros(N, dtype=np.complex128) if a0 is None else np.asarray(a0, dtype=np.complex128).reshape(N)
    return Workload(
        name="macrospin", nx=n, ny=n, nz=n, dx=5e-9, dy=5e-9, dz=5e-9, Ku=0.0, ku_axis=(0.0, 0.0, 1.0),
        alpha=alpha, B0=(0.0, 0.0, b0_for_ghz(f_kittel_ghz)), n_sub=1, B_exch_inter=0.0,
        u=np.ones((N, n, n, n)), m0=m0, a0=a, t_end=0.0, tol=0.0, fixed_dt=0.0, precision="f64",
        **_YIG, **md)
