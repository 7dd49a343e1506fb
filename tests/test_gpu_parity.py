"""GPU-vs-oracle parity (-m gpu): every test calls the CUDA path through the C ABI
(paper_2603_03706_b200.api -> libcavmag.so) and compares it with the fp64 CPU oracle element by
element on the same seeded inputs.

Bars (BASELINE.json north_star, reading G23):
  fixed step, fp64:  per component c: max_r |dm_c| <= 1e-10 * max_r |m_c^ref|;  |da_n| <= 1e-10 |a_n^ref|
  fixed step, fp32:  |dm| <= 1e-4 absolute;  | |a_n| - |a_n^ref| | <= 1e-4 |a_n^ref|
  adaptive:          observables (polariton frequencies within 1 MHz, Rabi period within 0.5 %)
"""
import math

import numpy as np
import pytest

import cavmag_workloads as W
from observables import fit_exponentials, dominant, rabi_period

pytestmark = pytest.mark.gpu

TWO_PI = 2 * math.pi
GAMMA = 1.76e11


@pytest.fixture(scope="module")
def api():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2603_03706_b200 import api as a      # raises if libcavmag.so is missing: no fallback
    return a


def oracle_of(w, **kw):
    from oracle import Oracle
    return Oracle(w, **kw)


PATHS = ["generic", "tma", "block", "coop"]


def open_sim(api, w, prec, path, **kw):
    """A Sim forced onto one implementation of the step: the generic or the TMA stage kernels, or the single-block
    integrator of grids up to 1024 cells (CAV_PATH_BLOCK), or the cooperative multi-block variant of it (CAV_PATH_COOP).
    Skips when the path is not eligible for this shape (TMA: nx*sizeof(T) not a multiple of 16 bytes; BLOCK: more than 1024
    cells; COOP: 1024 cells or fewer)."""
    sim = api.Sim(w, precision=prec, **kw)
    want = {"tma": api.CAV_PATH_TMA, "generic": api.CAV_PATH_GENERIC, "block": api.CAV_PATH_BLOCK, "coop": api.CAV_PATH_COOP}[path]
    try:
        api.cav_set_kernel_path(sim.h, want)
    except api.CavError as e:
        sim.close()
        assert e.status == api.CAV_E_UNSUPPORTED and path in ("tma", "block", "coop")
        if path == "coop":
            nc = w.nx * w.ny * w.nz
            assert nc <= 1024 or nc > 512 * 132, "COOP path refused although the grid is in its range"
            pytest.skip("cooperative path: grid outside 1025 .. 512 x SMs cells")
        if path == "block":
            assert w.nx * w.ny * w.nz > 1024, "BLOCK path refused although the grid has at most 1024 cells"
            pytest.skip("single-block path: grid too large")
        es = 4 if prec == "f32" else 8
        assert (w.nx * es) % 16 != 0, "TMA path refused although the row pitch is 16-byte aligned"
        pytest.skip("TMA kernel not eligible for this shape")
    assert api.cav_get_kernel_path(sim.h) == want
    return sim


def small_problem(nx, ny, nz, N, n_sub=1, seed=7, tilt=0.3, mixed=True, ku=2e3, dt_cells=(4e-9, 5e-9, 6e-9)):
    u = W.random_smooth_profiles(seed, max(N, 1), nx, ny, nz)[:N]
    if N:
        u[0] = 1.0       # one uniform mode so that the overlap of m ~ z^ + tilt is not tiny
    m0 = np.stack([W.tilted_state(seed, 1 + 2 * s, nx, ny, nz, tilt, sign=(1.0 if s == 0 else -1.0)) for s in range(n_sub)])
    f = np.linspace(9.0, 11.0, N) if N else np.zeros(0)
    g = 20.0 + 30.0 * W.uniform01(seed, 50, N)
    Gam = np.where(np.arange(N) % 2 == 1, 0.5 * g, 0.0) if mixed else np.zeros(N)
    Phi = np.where(np.arange(N) % 2 == 1, 1.1, 0.0) if mixed else np.zeros(N)
    md = W._modes(f, g, 5.0, Gam, Phi) if N else dict(omega=np.zeros(0), kappa=np.zeros(0), g=np.zeros(0), Gamma=np.zeros(0), Phi=np.zeros(0))
    a0 = (0.02 * (W.uniform01(seed, 60, N) - 0.5) + 0.02j * (W.uniform01(seed, 61, N) - 0.5)).astype(np.complex128)
    return W.Workload(name="small", nx=nx, ny=ny, nz=nz, dx=dt_cells[0], dy=dt_cells[1], dz=dt_cells[2], Ms=140e3,
                      Aex=3.7e-12, Ku=ku, ku_axis=(1.0, 0.5, 0.2), alpha=0.02, gamma=GAMMA, B0=(0.01, -0.02, 0.35),
                      n_sub=n_sub, B_exch_inter=(3.0 if n_sub == 2 else 0.0), u=u, m0=m0, a0=a0,
                      t_end=0, tol=0, fixed_dt=0, precision="f64", **md)


def assert_parity(m, a, ref, prec):
    if prec == "f64":
        for s in range(ref.m.shape[0]):
            for c in range(3):
                scale = np.abs(ref.m[s, c]).max()
                assert np.abs(m[s, c] - ref.m[s, c]).max() <= 1e-10 * scale, (s, c)
        for n in range(ref.a.shape[0]):
            assert abs(a[n] - ref.a[n]) <= 1e-10 * abs(ref.a[n]), n
    else:
        assert np.abs(m.astype(np.float64) - ref.m).max() <= 1e-4
        for n in range(ref.a.shape[0]):
            assert abs(abs(a[n]) - abs(ref.a[n])) <= 1e-4 * abs(ref.a[n]), n


# ----------------------------------------------------------------------------------------
# right-hand side, cell by cell
# ----------------------------------------------------------------------------------------
@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("shape,N,n_sub", [
    ((8, 8, 8), 1, 1),        # cfg1 shape
    ((40, 9, 7), 3, 1),       # several blocks + ragged tail, N between buckets
    ((13, 5, 3), 2, 1),       # nx not a multiple of the vector width -> scalar kernels
    ((12, 6, 5), 8, 1),       # rows shorter than a warp
    ((36, 10, 5), 9, 1),      # N = 9 -> 32-mode bucket
    ((64, 4, 3), 32, 1),      # max modes
    ((24, 6, 4), 0, 1),       # plain LLG
    ((20, 7, 6), 1, 2),       # antiferromagnet
    ((1, 1, 1), 1, 1),        # degenerate: a single cell
    ((2, 1, 9), 2, 2),        # thin in x,y
    ((72, 19, 5), 3, 1),      # TMA: two x tiles (ragged), three y tiles (ragged)
    ((132, 9, 11), 8, 1),     # TMA: three x tiles, the last 4 cells wide
    ((68, 17, 6), 1, 2),      # TMA: antiferromagnet, ragged in x and y
    ((4, 2, 40), 2, 1),       # TMA: one tile, long z march
])
@pytest.mark.parametrize("path", PATHS)
def test_rhs_matches_oracle(api, prec, shape, N, n_sub, path):
    w = small_problem(*shape, N, n_sub)
    dm_ref, da_ref, S_ref = oracle_of(w).rhs(w.m0, w.a0)
    with open_sim(api, w, prec, path) as sim:
        dm = np.empty(sim.shape_m, dtype=sim.np_dtype)
        api.cav_get_dmdt(sim.h, dm)
        da = api.cav_get_dadt(sim.h, N)
        S = api.cav_get_overlaps(sim.h, N)
    scale = np.abs(dm_ref).max()
    if prec == "f64":
        assert np.abs(dm - dm_ref).max() <= 2e-13 * scale
        if N:
            assert np.abs(S - S_ref).max() <= 1e-14
            assert np.abs(da - da_ref).max() <= 1e-13 * max(np.abs(da_ref).max(), 1.0)
    else:
        # fp32 inputs are rounded on upload: compare against the oracle evaluated on the same rounded inputs
        w32 = small_problem(*shape, N, n_sub)
        w32.m0 = w.m0.astype(np.float32).astype(np.float64)
        w32.m0 /= np.linalg.norm(w32.m0, axis=1, keepdims=True)
        w32.u = w.u.astype(np.float32).astype(np.float64)
        dm_ref, da_ref, S_ref = oracle_of(w32).rhs(w32.m0, w32.a0)
        assert np.abs(dm - dm_ref).max() <= 2e-5 * scale
        if N:
            assert np.abs(S - S_ref).max() <= 2e-6
            assert np.abs(da - da_ref).max() <= 2e-5 * max(np.abs(da_ref).max(), 1.0)


# ----------------------------------------------------------------------------------------
# fixed-step parity after 1000 steps (north_star)
# ----------------------------------------------------------------------------------------
@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("variant", ["a", "b"])
@pytest.mark.parametrize("path", PATHS)
def test_cfg1_fixed_1000_steps(api, prec, variant, path):
    w = W.cfg1(variant)
    if prec == "f32":
        w.m0 = w.m0.astype(np.float32).astype(np.float64)
    ref = oracle_of(w).run(w.m0, w.a0, fixed_dt=w.fixed_dt, max_steps=1000)
    with open_sim(api, w, prec, path) as sim:
        api.cav_run_steps(sim.h, math.inf, fixed_dt=w.fixed_dt, max_steps=1000)
        m, a = sim.get_m(), sim.get_a()
        st = api.cav_get_stats(sim.h)
    assert st["accepted"] == 1000 and st["rejected"] == 0 and st["rhs_evals"] == 6001
    assert abs(st["t"] - ref.t) <= 1e-24
    assert_parity(m, a, ref, prec)
    if variant == "a" and prec == "f64":
        assert np.abs(m - m[:, :, :1, :1, :1]).max() < 1e-13      # stays uniform


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("shape,N,n_sub,dt", [
    ((40, 9, 7), 3, 1, 0.1e-12),
    ((13, 5, 3), 2, 1, 0.1e-12),
    ((36, 10, 5), 9, 1, 0.1e-12),
    ((20, 7, 6), 1, 2, 0.05e-12),
    ((16, 8, 4), 2, 2, 0.05e-12),
    ((72, 19, 5), 3, 1, 0.1e-12),
    ((132, 9, 11), 8, 1, 0.1e-12),
    ((68, 17, 6), 1, 2, 0.05e-12),
    ((64, 8, 3), 32, 1, 0.1e-12),
    ((24, 6, 4), 0, 1, 0.1e-12),       # plain LLG: no modes to finish between the stages
    ((96, 20, 14), 0, 1, 0.1e-12),     # the same beyond the single-block range
])
@pytest.mark.parametrize("path", PATHS)
def test_busy_fixed_steps(api, prec, shape, N, n_sub, dt, path):
    """All terms on (off-axis field and anisotropy, profiled modes, mixed coupling, damping, AFM)."""
    w = small_problem(*shape, N, n_sub, tilt=0.2)
    if prec == "f32":
        w.m0 = w.m0.astype(np.float32).astype(np.float64)
        w.m0 /= np.linalg.norm(w.m0, axis=1, keepdims=True)
        w.u = w.u.astype(np.float32).astype(np.float64)
    ref = oracle_of(w).run(w.m0, w.a0, fixed_dt=dt, max_steps=300)
    with open_sim(api, w, prec, path) as sim:
        api.cav_run_steps(sim.h, math.inf, fixed_dt=dt, max_steps=300)
        m, a = sim.get_m(), sim.get_a()
    assert_parity(m, a, ref, prec)


@pytest.mark.parametrize("path", PATHS)
def test_cfg2_fixed_f64_and_f32(api, path):
    w = W.cfg2(nx=64, ny=64, nz=16)
    ref = oracle_of(w).run(w.m0, w.a0, fixed_dt=0.2e-12, max_steps=200)
    for prec in ("f64", "f32"):
        with open_sim(api, w, prec, path) as sim:
            api.cav_run_steps(sim.h, math.inf, fixed_dt=0.2e-12, max_steps=200)
            m, a = sim.get_m(), sim.get_a()
        if prec == "f64":
            assert_parity(m, a, ref, prec)
        else:
            assert np.abs(m - ref.m).max() <= 1e-4
            # a_n starts from zero and is still ~1e-6 here: compare on the scale of the driving overlap
            assert np.abs(a - ref.a).max() <= 1e-4 * np.abs(ref.a).max()


@pytest.mark.parametrize("path", PATHS)
def test_cfg4_afm_dissipative_fixed(api, path):
    w = W.cfg4(nx=32, ny=16, nz=8, dissipative=True)
    ref = oracle_of(w).run(w.m0, w.a0, fixed_dt=0.02e-12, max_steps=400)
    for prec in ("f64", "f32"):
        with open_sim(api, w, prec, path) as sim:
            api.cav_run_steps(sim.h, math.inf, fixed_dt=0.02e-12, max_steps=400)
            m, a = sim.get_m(), sim.get_a()
        if prec == "f64":
            assert_parity(m, a, ref, prec)
        else:
            assert np.abs(m - ref.m).max() <= 1e-4
            assert np.abs(a - ref.a).max() <= 1e-4 * np.abs(ref.a).max()


# ----------------------------------------------------------------------------------------
# full-size workloads, in the launch configuration bench.py times
# ----------------------------------------------------------------------------------------
FULL_SIZE_STEPS = 50      # parity on the full-size workloads over the fixed steps the oracle can afford


def test_cfg3_full_size_steps(api):
    """256x256x32, 8 modes, fp32: 50 fixed steps element by element against the oracle."""
    w = W.cfg3()
    w.m0 = w.m0.astype(np.float32).astype(np.float64)
    w.m0 /= np.linalg.norm(w.m0, axis=1, keepdims=True)
    w.u = w.u.astype(np.float32).astype(np.float64)
    # give the modes something to do from step 1
    w.a0 = (1e-3 * (1 + np.arange(8))).astype(np.complex128)
    ref = oracle_of(w).run(w.m0, w.a0, fixed_dt=0.1e-12, max_steps=FULL_SIZE_STEPS)
    with api.Sim(w, precision="f32") as sim:
        assert api.cav_get_kernel_path(sim.h) == api.CAV_PATH_TMA      # the configuration bench.py times
        api.cav_run_steps(sim.h, math.inf, fixed_dt=0.1e-12, max_steps=FULL_SIZE_STEPS)
        m, a = sim.get_m(), sim.get_a()
        S = api.cav_get_overlaps(sim.h, 8)
        st = api.cav_get_stats(sim.h)
    assert st["accepted"] == FULL_SIZE_STEPS and st["rhs_evals"] == 1 + 6 * FULL_SIZE_STEPS
    # fp32 rounding accumulates over 300 evaluations: ~1e-7 per step on |m| = 1 (north_star's bar is 1e-4)
    assert np.abs(m - ref.m).max() <= 1e-5
    assert np.abs(a - ref.a).max() <= 1e-5 * np.abs(ref.a).max()
    # invariants that hold at any size
    assert np.abs(np.linalg.norm(m.astype(np.float64), axis=1) - 1).max() < 3e-7
    mc = ref.m[0]
    S_direct = np.array([(w.u[n] * (mc[0] - 1j * mc[1])).mean() for n in range(8)])
    assert np.abs(S - S_direct).max() < 1e-7


def test_cfg4_full_size_steps(api):
    """128x128x64 two-sublattice antiferromagnet with dissipative coupling (BASELINE.json configs[3]), fp32 and fp64 on
    the TMA path as bench.py times it: 50 fixed steps element by element against the oracle."""
    w = W.cfg4(dissipative=True)
    w.m0 = w.m0.astype(np.float32).astype(np.float64)
    w.m0 /= np.linalg.norm(w.m0, axis=1, keepdims=True)
    w.a0 = np.array([2e-3 + 1e-3j])
    dt = 0.01e-12
    ref = oracle_of(w).run(w.m0, w.a0, fixed_dt=dt, max_steps=FULL_SIZE_STEPS)
    for prec, tol_m, tol_a in (("f64", 1e-11, 1e-11), ("f32", 1e-5, 1e-4)):
        with api.Sim(w, precision=prec) as sim:
            assert api.cav_get_kernel_path(sim.h) == api.CAV_PATH_TMA
            api.cav_run_steps(sim.h, math.inf, fixed_dt=dt, max_steps=FULL_SIZE_STEPS)
            m, a = sim.get_m(), sim.get_a()
        assert np.abs(m - ref.m).max() <= tol_m, prec
        assert np.abs(a - ref.a).max() <= tol_a * np.abs(ref.a).max(), prec
        assert np.abs(np.linalg.norm(m.astype(np.float64), axis=1) - 1).max() < (3e-7 if prec == "f32" else 1e-14)


def test_cfg5_slab_32_modes(api):
    """cfg5's 512x512 plane and 32 mixed-coupling modes on a thinner slab (oracle memory/time bound)."""
    w = W.cfg5(nz=4, dtype=np.float64)
    w.m0 = w.m0.astype(np.float32).astype(np.float64)
    w.m0 /= np.linalg.norm(w.m0, axis=1, keepdims=True)
    w.u = w.u.astype(np.float32).astype(np.float64)
    w.a0 = (1e-3 * (1 + np.arange(32)) * np.exp(0.3j * np.arange(32))).astype(np.complex128)
    ref = oracle_of(w).run(w.m0, w.a0, fixed_dt=0.1e-12, max_steps=2)
    with api.Sim(w, precision="f32") as sim:
        assert api.cav_get_kernel_path(sim.h) == api.CAV_PATH_TMA
        api.cav_run_steps(sim.h, math.inf, fixed_dt=0.1e-12, max_steps=2)
        m, a = sim.get_m(), sim.get_a()
    assert np.abs(m - ref.m).max() <= 2e-6
    assert np.abs(a - ref.a).max() <= 1e-6 * np.abs(ref.a).max()


@pytest.mark.timeout(2400)
def test_cfg5_full_size_steps(api):
    """BASELINE.json configs[4] at its stated size: 512x512x64 cells, 32 mixed-coupling modes, fp32, on the automatic
    (TMA) path as bench.py times it; two fixed steps element by element against the oracle.  This is the one workload
    whose profile array exceeds 2^31 bytes (32 x 16.8 M x 4 B = 2.1 GB) and whose plane-tile count (32 768) is far
    beyond any other test: a 32-bit byte offset or tile counter would show here and nowhere else.  The oracle needs
    about 10 GB of host memory for it."""
    w = W.cfg5(dtype=np.float32)
    w.m0 = w.m0.astype(np.float32).astype(np.float64)
    w.m0 /= np.linalg.norm(w.m0, axis=1, keepdims=True)
    w.a0 = (1e-3 * (1 + np.arange(32)) * np.exp(0.3j * np.arange(32))).astype(np.complex128)
    nc = w.n_cells
    assert w.u.nbytes >= 2 ** 31 and w.u.dtype == np.float32
    with api.Sim(w, precision="f32") as sim:
        assert api.cav_get_kernel_path(sim.h) == api.CAV_PATH_TMA
        # overlaps of the initial state first (stage 1 alone), against a direct numpy sum in fp64
        dm = np.empty(sim.shape_m, dtype=np.float32)
        api.cav_get_dmdt(sim.h, dm)
        S0 = api.cav_get_overlaps(sim.h, 32)
        api.cav_run_steps(sim.h, math.inf, fixed_dt=0.1e-12, max_steps=2)
        m, a = sim.get_m(), sim.get_a()
        S = api.cav_get_overlaps(sim.h, 32)
    mc0 = (w.m0[0, 0] - 1j * w.m0[0, 1]).reshape(-1)
    S0_direct = np.array([np.dot(w.u[n].reshape(-1).astype(np.float64), mc0) / nc for n in range(32)])
    # fp32 running sums per thread (221 planes x 2 cells x 32 modes), fp64 from the warp level up: |S| <= ~0.03 here
    assert np.abs(S0 - S0_direct).max() < 2e-7
    ref = oracle_of(w).run(w.m0, w.a0, fixed_dt=0.1e-12, max_steps=2)
    assert np.abs(m - ref.m).max() <= 2e-6
    assert np.abs(a - ref.a).max() <= 1e-6 * np.abs(ref.a).max()
    assert np.abs(dm - oracle_of(w).rhs(w.m0, w.a0)[0]).max() <= 2e-5 * np.abs(dm).max()
    assert np.abs(np.linalg.norm(m.astype(np.float64), axis=1) - 1).max() < 3e-7
    mc = (ref.m[0, 0] - 1j * ref.m[0, 1]).reshape(-1)
    S_direct = np.array([np.dot(w.u[n].reshape(-1).astype(np.float64), mc) / nc for n in range(32)])
    assert np.abs(S - S_direct).max() < 2e-7
    # the far corner of the grid and of the last profile really took part (offsets beyond 2^31 bytes)
    assert np.abs(m[0, :, -1, -1, -8:] - ref.m[0, :, -1, -1, -8:]).max() <= 2e-6


# ----------------------------------------------------------------------------------------
# the controller's reject branch (a7): forced rejections, step for step against the oracle
# ----------------------------------------------------------------------------------------
def _reject_case(n, driven):
    w = W.cfg1("b", n=n)
    dr = None
    if driven:      # a short strong pulse in mid-run: more rejections after the start-up ones
        dr = dict(amp=np.array([5e12 + 2e12j]), t0=np.array([4e-12]), sigma=np.array([0.15e-12]), omega_d=w.omega)
    return w, dr


@pytest.mark.parametrize("driven", [False, True])
@pytest.mark.parametrize("n", [8, 12])
@pytest.mark.parametrize("path", PATHS)
def test_forced_rejections_match_oracle(api, path, n, driven):
    """fp64, adaptive, dt_init = 2 ps (ten times the stability limit of the 5 nm grid): the first steps MUST be
    rejected (dt = h*fac, state and FSAL slope kept, the candidate buffer reused), and a 0.15 ps pulse in mid-run
    forces more.  Both implementations run the same controller in fp64, so accepted and rejected counts are equal
    and the final state agrees to 1e-10 (this also pins the 'parity unpinned' controller constants between the two)."""
    w, dr = _reject_case(n, driven)
    t_end = 8e-12
    ref = oracle_of(w, drive=dr).run(w.m0, w.a0, t_end=t_end, tol=1e-8, dt_init=2e-12)
    assert ref.rejected >= (8 if driven else 5)
    with open_sim(api, w, "f64", path) as sim:
        if dr:
            api.cav_set_drive(sim.h, dr["amp"], dr["t0"], dr["sigma"], dr["omega_d"])
        api.cav_run(sim.h, t_end, tol=1e-8, dt_init=2e-12)
        m, a = sim.get_m(), sim.get_a()
        st = api.cav_get_stats(sim.h)
    assert st["rejected"] > 0
    assert (st["accepted"], st["rejected"]) == (ref.accepted, ref.rejected)
    assert st["rhs_evals"] == ref.rhs_evals == 1 + 6 * (ref.accepted + ref.rejected)
    assert st["t"] == t_end
    # dt = h * 0.8 (tol/err)^(1/5), and err = |h sum_j d_j k_j| is a difference of slopes that cancel to ~1e-7 of their
    # size: rounding-order differences between the two implementations move err by ~1e-7 relative, dt by a fifth of that
    assert abs(st["dt_min"] / ref.dt_min - 1) < 1e-6 and abs(st["dt_max"] / ref.dt_max - 1) < 1e-6
    assert abs(st["dt_next"] / ref.dt - 1) < 1e-6
    assert_parity(m, a, ref, "f64")


@pytest.mark.parametrize("path", ["generic", "tma"])
def test_rejections_in_fp32_keep_state_and_slope(api, path):
    """fp32 on the stage kernels: step sequences may differ from the fp64 oracle, so compare what is unique - the run
    lands on t_end, rejections happened, every rejected step cost six evaluations, |m| = 1, and the final state agrees
    with the oracle's adaptive run to the accuracy the tolerance implies."""
    w = W.cfg1("b", n=12)
    w.m0 = w.m0.astype(np.float32).astype(np.float64)
    ref = oracle_of(w).run(w.m0, w.a0, t_end=8e-12, tol=1e-6, dt_init=2e-12)
    with open_sim(api, w, "f32", path) as sim:
        api.cav_run(sim.h, 8e-12, tol=1e-6, dt_init=2e-12)
        m, a = sim.get_m(), sim.get_a()
        st = api.cav_get_stats(sim.h)
    assert st["rejected"] >= 3 and st["t"] == 8e-12
    assert st["rhs_evals"] == 1 + 6 * (st["accepted"] + st["rejected"])
    assert abs(st["rejected"] - ref.rejected) <= 1 and abs(st["accepted"] - ref.accepted) <= 3
    assert np.abs(m - ref.m).max() < 2e-5
    assert np.abs(np.linalg.norm(m.astype(np.float64), axis=1) - 1).max() < 3e-7


# ----------------------------------------------------------------------------------------
# adaptive mode: observables
# ----------------------------------------------------------------------------------------
def _run_trace(api, w, prec, t_end, sample_dt, tol, path="generic"):
    cap = int(round(t_end / sample_dt))
    with open_sim(api, w, prec, path) as sim:
        api.cav_set_trace(sim.h, sample_dt, cap)
        api.cav_run(sim.h, t_end, tol=tol)
        tr = api.cav_get_trace(sim.h)
        st = api.cav_get_stats(sim.h)
    assert tr.shape[0] == cap
    return tr, st


@pytest.mark.parametrize("path", PATHS)
@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_adaptive_rabi_period(api, prec, path):
    """g/2pi = 50 MHz at resonance, a(0) = 0.01: T_R = pi/g = 10 ns within 0.5 %."""
    w = W.macrospin(5.0, [5.0], 50.0, 0.0, alpha=0.0, a0=[0.01], n=4)
    tol = 1e-8 if prec == "f64" else 1e-6
    tr, st = _run_trace(api, w, prec, 26e-9, 25e-12, tol, path)
    ref = oracle_of(w).run(w.m0, w.a0, t_end=26e-9, tol=tol, sample_dt=25e-12, trace_cap=1040)
    T_gpu = rabi_period(tr[:, 0], tr[:, 1] ** 2 + tr[:, 2] ** 2)
    T_ref = rabi_period(ref.trace[:, 0], ref.trace[:, 1] ** 2 + ref.trace[:, 2] ** 2)
    assert abs(T_gpu / T_ref - 1) < 5e-3
    assert abs(T_gpu / 10e-9 - 1) < 5e-3
    assert np.allclose(tr[:, 0], ref.trace[:, 0], rtol=0, atol=1e-22)
    assert st["accepted"] > 0 and st["rhs_evals"] == 1 + 6 * (st["accepted"] + st["rejected"])


@pytest.mark.parametrize("path", PATHS)
@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_adaptive_anticrossing_frequencies(api, prec, path):
    """Polariton branches of cfg1's tiny ferromagnet (per-cell tilt, exchange on) with g/2pi = 50 MHz:
    peak frequencies of GPU and oracle within 1 MHz, and both on Eq. 6."""
    w = W.cfg1("b")
    w.omega = np.array([TWO_PI * 10e9]); w.g = np.array([TWO_PI * 50e6]); w.kappa = np.array([TWO_PI * 1e6])
    w.a0 = np.array([1e-3 + 0j])
    w.B0 = (0.0, 0.0, W.b0_for_ghz(10.03))
    tol = 1e-8 if prec == "f64" else 1e-6
    t_end, sdt = 40e-9, 20e-12
    tr, _ = _run_trace(api, w, prec, t_end, sdt, tol, path)
    ref = oracle_of(w).run(w.m0, w.a0, t_end=t_end, tol=tol, sample_dt=sdt, trace_cap=2000)
    out = []
    for t in (tr, ref.trace):
        om, amp = fit_exponentials(t[:, 1] + 1j * t[:, 2], sdt, 4)
        out.append(dominant(om, amp, 2)[0].real / TWO_PI)
    assert np.abs(out[0] - out[1]).max() < 1e6
    wc, wm, g = TWO_PI * 10e9, GAMMA * w.B0[2], TWO_PI * 50e6
    eq6 = ((wc + wm) / 2 + np.array([-1, 1]) * math.sqrt(g * g + ((wc - wm) / 2) ** 2)) / TWO_PI
    assert np.abs(out[0] - eq6).max() < 1e6


def test_adaptive_afm_neel_line(api):
    """cfg4-like AFM: the Neel-vector line of GPU (fp32 and fp64) and oracle agree within 1e-5 relative."""
    w = W.cfg4(nx=8, ny=4, nz=4)
    t_end, sdt = 0.1e-9, 0.5e-12
    ref = oracle_of(w).run(w.m0, w.a0, t_end=t_end, tol=1e-7, sample_dt=sdt, trace_cap=200)

    def neel_freq(t):
        c = 1 + 4
        n = 0.5 * ((t[:, c] - t[:, c + 3]) - 1j * (t[:, c + 1] - t[:, c + 4]))
        om, amp = fit_exponentials(n, sdt, 4)
        return np.sort(np.abs(dominant(om, amp, 2)[0].real))
    f_ref = neel_freq(ref.trace)
    for prec in ("f64", "f32"):
        for path in PATHS:
            tr, _ = _run_trace(api, w, prec, t_end, sdt, 1e-7 if prec == "f64" else 1e-6, path)
            assert np.abs(neel_freq(tr) / f_ref - 1).max() < 1e-4


# ----------------------------------------------------------------------------------------
# launch modes, determinism, edge cases
# ----------------------------------------------------------------------------------------
@pytest.mark.parametrize("path", PATHS)
def test_graph_and_stream_modes_bitwise_identical_and_deterministic(api, path):
    w = small_problem(40, 9, 7, 3, 1)
    outs = []
    for mode in (api.CAV_LAUNCH_GRAPH, api.CAV_LAUNCH_STREAM, api.CAV_LAUNCH_GRAPH):
        with open_sim(api, w, "f32", path) as sim:
            api.cav_set_launch_mode(sim.h, mode)
            api.cav_run(sim.h, 5e-12, tol=1e-6)
            outs.append((sim.get_m(), sim.get_a(), api.cav_get_stats(sim.h)))
    for m, a, st in outs[1:]:
        assert np.array_equal(m, outs[0][0]) and np.array_equal(a, outs[0][1])
        assert st["accepted"] == outs[0][2]["accepted"] and st["rejected"] == outs[0][2]["rejected"]


def test_two_tma_sims_on_two_streams_equal_a_solo_run(api):
    """Distinct handles are independent (cavmag.h): two TMA simulations running concurrently on two streams share the
    SMs, so blocks of one stage kernel start at different times - each must still be bitwise identical to the same
    simulation run alone (block partials are double-buffered by stage parity)."""
    import torch
    ws = [small_problem(128, 64, 20, 3, 1, seed=7), small_problem(128, 64, 20, 3, 1, seed=11)]
    solo = []
    for w in ws:
        with open_sim(api, w, "f32", "tma") as sim:
            api.cav_run_steps(sim.h, math.inf, tol=1e-6, max_steps=40)
            solo.append((sim.get_m(), sim.get_a(), api.cav_get_stats(sim.h)))
    for _ in range(3):
        streams = [torch.cuda.Stream() for _ in ws]
        sims = [open_sim(api, w, "f32", "tma") for w in ws]
        try:
            for sim, st in zip(sims, streams):
                api.cav_set_stream(sim.h, st.cuda_stream)
            for sim in sims:                      # asynchronous: both graphs are in flight together
                api.cav_run_steps(sim.h, math.inf, tol=1e-6, max_steps=40)
            for sim, ref in zip(sims, solo):
                assert np.array_equal(sim.get_m(), ref[0]) and np.array_equal(sim.get_a(), ref[1])
                st = api.cav_get_stats(sim.h)
                assert (st["accepted"], st["rejected"]) == (ref[2]["accepted"], ref[2]["rejected"])
        finally:
            for sim in sims:
                sim.close()


def test_failed_set_modes_leaves_a_usable_handle(api):
    """CAV_E_SINGULAR_NORM from cav_set_modes must not leave tensor maps / graphs that point at freed profiles:
    afterwards the handle has no modes, runs as a plain LLG problem, and accepts a valid mode set again."""
    w = small_problem(64, 16, 6, 2, 1)
    w0 = small_problem(64, 16, 6, 0, 1)
    with api.Sim(w, precision="f64", overlap_norm=api.CAV_NORM_SUM_U) as sim:
        api.cav_run_steps(sim.h, math.inf, fixed_dt=0.1e-12, max_steps=5)
        bad = W.cfg2(nx=64, ny=16, nz=6)                         # sin(2 pi x/L) sums to zero
        with pytest.raises(api.CavError) as e:
            api.cav_set_modes(sim.h, np.ascontiguousarray(bad.u), bad.omega, bad.kappa, bad.g, bad.Gamma, bad.Phi)
        assert e.value.status == api.CAV_E_SINGULAR_NORM
        api.cav_set_m(sim.h, np.ascontiguousarray(w0.m0))
        api.cav_run_steps(sim.h, math.inf, fixed_dt=0.1e-12, max_steps=20)
        ref = oracle_of(w0).run(w0.m0, w0.a0, fixed_dt=0.1e-12, max_steps=20)
        assert np.abs(sim.get_m() - ref.m).max() < 1e-12
        # and a valid mode set works again on the same handle
        w.u = w.u + 0.5
        api.cav_set_modes(sim.h, np.ascontiguousarray(w.u), w.omega, w.kappa, w.g, w.Gamma, w.Phi)
        api.cav_set_m(sim.h, np.ascontiguousarray(w.m0)); api.cav_set_a(sim.h, w.a0)
        api.cav_run_steps(sim.h, math.inf, fixed_dt=0.1e-12, max_steps=20)
        ref = oracle_of(w, norm_sum_u=True).run(w.m0, w.a0, fixed_dt=0.1e-12, max_steps=20)
        assert_parity(sim.get_m(), sim.get_a(), ref, "f64")


def test_stage_overlap_is_bitwise_neutral(api):
    """Programmatic dependencies between the stage kernels of the loop body only move the data-independent
    prologue of a kernel under the tail of the previous one: results are bitwise identical with and without."""
    w = small_problem(96, 24, 12, 3, 1)
    outs, active = [], []
    for on in (1, 0, 1):
        with open_sim(api, w, "f32", "tma") as sim:
            api.cav_set_stage_overlap(sim.h, on)
            api.cav_run(sim.h, 5e-12, tol=1e-6)
            active.append(api.cav_get_stage_overlap(sim.h))
            outs.append((sim.get_m(), sim.get_a(), api.cav_get_stats(sim.h)))
    assert active[1] == 0
    for m, a, st in outs[1:]:
        assert np.array_equal(m, outs[0][0]) and np.array_equal(a, outs[0][1])
        assert st["accepted"] == outs[0][2]["accepted"] and st["rejected"] == outs[0][2]["rejected"]


def test_block_size_and_sweep_order_do_not_change_fp64_results_beyond_rounding(api):
    w = small_problem(40, 9, 7, 3, 1)
    res = []
    for cells, serp in ((0, 1), (512, 0), (2048, 1)):
        with api.Sim(w, precision="f64") as sim:
            api.cav_set_block_cells(sim.h, cells)
            api.cav_set_sweep_order(sim.h, serp)
            api.cav_run_steps(sim.h, math.inf, fixed_dt=0.1e-12, max_steps=50)
            res.append((sim.get_m(), sim.get_a()))
    for m, a in res[1:]:
        assert np.abs(m - res[0][0]).max() < 1e-13 and np.abs(a - res[0][1]).max() < 1e-15
    # the sweep order only permutes which block handles which cells: m is bitwise unchanged
    assert np.array_equal(res[0][0], res[2][0]) or np.abs(res[0][0] - res[2][0]).max() < 1e-13


@pytest.mark.parametrize("path", PATHS)
def test_resume_equals_single_run(api, path):
    """Stopping and continuing (FSAL slope kept on the device) gives the same trajectory."""
    w = small_problem(24, 6, 4, 2, 1)
    with open_sim(api, w, "f64", path) as sim:
        api.cav_run_steps(sim.h, math.inf, fixed_dt=0.1e-12, max_steps=40)
        m1, a1 = sim.get_m(), sim.get_a()
    with open_sim(api, w, "f64", path) as sim:
        api.cav_run_steps(sim.h, math.inf, fixed_dt=0.1e-12, max_steps=15)
        api.cav_run_steps(sim.h, math.inf, fixed_dt=0.1e-12, max_steps=25)
        m2, a2 = sim.get_m(), sim.get_a()
        st = api.cav_get_stats(sim.h)
    assert np.array_equal(m1, m2) and np.array_equal(a1, a2)
    # the single-block path keeps its slopes in registers and re-evaluates k1 at the start of every run
    assert st["rhs_evals"] == 1 + 6 * 40 + (1 if path in ("block", "coop") else 0)


def test_edge_cases(api):
    w = small_problem(8, 4, 2, 1, 1)
    with api.Sim(w, precision="f64") as sim:
        # t_end <= t: nothing happens
        api.cav_run(sim.h, 0.0, tol=1e-6)
        assert api.cav_get_stats(sim.h)["accepted"] == 0
        # argument validation
        for bad in (dict(tol=0.0, fixed_dt=0.0), dict(tol=1e-6, fixed_dt=1e-13)):
            with pytest.raises(api.CavError) as e:
                api.cav_run(sim.h, 1e-12, **bad)
            assert e.value.status == api.CAV_E_ARG
        with pytest.raises(api.CavError):
            api.cav_run(sim.h, math.inf, tol=1e-6)
        # set_m normalises
        api.cav_set_m(sim.h, np.ascontiguousarray(3.0 * w.m0))
        assert np.abs(np.linalg.norm(sim.get_m(), axis=1) - 1).max() < 1e-15
        # exact landing on t_end and on every trace sample
        api.cav_set_trace(sim.h, 1e-12, 5)
        api.cav_run(sim.h, 5e-12, tol=1e-7)
        t, _ = api.cav_get_time(sim.h)
        tr = api.cav_get_trace(sim.h)
        assert t == 5e-12 and tr.shape == (5, 1 + 4 + 3)
        assert np.allclose(tr[:, 0], 1e-12 * np.arange(1, 6), rtol=0, atol=1e-26)
        a = sim.get_a()
        assert tr[-1, 1] == a[0].real and tr[-1, 2] == a[0].imag
        mavg = sim.get_m().reshape(3, -1).mean(axis=1)
        assert np.abs(tr[-1, 5:8] - mavg).max() < 1e-14
    # a far too large fixed step blows up: reported, not hidden
    with api.Sim(w, precision="f32") as sim:
        api.cav_run_steps(sim.h, math.inf, fixed_dt=1e-9, max_steps=200)
        with pytest.raises(api.CavError) as e:
            api.cav_sync(sim.h)
        assert e.value.status == api.CAV_E_NONFINITE


def test_overlap_norm_sum_u_and_singular(api):
    w = small_problem(16, 4, 4, 2, 1)
    w.u = w.u + 0.5
    ref = oracle_of(w, norm_sum_u=True)
    _, _, S_ref = ref.rhs(w.m0, w.a0)
    with api.Sim(w, precision="f64", overlap_norm=api.CAV_NORM_SUM_U) as sim:
        dm = np.empty(sim.shape_m)
        api.cav_get_dmdt(sim.h, dm)
        S = api.cav_get_overlaps(sim.h, 2)
    assert np.abs(S - S_ref).max() < 1e-14
    w2 = W.cfg2(nx=16, ny=4, nz=2)      # sin(2 pi x/L) sums to zero
    with pytest.raises(api.CavError) as e:
        api.Sim(w2, precision="f64", overlap_norm=api.CAV_NORM_SUM_U)
    assert e.value.status == api.CAV_E_SINGULAR_NORM


def test_device_buffers_via_torch(api):
    """PyTorch only provides device memory and the stream: tensors cross the ABI as raw pointers."""
    import torch
    w = small_problem(24, 6, 4, 2, 1)
    stream = torch.cuda.Stream()
    with torch.cuda.stream(stream):
        m_dev = torch.tensor(w.m0, dtype=torch.float64, device="cuda")
        u_dev = torch.tensor(w.u, dtype=torch.float64, device="cuda")
    stream.synchronize()
    h = api.cav_create((w.nx, w.ny, w.nz, w.dx, w.dy, w.dz),
                       dict(Ms=w.Ms, Aex=w.Aex, Ku=w.Ku, ku_axis=w.ku_axis, alpha=w.alpha, gamma=w.gamma, B0=w.B0,
                            precision=api.CAV_F64))
    try:
        api.cav_set_stream(h, stream.cuda_stream)
        api.cav_set_modes(h, u_dev, w.omega, w.kappa, w.g, w.Gamma, w.Phi)
        api.cav_set_m(h, m_dev)
        api.cav_set_a(h, w.a0)
        api.cav_run_steps(h, math.inf, fixed_dt=0.1e-12, max_steps=20)
        out = torch.empty_like(m_dev)
        api.cav_get_m(h, out)
        a = api.cav_get_a(h, 2)
    finally:
        api.cav_destroy(h)
    ref = oracle_of(w).run(w.m0, w.a0, fixed_dt=0.1e-12, max_steps=20)
    assert np.abs(out.cpu().numpy() - ref.m).max() < 1e-12
    assert np.abs(a - ref.a).max() < 1e-13


# ----------------------------------------------------------------------------------------
# external drive eta_n(t) (cav_set_drive; G27)
# ----------------------------------------------------------------------------------------
def _drive_for(w, t0=3e-12, sigma=1.5e-12):
    N = w.omega.size
    amp = (2e10 * (1 + np.arange(N)) * np.exp(0.7j * np.arange(N))).astype(np.complex128)
    return dict(amp=amp, t0=np.full(N, t0), sigma=np.full(N, sigma), omega_d=np.asarray(w.omega) * 0.97)


@pytest.mark.parametrize("path", PATHS)
@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("shape,N,n_sub,dt", [((40, 9, 7), 3, 1, 0.1e-12), ((24, 6, 4), 1, 2, 0.02e-12)])
def test_driven_fixed_steps(api, prec, shape, N, n_sub, dt, path):
    """The pulse passes through the run (t0 = 30 / 150 steps in): every stage time t + c_s h matters."""
    w = small_problem(*shape, N, n_sub)
    if prec == "f32":
        w.m0 = w.m0.astype(np.float32).astype(np.float64)
    dr = _drive_for(w, t0=30 * dt, sigma=12 * dt)
    ref = oracle_of(w, drive=dr).run(w.m0, w.a0, fixed_dt=dt, max_steps=80)
    with open_sim(api, w, prec, path) as sim:
        api.cav_set_drive(sim.h, dr["amp"], dr["t0"], dr["sigma"], dr["omega_d"])
        api.cav_run_steps(sim.h, math.inf, fixed_dt=dt, max_steps=80)
        m, a = sim.get_m(), sim.get_a()
        # switching the drive off again restores the undriven slopes
        api.cav_set_drive(sim.h, None)
        dadt_off = api.cav_get_dadt(sim.h, N)
    assert_parity(m, a, ref, prec)
    undriven = oracle_of(w).run(w.m0, w.a0, fixed_dt=dt, max_steps=80)
    assert np.abs(ref.a - undriven.a).max() > 0.05 * np.abs(undriven.a).max()       # the drive is not a detail here
    _, da_ref, _ = oracle_of(w).rhs(ref.m, ref.a)
    assert np.abs(dadt_off - da_ref).max() <= (1e-9 if prec == "f64" else 1e-3) * np.abs(da_ref).max()


@pytest.mark.parametrize("path", PATHS)
def test_driven_adaptive_closed_form(api, path):
    """g = 0, fp64, adaptive: a(T) of the pulsed uncoupled cavity against the closed form the oracle is pinned with."""
    w = W.macrospin(10.0, [9.0, 10.5], 0.0, [1.0, 50.0], alpha=1e-3, a0=[0, 0], n=4)
    sig, t0, T = 20e-12, 0.2e-9, 0.5e-9
    amp = np.array([1e9 * (1 + 0.5j), 2e9 * (-0.3 + 1j)])
    wd = np.array([0.0, TWO_PI * 10.5e9])
    with open_sim(api, w, "f64", path) as sim:
        api.cav_set_drive(sim.h, amp, t0, sig, wd)
        api.cav_run(sim.h, T, tol=1e-12)
        a = sim.get_a()
    lam = w.kappa + 1j * w.omega
    exact = amp * sig * math.sqrt(TWO_PI) * np.exp((lam - 1j * wd) ** 2 * sig ** 2 / 2) * np.exp(-lam * (T - t0))
    assert np.all(np.abs(a - exact) <= 3e-9 * np.abs(exact))


# ----------------------------------------------------------------------------------------
# non-reciprocal coupling (cav_set_backaction; G31)
# ----------------------------------------------------------------------------------------
@pytest.mark.parametrize("path", PATHS)
@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_nonreciprocal_fixed_steps(api, prec, path):
    w = small_problem(40, 9, 7, 3, 1)
    if prec == "f32":
        w.m0 = w.m0.astype(np.float32).astype(np.float64)
    back = dict(g=0.25 * w.g, Gamma=2.0 * w.Gamma, Phi=w.Phi + 0.4)
    ref = oracle_of(w, backward=back).run(w.m0, w.a0, fixed_dt=0.1e-12, max_steps=80)
    with open_sim(api, w, prec, path) as sim:
        api.cav_set_backaction(sim.h, back["g"], back["Gamma"], back["Phi"])
        api.cav_run_steps(sim.h, math.inf, fixed_dt=0.1e-12, max_steps=80)
        m, a = sim.get_m(), sim.get_a()
    assert_parity(m, a, ref, prec)
    recip = oracle_of(w).run(w.m0, w.a0, fixed_dt=0.1e-12, max_steps=80)
    assert np.abs(ref.m - recip.m).max() > 1e-5            # the backward coupling is not a detail here
    # g_b = None restores reciprocal coupling
    with open_sim(api, w, prec, path) as sim:
        api.cav_set_backaction(sim.h, back["g"], back["Gamma"], back["Phi"])
        api.cav_set_backaction(sim.h, None)
        api.cav_run_steps(sim.h, math.inf, fixed_dt=0.1e-12, max_steps=80)
        assert_parity(sim.get_m(), sim.get_a(), recip, prec)


def test_nonreciprocal_rabi_period_geometric_mean(api):
    """g_f/2pi = 100 MHz, g_b/2pi = 25 MHz: T_R = pi / sqrt(g_f g_b) = 10 ns within 0.5 % (the oracle's pin, on the GPU)."""
    w = W.macrospin(5.0, [5.0], 100.0, 0.0, alpha=0.0, a0=[0.01], n=4)
    with api.Sim(w, precision="f64") as sim:
        api.cav_set_backaction(sim.h, np.array([TWO_PI * 25e6]))
        api.cav_set_trace(sim.h, 25e-12, 1040)
        api.cav_run(sim.h, 26e-9, tol=1e-8)
        tr = api.cav_get_trace(sim.h)
    assert abs(rabi_period(tr[:, 0], tr[:, 1] ** 2 + tr[:, 2] ** 2) / 10e-9 - 1) < 5e-3


# ----------------------------------------------------------------------------------------
# large grids whose rows are not a multiple of 16 bytes: padded rows inside the library, TMA path (no generic-kernel cliff)
# ----------------------------------------------------------------------------------------
@pytest.mark.parametrize("prec,nx", [("f32", 250), ("f32", 251), ("f64", 251), ("f32", 61)])
@pytest.mark.parametrize("n_sub,N", [(1, 3), (2, 1), (2, 4)])
def test_unaligned_rows_run_on_the_tma_path(api, prec, nx, n_sub, N):
    """nx * sizeof(T) % 16 != 0 on a grid beyond the cooperative kernel's range: the library pads the rows of its own
    buffers (the ABI arrays stay dense) and runs the TMA kernels.  Odd nx ends a row in the middle of a lane's pair of
    cells.  Right-hand side and 12 fixed steps element by element against the oracle."""
    ny, nz = (40, 8) if nx > 100 else (160, 8)
    w = small_problem(nx, ny, nz, N, n_sub)
    assert w.nx * w.ny * w.nz > 512 * 148
    if prec == "f32":
        w.m0 = w.m0.astype(np.float32).astype(np.float64)
        w.m0 /= np.linalg.norm(w.m0, axis=1, keepdims=True)
        w.u = w.u.astype(np.float32).astype(np.float64)
    dt = 0.05e-12 if n_sub == 1 else 0.01e-12
    o = oracle_of(w)
    dm_ref, da_ref, S_ref = o.rhs(w.m0, w.a0)
    ref = o.run(w.m0, w.a0, fixed_dt=dt, max_steps=12)
    with api.Sim(w, precision=prec) as sim:
        assert api.cav_get_kernel_path(sim.h) == api.CAV_PATH_TMA
        with pytest.raises(api.CavError) as e:
            api.cav_set_kernel_path(sim.h, api.CAV_PATH_GENERIC)
        assert e.value.status == api.CAV_E_UNSUPPORTED
        dm = np.empty(sim.shape_m, dtype=sim.np_dtype)
        api.cav_get_dmdt(sim.h, dm)
        S = api.cav_get_overlaps(sim.h, N)
        assert np.abs(sim.get_m().astype(np.float64) - w.m0).max() < (1e-15 if prec == "f64" else 2.5e-7)      # dense in, dense out (normalised on entry)
        api.cav_run_steps(sim.h, math.inf, fixed_dt=dt, max_steps=12)
        m, a = sim.get_m(), sim.get_a()
    scale = np.abs(dm_ref).max()
    assert np.abs(dm - dm_ref).max() <= (2e-13 if prec == "f64" else 2e-5) * scale
    assert np.abs(S - S_ref).max() <= (1e-14 if prec == "f64" else 2e-6)
    assert_parity(m, a, ref, prec)


# ----------------------------------------------------------------------------------------
# TMA path with several plane-tiles per block (marching in z, tile-column changes inside a run, serpentine sweep)
# ----------------------------------------------------------------------------------------
@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("n_sub,N", [(1, 3), (2, 1)])
@pytest.mark.parametrize("serpentine", [1, 0])
def test_tma_multi_plane_runs(api, prec, n_sub, N, serpentine):
    """128 x 64 x 20 cells: 320 (fp32) / 640 (fp64) plane-tiles over 148 persistent blocks, so every block marches over
    2-5 planes, most runs cross a tile-column boundary (nz = 20 does not divide the run length) and odd stages walk
    backwards.  Element by element against the oracle, with both sweep orders."""
    w = small_problem(128, 64, 20, N, n_sub)
    if prec == "f32":
        w.m0 = w.m0.astype(np.float32).astype(np.float64)
    dt = 0.05e-12 if n_sub == 1 else 0.01e-12
    ref = oracle_of(w).run(w.m0, w.a0, fixed_dt=dt, max_steps=6)
    with open_sim(api, w, prec, "tma") as sim:
        api.cav_set_sweep_order(sim.h, serpentine)
        api.cav_run_steps(sim.h, math.inf, fixed_dt=dt, max_steps=6)
        m, a = sim.get_m(), sim.get_a()
    assert_parity(m, a, ref, prec)


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("n_sub,N", [(1, 0), (1, 3), (1, 9), (1, 32), (2, 0), (2, 2), (2, 3), (2, 8), (2, 9), (2, 32)])
def test_every_mode_bucket_and_sublattice_count_runs_on_the_tma_kernels(api, prec, n_sub, N):
    """A grid with enough plane-tiles takes the TMA kernels under CAV_PATH_AUTO for every mode bucket (0, 1, 2, 8, 32) and one or
    two sublattices - also where the planner has to give a ring its minimum depth (two sublattices with more than two
    modes) - and matches the oracle there."""
    w = small_problem(64, 32, 80, N, n_sub)
    dt = 0.05e-12 if n_sub == 1 else 0.01e-12
    if prec == "f32":
        w.m0 = w.m0.astype(np.float32).astype(np.float64)
        w.m0 /= np.linalg.norm(w.m0, axis=1, keepdims=True)
        w.u = w.u.astype(np.float32).astype(np.float64)
    ref = oracle_of(w).run(w.m0, w.a0, fixed_dt=dt, max_steps=12)
    with api.Sim(w, precision=prec) as sim:
        assert api.cav_get_kernel_path(sim.h) == api.CAV_PATH_TMA
        api.cav_run_steps(sim.h, math.inf, fixed_dt=dt, max_steps=12)
        m, a = sim.get_m(), sim.get_a()
    assert_parity(m, a, ref, prec)


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("shape,n_sub,N", [
    ((512, 256, 1), 1, 2),      # a film: one plane, both z neighbours outside the grid
    ((512, 256, 1), 2, 1),      # the same with two sublattices
    ((256, 256, 2), 1, 3),      # two planes
    ((64, 2048, 1), 1, 2),      # one tile column per row of tiles, 256 tile rows
    ((8, 8, 2048), 1, 2),       # a needle along z: one tile, the longest z march
    ((2048, 8, 8), 2, 2),       # a needle along x: 32 tile columns, two sublattices
])
def test_extreme_aspect_ratios_on_the_tma_path(api, prec, shape, n_sub, N):
    w = small_problem(*shape, N, n_sub)
    dt = 0.05e-12 if n_sub == 1 else 0.01e-12
    if prec == "f32":
        w.m0 = w.m0.astype(np.float32).astype(np.float64)
        w.m0 /= np.linalg.norm(w.m0, axis=1, keepdims=True)
        w.u = w.u.astype(np.float32).astype(np.float64)
    ref = oracle_of(w).run(w.m0, w.a0, fixed_dt=dt, max_steps=8)
    with api.Sim(w, precision=prec) as sim:
        assert api.cav_get_kernel_path(sim.h) == api.CAV_PATH_TMA
        api.cav_run_steps(sim.h, math.inf, fixed_dt=dt, max_steps=8)
        m, a = sim.get_m(), sim.get_a()
    assert_parity(m, a, ref, prec)


def test_forced_rejections_with_two_sublattices_and_eight_modes(api):
    """The TMA configuration with a single aux slot (two sublattices, eight modes: DESIGN.md 5.3) through accepted and
    rejected steps: the step sequence of the oracle, state within 1e-10."""
    w = small_problem(64, 32, 80, 8, 2)
    ref = oracle_of(w).run(w.m0, w.a0, t_end=1.5e-12, tol=1e-9, dt_init=0.2e-12)
    assert ref.rejected > 0
    with api.Sim(w, precision="f64") as sim:
        assert api.cav_get_kernel_path(sim.h) == api.CAV_PATH_TMA
        api.cav_run(sim.h, 1.5e-12, tol=1e-9, dt_init=0.2e-12)
        st = api.cav_get_stats(sim.h)
        m, a = sim.get_m(), sim.get_a()
    assert (st["accepted"], st["rejected"]) == (ref.accepted, ref.rejected)
    assert_parity(m, a, ref, "f64")
