"""GPU parity of the batched small-grid integrator (cav_batch_*) against the fp64 CPU oracle:
every replica is an independent simulation, so the oracle is simply run once per replica on the same seeded
inputs.  Tolerances as for cav_run (north_star; G23): fp64 1e-10 relative per component / per mode after
1000 fixed steps, fp32 1e-4 absolute in m and 1e-4 relative in |a_n|; adaptive runs are compared on observables."""
import copy
import math
import os
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
for p in (ROOT, os.path.dirname(os.path.abspath(__file__))):
    if p not in sys.path:
        sys.path.insert(0, p)

import cavmag_workloads as W  # noqa: E402
from observables import rabi_period  # noqa: E402
from test_gpu_parity import api, assert_parity, oracle_of, small_problem  # noqa: E402,F401

pytestmark = pytest.mark.gpu
TWO_PI = 2.0 * math.pi


def with_field(w, ghz):
    w2 = copy.deepcopy(w)
    w2.B0 = (0.0, 0.0, W.b0_for_ghz(ghz))
    return w2


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("variant", ["a", "b"])
def test_cfg1_field_sweep_fixed_1000_steps(api, prec, variant):
    """BASELINE.json configs[0] as a 5-point field sweep: one launch, each replica against its own oracle run."""
    w = W.cfg1(variant)
    if prec == "f32":
        w.m0 = w.m0.astype(np.float32).astype(np.float64)
    ghz = np.linspace(9.9, 10.1, 5)
    B0 = np.array([[0.0, 0.0, W.b0_for_ghz(f)] for f in ghz])
    with api.Batch(w, 5, precision=prec, B0=B0) as b:
        b.run(math.inf, fixed_dt=w.fixed_dt, max_steps=1000)
        m, a, st = b.get_m(), b.get_a(), b.stats()
    for r, f in enumerate(ghz):
        wr = with_field(w, f)
        ref = oracle_of(wr).run(wr.m0, wr.a0, fixed_dt=w.fixed_dt, max_steps=1000)
        assert st[r]["accepted"] == 1000 and st[r]["rejected"] == 0 and st[r]["rhs_evals"] == 6001
        assert abs(st[r]["t"] - ref.t) <= 1e-24
        assert_parity(m[r], a[r], ref, prec)
    # the replicas really differ
    assert np.abs(a[0] - a[4]).max() > 1e-6 * np.abs(a[0]).max()


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("shape,N,n_sub,dt", [
    ((8, 8, 1), 1, 1, 0.1e-12),        # the paper's sweep grid
    ((5, 3, 2), 2, 1, 0.1e-12),        # 30 cells: a partly filled warp
    ((16, 8, 8), 3, 1, 0.05e-12),      # 1024 cells: the largest grid
    ((8, 4, 4), 1, 2, 0.02e-12),       # two-sublattice antiferromagnet
    ((6, 5, 4), 0, 1, 0.1e-12),        # no modes: plain LLG
])
def test_busy_fixed_steps(api, prec, shape, N, n_sub, dt):
    """All terms on (anisotropy off-axis, mixed coherent/dissipative coupling, non-cubic cells, large tilt)."""
    w = small_problem(*shape, N, n_sub)
    if prec == "f32":
        w.m0 = w.m0.astype(np.float32).astype(np.float64)
    ref = oracle_of(w).run(w.m0, w.a0, fixed_dt=dt, max_steps=60)
    with api.Batch(w, 3, precision=prec) as b:
        b.run(math.inf, fixed_dt=dt, max_steps=60)
        m, a = b.get_m(), b.get_a()
    for r in range(3):
        assert_parity(m[r], a[r], ref, prec)
    assert np.array_equal(m[0], m[1]) and np.array_equal(a[0], a[2])       # identical replicas: identical bits


def test_agrees_with_cav_run_on_the_same_inputs(api):
    """The batch kernel and the stage kernels are two implementations of the same step: fp64 results agree to
    rounding (only the summation order of the overlaps differs)."""
    w = small_problem(8, 8, 4, 2, 1)
    with api.Sim(w, precision="f64") as sim:
        api.cav_run_steps(sim.h, math.inf, fixed_dt=0.1e-12, max_steps=100)
        m1, a1 = sim.get_m(), sim.get_a()
    with api.Batch(w, 2, precision="f64") as b:
        b.run(math.inf, fixed_dt=0.1e-12, max_steps=100)
        m2, a2 = b.get_m(), b.get_a()
    assert np.abs(m2[1] - m1).max() < 1e-12 and np.abs(a2[1] - a1).max() < 1e-13 * np.abs(a1).max() + 1e-18


def test_per_replica_mode_parameters_and_states(api):
    """A coupling-strength sweep: g differs per replica, and so do the initial states."""
    w = small_problem(6, 4, 3, 2, 1)
    n_rep = 3
    scale = np.array([0.5, 1.0, 2.0])
    om = np.tile(w.omega, (n_rep, 1)); ka = np.tile(w.kappa, (n_rep, 1))
    g = scale[:, None] * w.g[None, :]; Gm = np.tile(w.Gamma, (n_rep, 1)); Ph = np.tile(w.Phi, (n_rep, 1))
    m0 = np.stack([np.roll(w.m0, r, axis=-1) for r in range(n_rep)])
    a0 = np.stack([w.a0 * (1 + r) for r in range(n_rep)])
    with api.Batch(w, n_rep, precision="f64") as b:
        api.cav_batch_set_modes(b.h, np.ascontiguousarray(w.u), om, ka, g, Gm, Ph, per_replica=True)
        api.cav_batch_set_m(b.h, np.ascontiguousarray(m0), per_replica=True)
        api.cav_batch_set_a(b.h, a0, per_replica=True)
        b.run(math.inf, fixed_dt=0.1e-12, max_steps=50)
        m, a = b.get_m(), b.get_a()
    for r in range(n_rep):
        wr = copy.deepcopy(w)
        wr.g = g[r]; wr.m0 = m0[r]; wr.a0 = a0[r]
        ref = oracle_of(wr).run(wr.m0, wr.a0, fixed_dt=0.1e-12, max_steps=50)
        assert_parity(m[r], a[r], ref, "f64")


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_adaptive_rabi_period_sweep(api, prec):
    """Vacuum Rabi oscillation at three coupling strengths in one launch: T_R = pi/g within 0.5 %
    for every replica, sample times exactly on the grid, and the same period as the oracle's trace."""
    w = W.macrospin(5.0, [5.0], 50.0, 0.0, alpha=0.0, a0=[0.01], n=4)
    gs = np.array([40.0, 50.0, 62.5])                               # MHz
    n_rep = len(gs)
    tol = 1e-8 if prec == "f64" else 1e-6
    t_end, sdt = 26e-9, 25e-12
    cap = int(round(t_end / sdt))
    with api.Batch(w, n_rep, precision=prec) as b:
        g = (TWO_PI * gs * 1e6)[:, None]
        api.cav_batch_set_modes(b.h, np.ascontiguousarray(w.u, dtype=b.np_dtype), np.tile(w.omega, (n_rep, 1)),
                                np.tile(w.kappa, (n_rep, 1)), g, None, None, per_replica=True)
        api.cav_batch_set_a(b.h, w.a0)
        api.cav_batch_set_trace(b.h, sdt, cap)
        b.run(t_end, tol=tol)
        trs = api.cav_batch_get_trace(b.h, n_rep, cap)
        st = b.stats()
    for r in range(n_rep):
        tr = trs[r]
        assert tr.shape[0] == cap
        assert np.allclose(tr[:, 0], sdt * np.arange(1, cap + 1), rtol=0, atol=1e-22)
        T = rabi_period(tr[:, 0], tr[:, 1] ** 2 + tr[:, 2] ** 2)
        assert abs(T / (math.pi / (TWO_PI * gs[r] * 1e6)) - 1) < 5e-3
        assert st[r]["accepted"] > 0 and st[r]["rhs_evals"] == 1 + 6 * (st[r]["accepted"] + st[r]["rejected"])
        assert st[r]["t"] == t_end
    wr = copy.deepcopy(w)
    ref = oracle_of(wr).run(wr.m0, wr.a0, t_end=t_end, tol=tol, sample_dt=sdt, trace_cap=cap)
    T_ref = rabi_period(ref.trace[:, 0], ref.trace[:, 1] ** 2 + ref.trace[:, 2] ** 2)
    T_gpu = rabi_period(trs[1][:, 0], trs[1][:, 1] ** 2 + trs[1][:, 2] ** 2)
    assert abs(T_gpu / T_ref - 1) < 5e-3


def test_resume_and_edge_cases(api):
    w = small_problem(8, 8, 2, 1, 1)
    with api.Batch(w, 2, precision="f64") as b:
        b.run(math.inf, fixed_dt=0.1e-12, max_steps=40)
        m1, a1 = b.get_m(), b.get_a()
    with api.Batch(w, 2, precision="f64") as b:
        b.run(math.inf, fixed_dt=0.1e-12, max_steps=15)
        b.run(math.inf, fixed_dt=0.1e-12, max_steps=25)
        m2, a2 = b.get_m(), b.get_a()
        st = b.stats()
        assert st[0]["accepted"] == 40 and st[0]["rhs_evals"] == 40 * 6 + 2      # k1 is re-evaluated per run
        # t_end already reached: nothing happens
        b.run(st[0]["t"], fixed_dt=0.1e-12)
        assert b.stats()[0]["accepted"] == 40
        # argument checks
        with pytest.raises(api.CavError):
            b.run(1e-9)                                  # neither tol nor fixed_dt
        with pytest.raises(api.CavError):
            b.run(1e-9, tol=1e-6, fixed_dt=1e-13)        # both
    assert np.array_equal(m1, m2) and np.array_equal(a1, a2)
    big = small_problem(33, 32, 1, 1, 1)                 # 1056 cells > 1024
    with pytest.raises(api.CavError) as e:
        api.Batch(big, 1)
    assert e.value.status == api.CAV_E_ARG


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_driven_sweep_fixed_steps(api, prec):
    """The paper's spectroscopy protocol in one launch: every replica (its own B0) gets the same Gaussian pulse on the
    cavity (cav_batch_set_drive), compared with the driven oracle replica by replica."""
    w = small_problem(8, 8, 2, 2, 1)
    if prec == "f32":
        w.m0 = w.m0.astype(np.float32).astype(np.float64)
    dt = 0.1e-12
    N = w.omega.size
    dr = dict(amp=np.array([3e10 + 1e10j, -2e10j]), t0=np.full(N, 30 * dt), sigma=np.full(N, 12 * dt), omega_d=w.omega * 1.02)
    ghz = np.array([9.0, 9.8, 10.6])
    B0 = np.array([[0.01, -0.02, W.b0_for_ghz(f)] for f in ghz])
    with api.Batch(w, 3, precision=prec, B0=B0) as b:
        api.cav_batch_set_drive(b.h, dr["amp"], dr["t0"], dr["sigma"], dr["omega_d"])
        b.run(math.inf, fixed_dt=dt, max_steps=80)
        m, a = b.get_m(), b.get_a()
    for r in range(3):
        wr = copy.deepcopy(w)
        wr.B0 = tuple(B0[r])
        ref = oracle_of(wr, drive=dr).run(wr.m0, wr.a0, fixed_dt=dt, max_steps=80)
        assert_parity(m[r], a[r], ref, prec)
    wr = copy.deepcopy(w); wr.B0 = tuple(B0[0])
    undriven = oracle_of(wr).run(wr.m0, wr.a0, fixed_dt=dt, max_steps=80)
    assert np.abs(a[0] - undriven.a).max() > 0.05 * np.abs(undriven.a).max()


def test_nonreciprocal_sweep(api):
    """cav_batch_set_backaction: every replica of a field sweep with g_b != g_f against the oracle."""
    w = small_problem(8, 8, 2, 2, 1)
    back = dict(g=0.25 * w.g, Gamma=2.0 * w.Gamma, Phi=w.Phi + 0.4)
    B0 = np.array([[0.01, -0.02, W.b0_for_ghz(f)] for f in (9.5, 10.5)])
    with api.Batch(w, 2, precision="f64", B0=B0) as b:
        api.cav_batch_set_backaction(b.h, back["g"], back["Gamma"], back["Phi"])
        b.run(math.inf, fixed_dt=0.1e-12, max_steps=80)
        m, a = b.get_m(), b.get_a()
    for r in range(2):
        wr = copy.deepcopy(w); wr.B0 = tuple(B0[r])
        ref = oracle_of(wr, backward=back).run(wr.m0, wr.a0, fixed_dt=0.1e-12, max_steps=80)
        assert_parity(m[r], a[r], ref, "f64")


@pytest.mark.parametrize("driven", [False, True])
def test_forced_rejections_match_oracle_per_replica(api, driven):
    """The controller's reject branch in the batch kernel: fp64, adaptive, dt_init = 2 ps on the 5 nm grid (ten times
    the stability limit) so the first steps are rejected, plus a 0.15 ps pulse in mid-run; three field values in one
    launch.  Accepted and rejected counts equal the oracle's for every replica, final state within 1e-10."""
    from test_gpu_parity import _reject_case
    w, dr = _reject_case(8, driven)
    ghz = np.array([9.9, 10.0, 10.1])
    B0 = np.array([[0.0, 0.0, W.b0_for_ghz(f)] for f in ghz])
    t_end = 8e-12
    with api.Batch(w, 3, precision="f64", B0=B0) as b:
        if dr:
            api.cav_batch_set_drive(b.h, dr["amp"], dr["t0"], dr["sigma"], dr["omega_d"])
        b.run(t_end, tol=1e-8, dt_init=2e-12)
        m, a, st = b.get_m(), b.get_a(), b.stats()
    for r, f in enumerate(ghz):
        wr = with_field(w, f)
        ref = oracle_of(wr, drive=dr).run(wr.m0, wr.a0, t_end=t_end, tol=1e-8, dt_init=2e-12)
        assert ref.rejected >= (8 if driven else 5)
        assert (st[r]["accepted"], st[r]["rejected"]) == (ref.accepted, ref.rejected), r
        assert st[r]["rhs_evals"] == ref.rhs_evals and st[r]["t"] == t_end
        assert abs(st[r]["dt_next"] / ref.dt - 1) < 1e-6
        assert_parity(m[r], a[r], ref, "f64")
