"""GPU parity of the joint launcher for sweeps of mid-size grids (cav_sweep_*, -m gpu): every member simulation
against its own fp64 oracle run (fixed step, north_star tolerances) and against the same simulation run alone."""
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
from test_gpu_parity import api, assert_parity, oracle_of, small_problem  # noqa: E402,F401

pytestmark = pytest.mark.gpu


@pytest.fixture()
def stream():
    import torch
    st = torch.cuda.Stream()            # the members of a sweep live on ONE stream
    yield st.cuda_stream
    st.synchronize()


def _members(n, shape=(64, 32, 8), N=2):
    ws = []
    for r in range(n):
        w = small_problem(*shape, N, 1, seed=7 + r)
        w.B0 = (0.01, -0.02, W.b0_for_ghz(9.6 + 0.2 * r))
        w.g = w.g * (1.0 + 0.1 * r)                       # mode parameters may differ too
        ws.append(w)
    return ws


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_sweep_fixed_steps_against_the_oracle(api, prec, stream):
    """Five simulations of 64 x 32 x 8 cells (32 plane-tiles each: blocks cross from one simulation into the next)."""
    ws = _members(5)
    for w in ws:
        if prec == "f32":
            w.m0 = w.m0.astype(np.float32).astype(np.float64)
            w.m0 /= np.linalg.norm(w.m0, axis=1, keepdims=True)
            w.u = w.u.astype(np.float32).astype(np.float64)
    sims = [api.Sim(w, precision=prec, stream=stream) for w in ws]
    sw = api.cav_sweep_create(sims)
    try:
        api.cav_sweep_run(sw, math.inf, fixed_dt=0.1e-12, max_steps=30)
        api.cav_sweep_run(sw, math.inf, fixed_dt=0.1e-12, max_steps=30)          # resume: FSAL slopes kept per simulation
        for w, sim in zip(ws, sims):
            ref = oracle_of(w).run(w.m0, w.a0, fixed_dt=0.1e-12, max_steps=60)
            st = api.cav_get_stats(sim.h)
            assert st["accepted"] == 60 and st["rhs_evals"] == 361
            assert_parity(sim.get_m(), sim.get_a(), ref, prec)
    finally:
        api.cav_sweep_destroy(sw)
        for sim in sims:
            sim.close()


def test_sweep_adaptive_members_keep_their_own_step_sequence(api, stream):
    """fp64, adaptive with dt_init far too large: every member rejects and adapts on its own (different B0 and coupling),
    lands exactly on t_end, fills its own trace, and agrees with the same simulation run alone (same controller, same
    bits up to the summation order of the overlap sums) and with the oracle's accepted / rejected counts."""
    ws = _members(6, shape=(64, 16, 8))
    t_end, sdt = 6e-12, 1e-12
    solo = []
    for w in ws:
        with api.Sim(w, precision="f64", path=api.CAV_PATH_TMA) as sim:
            api.cav_set_trace(sim.h, sdt, 6)
            api.cav_run(sim.h, t_end, tol=1e-8, dt_init=2e-12)
            solo.append((sim.get_m(), sim.get_a(), api.cav_get_stats(sim.h), api.cav_get_trace(sim.h)))
    sims = [api.Sim(w, precision="f64", stream=stream) for w in ws]
    for sim in sims:
        api.cav_set_trace(sim.h, sdt, 6)
    sw = api.cav_sweep_create(sims)
    try:
        api.cav_sweep_run(sw, t_end, tol=1e-8, dt_init=2e-12)
        counts = set()
        for w, sim, (m1, a1, st1, tr1) in zip(ws, sims, solo):
            st = api.cav_get_stats(sim.h)
            ref = oracle_of(w).run(w.m0, w.a0, t_end=t_end, tol=1e-8, dt_init=2e-12, sample_dt=sdt, trace_cap=6)
            assert st["t"] == t_end and st["rejected"] > 0
            assert (st["accepted"], st["rejected"]) == (st1["accepted"], st1["rejected"]) == (ref.accepted, ref.rejected)
            counts.add(st["accepted"])
            m, a = sim.get_m(), sim.get_a()
            assert np.abs(m - m1).max() < 1e-12 and np.abs(a - a1).max() < 1e-12 * np.abs(a1).max()
            assert_parity(m, a, ref, "f64")
            tr = api.cav_get_trace(sim.h)
            assert tr.shape == tr1.shape == (6, 1 + 8 + 3) and np.abs(tr - ref.trace).max() < 1e-9
        assert len(counts) > 1                   # the members really took different numbers of steps
    finally:
        api.cav_sweep_destroy(sw)
        for sim in sims:
            sim.close()


def test_sweep_of_cfg2_field_points(api, stream):
    """BASELINE.json configs[1] as (9 of) its field points, fp32, adaptive tol 1e-6: each member against its solo run."""
    ghz = W.cfg2_sweep_ghz()[::5]
    ws = [W.cfg2(f_kittel_ghz=float(f), seed=2000 + i) for i, f in enumerate(ghz)]
    solo = []
    for w in ws:
        with api.Sim(w, precision="f32", path=api.CAV_PATH_TMA) as sim:
            api.cav_run_steps(sim.h, math.inf, tol=1e-6, max_steps=80)
            solo.append((sim.get_m(), sim.get_a(), api.cav_get_stats(sim.h)))
    sims = [api.Sim(w, precision="f32", stream=stream) for w in ws]
    sw = api.cav_sweep_create(sims)
    try:
        api.cav_sweep_run(sw, math.inf, tol=1e-6, max_steps=80)
        for sim, (m1, a1, st1) in zip(sims, solo):
            st = api.cav_get_stats(sim.h)
            assert st["accepted"] + st["rejected"] == 80 and abs(st["t"] / st1["t"] - 1) < 1e-4
            assert np.abs(sim.get_m() - m1).max() < 2e-5
            assert np.abs(sim.get_a() - a1).max() <= 1e-3 * np.abs(a1).max() + 1e-12
    finally:
        api.cav_sweep_destroy(sw)
        for sim in sims:
            sim.close()


def test_sweep_argument_checks(api, stream):
    ws = _members(2)
    other = small_problem(64, 32, 4, 2, 1)
    sims = [api.Sim(w, precision="f64", stream=stream) for w in ws]
    so = api.Sim(other, precision="f64", stream=stream)
    lone = api.Sim(ws[1], precision="f64")                            # on its own stream
    try:
        with pytest.raises(api.CavError) as e:
            api.cav_sweep_create([sims[0], so])                       # different grids
        assert e.value.status == api.CAV_E_ARG
        with pytest.raises(api.CavError) as e:
            api.cav_sweep_create([sims[0], lone])                     # different streams
        assert e.value.status == api.CAV_E_ARG
        with pytest.raises(api.CavError) as e:
            api.cav_sweep_create([sims[0], sims[0]])                  # the same handle twice
        assert e.value.status == api.CAV_E_ARG
        with pytest.raises(api.CavError) as e:
            api.cav_sweep_create(sims)                                # 64 plane-tiles in total: fewer than SMs
        assert e.value.status == api.CAV_E_UNSUPPORTED
    finally:
        for s in sims + [so, lone]:
            s.close()


def test_sweep_refuses_members_with_a_variant_switched_on(api, stream):
    """Polarisation (and the dipolar field, the split integrator) live outside the joint kernels: refused when the sweep
    is created, and when it is switched on in a member afterwards."""
    ws = _members(6)
    sims = [api.Sim(w, precision="f64", stream=stream) for w in ws]
    sw = None
    try:
        api.cav_set_polarisation(sims[2].h, [[0.0, 1.0, 0.0], [1.0, 0.0, 0.0]])
        with pytest.raises(api.CavError) as e:
            api.cav_sweep_create(sims)
        assert e.value.status == api.CAV_E_UNSUPPORTED
        api.cav_set_polarisation(sims[2].h, None)
        sw = api.cav_sweep_create(sims)
        api.cav_sweep_run(sw, math.inf, fixed_dt=0.05e-12, max_steps=2)
        api.cav_set_polarisation(sims[4].h, [[0.0, 1.0, 0.0], [1.0, 0.0, 0.0]])
        with pytest.raises(api.CavError) as e:
            api.cav_sweep_run(sw, math.inf, fixed_dt=0.05e-12, max_steps=2)
        assert e.value.status == api.CAV_E_UNSUPPORTED
        api.cav_set_polarisation(sims[4].h, None)
        api.cav_sweep_run(sw, math.inf, fixed_dt=0.05e-12, max_steps=2)
        for sim in sims:
            assert api.cav_get_stats(sim.h)["accepted"] == 4
    finally:
        if sw is not None:
            api.cav_sweep_destroy(sw)
        for s in sims:
            s.close()


def test_members_stay_ordinary_handles(api, stream):
    """After a joint run a member can go on alone (cav_run on the single handle), a member that has already reached t_end
    is skipped by the next joint run, and the on-device Fourier sums accumulate per member."""
    from oracle import dft
    ws = _members(5)
    sims = [api.Sim(w, precision="f64", stream=stream) for w in ws]
    K, lo, hi = 17, 2 * math.pi * 9e9, 2 * math.pi * 11e9
    for sim in sims:
        api.cav_set_trace(sim.h, 1e-12, 8)
        api.cav_set_spectrum(sim.h, K, lo, hi)
    sw = api.cav_sweep_create(sims)
    try:
        api.cav_sweep_run(sw, math.inf, fixed_dt=0.1e-12, max_steps=40)
        # member 1 alone for 20 more steps, then everybody to t = 8 ps: member 1 has less to do
        api.cav_run_steps(sims[1].h, math.inf, fixed_dt=0.1e-12, max_steps=20)
        api.cav_sweep_run(sw, 8e-12, fixed_dt=0.1e-12)
        api.cav_sweep_run(sw, 8e-12, fixed_dt=0.1e-12)                 # everybody is at t_end: nothing happens
        for w, sim in zip(ws, sims):
            ref = oracle_of(w).run(w.m0, w.a0, fixed_dt=0.1e-12, max_steps=80, sample_dt=1e-12, trace_cap=8)
            st = api.cav_get_stats(sim.h)
            assert st["accepted"] == 80 and abs(st["t"] - 8e-12) < 1e-24
            assert_parity(sim.get_m(), sim.get_a(), ref, "f64")
            tr = api.cav_get_trace(sim.h)
            assert tr.shape[0] == 8 and np.abs(tr - ref.trace).max() < 1e-9
            X, ns = api.cav_get_spectrum(sim.h, K, 2)
            ref_a = dft(tr[:, 0], tr[:, 1] + 1j * tr[:, 2], np.linspace(lo, hi, K))
            assert ns == 8 and np.abs(X[:, 0] - ref_a).max() <= 1e-11 * np.abs(ref_a).max()
    finally:
        api.cav_sweep_destroy(sw)
        for sim in sims:
            sim.close()


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_sweep_of_antiferromagnets(api, prec, stream):
    """The paper's AFM protocol is a field sweep too: six two-sublattice members of cfg4's recipe on
    64 x 32 x 8 cells with dissipative coupling and different fields, each against its own oracle run."""
    ws = []
    for r in range(6):
        w = W.cfg4(nx=64, ny=32, nz=8, seed=4000 + r, dissipative=True)
        w.B0 = (0.0, 0.0, 0.05 * r)
        w.a0 = np.array([2e-3 + 1e-3j])
        if prec == "f32":
            w.m0 = w.m0.astype(np.float32).astype(np.float64)
            w.m0 /= np.linalg.norm(w.m0, axis=1, keepdims=True)
        ws.append(w)
    sims = [api.Sim(w, precision=prec, stream=stream) for w in ws]
    sw = api.cav_sweep_create(sims)
    try:
        api.cav_sweep_run(sw, math.inf, fixed_dt=0.02e-12, max_steps=60)
        for w, sim in zip(ws, sims):
            ref = oracle_of(w).run(w.m0, w.a0, fixed_dt=0.02e-12, max_steps=60)
            if prec == "f64":
                assert_parity(sim.get_m(), sim.get_a(), ref, prec)
            else:
                assert np.abs(sim.get_m() - ref.m).max() <= 1e-4
                assert np.abs(sim.get_a() - ref.a).max() <= 1e-4 * np.abs(ref.a).max()
    finally:
        api.cav_sweep_destroy(sw)
        for sim in sims:
            sim.close()
