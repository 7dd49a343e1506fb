"""Seeded random shapes (-m gpu): tile edges, ragged tails and transform lengths that no hand-picked case may hit.
(1) the TMA kernels against the generic kernels on ~100 random grids / mode counts / sublattice counts / precisions;
(2) the dipolar field (every pruned-transform length combination) against the oracle's direct sum on ~55 small grids."""
import copy
import math

import numpy as np
import pytest

from test_gpu_parity import api, oracle_of, small_problem  # noqa: F401

pytestmark = pytest.mark.gpu


def test_tma_and_generic_kernels_agree_on_random_shapes(api):
    rng = np.random.default_rng(12345)
    compared = 0
    for _ in range(120):
        prec = "f64" if rng.random() < 0.5 else "f32"
        es = 8 if prec == "f64" else 4
        nx = int(rng.integers(1, 40)) * (16 // es) if rng.random() < 0.7 else int(rng.integers(1, 300))
        ny, nz = int(rng.integers(1, 40)), int(rng.integers(1, 40))
        n_sub = int(rng.integers(1, 3))
        N = int(rng.choice([0, 1, 2, 3, 5, 8, 9, 20, 32]))
        w = small_problem(nx, ny, nz, N, n_sub, seed=int(rng.integers(1, 1000)))
        dt = 0.05e-12 if n_sub == 1 else 0.01e-12
        out = {}
        for name, path in (("tma", api.CAV_PATH_TMA), ("generic", api.CAV_PATH_GENERIC)):
            try:
                sim = api.Sim(w, precision=prec, path=path)
            except api.CavError as e:              # unaligned rows: a small grid has no TMA kernels, a large one (padded inside the library) only those
                assert e.status == api.CAV_E_UNSUPPORTED and (nx * es) % 16 != 0
                out = None
                break
            with sim:
                api.cav_run_steps(sim.h, math.inf, fixed_dt=dt, max_steps=4)
                out[name] = (sim.get_m().astype(np.float64), sim.get_a())
        if out is None:
            continue
        dm = np.abs(out["tma"][0] - out["generic"][0]).max()
        da = np.abs(out["tma"][1] - out["generic"][1]).max() if N else 0.0
        assert dm <= (1e-12 if prec == "f64" else 2e-6), (prec, nx, ny, nz, n_sub, N, dm)
        assert da <= (1e-12 if prec == "f64" else 1e-6) * max(np.abs(out["generic"][1]).max(), 1e-3) if N else True, (prec, nx, ny, nz, n_sub, N, da)
        compared += 1
    assert compared >= 80


def test_dipolar_field_on_random_small_grids(api):
    rng = np.random.default_rng(777)
    done = 0
    for _ in range(60):
        nx, ny, nz = int(rng.integers(1, 24)), int(rng.integers(1, 24)), int(rng.integers(1, 12))
        if nx * ny * nz > 2500:
            continue
        n_sub = int(rng.integers(1, 3))
        N = int(rng.choice([0, 1, 2]))
        w = small_problem(nx, ny, nz, N, n_sub, seed=int(rng.integers(1, 1000)))
        for prec in ("f64", "f32"):
            w2 = w
            if prec == "f32":
                w2 = copy.deepcopy(w)
                w2.m0 = w.m0.astype(np.float32).astype(np.float64)
                w2.m0 /= np.linalg.norm(w2.m0, axis=1, keepdims=True)
                w2.u = w.u.astype(np.float32).astype(np.float64)
            dm_ref, _, _ = oracle_of(w2, demag=True).rhs(w2.m0, w2.a0)
            with api.Sim(w2, precision=prec) as sim:
                api.cav_set_demag(sim.h, 1)
                dm = np.empty(sim.shape_m, dtype=sim.np_dtype)
                api.cav_get_dmdt(sim.h, dm)
            err = np.abs(dm - dm_ref).max() / np.abs(dm_ref).max()
            assert err <= (5e-13 if prec == "f64" else 3e-5), (prec, nx, ny, nz, n_sub, N, err)
        done += 1
    assert done >= 45


def test_small_grid_kernels_and_generic_kernels_agree_on_random_adaptive_runs(api):
    """Grids in the range of the single-block and the cooperative kernel (CAV_PATH_AUTO) against the generic stage kernels:
    short adaptive runs with a too large first step - in fp64 the same accepted / rejected counts and the same state."""
    rng = np.random.default_rng(4242)
    paths = set()
    for _ in range(100):
        prec = "f64" if rng.random() < 0.5 else "f32"
        if rng.random() < 0.5:
            nx, ny, nz = int(rng.integers(8, 70)), int(rng.integers(4, 40)), int(rng.integers(1, 30))
        else:
            nx, ny, nz = int(rng.integers(1, 17)), int(rng.integers(1, 9)), int(rng.integers(1, 9))
        if nx * ny * nz > 75000:
            continue
        n_sub = int(rng.integers(1, 3))
        N = int(rng.choice([0, 1, 2, 3, 8, 32]))
        w = small_problem(nx, ny, nz, N, n_sub, seed=int(rng.integers(1, 1000)))
        dt = 0.05e-12 if n_sub == 1 else 0.01e-12
        out = {}
        for name, path in (("auto", None), ("generic", api.CAV_PATH_GENERIC)):
            with api.Sim(w, precision=prec, path=path) as sim:
                api.cav_run(sim.h, 8 * dt, tol=1e-7 if prec == "f64" else 1e-5, dt_init=3 * dt)
                out[name] = (sim.get_m().astype(np.float64), sim.get_a(), api.cav_get_stats(sim.h))
                if name == "auto":
                    paths.add(api.cav_get_kernel_path(sim.h))
        dm = np.abs(out["auto"][0] - out["generic"][0]).max()
        assert dm <= (1e-11 if prec == "f64" else 5e-6), (prec, nx, ny, nz, n_sub, N, dm)
        if prec == "f64":
            sa, sg = out["auto"][2], out["generic"][2]
            assert (sa["accepted"], sa["rejected"]) == (sg["accepted"], sg["rejected"]), (nx, ny, nz, n_sub, N)
            if N:
                assert np.abs(out["auto"][1] - out["generic"][1]).max() <= 1e-11 * max(np.abs(out["generic"][1]).max(), 1e-3)
    assert {api.CAV_PATH_BLOCK, api.CAV_PATH_COOP} <= paths


def test_joint_sweeps_of_random_shapes_equal_solo_runs(api):
    """Random member counts, shapes, mode counts, sublattices and precisions: members of a joint sweep (adaptive, first step
    too large) take the step sequence of the same simulation run alone on the TMA kernels and end in the same state."""
    import torch
    import cavmag_workloads as W
    rng = np.random.default_rng(99)
    st = torch.cuda.Stream()
    done = 0
    for _ in range(25):
        prec = "f64" if rng.random() < 0.5 else "f32"
        es = 8 if prec == "f64" else 4
        n_sub = int(rng.integers(1, 3))
        N = int(rng.choice([1, 2])) if n_sub == 2 else int(rng.choice([1, 2, 3, 8]))
        nx = int(rng.integers(2, 12)) * 16 // es * (2 if es == 4 else 4) // 2
        ny, nz = int(rng.integers(4, 40)), int(rng.integers(2, 16))
        R = int(rng.integers(3, 40))
        dt = 0.05e-12 if n_sub == 1 else 0.01e-12
        tol = 1e-7 if prec == "f64" else 1e-5
        ws = []
        for r in range(R):
            w = small_problem(nx, ny, nz, N, n_sub, seed=7 + (r % 3))
            w.B0 = (0.01, -0.02, W.b0_for_ghz(9.0 + 0.05 * r))
            ws.append(w)
        sims = [api.Sim(w, precision=prec, stream=st.cuda_stream) for w in ws]
        sw = None
        try:
            try:
                sw = api.cav_sweep_create(sims)
            except api.CavError as e:                  # fewer plane-tiles in total than SMs
                assert e.status == api.CAV_E_UNSUPPORTED
                continue
            api.cav_sweep_run(sw, 10 * dt, tol=tol, dt_init=3 * dt)
            for r in sorted(set(int(x) for x in rng.integers(0, R, 2))):
                with api.Sim(ws[r], precision=prec, path=api.CAV_PATH_TMA) as solo:
                    api.cav_run(solo.h, 10 * dt, tol=tol, dt_init=3 * dt)
                    ms, as_, ss = solo.get_m(), solo.get_a(), api.cav_get_stats(solo.h)
                m, a, s1 = sims[r].get_m(), sims[r].get_a(), api.cav_get_stats(sims[r].h)
                assert (s1["accepted"], s1["rejected"]) == (ss["accepted"], ss["rejected"]), (prec, nx, ny, nz, n_sub, N, R, r)
                assert np.abs(m.astype(np.float64) - ms.astype(np.float64)).max() <= (1e-12 if prec == "f64" else 1e-6)
                assert np.abs(a - as_).max() <= (1e-12 if prec == "f64" else 1e-6) * max(np.abs(as_).max(), 1e-3)
            done += 1
        finally:
            if sw is not None:
                api.cav_sweep_destroy(sw)
            for s in sims:
                s.close()
    assert done >= 15


def test_random_feature_combinations_agree_across_kernel_families(api):
    """Drive, non-reciprocal coupling, per-mode polarisation, sum-u normalisation, renormalisation off, trace, Fourier sums,
    fixed or adaptive stepping - switched on at random - on the TMA kernels, the generic kernels and whatever CAV_PATH_AUTO
    picks (single-block / cooperative kernel here): the same state, trace, spectrum and step counts in fp64."""
    rng = np.random.default_rng(2024)
    two_pi = 2 * math.pi
    families = set()
    for _ in range(60):
        n_sub = int(rng.integers(1, 3))
        N = int(rng.choice([1, 2, 3, 8]))
        nx = int(rng.integers(2, 10)) * 8
        ny, nz = int(rng.integers(3, 30)), int(rng.integers(2, 24))
        w = small_problem(nx, ny, nz, N, n_sub, seed=int(rng.integers(1, 1000)))
        dt = 0.05e-12 if n_sub == 1 else 0.01e-12
        f = dict(drive=rng.random() < 0.5, back=rng.random() < 0.5, pol=rng.random() < 0.5, sumu=rng.random() < 0.3,
                 norenorm=rng.random() < 0.3, spec=rng.random() < 0.5, adaptive=rng.random() < 0.5)
        amp = (rng.normal(size=N) + 1j * rng.normal(size=N)) * 1e9
        gb = two_pi * 1e6 * rng.uniform(5, 40, size=N)
        p = rng.normal(size=(N, 3))
        p /= np.linalg.norm(p, axis=1, keepdims=True)
        if f["sumu"]:
            w.u = w.u + 0.7                              # keeps sum u away from zero
        out = {}
        for name, path in (("tma", api.CAV_PATH_TMA), ("generic", api.CAV_PATH_GENERIC), ("auto", None)):
            with api.Sim(w, precision="f64", path=path, renormalize=not f["norenorm"],
                         overlap_norm=api.CAV_NORM_SUM_U if f["sumu"] else api.CAV_NORM_NCELLS) as sim:
                if f["drive"]:
                    api.cav_set_drive(sim.h, amp, 2 * dt, 3 * dt, two_pi * 10e9)
                if f["back"]:
                    api.cav_set_backaction(sim.h, gb)
                if f["pol"]:
                    api.cav_set_polarisation(sim.h, p)
                api.cav_set_trace(sim.h, 2 * dt, 4)
                if f["spec"]:
                    api.cav_set_spectrum(sim.h, 5, two_pi * 9e9, two_pi * 11e9)
                if f["adaptive"]:
                    api.cav_run(sim.h, 8 * dt, tol=1e-8, dt_init=3 * dt)
                else:
                    api.cav_run_steps(sim.h, math.inf, fixed_dt=dt, max_steps=8)
                X = api.cav_get_spectrum(sim.h, 5, N)[0] if f["spec"] else np.zeros(1)
                out[name] = (sim.get_m(), sim.get_a(), api.cav_get_trace(sim.h), X, api.cav_get_stats(sim.h))
                families.add(api.cav_get_kernel_path(sim.h))
        ref = out["generic"]
        for name in ("tma", "auto"):
            o = out[name]
            what = (name, nx, ny, nz, n_sub, N, f)
            assert np.abs(o[0] - ref[0]).max() <= 1e-11, what
            assert np.abs(o[1] - ref[1]).max() <= 1e-11 * max(np.abs(ref[1]).max(), 1e-6), what
            assert o[2].shape == ref[2].shape and np.abs(o[2] - ref[2]).max() <= 1e-10 * max(np.abs(ref[2]).max(), 1e-6), what
            assert np.abs(o[3] - ref[3]).max() <= 1e-10 * max(np.abs(ref[3]).max(), 1e-6), what
            assert (o[4]["accepted"], o[4]["rejected"]) == (ref[4]["accepted"], ref[4]["rejected"]), what
    assert {api.CAV_PATH_TMA, api.CAV_PATH_GENERIC, api.CAV_PATH_COOP} <= families


def test_random_batches_equal_generic_single_runs(api):
    """cav_batch_run on random tiny grids (up to 1024 cells), replica counts, mode counts, sublattices, precisions, with a
    drive and a polarisation switched on at random: a replica equals the same problem run alone on the generic kernels."""
    import cavmag_workloads as W
    rng = np.random.default_rng(31)
    two_pi = 2 * math.pi
    for _ in range(40):
        prec = "f64" if rng.random() < 0.6 else "f32"
        n_sub = int(rng.integers(1, 3))
        N = int(rng.choice([0, 1, 2, 3, 8]))
        while True:
            nx, ny, nz = int(rng.integers(1, 17)), int(rng.integers(1, 12)), int(rng.integers(1, 12))
            if nx * ny * nz <= 1024:
                break
        R = int(rng.integers(1, 12))
        w = small_problem(nx, ny, nz, N, n_sub, seed=int(rng.integers(1, 1000)))
        dt = 0.05e-12 if n_sub == 1 else 0.01e-12
        B0 = np.array([[0.01 * r, -0.02, W.b0_for_ghz(9.0 + 0.3 * r)] for r in range(R)])
        f = dict(drive=N > 0 and rng.random() < 0.4, pol=N > 0 and rng.random() < 0.4, adaptive=rng.random() < 0.6)
        amp = (rng.normal(size=max(N, 1)) + 1j * rng.normal(size=max(N, 1)))[:N] * 1e9
        p = rng.normal(size=(max(N, 1), 3))[:N]
        if N:
            p /= np.linalg.norm(p, axis=1, keepdims=True)
        tol = 1e-8 if prec == "f64" else 1e-5
        with api.Batch(w, R, precision=prec, B0=B0) as b:
            if f["drive"]:
                api.cav_batch_set_drive(b.h, amp, 2 * dt, 3 * dt, two_pi * 10e9)
            if f["pol"]:
                api.cav_batch_set_polarisation(b.h, p)
            if f["adaptive"]:
                b.run(8 * dt, tol=tol, dt_init=3 * dt)
            else:
                b.run(math.inf, fixed_dt=dt, max_steps=8)
            mb, ab, sb = b.get_m(), b.get_a(), b.stats()
        for r in sorted(set(int(x) for x in rng.integers(0, R, 2))):
            w2 = copy.deepcopy(w)
            w2.B0 = tuple(B0[r])
            with api.Sim(w2, precision=prec, path=api.CAV_PATH_GENERIC) as sim:
                if f["drive"]:
                    api.cav_set_drive(sim.h, amp, 2 * dt, 3 * dt, two_pi * 10e9)
                if f["pol"]:
                    api.cav_set_polarisation(sim.h, p)
                if f["adaptive"]:
                    api.cav_run(sim.h, 8 * dt, tol=tol, dt_init=3 * dt)
                else:
                    api.cav_run_steps(sim.h, math.inf, fixed_dt=dt, max_steps=8)
                ms, as_, ss = sim.get_m(), sim.get_a(), api.cav_get_stats(sim.h)
            what = (prec, nx, ny, nz, n_sub, N, R, r, f)
            assert np.abs(mb[r].astype(np.float64) - ms.astype(np.float64)).max() <= (1e-11 if prec == "f64" else 5e-6), what
            if prec == "f64":
                assert (sb[r]["accepted"], sb[r]["rejected"]) == (ss["accepted"], ss["rejected"]), what
                if N:
                    assert np.abs(ab[r] - as_).max() <= 1e-11 * max(np.abs(as_).max(), 1e-6), what
