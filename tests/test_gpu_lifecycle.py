"""Handle life cycle on the device (-m gpu): creating, configuring, running and destroying handles of every kind over and
over returns all device memory (no leak in cav_destroy / cav_sweep_destroy / cav_batch_destroy, the run graphs, the
dipolar-field plan with its cuFFT plans, spectra, traces, polarisation tables)."""
import math

import numpy as np
import pytest

from test_gpu_parity import api, small_problem  # noqa: F401

pytestmark = pytest.mark.gpu


def _free(torch):
    torch.cuda.synchronize()
    return torch.cuda.mem_get_info()[0]


def _cycle(api, torch, k):
    w = small_problem(128, 32, 24, 2, 1)                       # TMA path (98 304 cells)
    st = torch.cuda.Stream()
    with api.Sim(w, precision="f32", stream=st.cuda_stream) as sim:
        api.cav_set_trace(sim.h, 1e-12, 64)
        api.cav_set_spectrum(sim.h, 33, 2 * math.pi * 9e9, 2 * math.pi * 11e9)
        api.cav_run_steps(sim.h, math.inf, tol=1e-6, max_steps=9)
        if k % 2:
            api.cav_set_polarisation(sim.h, [[0.0, 1.0, 0.0], [1.0, 0.0, 0.0]])
            api.cav_run_steps(sim.h, math.inf, tol=1e-6, max_steps=3)
        api.cav_sync(sim.h)
    wd = small_problem(24, 10, 6, 1, 1)
    with api.Sim(wd, precision="f64", stream=st.cuda_stream) as sim:
        api.cav_set_demag(sim.h, 1)                           # plan, tensor table, cuFFT plans, captured graph
        api.cav_run_steps(sim.h, math.inf, tol=1e-8, max_steps=3)
        api.cav_set_demag(sim.h, 0)
        api.cav_set_demag(sim.h, 1)
        api.cav_run_steps(sim.h, math.inf, fixed_dt=1e-14, max_steps=2)
        api.cav_sync(sim.h)
    ws = [small_problem(64, 32, 8, 2, 1, seed=11 + r) for r in range(5)]
    sims = [api.Sim(x, precision="f32", stream=st.cuda_stream) for x in ws]
    sw = api.cav_sweep_create(sims)
    api.cav_sweep_run(sw, math.inf, tol=1e-6, max_steps=5)
    for s in sims:
        api.cav_sync(s.h)
    api.cav_sweep_destroy(sw)
    for s in sims:
        s.close()
    wb = small_problem(8, 8, 4, 1, 1)
    with api.Batch(wb, 7, precision="f64") as b:
        b.run(math.inf, tol=1e-8, max_steps=5)
        b.get_a()
    st.synchronize()


def test_handles_give_their_device_memory_back(api):
    import torch
    _cycle(api, torch, 0)                                       # loads modules, creates cuFFT's and the allocator's one-time state
    _cycle(api, torch, 1)
    free0 = _free(torch)
    for k in range(12):
        _cycle(api, torch, k)
    free1 = _free(torch)
    # the driver hands memory out in 2 MiB granules and keeps a few cached: a leak of one handle per cycle would be >= 100 MB here
    assert free0 - free1 < 16 * 2 ** 20, (free0, free1)


def test_setters_in_any_order_leave_a_consistent_handle(api):
    """Settings that replace device tables or switch kernel families, applied between runs in orders a user might try: every
    run afterwards matches a fresh handle configured directly (bitwise: same kernels, same inputs)."""
    from test_gpu_parity import oracle_of
    w = small_problem(128, 32, 24, 2, 1)                        # 98 304 cells: beyond the cooperative kernel, TMA path
    p = [[0.0, 1.0, 0.0], [0.6, 0.0, 0.8]]

    def final(configure, steps=6):
        with api.Sim(w, precision="f64") as sim:
            configure(sim)
            api.cav_set_m(sim.h, np.ascontiguousarray(w.m0))
            api.cav_set_a(sim.h, w.a0)
            api.cav_set_time(sim.h, 0.0)
            api.cav_run_steps(sim.h, math.inf, fixed_dt=0.05e-12, max_steps=steps)
            return sim.get_m(), sim.get_a(), api.cav_get_kernel_path(sim.h)

    def modes(sim):
        api.cav_set_modes(sim.h, np.ascontiguousarray(w.u), w.omega, w.kappa, w.g, w.Gamma, w.Phi)

    # polarisation: direct / after a detour through the dipolar field, a spectrum, a run and a new mode set
    m0, a0, path0 = final(lambda s: api.cav_set_polarisation(s.h, p))

    def detour(sim):
        api.cav_set_demag(sim.h, 1)
        api.cav_run_steps(sim.h, math.inf, fixed_dt=0.05e-12, max_steps=2)
        api.cav_set_demag(sim.h, 0)
        api.cav_set_trace(sim.h, 0.1e-12, 8)
        api.cav_set_spectrum(sim.h, 9, 5e10, 7e10)
        api.cav_run_steps(sim.h, math.inf, fixed_dt=0.05e-12, max_steps=2)
        modes(sim)                                    # drops polarisation, spectrum, drive
        api.cav_set_spectrum(sim.h, 0)
        api.cav_set_trace(sim.h, 0.0, 0)
        api.cav_set_polarisation(sim.h, p)
    m1, a1, path1 = final(detour)
    assert path0 == path1 == api.CAV_PATH_TMA
    assert np.array_equal(m0, m1) and np.array_equal(a0, a1)
    ref = oracle_of(w, pol=p).run(w.m0, w.a0, fixed_dt=0.05e-12, max_steps=6)
    assert np.abs(m0 - ref.m).max() <= 1e-10 and np.abs(a0 - ref.a).max() <= 1e-10 * np.abs(ref.a).max()

    # the dipolar field: direct / after polarisation was set and taken back, on a forced generic path and back to auto
    md, ad, pathd = final(lambda s: api.cav_set_demag(s.h, 1), steps=3)

    def detour2(sim):
        api.cav_set_polarisation(sim.h, p)
        api.cav_run_steps(sim.h, math.inf, fixed_dt=0.05e-12, max_steps=2)
        api.cav_set_polarisation(sim.h, None)
        api.cav_set_kernel_path(sim.h, api.CAV_PATH_GENERIC)
        api.cav_set_kernel_path(sim.h, api.CAV_PATH_AUTO)
        api.cav_set_demag(sim.h, 1)
    me, ae, pathe = final(detour2, steps=3)
    assert pathd == pathe == api.CAV_PATH_GENERIC
    assert np.array_equal(md, me) and np.array_equal(ad, ae)
