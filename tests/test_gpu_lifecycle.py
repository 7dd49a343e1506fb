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
    w = small_problem(128, 24, 20, 2, 1)                       # TMA path (480 plane-tiles)
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
