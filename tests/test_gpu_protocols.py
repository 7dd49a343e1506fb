"""GPU runs of the paper's own protocols and of flags the other files do not reach (-m gpu): the anticrossing sweep read
out with the on-device Fourier sums, the mode-profile selection rule, and the
renormalisation switch (G13), all through the C ABI and against the oracle / the paper's closed forms."""
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
from test_gpu_parity import PATHS, api, assert_parity, open_sim, oracle_of, small_problem  # noqa: E402,F401

pytestmark = pytest.mark.gpu
TWO_PI = 2.0 * math.pi
GAMMA = 1.76e11


@pytest.mark.parametrize("path", PATHS)
@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_renormalisation_off_matches_oracle(api, path, prec):
    """cav_params.renormalize = 0: the 5th-order solution is taken as it is (|m| drifts at O(dt^5) per step)."""
    w = small_problem(40, 9, 7, 3, 1)
    if prec == "f32":
        w.m0 = w.m0.astype(np.float32).astype(np.float64)
        w.m0 /= np.linalg.norm(w.m0, axis=1, keepdims=True)
        w.u = w.u.astype(np.float32).astype(np.float64)
    ref = oracle_of(w, renormalize=False).run(w.m0, w.a0, fixed_dt=0.15e-12, max_steps=150)
    with open_sim(api, w, prec, path, renormalize=False) as sim:
        api.cav_run_steps(sim.h, math.inf, fixed_dt=0.15e-12, max_steps=150)
        m, a = sim.get_m(), sim.get_a()
    assert_parity(m, a, ref, prec)
    drift = np.abs(np.linalg.norm(ref.m, axis=1) - 1).max()
    assert drift > 1e-9                                           # the switch does something at this step size
    if prec == "f64":
        assert abs(np.abs(np.linalg.norm(m, axis=1) - 1).max() / drift - 1) < 1e-3


@pytest.mark.parametrize("path", PATHS)
def test_selection_rule_on_the_device(api, path):
    """PAPER.md:263-267 (Sim 4): a uniform precession does not couple to the profiles cos(n pi x/Lx), n >= 1, on the
    centred grid: their overlap vanishes to rounding and their amplitudes stay at zero, while the uniform mode exchanges
    energy with the magnet."""
    nx, ny, nz = 32, 8, 4
    w = W.macrospin(5.0, [5.0, 5.0, 5.0], 50.0, 1.0, alpha=1e-4, tilt=0.05, n=2)
    w.nx, w.ny, w.nz = nx, ny, nz
    w.m0 = np.broadcast_to(w.m0[:, :, :1, :1, :1], (1, 3, nz, ny, nx)).copy()
    w.u = np.stack([np.ones((nz, ny, nx)), W.cosine_profile(1, 0, 0, nx, ny, nz), W.cosine_profile(2, 0, 0, nx, ny, nz)])
    with open_sim(api, w, "f64", path) as sim:
        api.cav_set_trace(sim.h, 0.2e-9, 1)
        api.cav_run(sim.h, 0.2e-9, tol=1e-8)
        a = sim.get_a()
        row = api.cav_get_trace(sim.h)[0]
    S = row[1 + 6:1 + 12:2] + 1j * row[2 + 6:2 + 12:2]
    assert abs(S[0]) > 0.04                                        # <1 . m^-> = sin(tilt)
    assert abs(S[1]) < 1e-15 and abs(S[2]) < 1e-15
    assert abs(a[0]) > 1e-4 and abs(a[1]) < 1e-12 * abs(a[0]) and abs(a[2]) < 1e-12 * abs(a[0])


def test_anticrossing_sweep_read_out_on_the_device(api):
    """The paper's Sim 1 protocol in one launch: a field sweep across the cavity resonance
    (g/2pi = 50 MHz at 5 GHz, a(0) = 0.01), all members in one device-side loop (cav_sweep_run), spectra
    |X_a|^2 + |X_S|^2 accumulated on the device (cav_set_spectrum) - no trace leaves the GPU.  The two peaks of every
    member follow Eq. 6 within the frequency resolution; the minimum gap is 2g/2pi = 100 MHz."""
    import torch
    st = torch.cuda.Stream()
    f_m = np.linspace(4.90, 5.10, 9)
    g, f_c = 50e6, 5e9
    ws = []
    for f in f_m:
        w = W.macrospin(float(f), [5.0], 50.0, 0.2, alpha=2e-5, a0=[0.01], n=2)
        w.nx, w.ny, w.nz = 64, 32, 8
        w.m0 = np.broadcast_to(w.m0[:, :, :1, :1, :1], (1, 3, 8, 32, 64)).copy()
        w.u = np.ones((1, 8, 32, 64))
        ws.append(w)
    K = 601
    lo, hi = TWO_PI * 4.80e9, TWO_PI * 5.20e9
    T, sdt = 80e-9, 25e-12
    cap = int(round(T / sdt))
    sims = [api.Sim(w, precision="f64", stream=st.cuda_stream) for w in ws]
    for sim in sims:
        api.cav_set_trace(sim.h, sdt, cap)
        api.cav_set_spectrum(sim.h, K, lo, hi)
    sw = api.cav_sweep_create(sims)
    try:
        api.cav_sweep_run(sw, T, tol=1e-7)
        fk = np.linspace(4.80e9, 5.20e9, K)
        gaps = []
        for f, sim in zip(f_m, sims):
            X, ns = api.cav_get_spectrum(sim.h, K, 1)
            assert ns == cap and api.cav_get_stats(sim.h)["t"] == T
            P = np.abs(X[:, 0]) ** 2 + np.abs(X[:, 1]) ** 2
            mid = 0.5 * (f_c + f * 1e9)
            det = 0.5 * (f_c - f * 1e9)
            exp_lo, exp_hi = mid - math.sqrt(g * g + det * det), mid + math.sqrt(g * g + det * det)
            below, above = fk < mid, fk >= mid
            got_lo, got_hi = fk[below][P[below].argmax()], fk[above][P[above].argmax()]
            assert abs(got_lo - exp_lo) < 3e6 and abs(got_hi - exp_hi) < 3e6, (f, got_lo, exp_lo, got_hi, exp_hi)
            gaps.append(got_hi - got_lo)
        assert abs(min(gaps) - 2 * g) < 4e6 and int(np.argmin(gaps)) == 4          # minimum gap 2g at resonance
    finally:
        api.cav_sweep_destroy(sw)
        for sim in sims:
            sim.close()
