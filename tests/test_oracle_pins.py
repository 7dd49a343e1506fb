"""Pins for the fp64 CPU oracle (-m "not gpu").

The oracle is an integrator, so it is pinned to what the paper and the mathematics fix
independently of it: closed forms (Kittel line, exact damped macrospin, polariton branches,
Rabi period, arrowhead eigenvalues, level attraction, discrete spin-wave dispersion and the
overlap coupling, AFMR), invariants (m.f = 0, |m| drift order, selection rule, convergence
order 5, tableau identities), values the paper prints (tests/golden/paper_values.json) and a
library integrator (scipy DOP853).  Every linear model below is derived by hand from
PAPER.md Eqs. 1-5, 12-13, 19 in the docstrings — none calls the oracle to get its
expected value.
"""
import json
import math
import os

import numpy as np
import pytest

import cavmag_workloads as W
from oracle import Oracle, tableau
from observables import fit_exponentials, dominant, rabi_period

TWO_PI = 2 * math.pi
GAMMA = 1.76e11
GOLD = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "paper_values.json")))


# ----------------------------------------------------------------------------------------
# hand-derived small-signal model of the lumped system (uniform u, bit-uniform m ~ z^)
# ----------------------------------------------------------------------------------------
def lumped_spectrum(omega_c, kappa, G, omega_m, alpha, rwa=False):
    """Complex frequencies (x ~ exp(-i w t)) of N uniform cavity modes + one macrospin.

    Linearise  dm/dt = -gamma/(1+alpha^2)[m x B + alpha m x (m x B)]  about m = z^ with
    B = B0 z^ + x^ (2/gamma) sum_n Re[G_n a_n]  (Eqs. 3-5, 13):
        mu' = -(i+alpha) w_m/(1+alpha^2) mu + (i+alpha)/(1+alpha^2) sum_n (G_n a_n + G_n^* a_n^*)
        a_n' = -(i w_n + kappa_n) a_n + i G_n mu                      (Eq. 12 / Eq. 19)
    with mu = m_x - i m_y.  rwa=True drops the a_n^* term and alpha in the coupling:
    the (N+1)x(N+1) arrowhead matrix of Eq. 14 with w -> w - i*loss (Eq. 7).
    """
    omega_c, kappa, G = map(lambda v: np.atleast_1d(np.asarray(v, dtype=np.complex128)), (omega_c, kappa, G))
    N = omega_c.shape[0]
    if rwa:
        H = np.zeros((N + 1, N + 1), dtype=np.complex128)
        for n in range(N):
            H[n, n] = omega_c[n] - 1j * kappa[n]
            H[n, N] = -G[n]       # sign of the off-diagonal does not change the spectrum
            H[N, n] = -G[n]
        H[N, N] = omega_m - 1j * alpha * omega_m
        return np.sort_complex(np.linalg.eigvals(H))
    M = np.zeros((N + 1, N + 1), dtype=np.complex128)
    K = np.zeros((N + 1, N + 1), dtype=np.complex128)
    d = 1.0 + alpha * alpha
    for n in range(N):
        M[n, n] = -(1j * omega_c[n] + kappa[n])
        M[n, N] = 1j * G[n]
        M[N, n] = (1j + alpha) / d * G[n]
        K[N, n] = (1j + alpha) / d * np.conj(G[n])
    M[N, N] = -(1j + alpha) * omega_m / d
    big = np.block([[M, K], [K.conj(), M.conj()]])
    w = 1j * np.linalg.eigvals(big)
    w = w[w.real > 0]
    return np.sort_complex(w)


def simulate_lumped(w, t_end, sample_dt, tol=1e-10, **kw):
    o = Oracle(w, **kw)
    cap = int(round(t_end / sample_dt))
    r = o.run(w.m0, w.a0, t_end=t_end, tol=tol, sample_dt=sample_dt, trace_cap=cap)
    assert r.status == 0 and r.trace.shape[0] == cap
    return r


def trace_a(r, n=0):
    return r.trace[:, 1 + 2 * n] + 1j * r.trace[:, 2 + 2 * n]


def trace_mminus(r, N, sub=0):
    c = 1 + 4 * N + 3 * sub
    return r.trace[:, c] - 1j * r.trace[:, c + 1]


# ----------------------------------------------------------------------------------------
# P13 tableau identities
# ----------------------------------------------------------------------------------------
def test_tableau_identities():
    a, b, bh, c = tableau()
    assert np.allclose(a.sum(axis=1), c, atol=1e-15)
    assert abs(b.sum() - 1) < 1e-15 and abs(bh.sum() - 1) < 1e-15
    assert abs((b - bh).sum()) < 1e-16
    assert np.allclose(a[6], b)                     # FSAL: last stage row equals b
    # order conditions up to 3 for b and bhat (textbook, Hairer-Norsett-Wanner II.1)
    for wts in (b, bh):
        assert abs(wts @ c - 1 / 2) < 1e-15
        assert abs(wts @ c**2 - 1 / 3) < 1e-15
        assert abs(wts @ (a @ c) - 1 / 6) < 1e-15
    assert abs(b @ c**3 - 1 / 4) < 1e-15 and abs(b @ c**4 - 1 / 5) < 1e-15   # b is 5th order


# ----------------------------------------------------------------------------------------
# P1 Kittel line and the exact damped macrospin
# ----------------------------------------------------------------------------------------
def test_kittel_frequency_eq9():
    """alpha = 0, g = 0: m^- ~ exp(-i gamma B0 t)  (Eq. 9)."""
    w = W.macrospin(10.0, [10.0], 0.0, 0.0, alpha=0.0, tilt=0.01)
    r = simulate_lumped(w, 2e-9, 5e-12)
    om, amp = fit_exponentials(trace_mminus(r, 1), 5e-12, 1)
    assert abs(om[0].real / (GAMMA * w.B0[2]) - 1) < 1e-9
    assert om[0].real > 0          # co-rotating sign: m_x - i m_y ~ e^{-i w t}
    assert abs(om[0].imag) < 1e-9 * om[0].real


def test_macrospin_exact_damped_solution():
    """Textbook closed form of the LLG macrospin in a static field B z^:
    phi(t) = phi0 + w t, tan(theta/2)(t) = tan(theta0/2) exp(-lam t),
    w = gamma B/(1+alpha^2), lam = alpha w  (gives gamma_m = alpha w_m of PAPER.md:89)."""
    alpha, th0 = 0.05, 0.6
    w = W.macrospin(10.0, [10.0], 0.0, 0.0, alpha=alpha, tilt=th0)
    o = Oracle(w)
    T = 1.0e-9
    r = o.run(w.m0, w.a0, t_end=T, tol=1e-12)
    wm = GAMMA * w.B0[2] / (1 + alpha**2)
    th = 2 * math.atan(math.tan(th0 / 2) * math.exp(-alpha * wm * T))
    ph = wm * T
    exact = np.array([math.sin(th) * math.cos(ph), math.sin(th) * math.sin(ph), math.cos(th)])
    got = r.m[0, :, 0, 0, 0]
    assert np.abs(got - exact).max() < 2e-9
    assert np.abs(r.m - r.m[:, :, :1, :1, :1]).max() == 0.0      # stays bit-uniform (exchange = 0)


def test_resonance_field_printed():
    g = GOLD["resonance_field_mT"]
    B = TWO_PI * g["f_c_GHz"] * 1e9 / GOLD["gamma_rad_per_s_T"]["value"] * 1e3
    assert abs(B - g["B_res_mT"]) < g["tol_mT"]
    assert abs(W.b0_for_ghz(g["f_c_GHz"]) * 1e3 - B) < 1e-12


# ----------------------------------------------------------------------------------------
# P3 Rabi period, values printed by the paper
# ----------------------------------------------------------------------------------------
@pytest.mark.parametrize("case", GOLD["rabi_period_ns"])
def test_rabi_period_printed(case):
    """a(0) = 0.01 at resonance: |a|^2 and |m^-|^2 exchange with T_R = pi/g."""
    gM = case["g_over_2pi_MHz"]
    w = W.macrospin(5.0, [5.0], gM, 0.0, alpha=0.0, a0=[GOLD["rabi_initial_amplitude"]["value"]])
    T = 2.6 * case["T_R_ns"] * 1e-9
    r = simulate_lumped(w, T, 25e-12, tol=1e-9)
    t = r.trace[:, 0]
    pa = np.abs(trace_a(r)) ** 2
    pm = np.abs(trace_mminus(r, 1)) ** 2
    TR = rabi_period(t, pa)
    assert abs(TR * 1e9 / case["T_R_ns"] - 1) < 2e-3      # pi/g up to the non-RWA shift ~ (g/w)^2
    assert abs(TR * (TWO_PI * gM * 1e6) / math.pi - 1) < 2e-3
    # antiphase: the photon and magnon populations are anti-correlated and sum to ~const
    assert np.corrcoef(pa, pm)[0, 1] < -0.95


def test_wrong_handedness_gives_no_exchange():
    """coupling must be to the co-rotating m^-.  With B0 reversed the spin
    precesses the other way (m^- ~ e^{+iwt}); a ~ e^{-iwt} then cannot exchange energy."""
    w = W.macrospin(5.0, [5.0], 50.0, 0.0, alpha=0.0, a0=[0.01])
    w.B0 = (0.0, 0.0, -w.B0[2])
    w.m0 = -w.m0      # ground state follows the field
    r = simulate_lumped(w, 12e-9, 25e-12, tol=1e-9)
    pa = np.abs(trace_a(r)) ** 2
    assert pa.min() > 0.9 * pa[0]


# ----------------------------------------------------------------------------------------
# P2 polariton branches (Eq. 6 / Eq. 7) and the exact small-signal spectrum
# ----------------------------------------------------------------------------------------
@pytest.mark.parametrize("detune_ghz", [-0.06, 0.0, 0.045])
def test_polariton_branches_eq6_eq7(detune_ghz):
    fc, gM, kM, alpha = 5.0, 50.0, 0.5, 3e-4
    w = W.macrospin(fc + detune_ghz, [fc], gM, kM, alpha=alpha, a0=[1e-3], tilt=1e-3)
    r = simulate_lumped(w, 60e-9, 20e-12)
    om, amp = fit_exponentials(trace_a(r), 20e-12, 4)
    om2, _ = dominant(om, amp, 2)
    wc, wm, g, kap = TWO_PI * fc * 1e9, GAMMA * w.B0[2], TWO_PI * gM * 1e6, TWO_PI * kM * 1e6
    # Eq. 6, lossless RWA: within 1 MHz (north_star observable bound); non-RWA shift ~ g^2/2w = 250 kHz
    eq6 = (wc + wm) / 2 + np.array([-1, 1]) * math.sqrt(g**2 + ((wc - wm) / 2) ** 2)
    assert np.abs(om2.real - eq6).max() / TWO_PI < 1e6
    # Eq. 7 (lossy RWA): linewidths
    eq7 = lumped_spectrum([wc], [kap], [g], wm, alpha, rwa=True)
    assert np.abs(om2.imag - eq7.imag).max() / TWO_PI < 0.02e6
    # exact hand-derived small-signal model incl. counter-rotating terms: kHz agreement
    ex = lumped_spectrum([wc], [kap], [g], wm, alpha)
    assert np.abs(om2 - ex).max() / TWO_PI < 5e3
    # min gap 2g at resonance
    if detune_ghz == 0.0:
        gap = (om2[1].real - om2[0].real) / TWO_PI / 1e6
        assert abs(gap - GOLD["anticrossing_min_gap_MHz"]["gap_MHz"]) < 0.6


def test_h0_factor_two_matters():
    """without h0 = 2g/gamma the splitting is not 2g.  The model above
    uses exactly that factor; halving it would give sqrt(1/2) of the gap — the test of Eq. 6
    at < 1% of the gap (0.6 MHz of 100) therefore pins the factor.  Here: g -> 2g doubles it."""
    gaps = []
    for gM in (20.0, 40.0):
        w = W.macrospin(5.0, [5.0], gM, 0.0, alpha=0.0, a0=[1e-3])
        r = simulate_lumped(w, 80e-9, 20e-12)
        om, amp = fit_exponentials(trace_a(r), 20e-12, 4)
        om2, _ = dominant(om, amp, 2)
        gaps.append((om2[1].real - om2[0].real) / TWO_PI / 1e6)
    assert abs(gaps[0] - 40.0) < 0.1 and abs(gaps[1] - 80.0) < 0.3


def test_cooperativity_printed():
    """gamma_m = alpha w_m measured from the oracle's free decay reproduces the paper's C values."""
    g = GOLD["cooperativity"]
    w = W.macrospin(g["f_GHz"], [g["f_GHz"]], 0.0, 0.0, alpha=g["alpha"], tilt=1e-3)
    r = simulate_lumped(w, 40e-9, 20e-12)
    om, _ = fit_exponentials(trace_mminus(r, 1), 20e-12, 1)
    gamma_m = -om[0].imag
    assert abs(gamma_m / (g["alpha"] * TWO_PI * g["f_GHz"] * 1e9) - 1) < 1e-4
    for c in g["cases"]:
        C = (TWO_PI * c["g_MHz"] * 1e6) ** 2 / (TWO_PI * c["kappa_MHz"] * 1e6 * gamma_m)
        assert abs(C / c["C"] - 1) < c["rel_tol"]


# ----------------------------------------------------------------------------------------
# P4 N uniform modes: arrowhead matrix (Eq. 14 generalised), dark mode
# ----------------------------------------------------------------------------------------
def test_two_mode_eq14_printed_setup():
    tm = GOLD["two_mode"]
    f1, f2, gM = tm["f1_GHz"], tm["f2_GHz"], tm["g_MHz"]
    w = W.macrospin(0.5 * (f1 + f2), [f1, f2], gM, 0.0, alpha=0.0, a0=[tm["a1_0"] * 0.1, 0.0])
    r = simulate_lumped(w, 60e-9, 20e-12)
    g = TWO_PI * gM * 1e6
    H = np.array([[TWO_PI * f1 * 1e9, g, 0], [g, GAMMA * w.B0[2], g], [0, g, TWO_PI * f2 * 1e9]])   # Eq. 14
    ev = np.sort(np.linalg.eigvalsh(H))
    for n in (0, 1):
        om, amp = fit_exponentials(trace_a(r, n), 20e-12, 6)
        om3, _ = dominant(om, amp, 3)
        assert np.abs(om3.real - ev).max() / TWO_PI < 1e6
    # middle branch sits at the midpoint: sqrt(0.05^2 + 2*0.05^2) = 86.6 MHz from the others
    assert abs((ev[2] - ev[1]) / TWO_PI / 1e6 - 86.6025) < 1e-3
    # magnon-mediated transfer: mode 2 gets populated from zero
    assert np.abs(trace_a(r, 1)).max() > 0.5 * np.abs(trace_a(r, 0)).max()


def test_five_mode_arrowhead_exact():
    fcs = [9.7, 9.9, 10.0, 10.15, 10.3]
    gs = [12.0, 20.0, 8.0, 15.0, 25.0]
    ks = [1.0, 2.0, 0.5, 1.5, 1.0]
    alpha = 2e-4
    w = W.macrospin(10.02, fcs, gs, ks, alpha=alpha, a0=[1e-3, 5e-4, -3e-4, 2e-4j, 1e-3], tilt=5e-4)
    r = simulate_lumped(w, 120e-9, 20e-12)
    ex = lumped_spectrum(w.omega, w.kappa, w.g, GAMMA * w.B0[2], alpha)
    rw = lumped_spectrum(w.omega, w.kappa, w.g, GAMMA * w.B0[2], alpha, rwa=True)
    sig = sum((0.3 + n) * trace_a(r, n) for n in range(5))
    om, amp = fit_exponentials(sig, 20e-12, 12)
    om6, _ = dominant(om, amp, 6)
    assert np.abs(om6 - ex).max() / TWO_PI < 5e3
    assert np.abs(om6.real - rw.real).max() / TWO_PI < 1e6


# ----------------------------------------------------------------------------------------
# P5 dissipative coupling (Eq. 19/20): level attraction
# ----------------------------------------------------------------------------------------
def test_level_attraction_eq20_printed():
    """g = 0, g_d/2pi = 50 MHz.  The paper's (ig + g_d) is G = g - i g_d: Gamma = g_d, Phi = -pi/2
    (reading G6).  Eq. 20: at resonance Re parts coalesce, Im parts split by 2 g_d."""
    la = GOLD["level_attraction"]
    fc, gd = la["f_c_GHz"], la["g_d_MHz"]
    kM = fc * 1e3 / (2 * la["Q"])               # kappa = w_c/2Q = 0.5 MHz
    alpha = 3e-4
    w = W.macrospin(fc, [fc], 0.0, kM, alpha=alpha, a0=[1e-6], Gamma_mhz=[gd], Phi=[-math.pi / 2])
    r = simulate_lumped(w, 12e-9, 10e-12)
    om, amp = fit_exponentials(trace_a(r), 10e-12, 4)
    om2, _ = dominant(om, amp, 2)
    wc, Gd, kap = TWO_PI * fc * 1e9, TWO_PI * gd * 1e6, TWO_PI * kM * 1e6
    gt = -1j * Gd                                    # g~ = g - i g_d
    wct, wmt = wc - 1j * kap, wc - 1j * alpha * wc
    root = np.sqrt(gt**2 + ((wct - wmt) / 2) ** 2 + 0j)
    eq20 = np.sort_complex(np.array([(wct + wmt) / 2 - root, (wct + wmt) / 2 + root]))
    assert abs(om2[0].real - om2[1].real) / TWO_PI < 0.3e6                    # frequency gap closes
    split = abs(om2[0].imag - om2[1].imag) / TWO_PI / 1e6
    assert abs(split - la["linewidth_split_MHz"]) < 0.5                        # 2 g_d/2pi = 100 MHz
    assert np.abs(np.sort(om2.imag) - np.sort(eq20.imag)).max() / TWO_PI < 0.3e6
    assert om2.imag.max() > 0                                                  # one branch has gain (G29)
    ex = lumped_spectrum([wc], [kap], [gt], wc, alpha)
    assert np.abs(np.sort_complex(om2) - ex).max() / TWO_PI < 20e3


def test_mixed_coupling_phase_convention():
    """G = g + Gamma e^{i Phi}: Phi = 0 simply adds to g (gap 2(g+Gamma)); Phi = +-pi/2 give the
    same G^2 when g = 0 (Eq. 20 depends on g~^2 only)."""
    w = W.macrospin(5.0, [5.0], 30.0, 0.0, alpha=0.0, a0=[1e-3], Gamma_mhz=[20.0], Phi=[0.0])
    r = simulate_lumped(w, 60e-9, 20e-12)
    om, amp = fit_exponentials(trace_a(r), 20e-12, 4)
    om2, _ = dominant(om, amp, 2)
    assert abs((om2[1].real - om2[0].real) / TWO_PI / 1e6 - 100.0) < 0.6
    spec = []
    for ph in (+math.pi / 2, -math.pi / 2):
        w = W.macrospin(5.0, [5.0], 0.0, 1.0, alpha=1e-4, a0=[1e-6], Gamma_mhz=[40.0], Phi=[ph])
        r = simulate_lumped(w, 10e-9, 10e-12)
        om, amp = fit_exponentials(trace_a(r), 10e-12, 4)
        spec.append(np.sort_complex(dominant(om, amp, 2)[0]))
    assert np.abs(spec[0] - spec[1]).max() / TWO_PI < 20e3


# ----------------------------------------------------------------------------------------
# P6 discrete spin-wave dispersion and the overlap coupling (pins stencil, BC, 1/N_cells)
# ----------------------------------------------------------------------------------------
def _chain(nx, ny, nz, dx, dy, dz, f_k_ghz, modes, u, m0, a0, alpha=0.0, B0=None):
    md = W._modes(*modes)
    return W.Workload(name="chain", nx=nx, ny=ny, nz=nz, dx=dx, dy=dy, dz=dz, Ms=140e3, Aex=3.7e-12, Ku=0.0,
                      ku_axis=(0, 0, 1), alpha=alpha, gamma=GAMMA, B0=(0, 0, B0 if B0 is not None else W.b0_for_ghz(f_k_ghz)),
                      n_sub=1, B_exch_inter=0.0, u=u, m0=m0, a0=np.asarray(a0, dtype=np.complex128),
                      t_end=0, tol=0, fixed_dt=0, precision="f64", **md)


def test_exchange_dispersion_3d_anisotropic_cells():
    """Open-boundary (Neumann) Laplacian eigenvectors phi_k = prod_d cos(k_d pi (i_d+1/2)/n_d):
    w_k = gamma [B0 + (2A/Ms) sum_d (2/D_d^2)(1 - cos(k_d pi/n_d))]   (P6).
    Distinct n_d and D_d per axis catch a transposed axis, a wrong prefactor or a periodic wrap."""
    nx, ny, nz = 6, 5, 4
    dx, dy, dz = 4e-9, 5e-9, 7e-9
    kx, ky, kz = 2, 1, 3
    phi = W.cosine_profile(kx, ky, kz, nx, ny, nz)
    eps = 1e-4
    m0 = np.zeros((1, 3, nz, ny, nx))
    m0[0, 0] = eps * phi
    m0[0, 2] = np.sqrt(1 - m0[0, 0] ** 2)
    w = _chain(nx, ny, nz, dx, dy, dz, 10.0, ([10.0], 0.0, 0.0), phi[None], m0, [0.0])
    r = simulate_lumped(w, 1.0e-9, 1e-12, tol=1e-11)
    # the overlap S = <phi m^-> follows the k-mode amplitude (g = 0: S is just a probe here)
    S = r.trace[:, 3] + 1j * r.trace[:, 4]
    om, _ = fit_exponentials(S, 1e-12, 1)
    lap = sum((2 / d**2) * (1 - math.cos(k * math.pi / n)) for k, n, d in ((kx, nx, dx), (ky, ny, dy), (kz, nz, dz)))
    wk = GAMMA * (w.B0[2] + 2 * w.Aex / w.Ms * lap)
    assert abs(om[0].real / wk - 1) < 2e-8
    # and it is an eigenmode: the uniform average stays zero (orthogonal to k = 0)
    assert np.abs(trace_mminus(r, 1)).max() < 1e-15


def test_overlap_coupling_to_k1_spin_wave():
    """u = phi_1 = cos(pi (i+1/2)/n) on a 16-cell chain, cavity tuned to w_1:
    exact linear result g_eff = g <u phi_1>/sqrt(<phi_1^2>) = g/sqrt(2)  (P6/G30), so the
    gap is 2g/sqrt(2) and T_R = pi/(g/sqrt 2).  Pins W_n = N_cells (Eq. 18) and the u(r) feedback."""
    n, d, gM = 16, 5e-9, 50.0
    phi = W.cosine_profile(1, 0, 0, n, 1, 1)
    B0 = W.b0_for_ghz(9.0)
    w1 = GAMMA * (B0 + 2 * 3.7e-12 / 140e3 * (2 / d**2) * (1 - math.cos(math.pi / n)))
    m0 = np.zeros((1, 3, 1, 1, n)); m0[0, 2] = 1.0
    w = _chain(n, 1, 1, d, d, d, 0, ([w1 / TWO_PI / 1e9], gM, 0.0), phi[None], m0, [1e-3], B0=B0)
    r = simulate_lumped(w, 45e-9, 20e-12, tol=1e-10)
    om, amp = fit_exponentials(trace_a(r), 20e-12, 4)
    om2, _ = dominant(om, amp, 2)
    gap = (om2[1].real - om2[0].real) / TWO_PI / 1e6
    assert abs(gap - 2 * gM / math.sqrt(2)) < 0.3
    TR = rabi_period(r.trace[:, 0], np.abs(trace_a(r)) ** 2)
    assert abs(TR / (math.pi / (TWO_PI * gM * 1e6 / math.sqrt(2))) - 1) < 3e-3
    # full arrowhead over all chain modes: G_k = g <u phi_k>/sqrt(<phi_k^2>)
    ks = np.arange(n)
    phik = np.cos(np.outer(ks, math.pi * (np.arange(n) + 0.5) / n))
    Gk = TWO_PI * gM * 1e6 * (phik @ phi[0, 0]) / n / np.sqrt((phik**2).mean(axis=1))
    wk = GAMMA * (B0 + 2 * 3.7e-12 / 140e3 * (2 / d**2) * (1 - np.cos(ks * math.pi / n)))
    H = np.diag(np.concatenate([[w1], wk])).astype(np.float64)
    H[0, 1:] = Gk; H[1:, 0] = Gk
    ev = np.linalg.eigvalsh(H)
    near = ev[np.argsort(np.abs(ev - w1))[:2]]
    assert np.abs(np.sort(near) - om2.real).max() / TWO_PI < 0.3e6


def test_selection_rule_eq10_eq11_printed():
    """<cos(n pi x/Lx)> = 0 on the centred full grid, so a uniform
    magnetisation never excites those modes: a stays 0 to rounding; the uniform mode does."""
    po = GOLD["profile_overlaps"]
    nx, ny, nz = po["grid"]
    us = np.stack([W.cosine_profile(n, 0, 0, nx, ny, nz) for n in (0, 1, 2)])
    means = us.reshape(3, -1).mean(axis=1)
    assert abs(means[0] - po["uniform"]) < 1e-15 and abs(means[1]) < 1e-15 and abs(means[2]) < 1e-15
    m0 = W.tilted_state(7, 1, nx, ny, nz, 0.02, per_cell=False)[None]
    md = W._modes([5.0, 5.0, 5.0], 50.0, 0.5)
    w = W.Workload(name="sel", nx=nx, ny=ny, nz=nz, dx=10e-9, dy=10e-9, dz=10e-9, Ms=140e3, Aex=3.5e-12, Ku=0.0,
                   ku_axis=(0, 0, 1), alpha=3e-4, gamma=GAMMA, B0=(0, 0, W.b0_for_ghz(5.0)), n_sub=1,
                   B_exch_inter=0.0, u=us, m0=m0, a0=np.zeros(3, dtype=np.complex128), t_end=0, tol=0,
                   fixed_dt=0, precision="f64", **md)
    o = Oracle(w)
    r = o.run(w.m0, w.a0, t_end=3e-9, tol=1e-9)
    assert abs(r.a[0]) > 1e-4
    assert abs(r.a[1]) < 1e-16 and abs(r.a[2]) < 1e-16


def test_overlap_normalisation_options():
    """Eq. 18 divides by N_cells; the north_star variant divides by sum u.  They agree for u = 1 and
    differ by <u> otherwise."""
    nx, ny, nz = 5, 4, 3
    u = W.random_smooth_profiles(11, 1, nx, ny, nz) + 0.5
    m0 = W.tilted_state(11, 1, nx, ny, nz, 0.3)[None]
    md = W._modes([5.0], 10.0, 1.0)
    kw = dict(nx=nx, ny=ny, nz=nz, dx=5e-9, dy=5e-9, dz=5e-9, Ms=140e3, Aex=3.7e-12, Ku=0.0, ku_axis=(0, 0, 1),
              alpha=0.0, gamma=GAMMA, B0=(0, 0, 0.1), n_sub=1, B_exch_inter=0.0, u=u, **md)
    _, _, S1 = Oracle(**kw).rhs(m0, [0j])
    _, _, S2 = Oracle(norm_sum_u=True, **kw).rhs(m0, [0j])
    direct = (u[0] * (m0[0, 0] - 1j * m0[0, 1])).sum()
    assert abs(S1[0] - direct / (nx * ny * nz)) < 1e-15
    assert abs(S2[0] - direct / u.sum()) < 1e-15


# ----------------------------------------------------------------------------------------
# P9 antiferromagnetic resonance (Eq. 15/16) and the paper's printed example
# ----------------------------------------------------------------------------------------
def _afm(B_E, B_A, B0z, Ms=400e3, alpha=0.0, n=2, g_mhz=0.0, f_c_ghz=100.0, tilt=1e-3, a0=0.0, kappa_mhz=0.0):
    Ku = 0.5 * B_A * Ms
    m1 = np.zeros((3, n, n, n)); m2 = np.zeros((3, n, n, n))
    m1[0] = math.sin(tilt); m1[2] = math.cos(tilt)
    m2[0] = math.sin(0.4 * tilt); m2[1] = 0.3 * tilt; m2[2] = -math.sqrt(1 - m2[0, 0, 0, 0] ** 2 - (0.3 * tilt) ** 2)
    md = W._modes([f_c_ghz], g_mhz, kappa_mhz)
    return W.Workload(name="afm", nx=n, ny=n, nz=n, dx=2e-9, dy=2e-9, dz=2e-9, Ms=Ms, Aex=10e-12, Ku=Ku,
                      ku_axis=(0, 0, 1), alpha=alpha, gamma=GAMMA, B0=(0, 0, B0z), n_sub=2, B_exch_inter=B_E,
                      u=np.ones((1, n, n, n)), m0=np.stack([m1, m2]), a0=np.array([a0], dtype=np.complex128),
                      t_end=0, tol=0, fixed_dt=0, precision="f64", **md)


def _neel_minus(r, N=1):
    c = 1 + 4 * N
    nx_ = 0.5 * (r.trace[:, c] - r.trace[:, c + 3])
    ny_ = 0.5 * (r.trace[:, c + 1] - r.trace[:, c + 4])
    return nx_ - 1j * ny_


@pytest.mark.parametrize("B0z", [0.0, 0.02])
def test_afmr_eq15_eq16(B0z):
    """w_AFMR = gamma sqrt(2 B_E B_A + B_A^2) (Eq. 15); a field along the easy axis splits it
    into w_AFMR +- gamma B (Eq. 16); the two branches have opposite handedness in n^-.
    CFG4 numbers: B_E = 50 T, B_A = 2Ku/Ms = 0.25 T -> 140.23 GHz."""
    B_E, B_A = 50.0, 0.25
    w = _afm(B_E, B_A, B0z, tilt=1e-5)       # the closed form is the small-angle limit: error ~ tilt^2 B_E/B_A
    r = simulate_lumped(w, 0.25e-9, 0.5e-12, tol=1e-12)
    om, amp = fit_exponentials(_neel_minus(r), 0.5e-12, 2)
    w0 = GAMMA * math.sqrt(2 * B_E * B_A + B_A * B_A)
    assert abs(w0 / TWO_PI / 1e9 - 140.23) < 0.01
    expect = np.sort([-(w0 - GAMMA * B0z), w0 + GAMMA * B0z])
    assert np.abs(np.sort(om.real) / expect - 1).max() < 1e-7


def test_afmr_printed_example():
    ex = GOLD["afmr_example"]
    w = _afm(ex["mu0_HE_T"], ex["mu0_HA_T"], 0.0, Ms=200e3, tilt=1e-6)
    r = simulate_lumped(w, 2e-9, 4e-12, tol=1e-12)
    om, amp = fit_exponentials(_neel_minus(r), 4e-12, 2)
    f = np.abs(om.real) / TWO_PI / 1e9
    assert np.abs(f - ex["f_AFMR_GHz"]).max() < ex["tol_GHz"]
    assert np.abs(f - 4.9952).max() < 1e-4        # gamma sqrt(2*15.9*1e-3 + 1e-6)/2pi


def test_sublattice_exchange_symmetry():
    """Swapping the two sublattices swaps their torques and leaves the cavity drive unchanged
    (the cavity sees only (m1+m2)/2)."""
    w = _afm(50.0, 0.25, 0.03, g_mhz=1000.0, f_c_ghz=140.23, kappa_mhz=500.0, tilt=0.2, a0=0.01 + 0.02j)
    o = Oracle(w)
    dm, da, S = o.rhs(w.m0, w.a0)
    dm2, da2, S2 = o.rhs(w.m0[::-1], w.a0)
    assert np.array_equal(dm2, dm[::-1]) and np.array_equal(da2, da) and np.array_equal(S2, S)
    # S is the overlap of the NET magnetisation
    mc = 0.5 * (w.m0[0] + w.m0[1])
    assert abs(S[0] - (mc[0] - 1j * mc[1]).mean()) < 1e-16


# ----------------------------------------------------------------------------------------
# P8 brute-force Jacobian spectrum on a tiny grid (AFM + anisotropy + cavity, non-RWA)
# ----------------------------------------------------------------------------------------
def test_jacobian_spectrum_matches_trace_afm_cavity():
    w = _afm(50.0, 0.25, 0.01, n=1, g_mhz=3000.0, f_c_ghz=141.0, tilt=2e-5, a0=1e-5, kappa_mhz=100.0, alpha=1e-3)
    o = Oracle(w, renormalize=False)
    meq = np.zeros((2, 3, 1, 1, 1)); meq[0, 2] = 1; meq[1, 2] = -1
    x0 = np.concatenate([meq.ravel(), [0.0, 0.0]])

    def f(x):
        dm, da, _ = o.rhs(x[:6].reshape(2, 3, 1, 1, 1), x[6:].view(np.complex128))
        return np.concatenate([dm.ravel(), da.view(np.float64)])
    h = 1e-6
    J = np.stack([(f(x0 + h * e) - f(x0 - h * e)) / (2 * h) for e in np.eye(8)], axis=1)
    lam = np.linalg.eigvals(J)
    wj = 1j * lam
    wj = wj[np.abs(wj) > 1e9]                     # drop the two |m| = const zero modes
    r = simulate_lumped(w, 0.4e-9, 0.5e-12, tol=1e-12, renormalize=False)
    om, amp = fit_exponentials(trace_a(r), 0.5e-12, 6)
    om3, _ = dominant(om, amp, 3)
    for wfit in om3:
        assert np.abs(wj - wfit).min() / abs(wfit) < 5e-6


# ----------------------------------------------------------------------------------------
# P10 invariants, P11 order, P12 library integrator
# ----------------------------------------------------------------------------------------
def _busy_problem(nx=3, ny=2, nz=2, n_sub=1, seed=5):
    N = 2
    u = W.random_smooth_profiles(seed, N, nx, ny, nz)
    m0 = np.stack([W.tilted_state(seed, 1 + 2 * s, nx, ny, nz, 0.4, sign=(1.0 if s == 0 else -1.0)) for s in range(n_sub)])
    md = W._modes([9.0, 11.0], [40.0, 25.0], [5.0, 3.0], [0.0, 15.0], [0.0, 1.1])
    return W.Workload(name="busy", nx=nx, ny=ny, nz=nz, dx=4e-9, dy=5e-9, dz=6e-9, Ms=140e3, Aex=3.7e-12, Ku=2e3,
                      ku_axis=(1.0, 0.5, 0.2), alpha=0.02, gamma=GAMMA, B0=(0.01, -0.02, 0.35), n_sub=n_sub,
                      B_exch_inter=(3.0 if n_sub == 2 else 0.0), u=u, m0=m0,
                      a0=np.array([0.02 + 0.01j, -0.015j]), t_end=0, tol=0, fixed_dt=0, precision="f64", **md)


@pytest.mark.parametrize("n_sub", [1, 2])
def test_torque_is_perpendicular_to_m(n_sub):
    w = _busy_problem(4, 3, 3, n_sub)
    dm, da, S = Oracle(w).rhs(w.m0, w.a0)
    dot = (dm * w.m0).sum(axis=1)
    assert np.abs(dot).max() < 1e-15 * np.abs(dm).max() * 10


def test_norm_drift_is_fifth_order_without_renormalisation():
    w = W.cfg1("b", n=4)
    w.alpha = 0.0
    drifts = []
    for dt in (0.1e-12, 0.05e-12):
        r = Oracle(w, renormalize=False).run(w.m0, w.a0, fixed_dt=dt, max_steps=int(round(4e-12 / dt)))
        drifts.append(np.abs(np.linalg.norm(r.m, axis=1) - 1).max())
    assert drifts[0] < 1e-9 and 16 < drifts[0] / drifts[1] < 80          # ~2^5 = 32 (dt^5 per unit time)
    r = Oracle(w, renormalize=True).run(w.m0, w.a0, fixed_dt=0.1e-12, max_steps=40)
    assert np.abs(np.linalg.norm(r.m, axis=1) - 1).max() < 4e-16


def test_convergence_order_five():
    w = _busy_problem()
    o = Oracle(w, renormalize=False)
    T = 8e-12
    ref = o.run(w.m0, w.a0, fixed_dt=T / 1024, max_steps=1024)
    errs = []
    for n in (32, 64, 128):
        r = o.run(w.m0, w.a0, fixed_dt=T / n, max_steps=n)
        errs.append(max(np.abs(r.m - ref.m).max(), np.abs(r.a - ref.a).max()))
    assert 24 < errs[0] / errs[1] < 42 and 24 < errs[1] / errs[2] < 42


@pytest.mark.parametrize("n_sub", [1, 2])
def test_against_scipy_dop853(n_sub):
    """2x2x2 grid, every term on (exchange, Ku off-axis, Zeeman off-axis, 2 profiled modes, mixed
    coupling, damping [, AFM]): the oracle's own DP5(4) vs scipy's DOP853 at rtol = atol = 1e-13."""
    from scipy.integrate import solve_ivp
    w = _busy_problem(2, 2, 2, n_sub)
    o = Oracle(w, renormalize=False)
    nm = w.m0.size

    def f(t, x):
        dm, da, _ = o.rhs(x[:nm], x[nm:].view(np.complex128))
        return np.concatenate([dm.ravel(), da.view(np.float64)])
    T = 30e-12
    x0 = np.concatenate([w.m0.ravel(), w.a0.view(np.float64)])
    sol = solve_ivp(f, (0, T), x0, method="DOP853", rtol=1e-13, atol=1e-13)
    r = o.run(w.m0, w.a0, t_end=T, tol=1e-12)
    assert np.abs(r.m.ravel() - sol.y[:nm, -1]).max() < 5e-10
    assert np.abs(r.a.view(np.float64) - sol.y[nm:, -1]).max() < 5e-10
    # renormalising only removes the O(err) drift of |m|
    r2 = Oracle(w, renormalize=True).run(w.m0, w.a0, t_end=T, tol=1e-12)
    assert np.abs(r2.m - r.m).max() < 1e-9
    # fixed-step mode lands on the same solution
    r3 = o.run(w.m0, w.a0, fixed_dt=T / 3000, max_steps=3000)
    assert np.abs(r3.m.ravel() - sol.y[:nm, -1]).max() < 5e-10


def test_adaptive_controller_bookkeeping():
    w = W.cfg1("b", n=4)
    o = Oracle(w)
    r = o.run(w.m0, w.a0, t_end=20e-12, tol=1e-8, sample_dt=2e-12, trace_cap=10)
    assert r.status == 0 and r.t == 20e-12
    assert r.rhs_evals == 1 + 6 * (r.accepted + r.rejected)
    assert np.allclose(r.trace[:, 0], 2e-12 * np.arange(1, 11), rtol=0, atol=1e-24)
    # last trace row holds the final amplitudes
    assert r.trace[-1, 1] == r.a[0].real and r.trace[-1, 2] == r.a[0].imag
    # fixed-step trace: every 5th step
    r = o.run(w.m0, w.a0, fixed_dt=0.2e-12, max_steps=50, sample_dt=1e-12, trace_cap=100)
    assert r.trace.shape[0] == 10 and r.accepted == 50 and r.rejected == 0


# ----------------------------------------------------------------------------------------
# external drive eta_n(t) (PAPER.md:43 Eq. 1, :119 Eq. 12; Gaussian pulse of PAPER.md:229)
# ----------------------------------------------------------------------------------------
def _pulse(N, sigma=20e-12, t0=0.2e-9):
    amp = np.array([1e9 * (1 + 0.5j), 2e9 * (-0.3 + 1j), 0.5e9 * (0.2 - 1j)])[:N]
    return dict(amp=amp, t0=np.full(N, t0), sigma=np.full(N, sigma))


@pytest.mark.parametrize("mode", ["fixed", "adaptive"])
def test_gaussian_pulse_closed_form_uncoupled_cavity(mode):
    """g = 0: da/dt = -lambda a + A exp(-(t-t0)^2/(2 s^2)) exp(-i w_d (t-t0)), lambda = kappa + i w, has, once the pulse
    is over (t0 = 10 sigma, T - t0 = 15 sigma: truncation < 1e-20),
        a(T) = A s sqrt(2 pi) exp((lambda - i w_d)^2 s^2 / 2) exp(-lambda (T - t0)).
    Pins the drive's amplitude, envelope, carrier sign and the stage times t + c_s h (with all stages evaluated at t
    the result would be off by O(h / sigma))."""
    w = W.macrospin(10.0, [9.0, 10.5, 10.0], 0.0, [1.0, 50.0, 10.0], alpha=1e-3, a0=[0, 0, 0], n=2)
    dr = _pulse(3)
    dr["omega_d"] = np.array([0.0, TWO_PI * 10.5e9, TWO_PI * 9.7e9])     # baseband, resonant and detuned carrier
    o = Oracle(w, drive=dr)
    T = 0.5e-9
    r = o.run(w.m0, w.a0, t_end=T, fixed_dt=0.25e-12) if mode == "fixed" else o.run(w.m0, w.a0, t_end=T, tol=1e-12)
    lam = w.kappa + 1j * w.omega
    s = dr["sigma"]
    exact = dr["amp"] * s * math.sqrt(TWO_PI) * np.exp((lam - 1j * dr["omega_d"]) ** 2 * s ** 2 / 2) * np.exp(-lam * (T - dr["t0"]))
    assert np.all(np.abs(r.a - exact) <= (1e-10 if mode == "fixed" else 3e-9) * np.abs(exact))
    # the resonant carrier delivers the most: |a| = |A| s sqrt(2 pi) exp(kappa^2 s^2/2) exp(-kappa (T-t0))
    assert abs(abs(exact[1]) / (abs(dr["amp"][1]) * s[1] * math.sqrt(TWO_PI) * math.exp(-w.kappa[1] * (T - 0.2e-9))) - 1) < 1e-4


def test_drive_enters_at_the_stage_times_order_five():
    """With a time-dependent drive the scheme stays 5th order only if stage s is evaluated at t + c_s h."""
    w = _busy_problem()
    N = w.omega.size
    o = Oracle(w, renormalize=False, drive=dict(amp=np.full(N, 4e10 * (1 - 1j)), t0=np.full(N, 4e-12),
                                                  sigma=np.full(N, 2e-12), omega_d=w.omega))
    T = 8e-12
    ref = o.run(w.m0, w.a0, fixed_dt=T / 1024, max_steps=1024)
    errs = []
    for n in (32, 64, 128):
        r = o.run(w.m0, w.a0, fixed_dt=T / n, max_steps=n)
        errs.append(max(np.abs(r.m - ref.m).max(), np.abs(r.a - ref.a).max()))
    assert 22 < errs[0] / errs[1] < 44 and 22 < errs[1] / errs[2] < 44
    undriven = Oracle(w, renormalize=False).run(w.m0, w.a0, fixed_dt=T / 128, max_steps=128)
    assert np.abs(ref.a - undriven.a).max() > 1e3 * errs[2]          # the drive matters at this accuracy


def test_pulse_spectroscopy_shows_both_polariton_branches():
    """The paper's protocol: a short Gaussian pulse (sigma = 20 ps, t0 = 0.1 ns) on the cavity at
    resonance, then free evolution; the ring-down of a(t) holds both branches w_c +- g of Eq. 6 with equal weight."""
    g_mhz = 50.0
    w = W.macrospin(10.0, [10.0], g_mhz, 1.0, alpha=1e-4, a0=[0.0], n=2)
    o = Oracle(w, drive=dict(amp=np.array([1e8 + 0j]), t0=np.array([0.1e-9]), sigma=np.array([20e-12])))
    sdt = 20e-12
    r = o.run(w.m0, w.a0, t_end=40e-9, tol=1e-9, sample_dt=sdt, trace_cap=2000)
    tr = r.trace[r.trace[:, 0] > 0.3e-9]                              # after the pulse
    z = tr[:, 1] + 1j * tr[:, 2]
    om, amp = fit_exponentials(z, sdt, 4)
    om2, amp2 = dominant(om, amp, 2)
    f = om2.real / TWO_PI
    assert abs(f[0] - (10e9 - g_mhz * 1e6)) < 1e6 and abs(f[1] - (10e9 + g_mhz * 1e6)) < 1e6
    assert 0.8 < abs(amp2[0]) / abs(amp2[1]) < 1.25


# ----------------------------------------------------------------------------------------
# non-reciprocal coupling g_f != g_b (h0 = 2 g_b / gamma for the backward channel)
# ----------------------------------------------------------------------------------------
def test_nonreciprocal_coupling_geometric_mean():
    """Forward coefficient i g_f (Eq. 1), backward field h0 = 2 g_b/gamma: the linearised pair has
    (w - w_c)(w - w_m) = g_f g_b, i.e. the splitting and the Rabi period of a reciprocal system with g = sqrt(g_f g_b):
    g_f/2pi = 100 MHz, g_b/2pi = 25 MHz  ->  T_R = pi / (2pi 50 MHz) = 10 ns, like PAPER.md:237-239's g/2pi = 50 MHz."""
    w = W.macrospin(5.0, [5.0], 100.0, 0.0, alpha=0.0, a0=[0.01], n=2)
    o = Oracle(w, backward=dict(g=np.array([TWO_PI * 25e6])))
    r = o.run(w.m0, w.a0, t_end=26e-9, tol=1e-9, sample_dt=25e-12, trace_cap=1040)
    T = rabi_period(r.trace[:, 0], r.trace[:, 1] ** 2 + r.trace[:, 2] ** 2)
    assert abs(T / 10e-9 - 1) < 2e-3
    # the reciprocal system with g_f alone would oscillate twice as fast
    r2 = Oracle(w).run(w.m0, w.a0, t_end=26e-9, tol=1e-9, sample_dt=25e-12, trace_cap=1040)
    T2 = rabi_period(r2.trace[:, 0], r2.trace[:, 1] ** 2 + r2.trace[:, 2] ** 2)
    assert abs(T2 / 5e-9 - 1) < 2e-3
    # energy bookkeeping is asymmetric: the magnon amplitude reached is scaled by sqrt(g_b/g_f) relative to the
    # reciprocal case with the geometric-mean coupling (same a(0))
    w3 = W.macrospin(5.0, [5.0], 50.0, 0.0, alpha=0.0, a0=[0.01], n=2)
    r3 = Oracle(w3).run(w3.m0, w3.a0, t_end=26e-9, tol=1e-9, sample_dt=25e-12, trace_cap=1040)
    S_max, S3_max = np.abs(r.trace[:, 3] + 1j * r.trace[:, 4]).max(), np.abs(r3.trace[:, 3] + 1j * r3.trace[:, 4]).max()
    assert abs(S_max / S3_max - math.sqrt(25.0 / 100.0)) < 0.01
    # giving the backward coupling equal to the forward one changes nothing
    r4 = Oracle(w, backward=dict(g=w.g, Gamma=w.Gamma, Phi=w.Phi)).run(w.m0, w.a0, fixed_dt=0.5e-12, max_steps=200)
    r5 = Oracle(w).run(w.m0, w.a0, fixed_dt=0.5e-12, max_steps=200)
    assert np.array_equal(r4.m, r5.m) and np.array_equal(r4.a, r5.a)


# ----------------------------------------------------------------------------------------
# per-mode polarisation (the paper fixes x^; reading G32)
# ----------------------------------------------------------------------------------------
def _rot_z(v, phi):
    c, s = math.cos(phi), math.sin(phi)
    out = np.array(v, dtype=np.float64, copy=True)
    out[..., 0, :, :, :] = c * v[..., 0, :, :, :] - s * v[..., 1, :, :, :]
    out[..., 1, :, :, :] = s * v[..., 0, :, :, :] + c * v[..., 1, :, :, :]
    return out


def test_polarisation_y_reproduces_the_rabi_period():
    """A mode polarised along y^ (quadrature axis z^ x y^ = -x^) couples to m.y^ + i m.x^ and drives B_y: the problem is
    the paper's rotated by 90 degrees about the static field, so T_R = pi/g must come out again -
    nothing in this run touches the x^-polarised code path the other pins cover."""
    w = W.macrospin(5.0, [5.0], 50.0, 0.0, alpha=0.0, a0=[0.01], n=2)
    r = Oracle(w, pol=[[0.0, 1.0, 0.0]]).run(w.m0, w.a0, t_end=26e-9, tol=1e-9, sample_dt=25e-12, trace_cap=1040)
    T = rabi_period(r.trace[:, 0], r.trace[:, 1] ** 2 + r.trace[:, 2] ** 2)
    assert abs(T / 10e-9 - 1) < 2e-3
    # with the wrong quadrature sign (q = +x^: the counter-rotating component) there is no exchange
    r2 = Oracle(w, pol=[[0.0, 1.0, 0.0]], quad=[[1.0, 0.0, 0.0]]).run(w.m0, w.a0, t_end=26e-9, tol=1e-9,
                                                                       sample_dt=25e-12, trace_cap=1040)
    pa = r2.trace[:, 1] ** 2 + r2.trace[:, 2] ** 2
    assert pa.min() > 0.8 * pa.max()                      # only the fast counter-rotating ripple, no population exchange


def test_polarisation_is_covariant_under_rotation_about_the_field():
    """B0 along z^, anisotropy axis z^: rotating the initial magnetisation AND every mode's polarisation by phi about z^
    rotates the whole trajectory (the equations are covariant; a_n is a scalar).  Three profiled modes with different
    axes, exchange on, mixed coupling."""
    w = W.cfg3(nx=6, ny=5, nz=4)
    N = 3
    w.u, w.omega, w.kappa, w.g, w.Gamma, w.Phi = w.u[:N], w.omega[:N], w.kappa[:N], w.g[:N] * 30, w.g[:N] * 10, np.array([0.3, 0.0, 1.0])
    w.ku_axis = (0.0, 0.0, 1.0)
    w.m0 = W.tilted_state(5, 1, 6, 5, 4, 0.3)[None]
    w.a0 = np.array([1e-2, 2e-2j, -1e-2 + 1e-2j])
    ang = np.array([0.0, 0.7, 2.1])
    pol = np.stack([np.cos(ang), np.sin(ang), np.zeros(3)], axis=1)
    phi = 0.9
    pol_r = np.stack([np.cos(ang + phi), np.sin(ang + phi), np.zeros(3)], axis=1)
    r1 = Oracle(w, pol=pol).run(w.m0, w.a0, fixed_dt=0.1e-12, max_steps=200)
    r2 = Oracle(w, pol=pol_r).run(_rot_z(w.m0, phi), w.a0, fixed_dt=0.1e-12, max_steps=200)
    assert np.abs(r2.m - _rot_z(r1.m, phi)).max() < 1e-12
    assert np.abs(r2.a - r1.a).max() < 1e-12 * np.abs(r1.a).max()
    # the polarisation matters: all modes along x^ give another trajectory
    r0 = Oracle(w).run(w.m0, w.a0, fixed_dt=0.1e-12, max_steps=200)
    assert np.abs(r0.a - r1.a).max() > 1e-4 * np.abs(r1.a).max()
    # p = x^ given explicitly is the default, bit for bit
    rx = Oracle(w, pol=np.tile([1.0, 0.0, 0.0], (N, 1))).run(w.m0, w.a0, fixed_dt=0.1e-12, max_steps=50)
    rd = Oracle(w).run(w.m0, w.a0, fixed_dt=0.1e-12, max_steps=50)
    assert np.abs(rx.m - rd.m).max() < 1e-15 and np.abs(rx.a - rd.a).max() < 1e-15 * np.abs(rd.a).max()


def test_longitudinal_polarisation_closed_form():
    """p = z^ (along the static field, q = z^ x p = 0): the mode sees the constant S = <u m_z> = 1 and its field points
    along z^, so m = z^ never moves and a(t) = a_p + (a_0 - a_p) exp(-(i w + kappa) t), a_p = i G/(i w + kappa)
    (Eq. 12 with a constant source).  Pins the m.p projection and the q default."""
    w = W.macrospin(5.0, [5.0], 50.0, 20.0, alpha=1e-3, a0=[0.01], n=2)
    T = 0.4e-9
    r = Oracle(w, pol=[[0.0, 0.0, 1.0]]).run(w.m0, w.a0, t_end=T, tol=1e-12)
    lam = 1j * w.omega[0] + w.kappa[0]
    a_p = 1j * w.g[0] / lam
    exact = a_p + (w.a0[0] - a_p) * np.exp(-lam * T)
    assert abs(r.a[0] - exact) < 1e-9 * abs(exact)
    assert np.abs(r.m[0, 2] - 1.0).max() < 1e-15 and np.abs(r.m[0, :2]).max() < 1e-15


# ----------------------------------------------------------------------------------------
# the paper's tier-2 operator-split loop as a comparison integrator (reading G33)
# ----------------------------------------------------------------------------------------
def _rk4_R(z):
    return 1 + z + z ** 2 / 2 + z ** 3 / 6 + z ** 4 / 24


def test_split_cavity_half_is_classic_rk4():
    """g = 0: the cavity half alone.  Classic RK4 on a' = lambda a multiplies by R(z) = 1 + z + z^2/2 + z^3/6 + z^4/24,
    z = lambda dt, every step (PAPER.md:199 'fourth-order Runge-Kutta'): a_n = a_0 R(z)^n exactly."""
    w = W.macrospin(5.0, [5.0, 5.3], 0.0, [1.0, 30.0], alpha=1e-3, a0=[0.01, 0.02j], tilt=0.1, n=2)
    dt, n = 1e-12, 500
    r = Oracle(w).run_split(w.m0, w.a0, dt, n)
    z = -(1j * w.omega + w.kappa) * dt
    assert np.abs(r.a - w.a0 * _rk4_R(z) ** n).max() < 1e-13
    assert abs(r.t - n * dt) < 1e-24


def test_split_llg_half_is_the_unified_step_without_modes():
    """g = 0: the LLG half alone is n_llg Dormand-Prince steps of dt/n_llg with per-cell renormalisation, i.e. exactly
    what the (independently pinned) unified integrator does on the same plain-LLG problem at fixed step dt/n_llg."""
    w = W.cfg1("b", n=4)
    w.g = np.zeros(1)
    h = 0.1e-12
    r = Oracle(w).run_split(w.m0, w.a0, 2 * h, 50, n_llg=2)
    ref = Oracle(w).run(w.m0, w.a0, fixed_dt=h, max_steps=100)
    assert np.abs(r.m - ref.m).max() < 1e-15


def _split_one_step_map(wc, kap, g, wm, dt, field_from_new_a=True):
    """Hand-derived linear one-step map of Listing 1 for the macrospin at small angle, alpha = 0,
    on the vector (a, a*, mu, mu*), mu = m_x - i m_y:
      cavity half (RK4, mu frozen):  a' = R(z) a + i g dt phi(z) mu,  z = -(i wc + kappa) dt,
                                     phi(z) = 1 + z/2 + z^2/6 + z^3/24   (RK4 on a' = lambda a + const)
      LLG half (field b = (2/gamma) g Re a' frozen):  mu' = -i wm mu + i g (a' + a'*)  integrated
                                     exactly over dt:  mu(dt) = E mu + g (a' + a'*) (1 - E)/wm,  E = exp(-i wm dt)."""
    z = -(1j * wc + kap) * dt
    R, phi = _rk4_R(z), 1 + z / 2 + z ** 2 / 6 + z ** 3 / 24
    E = np.exp(-1j * wm * dt)
    c = g * (1 - E) / wm
    M = np.zeros((4, 4), dtype=np.complex128)
    M[0] = [R, 0, 1j * g * dt * phi, 0]
    M[1] = np.conj([0, R, 0, 1j * g * dt * phi])
    src = M[0] + M[1] if field_from_new_a else np.array([1, 1, 0, 0], dtype=np.complex128)
    M[2] = c * src + np.array([0, 0, E, 0])
    M[3] = np.conj(c) * (M[0] + M[1] if field_from_new_a else src) + np.array([0, 0, 0, np.conj(E)])
    return M


@pytest.mark.parametrize("dt_ps", [2.0, 4.0])
def test_split_rabi_period_follows_the_exact_one_step_map(dt_ps):
    """g/2pi = 50 MHz at 5 GHz, a(0) = 0.01 (Fig. 11): the Rabi period of the operator-split
    loop is 2 pi / (W+ - W-) with exp(-i W dt) the eigenvalues of the hand-derived one-step map above - NOT pi/g: the
    splitting error is what this integrator is kept for.  The map with the field taken from the OLD amplitudes (the
    other possible reading of Listing 1) gives a period that differs by several times the tolerance."""
    dt = dt_ps * 1e-12
    w = W.macrospin(5.0, [5.0], 50.0, 0.0, alpha=0.0, a0=[0.01], n=2)
    T = 32e-9
    n = int(round(T / dt))
    se = max(1, int(round(24e-12 / dt)))
    r = Oracle(w).run_split(w.m0, w.a0, dt, n, sample_every=se, trace_cap=n // se)
    T_sim = rabi_period(r.trace[:, 0], r.trace[:, 1] ** 2 + r.trace[:, 2] ** 2)

    def period(new):
        lam = np.linalg.eigvals(_split_one_step_map(w.omega[0], 0.0, w.g[0], GAMMA * w.B0[2], dt, new))
        W_ = np.sort((1j * np.log(lam) / dt).real)
        Wp = W_[W_ > 0]                       # the two polariton branches near +wc
        return TWO_PI / (Wp[1] - Wp[0])
    T_new, T_old = period(True), period(False)
    assert abs(T_sim / T_new - 1) < 3e-5
    assert abs(T_old / T_new - 1) > 3e-4                  # the pin tells the two readings apart
    assert abs(T_new / 10e-9 - 1) > 1e-4                  # and the splitting error is visible at this step size
    # the paper's bound: "the error remains below 3 % for all tested step sizes" up to 4 ps
    assert abs(T_sim / 10e-9 - 1) < 0.03


def test_split_converges_to_the_unified_integrator():
    """dt -> 0: the operator-split state approaches the unified RK45 one, and "the operator splitting is first order in
    dt": halving dt halves the distance.  (The Rabi PERIOD converges faster - reading m before and
    setting the field after the cavity step cancels its first-order term, see the one-step map above.)"""
    w = W.macrospin(5.0, [5.0], 50.0, 1.0, alpha=1e-3, a0=[0.01], tilt=0.02, n=2)
    T = 2e-9
    ref = Oracle(w).run(w.m0, w.a0, t_end=T, tol=1e-12)
    errs = []
    for dt in (2e-12, 1e-12, 0.5e-12):
        r = Oracle(w).run_split(w.m0, w.a0, dt, int(round(T / dt)))
        errs.append(abs(r.a[0] - ref.a[0]))
    assert 1.8 < errs[0] / errs[1] < 2.2 and 1.8 < errs[1] / errs[2] < 2.2 and errs[2] < 1e-4


# ----------------------------------------------------------------------------------------
# the plain Fourier sum behind the paper's spectra
# ----------------------------------------------------------------------------------------
def test_dft_equals_numpy_fft_on_the_fft_grid_and_peaks_at_the_signal_frequency():
    from oracle import dft
    rng = np.random.default_rng(3)
    n, d = 256, 20e-12
    x = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    t = d * np.arange(n)
    k = np.arange(n)
    X = dft(t, x, TWO_PI * k / (n * d))                   # sum_j x_j exp(+2 pi i j k / n) = n * ifft(x)
    assert np.abs(X - n * np.fft.ifft(x)).max() < 1e-10 * n
    # a time origin t0 only multiplies by exp(i w t0)
    X2 = dft(t + 3e-9, x, TWO_PI * k / (n * d))
    assert np.abs(X2 - X * np.exp(1j * TWO_PI * k / (n * d) * 3e-9)).max() < 1e-9 * n
    # x ~ exp(-i w0 t) peaks at +w0, off the FFT grid (the paper zero-pads 4x for that)
    w0 = TWO_PI * 5.013e9
    ws = TWO_PI * np.linspace(4.9e9, 5.1e9, 401)
    P = np.abs(dft(t, np.exp(-1j * w0 * t), ws)) ** 2
    assert abs(ws[P.argmax()] - w0) <= TWO_PI * 0.5e6 + 1e-3


# ----------------------------------------------------------------------------------------
# dipolar (demagnetising) field, SURVEY.md 8(f4) - off in the paper; reading G34
# ----------------------------------------------------------------------------------------
MU0 = 4e-7 * math.pi


def test_demag_tensor_identities():
    """Newell tensor: a cube's self term is 1/3 per axis, off-diagonals vanish there; the trace is 1 at the origin and 0
    for every other offset (div B = 0 outside the source cell); N_ij(-r) = N_ij(r); N_xy is odd in x and in y."""
    from oracle import demag_tensor
    T = demag_tensor(4, 3, 5, 2e-9, 2e-9, 2e-9)
    c = T[4, 2, 3]
    assert np.abs(c[:3] - 1.0 / 3.0).max() < 1e-12 and np.abs(c[3:]).max() < 1e-12
    tr = T[..., :3].sum(axis=-1)
    tr[4, 2, 3] -= 1.0
    assert np.abs(tr).max() < 1e-11
    assert np.abs(T - T[::-1, ::-1, ::-1]).max() < 1e-12
    assert np.abs(T[:, :, :, 3] + T[:, :, ::-1, 3]).max() < 1e-12 and np.abs(T[:, :, :, 3] + T[:, ::-1, :, 3]).max() < 1e-12
    # anisotropic cell: the thin direction carries almost all of the self demagnetisation
    Tp = demag_tensor(1, 1, 1, 100e-9, 100e-9, 1e-9)[0, 0, 0]
    assert abs(Tp[:3].sum() - 1.0) < 1e-10 and Tp[2] > 0.95 and abs(Tp[0] - Tp[1]) < 1e-10


def test_demag_tensor_far_field_and_brute_force():
    """Far away the cell pair is a pair of point dipoles, N_ij -> V/(4 pi) (delta_ij/r^3 - 3 r_i r_j/r^5), with a
    relative correction ~ (cell/r)^2; nearby, the tensor equals the average over sub-cell dipole pairs (brute force)."""
    from oracle import demag_tensor
    d = np.array([1.0, 1.5, 0.7])
    T = demag_tensor(12, 12, 12, *d)
    idx = {0: (0, 0), 1: (1, 1), 2: (2, 2), 3: (0, 1), 4: (0, 2), 5: (1, 2)}

    def dip(r):
        R = np.linalg.norm(r)
        return (np.eye(3) / R ** 3 - 3 * np.outer(r, r) / R ** 5) / (4 * math.pi)
    for off in ((11, 4, -7), (-9, 10, 11)):
        r = np.array(off) * d
        D = dip(r) * d.prod()
        got = T[11 + off[2], 11 + off[1], 11 + off[0]]
        for k, (i, j) in idx.items():
            assert abs(got[k] - D[i, j]) < 0.02 * np.abs(D).max()
    n = 6
    sub = (np.arange(n) + 0.5) / n - 0.5
    g = np.stack(np.meshgrid(sub, sub, sub, indexing="ij"), -1).reshape(-1, 3) * d
    for off in ((2, 1, 0), (1, 1, 1), (0, 0, 2)):
        r0 = np.array(off) * d
        acc = np.zeros((3, 3))
        for a in g:
            rr = r0 + a - g                                    # target sub-point minus source sub-points
            R = np.linalg.norm(rr, axis=1)
            acc += (np.eye(3)[None] / R[:, None, None] ** 3 - 3 * rr[:, :, None] * rr[:, None, :] / R[:, None, None] ** 5).sum(0)
        D = acc / (4 * math.pi) * d.prod() / n ** 6
        got = T[11 + off[2], 11 + off[1], 11 + off[0]]
        for k, (i, j) in idx.items():
            assert abs(got[k] - D[i, j]) < 0.02 * np.abs(D).max(), (off, k)


def test_demag_field_of_uniform_bodies():
    """Uniformly magnetised cube of n^3 cells: the volume-averaged demagnetising factor is exactly 1/3 per axis (sum over
    all cell pairs of N_aa / n^3).  A 41 x 41 x 1 slab: the field at the centre cell, read through the torque on a slightly
    tilted uniform state, has N_zz - N_xx close to 1 (thin-film limit) - the oracle's direct sum, not the table alone."""
    from oracle import demag_tensor
    T = demag_tensor(5, 5, 5, 5e-9, 5e-9, 5e-9)
    cnt = np.array([[[(5 - abs(i)) * (5 - abs(j)) * (5 - abs(k)) for i in range(-4, 5)] for j in range(-4, 5)] for k in range(-4, 5)])
    for axis in range(3):
        assert abs((T[..., axis] * cnt).sum() / 125.0 - 1.0 / 3.0) < 1e-12
    ws = W.macrospin(5.0, [5.0], 0.0, 0.0, alpha=0.0, n=2)
    ws.nx = ws.ny = 41; ws.nz = 1
    ws.u = np.ones((1, 1, 41, 41)); ws.B0 = (0.0, 0.0, 0.0)
    o = Oracle(ws, demag=True)
    eps = 1e-6
    m0 = np.zeros((1, 3, 1, 41, 41)); m0[0, 2] = 1.0; m0[0, 0] = eps           # m = z^ + eps x^
    dm, _, _ = o.rhs(m0 / math.sqrt(1 + eps * eps), np.zeros(1, dtype=np.complex128))
    # B_d = -mu0 Ms (N_zz z^ + eps N_xx x^) at the centre;  (m x B)_y = m_z B_x - m_x B_z = eps mu0 Ms (N_zz - N_xx)
    # dm_y/dt = -gamma (m x B)_y
    diff = dm[0, 1, 0, 20, 20] / (-GAMMA * eps * MU0 * ws.Ms)
    assert 0.90 < diff < 1.0
    # the same number from the table: sum over the slab of N_zz - N_xx seen from the centre cell
    Ts = demag_tensor(41, 41, 1, ws.dx, ws.dy, ws.dz)[0, 20:61, 20:61]
    assert abs(diff - (Ts[..., 2] - Ts[..., 0]).sum()) < 1e-6


def test_demag_shifts_the_kittel_line_of_a_platelet():
    """One flat cell (100 x 100 x 2 nm) magnetised along its normal in B0 z^: the macrospin precesses at
    w = gamma (B0 - mu0 Ms (N_zz - N_xx)) (Kittel's formula for a body with demagnetising factors N; small angle,
    alpha = 0).  Pins the sign and size of the dipolar term inside the LLG right-hand side."""
    from oracle import demag_tensor
    w = W.macrospin(10.0, [5.0], 0.0, 0.0, alpha=0.0, tilt=1e-3, n=1)
    w.dx = w.dy = 100e-9; w.dz = 2e-9
    N = demag_tensor(1, 1, 1, w.dx, w.dy, w.dz)[0, 0, 0]
    om = GAMMA * (w.B0[2] - MU0 * w.Ms * (N[2] - N[0]))
    T = 2e-9
    r = Oracle(w, demag=True).run(w.m0, w.a0, t_end=T, tol=1e-11)
    phase = math.atan2(r.m[0, 1, 0, 0, 0], r.m[0, 0, 0, 0, 0])
    expect = (om * T + math.pi) % TWO_PI - math.pi
    assert abs(((phase - expect) + math.pi) % TWO_PI - math.pi) < 2e-4
    assert abs(om / (GAMMA * w.B0[2]) - 1) > 0.3                   # the shift is large here (mu0 Ms = 0.176 T)
    # and off by default: the paper's setting
    r0 = Oracle(w).run(w.m0, w.a0, t_end=T, tol=1e-11)
    ph0 = math.atan2(r0.m[0, 1, 0, 0, 0], r0.m[0, 0, 0, 0, 0])
    e0 = (GAMMA * w.B0[2] * T + math.pi) % TWO_PI - math.pi
    assert abs(((ph0 - e0) + math.pi) % TWO_PI - math.pi) < 2e-4
