"""Observable extraction shared by the oracle pins and the GPU-vs-oracle observable parity
tests (harness only; neither the oracle nor the CUDA path imports it).

SURVEY.md G25: polariton frequencies are extracted by fitting a uniformly sampled complex
trace to a sum of damped complex exponentials (matrix pencil), not by FFT peak picking —
the paper's FFT bins (62.5 MHz) are coarser than the splittings here.
"""
from __future__ import annotations

import numpy as np


def fit_exponentials(x: np.ndarray, dt: float, n_poles: int, pencil: int | None = None):
    """Matrix-pencil fit  x[k] ~ sum_j A_j z_j^k.

    Returns (omega, amp): complex angular frequencies with the paper's sign convention
    x(t) ~ A exp(-i omega t), i.e. omega = i log(z)/dt, Re = frequency,
    -Im = amplitude decay rate; sorted by Re(omega).
    """
    x = np.asarray(x, dtype=np.complex128)
    n = x.shape[0]
    L = pencil if pencil is not None else n // 3
    Y = np.lib.stride_tricks.sliding_window_view(x, L + 1)          # (n-L) x (L+1) Hankel
    U, s, Vh = np.linalg.svd(Y, full_matrices=False)
    V = Vh[:n_poles].T                                               # (L+1) x M
    V1, V2 = V[:-1], V[1:]
    z = np.linalg.eigvals(np.linalg.pinv(V1) @ V2)
    # amplitudes by least squares
    k = np.arange(n)[:, None]
    Z = z[None, :] ** k
    amp = np.linalg.lstsq(Z, x, rcond=None)[0]
    omega = 1j * np.log(z) / dt
    order = np.argsort(omega.real)
    return omega[order], amp[order]


def dominant(omega: np.ndarray, amp: np.ndarray, n: int):
    """The n components of largest |amplitude|, sorted by frequency."""
    idx = np.argsort(-np.abs(amp))[:n]
    idx = idx[np.argsort(omega[idx].real)]
    return omega[idx], amp[idx]


def _parabolic_extremum(t, y, i):
    if i <= 0 or i >= len(y) - 1:
        return t[i]
    d = (y[i - 1] - 2 * y[i] + y[i + 1])
    if d == 0:
        return t[i]
    off = 0.5 * (y[i - 1] - y[i + 1]) / d
    return t[i] + off * (t[1] - t[0])


def rabi_period(t: np.ndarray, pop: np.ndarray) -> float:
    """Period of the population exchange |a|^2(t): mean spacing of successive minima
    (parabolic interpolation); PAPER.md:239 T_R = pi/g."""
    y = np.asarray(pop, dtype=np.float64)
    mins = [i for i in range(1, len(y) - 1) if y[i] < y[i - 1] and y[i] <= y[i + 1]]
    # keep deep minima only (population exchange), not the fast wiggles
    thr = y.min() + 0.2 * (y.max() - y.min())
    mins = [i for i in mins if y[i] < thr]
    # merge minima closer than 1/4 of the largest gap (counter-rotating ripple)
    tm = np.array([_parabolic_extremum(t, y, i) for i in mins])
    if len(tm) < 2:
        raise ValueError("need at least two Rabi minima")
    gaps = np.diff(tm)
    keep = [0]
    for j in range(1, len(tm)):
        if tm[j] - tm[keep[-1]] > 0.5 * gaps.max():
            keep.append(j)
    tm = tm[keep]
    return float(np.mean(np.diff(tm)))
