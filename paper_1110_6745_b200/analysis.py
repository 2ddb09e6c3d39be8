"""Host post-processing of the per-replica W^2 samples the hot path produces (steady-state study).

Nothing here runs on the hot path: these are the few scalar formulas the paper applies to the measured widths.
  * cumulants           -- eq. (18): kappa_1..kappa_4 from the non-central moments nu_n of W^2
  * width_distribution  -- Psi_L(x) = <W^2> P_L(W^2 / <W^2>), as a normalised histogram
  * steady_state_t_end  -- run length of BASELINE config 4: t = 20 L^1.61 MCS, rounded up
  * sampling_times      -- eq. (8): t_{i+1} = (t_i + 10) e^m, t_0 = 0, as distinct integers floor(t_i)
"""
from __future__ import annotations

import math

import numpy as np


def noncentral_moments(w2, n_max=4):
    """nu_n = <(W^2)^n>, n = 1..n_max, over all samples (float64)."""
    x = np.asarray(w2, dtype=np.float64).ravel()
    return [float(np.mean(x ** n)) for n in range(1, n_max + 1)]


def cumulants(w2):
    """(kappa_1, kappa_2, kappa_3, kappa_4) of the W^2 samples by eq. (18)."""
    n1, n2, n3, n4 = noncentral_moments(w2, 4)
    k1 = n1
    k2 = n2 - n1 ** 2
    k3 = n3 - 3.0 * n1 * n2 + 2.0 * n1 ** 3
    k4 = n4 - 4.0 * n3 * n1 - 3.0 * n2 ** 2 + 12.0 * n1 ** 2 * n2 - 6.0 * n1 ** 4
    return k1, k2, k3, k4


def width_distribution(w2, bins=50, x_range=(0.0, 3.0)):
    """Psi_L(x) = <W^2> P_L(W^2 / <W^2>) on a uniform grid of x = W^2 / <W^2>.
    Returns (x_centres, psi) with sum(psi) * dx = fraction of the samples inside x_range."""
    x = np.asarray(w2, dtype=np.float64).ravel()
    x = x / x.mean()
    hist, edges = np.histogram(x, bins=bins, range=x_range)
    dx = edges[1] - edges[0]
    return 0.5 * (edges[:-1] + edges[1:]), hist / (x.size * dx)


def steady_state_t_end(L):
    """BASELINE config 4: 'run to t = 20 * L^1.61 MCS' (rounded up)."""
    return int(math.ceil(20.0 * float(L) ** 1.61))


def sampling_times(m, t_max):
    """eq. (8): t_{i+1} = (t_i + 10) e^m, t_0 = 0; returns the distinct integers floor(t_i) in (0, t_max]."""
    out, t = [], 0.0
    while True:
        t = (t + 10.0) * math.exp(m)
        ti = int(math.floor(t))
        if ti > t_max:
            return out
        if not out or ti != out[-1]:
            out.append(ti)
