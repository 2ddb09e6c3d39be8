"""TEST INFRASTRUCTURE, NOT THE PRODUCT -- plain definition of the power spectrum of a height field.

Kelling & Odor, arXiv:1110.6745, eq. (15)-(16):
    S(k) = <h(k) h(-k)>,   h(k) = L^(-d/2) sum_x [h(x) - <h>] exp(i k.x),   d = 2,
"computed from the surface profiles with the FFT method ... averaging over x and y directions".  Reading taken
(DESIGN.md "Power spectrum"): the full two-dimensional transform (numpy.fft.fft2, fp64) of the height field of ONE
surface, read off along the two lattice axes, S_x(n) = |h(k_n, 0)|^2 and S_y(n) = |h(0, k_n)|^2 with k_n = 2 pi n / L,
n = 0..L/2, and S(n) = (S_x(n) + S_y(n)) / 2; the ensemble average <.> is the caller's mean over surfaces.
Shares no code with the CUDA path (which never forms the 2-D transform).  Pinned by tests/test_oracle_spectrum.py:
closed-form spectrum of triangle-wave surfaces, Parseval on the axes, invariance under a constant shift.
"""
from __future__ import annotations

import numpy as np


def power_spectrum(h):
    """h: integer height field indexed [y, x], L x L.  Returns (S, Sx, Sy), float64 arrays of length L/2 + 1."""
    h = np.asarray(h, dtype=np.float64)
    L = h.shape[0]
    assert h.shape == (L, L)
    hk = np.fft.fft2(h - h.mean()) / L          # L^(-d/2) with d = 2; the sign of the exponent does not enter |.|^2
    P = (hk * hk.conj()).real
    n = L // 2 + 1
    Sx = P[0, :n].copy()                         # k_y = 0 (axis 0 of the array is y)
    Sy = P[:n, 0].copy()                         # k_x = 0
    return 0.5 * (Sx + Sy), Sx, Sy


def profiles(h):
    """Exact column sums sum_y h(x,y) and row sums sum_x h(x,y) (int64) of a height field indexed [y, x]."""
    h = np.asarray(h, dtype=np.int64)
    return h.sum(axis=0), h.sum(axis=1)
