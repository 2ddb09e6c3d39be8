"""Pins of oracle/spectrum.py (eq. 15-16) against what the mathematics fixes."""
import numpy as np
import pytest

from oracle.spectrum import power_spectrum, profiles
from kpz_inputs import triangle_heights, staircase_heights, raised_flat_heights


@pytest.mark.parametrize("L,A", [(32, 2), (64, 4), (64, 16), (96, 3), (128, 8)])
def test_triangle_wave_closed_form(L, A):
    """h = tri_A(x) + tri_A(y): tri_A is a box of length A convolved with itself, so its DFT over one period 2A has
    modulus sin^2(pi j / 2) / sin^2(pi j / 2A).  On the k_x axis only the x-dependent part survives:
    S_x(n) = (L / 2A)^2 / sin^4(pi j / 2A) for n = j L / 2A with j odd, and 0 for every other n (same for S_y)."""
    S, Sx, Sy = power_spectrum(triangle_heights(L, A))
    expect = np.zeros(L // 2 + 1)
    for j in range(1, 2 * A, 2):
        n = j * L // (2 * A)
        if n <= L // 2:
            expect[n] = (L / (2 * A)) ** 2 / np.sin(np.pi * j / (2 * A)) ** 4
    scale = expect.max()
    assert np.allclose(Sx, expect, rtol=0, atol=1e-10 * scale)
    assert np.allclose(Sy, expect, rtol=0, atol=1e-10 * scale)
    assert np.allclose(S, expect, rtol=0, atol=1e-10 * scale)


@pytest.mark.parametrize("seed", [1, 2])
def test_parseval_on_the_axes_and_shift_invariance(seed):
    L = 64
    h = staircase_heights(L, seed) + raised_flat_heights(L, seed + 10) - (np.add.outer(np.arange(L), np.arange(L)) & 1)
    S, Sx, Sy = power_spectrum(h)
    c, r = profiles(h)
    # sum over the whole k_x axis of |h(k,0)|^2 = (1/L) sum_x (c(x) - mean c)^2 ; modes n and L-n are conjugates
    full_x = Sx[0] + 2 * Sx[1:L // 2].sum() + Sx[L // 2]
    full_y = Sy[0] + 2 * Sy[1:L // 2].sum() + Sy[L // 2]
    assert full_x == pytest.approx(((c - c.mean()) ** 2).sum() / L, rel=1e-12)
    assert full_y == pytest.approx(((r - r.mean()) ** 2).sum() / L, rel=1e-12)
    assert Sx[0] == pytest.approx(0.0, abs=1e-9) and Sy[0] == pytest.approx(0.0, abs=1e-9)
    S2, Sx2, Sy2 = power_spectrum(h + 12345)
    assert np.allclose(Sx2, Sx, rtol=1e-9, atol=1e-9) and np.allclose(Sy2, Sy, rtol=1e-9, atol=1e-9)
    # x <-> y exchanges the two axes
    St, Sxt, Syt = power_spectrum(h.T)
    assert np.allclose(Sxt, Sy) and np.allclose(Syt, Sx) and np.allclose(St, S)


def test_separable_surface_has_independent_axes():
    """h = u(x) + v(y): S_x depends on u only and equals the 1-D spectrum of L*u / L."""
    L = 64
    h = staircase_heights(L, 5)
    u = h[0, :] - h[0, 0]
    S, Sx, Sy = power_spectrum(h)
    uk = np.fft.fft(u - u.mean())          # h(k,0) = (1/L) * L * u(k)
    assert np.allclose(Sx, (np.abs(uk) ** 2)[:L // 2 + 1], rtol=1e-10, atol=1e-8)
