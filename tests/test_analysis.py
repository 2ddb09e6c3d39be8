"""Host post-processing formulas (paper_1110_6745_b200/analysis.py) against what the paper and textbooks fix."""
from fractions import Fraction
import math

import numpy as np
import pytest

from paper_1110_6745_b200 import analysis


def test_cumulants_eq18_on_an_exact_discrete_distribution():
    """eq. (18).  Samples = a multiset whose moments are exact rationals; the cumulants of a sum of
    independent variables add, so the cumulants of {0,1} x {0,2,5} (all 6 sums equally likely) are the sums of the
    cumulants of the two factors, computed here from central moments (kappa_2 = mu_2, kappa_3 = mu_3,
    kappa_4 = mu_4 - 3 mu_2^2)."""
    def central_cumulants(vals):
        n = len(vals)
        m = Fraction(sum(vals), n)
        mu = [sum((Fraction(v) - m) ** k for v in vals) / n for k in (2, 3, 4)]
        return [m, mu[0], mu[1], mu[2] - 3 * mu[0] ** 2]
    a, b = [0, 1], [0, 2, 5]
    expect = [x + y for x, y in zip(central_cumulants(a), central_cumulants(b))]
    samples = [x + y for x in a for y in b]
    got = analysis.cumulants(samples)
    for g, e in zip(got, expect):
        assert g == pytest.approx(float(e), rel=1e-12, abs=1e-12)


def test_cumulants_of_an_exponential_sample():
    """Exponential(1): kappa_n = (n-1)!  (statistical, 2e6 samples)."""
    rng = np.random.default_rng(5)
    k = analysis.cumulants(rng.exponential(1.0, 2_000_000))
    for n, kn in enumerate(k, start=1):
        assert kn == pytest.approx(math.factorial(n - 1), rel=0.03)


def test_width_distribution_is_normalised_with_unit_mean():
    rng = np.random.default_rng(6)
    w2 = rng.gamma(9.0, 0.3, 400_000)
    x, psi = analysis.width_distribution(w2, bins=120, x_range=(0.0, 4.0))
    dx = x[1] - x[0]
    assert psi.sum() * dx == pytest.approx(1.0, abs=1e-3)          # P(W^2 / <W^2>) integrates to 1
    assert (x * psi).sum() * dx == pytest.approx(1.0, abs=2e-3)     # and has mean 1 by construction


def test_config4_run_lengths_and_eq8_sampling_times():
    """BASELINE config 4: t = 20 L^1.61 (the integers SURVEY section 8(d) pins); eq. (8) with m = 0.01."""
    assert [analysis.steady_state_t_end(L) for L in (128, 256, 512, 1024, 2048)] == \
        [49390, 150764, 460209, 1404795, 4288163]
    t = analysis.sampling_times(0.01, 70000)
    assert t[:4] == [10, 20, 30, 41] and t[-1] <= 70000
    assert all(b > a for a, b in zip(t, t[1:]))
    # late times grow geometrically with ratio e^m
    assert t[-1] / t[-2] == pytest.approx(math.exp(0.01), rel=2e-3)


def test_growth_sampling_times():
    from paper_1110_6745_b200 import growth_run
    assert growth_run.sampling_times(64) == [1, 2, 4, 5, 8, 10, 16, 20, 32, 50, 64]
    ts = growth_run.sampling_times(10000)
    assert ts[-1] == 10000 and all(t in ts for t in (1, 2, 5, 10, 20, 50, 100, 200, 500, 1000, 2000, 5000, 8192))
    assert ts == sorted(set(ts))
