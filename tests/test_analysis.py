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
    assert growth_run.sampling_times(64) == [1, 2, 4, 5, 8, 10, 16, 20, 25, 32, 50, 64]
    ts = growth_run.sampling_times(10000)
    assert ts[-1] == 10000 and all(t in ts for t in (1, 2, 5, 10, 20, 50, 100, 200, 500, 1000, 2000, 5000, 8192))
    assert ts == sorted(set(ts))


def test_beta_eff_eq11_and_fit_eq12_recover_the_generating_parameters():
    """eq. (9), (11), (12).  W(t) = b t^beta (1 + b1 t^phi1) with the paper's own numbers (beta = 0.2415,
    b1 = -0.12, |phi1| = 1.05) on top of the intrinsic 1/4: the local slopes with t/t' = 2 tend to
    beta, and the fit of the form (12) returns beta, b1, phi1.  The discrete slope of eq. (11) differs from the
    derivative in eq. (12) by the known factor (2^-phi1 ... ) -- so the fit is pinned on the exact derivative, and the
    discrete slopes on their own closed form."""
    beta, b1, phi1, b = 0.2415, -0.12, -1.05, 0.7
    t = np.array([2 ** i for i in range(4, 18)], dtype=np.float64)
    W = b * t ** beta * (1.0 + b1 * t ** phi1)
    be = analysis.beta_eff(t.astype(int), W ** 2 + 0.25)
    assert [x[0] for x in be] == [int(v) for v in t[1:]]
    for (tt, v) in be:
        exact = beta + math.log2((1 + b1 * tt ** phi1) / (1 + b1 * (tt / 2) ** phi1))
        assert v == pytest.approx(exact, abs=1e-12)
    assert be[-1][1] == pytest.approx(beta, abs=2e-6)
    # eq. (12) is the logarithmic derivative to first order in the correction: generate it exactly and refit
    y = beta + b1 * phi1 * t ** phi1
    f = analysis.fit_correction(t, y)
    assert f["asymptote"] == pytest.approx(beta, abs=1e-9)
    assert f["amplitude"] == pytest.approx(b1, rel=1e-6) and f["exponent"] == pytest.approx(phi1, rel=1e-6)
    # with noise of the size of the paper's error bar (1.5e-3) beta is still recovered within it
    rng = np.random.default_rng(12)
    tt = np.array([50 * 1.3 ** i for i in range(28)])
    f = analysis.fit_correction(tt, beta + b1 * phi1 * tt ** phi1 + rng.normal(0, 2e-4, tt.size))
    assert f["asymptote"] == pytest.approx(beta, abs=1.5e-3)


def test_alpha_eff_eq13_and_fit_eq14():
    """eq. (10), (13), (14), P:119-127 with the paper's numbers (alpha = 0.393, a1 = -1.24, |omega1| = 1.16)."""
    alpha, a1, om = 0.393, -1.24, -1.16
    sizes = [2 ** i for i in range(7, 14)]
    W = [0.4 * L ** alpha * (1 + a1 * L ** om) for L in sizes]
    ae = analysis.alpha_eff(sizes, [w * w for w in W], intrinsic=0.0)
    assert [x[0] for x in ae] == sizes[1:]
    for L, v in ae:
        assert v == pytest.approx(alpha + math.log2((1 + a1 * L ** om) / (1 + a1 * (L / 2) ** om)), abs=1e-12)
    # pure power law: every local slope equals alpha; the intrinsic width is removed before the logarithm
    ae = analysis.alpha_eff(sizes, [0.25 + 0.16 * L ** (2 * alpha) for L in sizes])
    assert all(v == pytest.approx(alpha, abs=1e-12) for _, v in ae)
    Ls = np.array(sizes, dtype=np.float64)
    f = analysis.fit_correction(Ls, alpha + a1 * om * Ls ** om)
    assert (f["asymptote"], f["amplitude"], f["exponent"]) == pytest.approx((alpha, a1, om), rel=1e-6)
    assert f["at_bound"] is False
    flat = analysis.fit_correction(Ls, alpha + 1e-3 * (-1.0) ** np.arange(Ls.size))      # no trend: not resolvable
    assert flat["at_bound"] is True and flat["asymptote"] == pytest.approx(alpha, abs=2e-3)
    with pytest.raises(ValueError):
        analysis.fit_correction([1, 2], [1, 2])


def test_cumulant_power_laws_eq19_eq20():
    """eq. (19)-(20): kappa_n = L^(2 n alpha) (k0 + k1 L^-omega1)."""
    alpha, om = 0.393, 1.16
    sizes = np.array([512, 1024, 2048, 4096, 8192], dtype=np.float64)       # the sizes of Fig. 7
    for n, (k0, k1) in enumerate([(0.05, 0.3), (2e-3, -0.01), (1e-4, 2e-3), (4e-6, 1e-4)], start=1):
        pure = k0 * sizes ** (2 * n * alpha)
        c, s = analysis.fit_power_law(sizes, pure)
        assert c == pytest.approx(k0, rel=1e-9) and s / (2 * n) == pytest.approx(alpha, abs=1e-12)
        kap = sizes ** (2 * n * alpha) * (k0 + k1 * sizes ** (-om))
        f = analysis.fit_cumulant_fss(sizes, kap, n, alpha, omega1=om)
        assert f["kappa0"] == pytest.approx(k0, rel=1e-8) and f["kappa1"] == pytest.approx(k1, rel=1e-6)
        g = analysis.fit_cumulant_fss(sizes, kap, n, alpha)
        assert g["omega1"] == pytest.approx(om, rel=1e-5) and g["kappa0"] == pytest.approx(k0, rel=1e-6)


def test_finite_size_scaling_reduces_run_outputs():
    """steady_state.finite_size_scaling on synthetic run() outputs: <W^2> = 1/4 + a L^(2 alpha) gives alpha_eff = alpha
    at every size after the subtraction of the intrinsic width, and less without it (eq. 13); the cumulant power
    laws of eq. (19) return alpha_n = alpha."""
    from paper_1110_6745_b200 import steady_state
    alpha = 0.393
    runs = [{"L": L, "cumulants": [0.25 + 0.15 * L ** (2 * alpha), 2e-3 * L ** (4 * alpha), 1e-4 * L ** (6 * alpha),
                                   -1.0]} for L in (128, 256, 512, 1024, 2048)]
    f = steady_state.finite_size_scaling(runs)
    assert [a["L"] for a in f["alpha_eff"]] == [256, 512, 1024, 2048]
    assert all(a["alpha_eff"] == pytest.approx(alpha, abs=1e-12) for a in f["alpha_eff"])
    assert all(a["alpha_eff"] < alpha for a in f["alpha_eff_raw"])
    assert [c["n"] for c in f["cumulant_power_laws"]] == [1, 2, 3]    # kappa_4 < 0 here: no power law
    assert all(c["alpha_n"] == pytest.approx(alpha, abs=1e-12) for c in f["cumulant_power_laws"][1:])
    assert f["cumulant_power_laws"][0]["alpha_n"] < alpha               # kappa_1 still carries the additive 1/4
    assert "eq14_fit" in f
    assert "eq14_fit" not in steady_state.finite_size_scaling(runs[:4])     # three slopes cannot fix three parameters


def test_pool_cumulants_equals_cumulants_of_the_union():
    """eq. (18) on batches: pooling (n, cumulants) of three unequal batches reproduces the cumulants of all samples
    together, and the inversion cumulants -> moments is exact on a rational example."""
    rng = np.random.default_rng(8)
    parts = [rng.gamma(7.0, 1.3, n) for n in (6400, 19200, 1000)]
    pooled = analysis.pool_cumulants([(len(p), analysis.cumulants(p)) for p in parts])
    direct = analysis.cumulants(np.concatenate(parts))
    for a, b in zip(pooled, direct):
        assert a == pytest.approx(b, rel=1e-9)
    vals = [0, 1, 1, 3]                                    # nu = 5/4, 11/4, 29/4, 83/4
    assert analysis.moments_from_cumulants(analysis.cumulants(vals)) == pytest.approx((1.25, 2.75, 7.25, 20.75), rel=1e-12)


def test_pool_batches_and_fss_with_the_pooled_size():
    """steady_state.pool_batches: four batches of one size pool to the cumulants of all their samples; a pooled size
    joins the other sizes in the finite-size scaling; sizes cannot be mixed."""
    from paper_1110_6745_b200 import steady_state
    rng = np.random.default_rng(9)
    parts = [rng.gamma(9.0, 5.6, 6400) for _ in range(4)]
    batches = [{"L": 2048, "replicas": 64, "seed": 4 + i, "n_samples": p.size, "cumulants": list(analysis.cumulants(p))}
               for i, p in enumerate(parts)]
    pooled = steady_state.pool_batches(batches)
    assert pooled["replicas"] == 256 and pooled["n_samples"] == 25600 and pooled["seeds"] == [4, 5, 6, 7]
    for a, b in zip(pooled["cumulants"], analysis.cumulants(np.concatenate(parts))):
        assert a == pytest.approx(b, rel=1e-9)
    alpha = 0.39
    runs = [{"L": L, "cumulants": [0.25 + 0.15 * L ** (2 * alpha), 1.0, 1.0, 1.0]} for L in (128, 256, 512, 1024)]
    big = dict(pooled, cumulants=[0.25 + 0.15 * 2048 ** (2 * alpha), 1.0, 1.0, 1.0])
    f = steady_state.finite_size_scaling(runs + [big])
    assert [a["L"] for a in f["alpha_eff"]] == [256, 512, 1024, 2048] and "eq14_fit" in f
    assert all(a["alpha_eff"] == pytest.approx(alpha, abs=1e-12) for a in f["alpha_eff"])
    with pytest.raises(ValueError):
        steady_state.pool_batches(batches + [dict(batches[0], L=1024)])
