"""Host post-processing of the per-replica W^2 samples the hot path produces (steady-state study).

Nothing here runs on the hot path: these are the few scalar formulas the paper applies to the measured widths.
  * cumulants           -- eq. (18): kappa_1..kappa_4 from the non-central moments nu_n of W^2
  * pool_cumulants      -- eq. (18) over the union of several batches (moments pool as weighted averages)
  * width_distribution  -- Psi_L(x) = <W^2> P_L(W^2 / <W^2>), as a normalised histogram
  * steady_state_t_end  -- run length of BASELINE config 4: t = 20 L^1.61 MCS, rounded up
  * sampling_times      -- eq. (8): t_{i+1} = (t_i + 10) e^m, t_0 = 0, as distinct integers floor(t_i)
  * beta_eff            -- eq. (11): local slopes of ln W against ln t with t / t' = 2, after W^2(0) = 1/4 is
                           subtracted
  * alpha_eff           -- eq. (13): local slopes of the saturated width against ln L between L and L/2
  * fit_correction      -- the common shape of eq. (12), P:107-111 and eq. (14), P:125-127:
                           y(x) = y_inf + c1 e x^e  (beta_eff = beta + b1 phi1 t^phi1, alpha_eff = alpha + a1 omega1 L^omega1)
  * fit_power_law       -- eq. (19): kappa_n ~ L^(2 n alpha), straight line in logarithms
  * fit_cumulant_fss    -- eq. (20): kappa_n = L^(2 n alpha) (kappa_n^0 + kappa_n^1 L^(-omega1))

Reading of eq. (12) and (14) (R19): the printed forms are the exact logarithmic derivatives of
W = b t^beta (1 + b1 t^phi1) and W = a L^alpha (1 + a1 L^omega1) to first order in the correction, so the exponent
phi1 / omega1 is SIGNED here and negative for a correction that dies out; the paper quotes the magnitudes (phi1 = 1.05,
omega1 = 1.16) and writes the sign explicitly only in eq. (20) (L^(-omega1)).
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


def moments_from_cumulants(k):
    """Inverse of eq. (18): (nu_1..nu_4) from (kappa_1..kappa_4)."""
    k1, k2, k3, k4 = k
    n1 = k1
    n2 = k2 + k1 ** 2
    n3 = k3 + 3.0 * n1 * n2 - 2.0 * n1 ** 3
    n4 = k4 + 4.0 * n3 * n1 + 3.0 * n2 ** 2 - 12.0 * n1 ** 2 * n2 + 6.0 * n1 ** 4
    return n1, n2, n3, n4


def pool_cumulants(batches):
    """Cumulants of the union of several batches of samples, each given as (n_samples, (kappa_1..kappa_4)): the
    non-central moments of eq. (18) are plain averages, so they pool with the sample counts as weights.  For
    ensembles run as several independent batches (e.g. config 4's 256 replicas of L = 2048 as four runs of 64)."""
    n_tot = float(sum(n for n, _ in batches))
    nu = [sum(n * m for n, m in zip([b[0] for b in batches], col)) / n_tot
          for col in zip(*[moments_from_cumulants(k) for _, k in batches])]
    n1, n2, n3, n4 = nu
    return (n1, n2 - n1 ** 2, n3 - 3.0 * n1 * n2 + 2.0 * n1 ** 3,
            n4 - 4.0 * n3 * n1 - 3.0 * n2 ** 2 + 12.0 * n1 ** 2 * n2 - 6.0 * n1 ** 4)


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


def beta_eff(times, w2, ratio=2, intrinsic=0.25):
    """eq. (11) with t / t' = ratio: beta_eff(t) = [ln W(t) - ln W(t/ratio)] / ln(ratio), W^2 := w2 - intrinsic (the
    zig-zag start's W^2(L,0) = 1/4, "a leading order constant correction ... that we subtract").
    Returns [(t, beta_eff)] for every sampled t whose partner t/ratio was sampled too."""
    w = {int(t): float(v) - intrinsic for t, v in zip(times, w2)}
    out = []
    for t in sorted(w):
        if t % ratio == 0 and t // ratio in w and w[t // ratio] > 0.0 and w[t] > 0.0:
            out.append((t, 0.5 * math.log(w[t] / w[t // ratio]) / math.log(ratio)))
    return out


def alpha_eff(sizes, w2_sat, intrinsic=0.25):
    """eq. (13): alpha_eff(L) = [ln W(inf, L) - ln W(inf, L/2)] / [ln L - ln(L/2)] for every L whose half size is in
    `sizes`; W^2 := w2_sat - intrinsic (same subtraction as in the growth analysis; intrinsic = 0 gives the
    slopes of the raw widths).  Returns [(L, alpha_eff)]."""
    w = {int(L): float(v) - intrinsic for L, v in zip(sizes, w2_sat)}
    return [(L, 0.5 * math.log(w[L] / w[L // 2]) / math.log(2.0))
            for L in sorted(w) if L % 2 == 0 and L // 2 in w and w[L // 2] > 0.0 and w[L] > 0.0]


def fit_correction(x, y, exponent_range=(-4.0, -0.05), weights=None):
    """Least-squares fit of y(x) = y_inf + c1 e x^e (eq. 12: x = t, y = beta_eff, y_inf = beta, c1 = b1, e = phi1;
    eq. 14: x = L, y = alpha_eff, y_inf = alpha, c1 = a1, e = omega1; e signed, see the module docstring).
    For a fixed e the model is linear in (y_inf, c1 e): the exponent is found by a bounded 1-D search over the
    profiled residual.  Returns {"asymptote", "amplitude" (= c1), "exponent", "rss", "at_bound"}; at_bound = the exponent
    ran into the edge of exponent_range, i.e. the correction is not resolved by the data."""
    from scipy.optimize import minimize_scalar
    x = np.asarray(x, dtype=np.float64)
    y = np.asarray(y, dtype=np.float64)
    if x.size < 3:
        raise ValueError("three parameters need at least three points")
    w = np.ones_like(y) if weights is None else np.sqrt(np.asarray(weights, dtype=np.float64))

    def solve(e):
        A = np.stack([np.ones_like(x), x ** e], axis=1) * w[:, None]
        coef, *_ = np.linalg.lstsq(A, y * w, rcond=None)
        r = A @ coef - y * w
        return coef, float(r @ r)

    grid = np.linspace(exponent_range[0], exponent_range[1], 80)
    rss = [solve(e)[1] for e in grid]
    i = int(np.argmin(rss))
    lo, hi = grid[max(0, i - 1)], grid[min(len(grid) - 1, i + 1)]
    res = minimize_scalar(lambda e: solve(e)[1], bounds=(lo, hi), method="bounded", options={"xatol": 1e-10})
    e = float(res.x)
    coef, r = solve(e)
    # an exponent on the edge of the search range means the data do not resolve the correction term (e.g. local slopes
    # that are flat within their noise): only the asymptote is meaningful then
    at_bound = min(abs(e - exponent_range[0]), abs(e - exponent_range[1])) < 1e-3 * (exponent_range[1] - exponent_range[0])
    return {"asymptote": float(coef[0]), "amplitude": float(coef[1]) / e, "exponent": e, "rss": r, "at_bound": bool(at_bound)}


def fit_power_law(x, y):
    """y = c x^s as a straight line in logarithms (eq. 19: x = L, y = kappa_n, s = 2 n alpha).  Returns (c, s)."""
    lx, ly = np.log(np.asarray(x, dtype=np.float64)), np.log(np.asarray(y, dtype=np.float64))
    s, lc = np.polyfit(lx, ly, 1)
    return float(math.exp(lc)), float(s)


def fit_cumulant_fss(sizes, kappa, n, alpha, omega1=None):
    """eq. (20): kappa_n L^(-2 n alpha) = kappa_n^0 + kappa_n^1 L^(-omega1).  With omega1 given the fit is linear;
    otherwise the exponent is fitted too (fit_correction).  Returns {"kappa0", "kappa1", "omega1", "rss"}."""
    L = np.asarray(sizes, dtype=np.float64)
    y = np.asarray(kappa, dtype=np.float64) * L ** (-2.0 * n * alpha)
    if omega1 is not None:
        A = np.stack([np.ones_like(L), L ** (-float(omega1))], axis=1)
        coef, *_ = np.linalg.lstsq(A, y, rcond=None)
        r = A @ coef - y
        return {"kappa0": float(coef[0]), "kappa1": float(coef[1]), "omega1": float(omega1), "rss": float(r @ r)}
    f = fit_correction(L, y)
    return {"kappa0": f["asymptote"], "kappa1": f["amplitude"] * f["exponent"], "omega1": -f["exponent"], "rss": f["rss"]}
