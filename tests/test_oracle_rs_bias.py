"""Oracle schedule vs true single-site random-sequential dynamics (north star: ensemble W^2(t) within 3 sigma).

SURVEY App. D measured a real, T-dependent bias of the domain decomposition (-2 % at T=16, <1 % at T>=32 for
p=1; none detectable at p=0.75/q=0.25; exactly none in the stationary state for p=q).  Following its
recommendation the assertion is |bias| <= 3 sigma OR <= 3 %, with the run count stated, at the config's own T.
"""
import numpy as np
import pytest

from oracle import Oracle


def _ensemble(L, T, p, q, runs, t_end, rs, schedule="colours", sub_sweeps=1, poisson=False):
    w = np.zeros(runs)
    for r in range(runs):
        o = Oracle(L, p, q, T, seed=900 + r, threads=2)
        o.set_schedule(schedule)
        o.set_sub_sweeps(sub_sweeps)
        o.set_poisson(poisson)
        o.init_flat()
        (o.run_rs if rs else o.run)(t_end)
        w[r] = o.measure()[2]
    return w.mean(), w.std(ddof=1) / np.sqrt(runs)


@pytest.mark.parametrize("L,T,p,q,runs,t_end", [
    (128, 32, 1.0, 0.0, 48, 32),
    (128, 64, 1.0, 0.0, 48, 32),
    (128, 32, 0.75, 0.25, 48, 32),
    (128, 16, 1.0, 0.0, 48, 32),
])
def test_schedule_bias_vs_true_random_sequential(L, T, p, q, runs, t_end):
    dd, e1 = _ensemble(L, T, p, q, runs, t_end, rs=False)
    rs, e2 = _ensemble(L, T, p, q, runs, t_end, rs=True)
    sigma = np.hypot(e1, e2)
    bias = dd - rs
    assert abs(bias) <= 3 * sigma or abs(bias) <= 0.03 * rs, (dd, rs, sigma)
    assert 1.0 < rs < 3.0          # growth really happened (W^2 well above the flat 1/4)


def test_dead_border_schedule_bias_vs_true_random_sequential():
    """Schedule S5 loses 1 - (1-1/T)^2 of the attempts ("impacts the pre-factors of the scaling, but not
    exponents"): at T = 64 the width after 32 MCS stays within 3 sigma or 5 % of true RS dynamics."""
    L, T, runs, t_end = 128, 64, 48, 32
    dd, e1 = _ensemble(L, T, 1.0, 0.0, runs, t_end, rs=False, schedule="dead_border")
    rs, e2 = _ensemble(L, T, 1.0, 0.0, runs, t_end, rs=True)
    bias, sigma = dd - rs, np.hypot(e1, e2)
    assert abs(bias) <= 3 * sigma or abs(bias) <= 0.05 * rs, (dd, rs, sigma)


def test_bias_knobs_bring_the_small_tile_schedule_within_three_sigma():
    """S:App. D: at T = 16 the default schedule sits about 2 % below true RS dynamics (frozen neighbours +
    stratified attempt counts); 16 sub-sweeps with Poissonised counts (S6 + S7) remove that.  L = 256, 64 MCS,
    64 runs each: the knobs' ensemble is within 3 sigma of RS (measured: +0.7 % +- 0.6 %; default -1.7 %)."""
    L, T, runs, t_end = 256, 16, 64, 64
    kn, e1 = _ensemble(L, T, 1.0, 0.0, runs, t_end, rs=False, sub_sweeps=16, poisson=True)
    rs, e2 = _ensemble(L, T, 1.0, 0.0, runs, t_end, rs=True)
    assert abs(kn - rs) <= 3 * np.hypot(e1, e2), (kn, rs, e1, e2)


def test_rs_reference_itself_against_exact_L4():
    """The RS reference is pinned too: its stationary <W^2> on L=4, p=1, q=0 is 0.583896 (exact chain)."""
    import exact_small as E
    ch = E.ExactChain(4, 2, 1.0, 0.0)
    pi = ch.stationary(ch.rs_mcs_kernel())
    o = Oracle(4, 1.0, 0.0, 2, seed=5)
    o.init_flat(); o.run_rs(100)
    w = np.zeros(100000)
    for i in range(len(w)):
        o.run_rs(1)
        w[i] = o.measure()[2]
    b = w.reshape(100, -1).mean(axis=1)
    assert abs(b.mean() - float(pi @ ch.w2)) < 5 * b.std(ddof=1) / 10
    assert abs(float(pi @ ch.w2) - 0.583896) < 1.5e-6
