"""Exact Markov chains on L=4 and L=6 tori vs the oracle (north star: brute-force enumeration of the exact
stationary distribution compared with long-run visit frequencies)."""
from fractions import Fraction
from pathlib import Path

import numpy as np
import pytest

from oracle import Oracle
import exact_small as E

GOLD = {}
for _l in (Path(__file__).parent / "golden" / "exact_small_chains.txt").read_text().splitlines():
    if _l and not _l.startswith("#"):
        k, v = _l.split()
        GOLD[k] = v


def test_enumeration_matches_recorded_exact_values():
    for L in (2, 4, 6):
        B, PI, pats = E.enumerate_states(L)
        assert len(B) == int(GOLD["zero_tilt_states_L%d" % L])
        if L > 2:
            S1, S2 = E.sums_per_state(B, PI, pats)
            N = L * L
            mean = Fraction(int((N * S2 - S1 * S1).sum()), N * N * len(B))
            a, b = GOLD["mean_W2_uniform_L%d" % L].split("/")
            assert mean == Fraction(int(a), int(b))
            w2 = (N * S2 - S1 * S1) / float(N * N)
            assert w2.min() == 0.25 and (w2 == 0.25).sum() == 2            # the two checkerboards (reading R7)
            assert w2.max() == {4: 1.0, 6: 11 / 6}[L]


@pytest.fixture(scope="module")
def chains():
    out = {}
    for (p, q) in ((1.0, 0.0), (0.75, 0.25), (0.5, 0.5)):
        ch = E.ExactChain(4, 2, p, q)
        out[(p, q)] = (ch, ch.mcs_kernel())
    return out


def _flat_index(ch):
    flat = np.array([[(x + y) & 1 for x in range(4)] for y in range(4)])
    return ch.index[E.key_of(flat)]


@pytest.mark.parametrize("p,q,tag", [(1.0, 0.0, "DD_p1_q0"), (0.75, 0.25, "DD_p075_q025")])
def test_exact_chain_reproduces_recorded_transients(chains, p, q, tag):
    """My own matrix construction reproduces the independently recorded E[W^2(t)] of SURVEY App. C to 6 digits."""
    ch, M = chains[(p, q)]
    v = np.zeros(ch.n); v[_flat_index(ch)] = 1.0
    got = {}
    for t in range(1, 9):
        v = v @ M
        got[t] = float(v @ ch.w2)
    for t in (1, 2, 4, 8):
        assert abs(got[t] - float(GOLD["%s_EW2_t%d" % (tag, t)])) < 1.5e-6
    pi = ch.stationary(M)
    assert abs(float(pi @ ch.w2) - float(GOLD[tag + "_EW2_stationary"])) < 1.5e-6
    assert abs(float(pi @ ch.min_density()) - float(GOLD[tag + "_min_density_stationary"])) < 1.5e-6


@pytest.mark.parametrize("p,q", [(1.0, 0.0), (0.75, 0.25)])
def test_oracle_transient_ensemble_vs_exact(chains, p, q):
    """E[W^2(t)] from the flat state, t = 1..8: ensemble of oracle runs (different seeds) vs the exact chain."""
    ch, M = chains[(p, q)]
    v = np.zeros(ch.n); v[_flat_index(ch)] = 1.0
    exact, var = [], []
    for t in range(1, 9):
        v = v @ M
        mu = float(v @ ch.w2)
        exact.append(mu); var.append(float(v @ (ch.w2 - mu) ** 2))
    n = 20000
    acc = np.zeros(8)
    for s in range(n):
        o = Oracle(4, p, q, 2, seed=1000 + s)
        o.init_flat()
        for t in range(8):
            o.run(1)
            acc[t] += o.measure()[2]
    mean = acc / n
    for t in range(8):
        sigma = np.sqrt(var[t] / n)
        assert abs(mean[t] - exact[t]) < 4.5 * sigma, (t, mean[t], exact[t], sigma)


@pytest.mark.parametrize("p,q", [(1.0, 0.0), (0.75, 0.25), (0.5, 0.5)])
def test_oracle_visit_frequencies_vs_exact_stationary_L4(chains, p, q):
    """Long-run visit frequencies over the 990 states vs the stationary vector of the oracle's own schedule."""
    ch, M = chains[(p, q)]
    pi = ch.stationary(M)
    if p == q:
        assert np.abs(pi - 1.0 / ch.n).sum() < 1e-10           # uniform over the zero-tilt sector, exactly
        assert abs(float(pi @ ch.w2) - 92 / 165) < 1e-12
    o = Oracle(4, p, q, 2, seed=31337)
    o.init_flat()
    o.run(200)
    n = 300000
    counts = np.zeros(ch.n)
    w2acc = []
    for i in range(n):
        o.run(1)
        sx, sy = o.slopes()
        # heights in the gauge h(0,0)=0 from the slopes (eq. 3 walk)
        hx0 = np.concatenate([[0], np.cumsum(sx[0, 1:].astype(np.int64))])
        h = hx0[None, :] + np.concatenate([np.zeros((1, 4), dtype=np.int64),
                                           np.cumsum(sy[1:, :].astype(np.int64), axis=0)], axis=0)
        counts[ch.index[E.key_of(h)]] += 1
        w2acc.append(ch.w2[ch.index[E.key_of(h)]])
    freq = counts / n
    tv = 0.5 * np.abs(freq - pi).sum()
    # expected TV of n iid draws ~ 0.5*sum sqrt(2 pi_i/(pi n)) ~ 0.023; samples are correlated -> allow 2x
    assert tv < 0.05, tv
    # scalar check with batch means (robust to autocorrelation); discriminates DD (0.552) from RS (0.584) at p=1
    w = np.array(w2acc).reshape(100, -1).mean(axis=1)
    assert abs(w.mean() - float(pi @ ch.w2)) < 5 * w.std(ddof=1) / np.sqrt(len(w))
    assert w.std(ddof=1) / np.sqrt(len(w)) < 2e-3


@pytest.mark.parametrize("T", [3, 1])
def test_oracle_L6_p_equals_q_uniform_stationary(T):
    """p = q: every single-site kernel is symmetric, so the stationary law is uniform over the 5 482 716
    zero-tilt states for ANY schedule.  Compare the long-run W^2 histogram with exact enumeration."""
    B, PI, pats = E.enumerate_states(6)
    S1, S2 = E.sums_per_state(B, PI, pats)
    num = 36 * S2 - S1 * S1                         # W^2 * 36^2, integer
    vals, cnts = np.unique(num, return_counts=True)
    exact = cnts / cnts.sum()
    o = Oracle(6, 0.5, 0.5, T, seed=2024 + T)
    o.init_flat()
    o.run(500)
    n = 200000
    got = np.zeros(n, dtype=np.int64)
    for i in range(n):
        o.run(2)
        s1, s2, _ = o.measure()
        got[i] = 36 * s2 - s1 * s1
    assert np.all(np.isin(got, vals))
    means = (got / 1296.0).reshape(100, -1).mean(axis=1)
    assert abs(means.mean() - 1218213 / 1827572) < 5 * means.std(ddof=1) / 10
    # histogram over coarse bins of W^2 (each with >= 2% mass)
    order = np.argsort(vals)
    cdf = np.cumsum(exact[order])
    edges = [vals[order][np.searchsorted(cdf, qv)] for qv in np.linspace(0.1, 0.9, 9)]
    eb = np.bincount(np.searchsorted(edges, vals), weights=exact, minlength=10)
    gb = np.bincount(np.searchsorted(edges, got), minlength=10) / n
    assert np.abs(eb - gb).max() < 0.01
