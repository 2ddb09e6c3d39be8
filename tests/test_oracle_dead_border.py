"""Dead-border schedule S5 (the paper's own device-level scheme) in the oracle: pins."""
import numpy as np
import pytest

from oracle import Oracle
from oracle import kpz_twin


@pytest.mark.parametrize("L,T,p,q,seed,n", [(16, 4, 1.0, 0.0, 5, 4), (24, 3, 0.6, 0.3, 6, 3), (32, 8, 0.75, 0.25, 7, 3),
                                            (32, 16, 1.0, 0.0, 8, 3)])
def test_oracle_equals_twin(L, T, p, q, seed, n):
    o = Oracle(L, p, q, T, seed)
    o.set_schedule("dead_border")
    o.init_flat()
    t = kpz_twin.Twin(L, p, q, T, seed, schedule="dead_border")
    t.init_flat()
    for _ in range(n):
        o.run(1)
        t.run(1)
        sx, sy = o.slopes()
        tx, ty = t.slopes()
        assert np.array_equal(sx, np.array(tx)) and np.array_equal(sy, np.array(ty))
        assert o.measure()[:2] == t.sums()
        assert o.check() == 0                      # conservation, curl-free, +-1 slopes


def test_edge_sites_of_a_tile_never_change_within_one_mcs():
    """P:60 'conflicts at the subsystem borders are avoided simply by not updating them'; Fig. 1: two edges are
    inactive.  Heights on the +x / +y edge of every tile of the shifted frame are unchanged by that MCS."""
    L, T = 64, 16
    o = Oracle(L, 1.0, 0.0, T, 3)
    o.set_schedule("dead_border")
    o.init_flat()
    for m in range(6):
        ox, oy, _ = o.global_draw(m)
        before = o.heights().astype(np.int64)
        o.run(1)
        after = o.heights().astype(np.int64)
        changed = before != after
        xs = (np.arange(L) - ox) % T == T - 1
        ys = (np.arange(L) - oy) % T == T - 1
        assert not changed[:, xs].any() and not changed[ys, :].any()
        assert changed.any()


def test_lost_attempts_fraction_and_thread_independence():
    """With p = 1 on the flat start of MCS 0 every attempt on a live even site flips unless an earlier flip of the
    same MCS touched it; the count with dead borders is below the colour schedule's and results do not depend on
    the number of OpenMP threads (tiles are independent)."""
    L, T = 128, 16
    res = []
    for threads in (1, 4):
        o = Oracle(L, 1.0, 0.0, T, 11, threads=threads)
        o.set_schedule("dead_border")
        o.init_flat()
        o.run(3)
        res.append((o.state_hash(), o.measure()[:2], o.counters()["deposits"]))
    assert res[0] == res[1]
    c = Oracle(L, 1.0, 0.0, T, 11)
    c.init_flat()
    c.run(3)
    live = (1 - 1 / T) ** 2
    ratio = res[0][2] / c.counters()["deposits"]
    assert live - 0.05 < ratio < 1.0
    assert c.counters()["attempts"] == 3 * L * L == Oracle.counters(o)["attempts"]


@pytest.mark.parametrize("L,T,p,q,K,sched", [(16, 4, 1.0, 0.0, 2, "colours"), (24, 3, 0.6, 0.3, 3, "colours"),
                                             (32, 8, 0.75, 0.25, 8, "dead_border"), (32, 4, 1.0, 0.0, 16, "colours")])
def test_sub_sweeps_oracle_equals_twin(L, T, p, q, K, sched):
    """Schedule S6: K sub-sweeps per MCS, each with its own draw, over consecutive slices of the tile streams."""
    o = Oracle(L, p, q, T, 5)
    o.set_schedule(sched); o.set_sub_sweeps(K)
    o.init_flat(); o.run(3)
    t = kpz_twin.Twin(L, p, q, T, 5, schedule=sched, sub_sweeps=K)
    t.init_flat(); t.run(3)
    sx, sy = o.slopes()
    tx, ty = t.slopes()
    assert np.array_equal(sx, np.array(tx)) and np.array_equal(sy, np.array(ty))
    assert o.measure()[:2] == t.sums() and o.check() == 0
    assert o.counters()["attempts"] == 3 * L * L


def test_sub_sweeps_one_is_the_default_and_bad_values_are_rejected():
    a = Oracle(64, 1.0, 0.0, 16, 9); a.init_flat(); a.run(2)
    b = Oracle(64, 1.0, 0.0, 16, 9); b.set_sub_sweeps(1); b.init_flat(); b.run(2)
    c = Oracle(64, 1.0, 0.0, 16, 9); c.set_sub_sweeps(4); c.init_flat(); c.run(2)
    assert a.state_hash() == b.state_hash() != c.state_hash()
    with pytest.raises(ValueError):
        a.set_sub_sweeps(7)


def test_poisson_table_is_the_poisson_law():
    """Schedule S7: the integer-defined count table equals the Poisson(lambda = T*T/K) distribution function to
    the 2^-32 resolution of its thresholds (scipy's regularised gamma function as the independent reference)."""
    from scipy.stats import poisson
    for (T, K) in ((16, 1), (64, 1), (64, 16), (32, 4), (4, 2)):
        o = Oracle(2 * T, 1.0, 0.0, T, 1)
        o.set_sub_sweeps(K); o.set_poisson(True)
        kmin, thr = o.poisson_table()
        lam = T * T // K
        cdf = poisson.cdf(kmin + np.arange(len(thr)), lam)
        assert np.max(np.abs(thr.astype(np.float64) / 2.0 ** 32 - cdf)) < 3e-10
        assert thr[-1] == 2 ** 32 and np.all(np.diff(thr.astype(np.int64)) >= 0)
        assert kmin <= lam < kmin + len(thr)


@pytest.mark.parametrize("L,T,p,q,K,sched", [(16, 4, 1.0, 0.0, 1, "colours"), (24, 3, 0.6, 0.3, 3, "colours"),
                                             (32, 8, 0.75, 0.25, 2, "dead_border"), (32, 4, 1.0, 0.0, 4, "colours")])
def test_poissonised_counts_oracle_equals_twin(L, T, p, q, K, sched):
    o = Oracle(L, p, q, T, 5)
    o.set_schedule(sched); o.set_sub_sweeps(K); o.set_poisson(True)
    o.init_flat(); o.run(3)
    t = kpz_twin.Twin(L, p, q, T, 5, schedule=sched, sub_sweeps=K, poisson=True)
    t.init_flat(); t.run(3)
    sx, sy = o.slopes()
    tx, ty = t.slopes()
    assert np.array_equal(sx, np.array(tx)) and np.array_equal(sy, np.array(ty))
    assert o.measure()[:2] == t.sums() and o.check() == 0
    assert o.counters()["attempts"] == t.attempts
    kmin, thr = o.poisson_table()
    assert kmin == t.kmin and [int(v) for v in thr] == t.thr


def test_poissonised_attempt_counts_have_poisson_mean_and_variance():
    """Per MCS the number of attempts is a sum of NT^2 independent Poisson(T*T) counts: mean L*L, variance L*L."""
    L, T, n = 64, 8, 400
    o = Oracle(L, 0.0, 0.0, T, 77)         # p = q = 0: only the counting matters, the surface never changes
    o.set_poisson(True)
    o.init_flat()
    per_mcs = []
    last = 0
    for _ in range(n):
        o.run(1)
        a = o.counters()["attempts"]
        per_mcs.append(a - last)
        last = a
    per_mcs = np.array(per_mcs, dtype=np.float64)
    lam = L * L
    assert abs(per_mcs.mean() - lam) < 4 * np.sqrt(lam / n)
    assert 0.8 * lam < per_mcs.var(ddof=1) < 1.25 * lam
    assert o.measure()[2] == 0.25
