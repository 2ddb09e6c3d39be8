"""Pins of the CPU oracle against what the paper and the mathematics fix (no GPU, no CUDA path)."""
from fractions import Fraction
from pathlib import Path

import numpy as np
import pytest

import oracle
from oracle import Oracle
from oracle import kpz_twin
import kpz_inputs as gen

GOLDEN = Path(__file__).parent / "golden"


def _kat():
    rows = []
    for line in (GOLDEN / "philox4x32_10_kat.txt").read_text().splitlines():
        if line.startswith("#") or not line.strip():
            continue
        v = [int(t, 16) for t in line.split()]
        rows.append((v[0:4], v[4:6], v[6:10]))
    return rows


def test_philox_known_answers_cpp_and_twin():
    rows = _kat()
    assert len(rows) == 3
    for ctr, key, out in rows:
        assert [int(v) for v in oracle.philox4x32_10(ctr, key)] == out
        assert kpz_twin.philox4x32_10(ctr, key) == out


def test_philox_counter_and_key_positions_matter():
    # a transposed counter/key word must change the output (guards against symmetric-looking mistakes)
    base = [int(v) for v in oracle.philox4x32_10([1, 2, 3, 4], [5, 6])]
    assert base != [int(v) for v in oracle.philox4x32_10([2, 1, 3, 4], [5, 6])]
    assert base != [int(v) for v in oracle.philox4x32_10([1, 2, 4, 3], [5, 6])]
    assert base != [int(v) for v in oracle.philox4x32_10([1, 2, 3, 4], [6, 5])]
    assert base == kpz_twin.philox4x32_10([1, 2, 3, 4], [5, 6])


def test_thresholds_exact():
    assert oracle.threshold(1.0) == 1 << 32
    assert oracle.threshold(0.0) == 0
    assert oracle.threshold(0.75) == 3 << 30
    assert oracle.threshold(0.25) == 1 << 30
    assert oracle.threshold(0.5) == 1 << 31
    for pr in (1.0, 0.0, 0.75, 0.25, 0.3):
        assert kpz_twin.threshold(pr) == oracle.threshold(pr)


@pytest.mark.parametrize("L,T", [(8, 4), (64, 16), (256, 16), (12, 3)])
def test_flat_state_paper_pin(L, T):
    """zig-zag start has W^2(L,0) = 1/4 exactly; sum h = sum h^2 = L^2/2 for h in {0,1}."""
    pins = dict(l.split()[:2] for l in (GOLDEN / "paper_pins.txt").read_text().splitlines() if l and l[0] != "#")
    o = Oracle(L, 1.0, 0.0, T, seed=1, shadow=True)
    o.init_flat()
    s1, s2, w2 = o.measure()
    assert s1 == L * L // 2 and s2 == L * L // 2
    assert w2 == float(pins["W2_flat"]) == 0.25
    assert o.check() == 0
    sx, sy = o.slopes()
    # every even-parity site is a local minimum (-1,+1;-1,+1), every odd one a local maximum
    a, b, c, d = sx, np.roll(sx, -1, axis=1), sy, np.roll(sy, -1, axis=0)
    y, x = np.mgrid[0:L, 0:L]
    even = ((x + y) & 1) == 0
    assert np.all((a == -1) & (b == 1) & (c == -1) & (d == 1) == even)
    assert np.all((a == 1) & (b == -1) & (c == 1) & (d == -1) == ~even)
    assert np.array_equal(o.heights(), gen.flat_heights(L))
    assert np.array_equal(o.shadow_heights(), gen.flat_heights(L))


def test_striped_separable_state_is_rejected_reading():
    """Reading R7: the separable 'striped' state (sx depends on x only, sy on y only) has W^2 = 1/2, not 1/4."""
    L = 16
    h = gen.triangle_heights(L, 1)
    o = Oracle(L, 1.0, 0.0, 4, seed=1)
    o.set_slopes(*gen.heights_to_slopes(h), h00=int(h[0, 0]))
    assert o.measure()[2] == 0.5


@pytest.mark.parametrize("L,A", [(16, 1), (16, 2), (16, 4), (32, 8), (64, 16), (48, 3)])
def test_triangle_wave_closed_form(L, A):
    """h = tri_A(x) + tri_A(y): W^2 = (A^2 + 2)/6 exactly, mean = A (closed form)."""
    h = gen.triangle_heights(L, A)
    T = 4 if L % 8 == 0 else 3
    o = Oracle(L, 1.0, 0.0, T, seed=1)
    o.set_slopes(*gen.heights_to_slopes(h), h00=int(h[0, 0]))
    s1, s2, w2 = o.measure()
    N = L * L
    assert Fraction(s1, N) == A
    assert Fraction(N * s2 - s1 * s1, N * N) == Fraction(A * A + 2, 6)
    assert w2 == float(Fraction(A * A + 2, 6)) or abs(w2 - (A * A + 2) / 6) < 1e-15
    assert np.array_equal(o.heights(), h)


@pytest.mark.parametrize("seed", [0, 1, 2])
def test_measure_equals_direct_definition_and_path_independence(seed):
    """eq. 3 reading R4 vs (i) the generating height field itself, (ii) the y-then-x walk, on random surfaces."""
    L = 32
    h = gen.raised_flat_heights(L, seed) + 7          # h00 = 7 or 9
    sx, sy = gen.heights_to_slopes(h)
    o = Oracle(L, 1.0, 0.0, 4, seed=1)
    o.set_slopes(sx, sy, h00=int(h[0, 0]))
    assert np.array_equal(o.heights(), h)
    s1, s2, w2 = o.measure()
    assert s1 == int(h.sum()) and s2 == int((h * h).sum())
    assert Fraction(w2) == Fraction(L * L * s2 - s1 * s1, (L * L) ** 2)   # power-of-two N: division exact
    # other path: walk y along column 0 first, then x along row y
    col0 = h[0, 0] + np.concatenate([[0], np.cumsum(sy[1:, 0].astype(np.int64))])
    h2 = col0[:, None] + np.concatenate([np.zeros((L, 1), dtype=np.int64),
                                         np.cumsum(sx[:, 1:].astype(np.int64), axis=1)], axis=1)
    assert np.array_equal(h2, h)


def test_large_heights_int128_sums():
    L = 64
    h = gen.staircase_heights(L, 5) + 3_000_000_000      # |h| > 2^31: needs 64-bit heights, 128-bit sums safe
    o = Oracle(L, 1.0, 0.0, 16, seed=1)
    o.set_slopes(*gen.heights_to_slopes(h), h00=int(h[0, 0]))
    s1, s2, w2 = o.measure()
    assert s1 == int(h.sum())
    assert s2 == sum(int(v) ** 2 for v in h.ravel())
    ref = Fraction(L * L * s2 - s1 * s1, (L * L) ** 2)
    assert Fraction(w2) == ref or abs(w2 - float(ref)) <= 1e-12 * float(ref)


@pytest.mark.parametrize("L,T,p,q", [(8, 4, 1.0, 0.0), (8, 4, 0.75, 0.25), (8, 2, 0.5, 0.5), (12, 3, 0.3, 0.9),
                                     (16, 4, 1.0, 1.0), (6, 1, 0.6, 0.2)])
def test_invariants_after_every_single_attempt(L, T, p, q):
    """After EVERY attempt: slopes +-1, row sums of sx and column sums of sy conserved (Kawasaki exchange, eq. 2),
    curl-free on all plaquettes, shadow heights consistent, and the surface total moves by exactly 2*dir."""
    o = Oracle(L, p, q, T, seed=11, shadow=True)
    o.init_flat()
    assert o.run_checked(6) == 0
    c = o.counters()
    assert c["mcs"] == 6 and c["attempts"] == 6 * L * L
    s1, s2, _ = o.measure()
    assert s1 - L * L // 2 == 2 * (c["deposits"] - c["removals"])
    assert c["deposits"] > 0
    if q > 0:
        assert c["removals"] > 0


def test_invariants_random_start():
    L = 16
    h = gen.raised_flat_heights(L, 3, 0.3)
    o = Oracle(L, 0.7, 0.4, 4, seed=5, shadow=True)
    o.set_slopes(*gen.heights_to_slopes(h), h00=int(h[0, 0]))
    s1a = o.measure()[0]
    assert o.run_checked(4) == 0
    c = o.counters()
    assert o.measure()[0] - s1a == 2 * (c["deposits"] - c["removals"])


def test_p1_q0_monotone_growth_two_per_flip():
    L, T = 64, 16
    o = Oracle(L, 1.0, 0.0, T, seed=3, shadow=True)
    o.init_flat()
    prev_s1, prev_dep = L * L // 2, 0
    hprev = o.heights()
    for t in range(1, 9):
        o.run(1)
        s1, _, _ = o.measure()
        c = o.counters()
        assert c["removals"] == 0
        assert s1 - prev_s1 == 2 * (c["deposits"] - prev_dep) and s1 >= prev_s1
        hnow = o.heights()
        assert np.all(hnow >= hprev) and np.all((hnow - hprev) % 2 == 0)
        assert np.array_equal(hnow, o.shadow_heights())          # h00 bookkeeping anchors eq. 3 correctly
        prev_s1, prev_dep, hprev = s1, c["deposits"], hnow
    assert o.check() == 0


def test_p0_q0_never_changes():
    o = Oracle(32, 0.0, 0.0, 8, seed=9)
    o.init_flat()
    a = o.slopes()
    o.run(5)
    b = o.slopes()
    assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1])
    assert o.counters()["deposits"] == 0 and o.counters()["removals"] == 0


def test_first_mcs_from_flat_p1_flips_only_minima_once_each_at_most_in_sequence():
    """From the flat start with p=1: a site can be raised only while it is a local minimum; after one MCS every
    height is 0/1 (untouched), 2 (even site raised) or 3 (odd site raised after its 4 neighbours) ..."""
    L = 64
    o = Oracle(L, 1.0, 0.0, 16, seed=2)
    o.init_flat()
    o.run(1)
    h = o.heights()
    assert h.min() >= 0 and o.check() == 0
    assert np.all(np.abs(h - np.roll(h, 1, 0)) == 1) and np.all(np.abs(h - np.roll(h, 1, 1)) == 1)


def test_run_split_equals_run_whole_and_thread_independence():
    a = Oracle(64, 0.75, 0.25, 16, seed=21)
    b = Oracle(64, 0.75, 0.25, 16, seed=21, threads=4)
    a.init_flat(); b.init_flat()
    a.run(7)
    b.run(3); b.run(4)
    assert a.state_hash() == b.state_hash()
    assert a.measure() == b.measure()
    assert a.counters() == b.counters()
    c = Oracle(64, 0.75, 0.25, 16, seed=22)
    c.init_flat(); c.run(7)
    assert c.state_hash() != a.state_hash()
    d = Oracle(64, 0.75, 0.25, 16, seed=21, replica=1)
    d.init_flat(); d.run(7)
    assert d.state_hash() != a.state_hash()


def test_window_oracle_matches_full_oracle_inside_light_cone():
    """A windowed run (garbage outside) equals the full run on the inner block shrunk by 4*(T+1) per MCS."""
    L, T, n = 256, 16, 2
    full = Oracle(L, 0.75, 0.25, T, seed=5)
    full.init_flat(); full.run(n)
    fsx, fsy = full.slopes()
    wx0, wy0, W = 200, 230, 200          # wraps around both edges
    win = Oracle(L, 0.75, 0.25, T, seed=5, window=(wx0, wy0, W, W))
    win.init_flat(); win.run(n)
    wsx, wsy = win.slopes()
    M = 4 * (T + 1) * n
    ys = (wy0 + np.arange(W)) % L
    xs = (wx0 + np.arange(W)) % L
    sub_x = fsx[np.ix_(ys, xs)]
    sub_y = fsy[np.ix_(ys, xs)]
    assert np.array_equal(wsx[M:W - M, M:W - M], sub_x[M:W - M, M:W - M])
    assert np.array_equal(wsy[M:W - M, M:W - M], sub_y[M:W - M, M:W - M])
    assert not np.array_equal(wsx, sub_x)     # the margin really is garbage, i.e. the test is not vacuous


def test_mcs_is_exactly_L2_attempts_and_each_tile_gets_T2():
    L, T = 16, 4
    tw = kpz_twin.Twin(L, 1.0, 0.0, T, seed=4)
    tw.init_flat(); tw.trace = []
    tw.run(1)
    assert len(tw.trace) == L * L
    ox, oy, perm = tw.global_draw(0)
    assert ox % 4 == 0 and oy % 4 == 0 and sorted(perm) == [0, 1, 2, 3]
    counts = {}
    for (x, y, d) in tw.trace:
        tx, ty = ((x - ox) % L) // T, ((y - oy) % L) // T
        counts[(tx, ty)] = counts.get((tx, ty), 0) + 1
    assert len(counts) == (L // T) ** 2 and set(counts.values()) == {T * T}
    # colour passes come in the drawn order
    order = []
    for (x, y, d) in tw.trace:
        tx, ty = ((x - ox) % L) // T, ((y - oy) % L) // T
        col = (tx & 1) + 2 * (ty & 1)
        if not order or order[-1] != col:
            order.append(col)
    assert order == perm


def test_set_clock_restarts_a_trajectory_and_parallel_measure_is_thread_independent():
    """set_clock only moves the MCS clock (S1: counter word c2): a lattice copied out after 2 MCS and
    restarted at clock 2 continues the original trajectory bit for bit; the clock stops at 2^32 - 1.  The
    measurement and the hash do not depend on the number of threads of their column / site loops."""
    L, T, seed = 64, 16, 9
    a = Oracle(L, 0.75, 0.25, T, seed)
    a.init_flat(); a.run(2)
    sx, sy = a.slopes()
    h00 = a.counters()["h00"]
    a.run(1)
    b = Oracle(L, 0.75, 0.25, T, seed, threads=4)
    b.set_slopes(sx, sy, h00=h00)
    b.set_clock(2)
    b.run(1)
    bx, by = b.slopes()
    ax, ay = a.slopes()
    assert np.array_equal(ax, bx) and np.array_equal(ay, by)
    assert a.measure() == b.measure() and a.state_hash() == b.state_hash()
    assert b.counters()["mcs"] == 3 and b.counters()["attempts"] == 3 * L * L
    h = gen.heights_to_slopes(ax.astype(np.int64).cumsum(axis=1) * 0 + Oracle.heights(a).astype(np.int64))
    assert np.array_equal(h[0], ax) and np.array_equal(h[1], ay)        # heights() inverts to the same slopes
    c = Oracle(L, 1.0, 0.0, T, seed)
    c.init_flat(); c.set_clock(2**32 - 2)
    c.run(1)
    with pytest.raises(RuntimeError):
        c.run(1)
    with pytest.raises(ValueError):
        c.set_clock(2**32)
