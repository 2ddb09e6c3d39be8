"""Host logic of kpz_step_host_overlapped, checked exhaustively on the CPU: the schedule that
kpz_overlap_plan returns is replayed as sets of lattice rows, with no GPU and no kernel.

What makes the overlapped step exact is a statement about ORDER only: the kernels, tile ids and random streams are those
of kpz_run, so the trajectory is the same iff
  (1) every tile row of every colour pass is launched exactly once,
  (2) a launch only touches rows that have arrived,
  (3) two tiles of different passes whose footprints share a lattice row run in pass order,
  (4) a row is copied back only after the last launch that touches it, and every row is copied back exactly once.
A colour pass on a tile touches the T + 1 storage rows oy + t T .. oy + t T + T (mod L) of both planes (its own rows and
the row above, whose sigma_y it rewrites; DESIGN.md section 7.1 "Write-back without races")."""
import numpy as np
import pytest

import __graft_entry__ as g


@pytest.fixture(scope="module")
def pkg():
    g.build()
    import paper_1110_6745_b200 as pkg
    return pkg


def _touch_table(L, T, oy, cy):
    """touch[p, r]: does colour pass p (MCS p // 4 with y offset oy, tile-row parity cy[p]) touch lattice row r?  The active
    tile rows t = cy (mod 2) cover the local rows t T .. t T + T of the frame shifted by oy."""
    r = np.arange(L)
    touch = np.zeros((len(cy), L), dtype=bool)
    for p in range(len(cy)):
        loc = (r - int(oy[p // 4])) % L % (2 * T)
        touch[p] = (loc <= T) if cy[p] == 0 else ((loc >= T) | (loc == 0))
    return touch


def _replay(L, T, oy, cy, plan):
    bnd, launches, copies = plan
    NT, mcs = L // T, len(oy)
    S = len(bnd) - 1
    assert bnd[0] == 0 and bnd[-1] == L and np.all(np.diff(bnd) > 0)
    assert np.all(bnd[:-1] % (2 * T) == 0)
    # issue order: stages ascending, passes ascending inside a stage
    key = launches[:, 0] * (4 * mcs) + launches[:, 1]
    assert np.all(np.diff(key) > 0)
    touch = _touch_table(L, T, oy, cy)
    before = np.cumsum(touch, axis=0) - touch          # before[p, r] = number of passes p' < p that touch row r
    seen = np.zeros(L, dtype=np.int64)                 # touches row r has received so far
    last_touch = np.full(L, -1, dtype=np.int64)        # issue index of the last launch that touches a row
    done = np.zeros((4 * mcs, NT), dtype=np.int64)
    for i, (s, p, a, b) in enumerate(launches):
        o, c = int(oy[p // 4]), int(cy[p])
        assert 0 <= a <= b < 2 * NT
        for t in range(a, b + 1):
            if (t - c) % 2:
                continue
            tr = t % NT
            done[p, tr] += 1
            rows = (o + tr * T + np.arange(T + 1)) % L
            assert np.all(touch[p, rows])
            assert rows.max() < bnd[s + 1], "launch touches rows that have not arrived"           # (2)
            # (3) every row of the footprint has been touched by exactly the earlier passes that touch it -- none of
            # them is still to come, and no later pass has been here first
            assert np.array_equal(seen[rows], before[p, rows]), "stage %d pass %d tile row %d out of order" % (s, p, tr)
            seen[rows] += 1
            last_touch[rows] = i
    # (1)
    for p in range(4 * mcs):
        c = int(cy[p])
        want = np.array([(t - c) % 2 == 0 for t in range(NT)], dtype=np.int64)
        assert np.array_equal(done[p], want), "pass %d: tile rows launched %s" % (p, done[p])
    assert np.array_equal(seen, touch.sum(axis=0))
    # (4)
    copied = np.zeros(L, dtype=np.int64)
    stage_of = launches[:, 0]
    for s, r0, r1 in copies:
        assert 0 <= r0 <= r1 < L
        copied[r0:r1 + 1] += 1
        lt = last_touch[r0:r1 + 1]
        assert np.all(lt >= 0)
        assert np.all(stage_of[lt] <= s), "rows %d..%d copied back after stage %d are touched later" % (r0, r1, s)
    assert np.all(copied == 1)
    return S


SHAPES = [
    # L, T, mcs, n_slabs
    (4096, 16, 1, 2), (4096, 16, 2, 4), (4096, 16, 3, 8), (8192, 32, 2, 6), (8192, 64, 1, 4), (16384, 64, 2, 5),
    (16384, 64, 3, 8), (32768, 64, 10, 3), (2048, 4, 5, 7), (2048, 8, 1, 16),
]


@pytest.mark.parametrize("L,T,mcs,n_slabs", SHAPES)
def test_overlap_plan_is_a_valid_schedule(pkg, L, T, mcs, n_slabs):
    rng = np.random.default_rng(L + 7 * T + 31 * mcs + n_slabs)
    n_ok = 0
    for trial in range(6):
        g4 = max(1, T // 4)
        oy = (4 * rng.integers(0, g4, size=mcs)).astype(np.uint32) if T >= 4 else rng.integers(0, T, size=mcs).astype(np.uint32)
        if trial == 0:
            oy[:] = 0
        if trial == 1:
            oy[:] = T - 4 if T >= 4 else T - 1
        cy = np.concatenate([(rng.permutation(4) >> 1) for _ in range(mcs)]).astype(np.uint32)
        # blocks in proportion 1 : 2 : 4 .. (wave_tiles = 0) or as whole waves of a GPU that holds wave_tiles tiles
        wave_tiles = (0, 148 * 288, 148 * 512, 1000, 37 * L // (2 * T))[(trial + mcs) % 5]
        plan = pkg.overlap_plan(L, T, oy, n_slabs, wave_tiles)
        assert plan is not None
        S = _replay(L, T, oy, cy, plan)
        assert 2 <= S <= n_slabs
        n_ok += 1
    assert n_ok == 6


def test_overlap_plan_refuses_shapes_that_cannot_overlap(pkg):
    # blocks would have to be taller than 8 mcs (T + 1) + 4 T rows: L = 1024, T = 64, 2 MCS -> 1296 rows per block
    assert pkg.overlap_plan(1024, 64, np.zeros(2, dtype=np.uint32), 2) is None
    assert pkg.overlap_plan(4096, 64, np.zeros(10, dtype=np.uint32), 4) is None
    assert pkg.overlap_plan(4096, 16, np.zeros(1, dtype=np.uint32), 1) is None            # one block: nothing to overlap
    with pytest.raises(pkg.KpzError):
        pkg.overlap_plan(4096, 16, np.array([16], dtype=np.uint32), 4)                    # offset >= tile
    with pytest.raises(pkg.KpzError):
        pkg.overlap_plan(4100, 16, np.zeros(1, dtype=np.uint32), 4)                       # L not a multiple of 2 T
    # the number of blocks is reduced until every block is tall enough
    plan = pkg.overlap_plan(8192, 64, np.zeros(2, dtype=np.uint32), 16)
    assert plan is not None and 2 <= len(plan[0]) - 1 < 16
    assert np.all(np.diff(plan[0]) >= 8 * 2 * 65 + 4 * 64)


def test_overlap_plan_blocks_ramp_up_from_both_ends(pkg):
    bnd, _, _ = pkg.overlap_plan(1 << 17, 64, np.zeros(10, dtype=np.uint32), 8)
    h = np.diff(bnd)
    mid = len(h) // 2
    assert np.all(np.diff(h[:mid + 1]) >= 0) and np.all(np.diff(h[mid:]) <= 0)
    assert h[0] < h[mid] / 2 and h[-1] < h[mid] / 2
    # whole waves: with 148 SMs x 288 tiles a wave is 41.625 tile rows of one colour at L = 2^17, T = 64; every block but
    # the middle one is the largest whole number of tile-row pairs below 2, 4, 8 .. waves
    wave = 148 * 288
    bnd, launches, _ = pkg.overlap_plan(1 << 17, 64, np.zeros(10, dtype=np.uint32), 8, wave)
    h = np.diff(bnd)
    mid = len(h) // 2
    per_row = (1 << 17) // 128                     # tiles of one colour in a tile row
    for i, rows in enumerate(h):
        if i == mid:
            continue
        k = 2 << min(i, len(h) - 1 - i)
        assert rows == (k * wave // per_row) * 128
    # a middle stage launches (block height / 128) colour rows per pass: just under a whole number of waves
    st = launches[launches[:, 0] == 1]
    assert len(st) == 40
    for _, _, a, b in st:
        colour_rows = (b - a + 1 + 1) // 2
        assert colour_rows * per_row <= 4 * wave
