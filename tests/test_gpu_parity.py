"""GPU parity tests proper: the CUDA path (through the C ABI) vs the CPU oracle, element by element, bit-exact.
Tolerance: 0 for the lattice state, the int64 sums and W^2 (derived in double from exact integers)."""
import os

import numpy as np
import pytest

from oracle import Oracle
import oracle as oracle_mod
import kpz_inputs as gen

pytestmark = pytest.mark.gpu

NTHREADS = max(1, min(32, os.cpu_count() or 1))


@pytest.fixture(scope="module")
def pkg():
    import __graft_entry__ as g
    g.build()
    import paper_1110_6745_b200 as pkg
    return pkg


def _kat():
    from pathlib import Path
    rows = []
    for line in (Path(__file__).parent / "golden" / "philox4x32_10_kat.txt").read_text().splitlines():
        if line.startswith("#") or not line.strip():
            continue
        v = [int(t, 16) for t in line.split()]
        rows.append(v)
    return np.array(rows, dtype=np.uint64)


def test_device_philox_known_answers(pkg):
    k = _kat()
    out = pkg.philox_selftest(k[:, 0:4].astype(np.uint32), k[:, 4:6].astype(np.uint32))
    assert np.array_equal(out, k[:, 6:10].astype(np.uint32))
    rng = np.random.default_rng(0)
    ctr = rng.integers(0, 2**32, size=(257, 4), dtype=np.uint64).astype(np.uint32)
    key = rng.integers(0, 2**32, size=(257, 2), dtype=np.uint64).astype(np.uint32)
    out = pkg.philox_selftest(ctr, key)
    for i in range(0, 257, 16):
        assert np.array_equal(out[i], oracle_mod.philox4x32_10(ctr[i], key[i]))


@pytest.mark.parametrize("L,T", [(32, 4), (64, 8), (256, 16), (128, 64), (4096, 32), (96, 16)])
def test_flat_init(pkg, L, T):
    k = pkg.KPZ(L, 1.0, 0.0, T, 1)
    k.init_flat()
    s1, s2, w2 = k.measure()
    assert s1[0] == L * L // 2 and s2[0] == L * L // 2 and w2[0] == 0.25
    if L <= 256:
        sx, sy = k.get_slopes()
        ex, ey = gen.heights_to_slopes(gen.flat_heights(L))
        assert np.array_equal(sx, ex) and np.array_equal(sy, ey)
    o = Oracle(L, 1.0, 0.0, T, 1)
    o.init_flat()
    assert k.state_hash() == o.state_hash()
    c = k.counters()
    assert c == {"attempts": 0, "deposits": 0, "removals": 0, "h00": 0, "mcs": 0}


@pytest.mark.parametrize("L,kind", [(64, "tri1"), (64, "tri8"), (256, "raised"), (128, "stair"), (96, "raised"),
                                    (1024, "raised"), (2048, "stair")])
def test_measure_pack_unpack_hash_parity(pkg, L, kind):
    if kind == "tri1":
        h = gen.triangle_heights(L, 1)
    elif kind == "tri8":
        h = gen.triangle_heights(L, 8)
    elif kind == "raised":
        h = gen.raised_flat_heights(L, 11, 0.4) - 5
    else:
        h = gen.staircase_heights(L, 3) + 1_000_000
    sx, sy = gen.heights_to_slopes(h)
    k = pkg.KPZ(L, 1.0, 0.0, 16, 1)
    k.init_flat()
    k.set_slopes(sx, sy, h00=int(h[0, 0]))
    gx, gy = k.get_slopes()
    assert np.array_equal(gx, sx) and np.array_equal(gy, sy)
    o = Oracle(L, 1.0, 0.0, 16, 1)
    o.set_slopes(sx, sy, h00=int(h[0, 0]))
    s1, s2, w2 = k.measure()
    os1, os2, ow2 = o.measure()
    assert int(s1[0]) == os1 == int(h.sum())
    assert int(s2[0]) == os2
    assert float(w2[0]) == ow2
    assert k.state_hash() == o.state_hash()
    if kind == "tri8":
        assert abs(w2[0] - (64 + 2) / 6) < 1e-12
    # window with wrap
    wx, wy = k.get_window(L - 5, L - 3, 17, 9)
    ys = (L - 3 + np.arange(9)) % L
    xs = (L - 5 + np.arange(17)) % L
    assert np.array_equal(wx, sx[np.ix_(ys, xs)]) and np.array_equal(wy, sy[np.ix_(ys, xs)])


def test_measure_overflow_and_set_slopes_validation(pkg):
    L = 64
    k = pkg.KPZ(L, 1.0, 0.0, 16, 1)
    k.init_flat()
    h = gen.flat_heights(L)
    sx, sy = gen.heights_to_slopes(h)
    k.set_slopes(sx, sy, h00=2**62)                       # sum h overflows int64
    with pytest.raises(pkg.KpzError) as e:
        k.measure()
    assert e.value.code == pkg.KPZ_EOVERFLOW
    bad = sx.copy(); bad[3, 3] = 0
    with pytest.raises(pkg.KpzError) as e:
        k.set_slopes(bad, sy)
    assert e.value.code == pkg.KPZ_EINVAL
    bad = sx.copy(); bad[3, 3] = -bad[3, 3]               # breaks curl-free / zero tilt
    with pytest.raises(pkg.KpzError) as e:
        k.set_slopes(bad, sy)
    assert e.value.code == pkg.KPZ_ESTATE
    k.set_slopes(sx, sy, h00=0)
    assert k.measure()[2][0] == 0.25


def _compare_full(k, o, replica=0):
    sx, sy = k.get_slopes(replica)
    osx, osy = o.slopes()
    assert np.array_equal(sx, osx), "sigma_x differs at %d sites" % int((sx != osx).sum())
    assert np.array_equal(sy, osy), "sigma_y differs at %d sites" % int((sy != osy).sum())


def _compare_scalars(k, os_, replica_slice=None):
    s1, s2, w2 = k.measure()
    for r, o in enumerate(os_):
        os1, os2, ow2 = o.measure()
        assert int(s1[r]) == os1 and int(s2[r]) == os2, (r, int(s1[r]), os1, int(s2[r]), os2)
        assert float(w2[r]) == ow2
        c, oc = k.counters(r), o.counters()
        assert c == oc, (c, oc)


@pytest.mark.parametrize("L,T,p,q,seed,n", [
    (32, 4, 1.0, 0.0, 1, 6),
    (64, 8, 0.75, 0.25, 2, 6),
    (64, 16, 1.0, 0.0, 3, 8),
    (96, 16, 0.5, 0.5, 4, 5),          # L not a power of two
    (128, 32, 1.0, 0.0, 5, 6),
    (128, 64, 0.75, 0.25, 6, 6),       # a single tile per colour
    (192, 32, 0.3, 0.9, 7, 4),
    (384, 64, 1.0, 0.0, 2**40 + 17, 5),
    (512, 64, 0.75, 0.25, 9, 5),       # blocked lane mapping needs HN % 8 == 0: HN = 4 -> linear
    (1024, 64, 1.0, 0.0, 10, 4),       # HN = 8 -> blocked lane mapping
    (1024, 32, 0.6, 0.1, 11, 3),
    (1024, 16, 1.0, 0.0, 12, 3),
    (64, 16, 0.5, 0.0, 13, 4),         # a probability of exactly 0: the 64-bit threshold path
    (128, 64, 0.0, 0.7, 14, 3),
    (128, 32, 1.0, 0.4, 15, 3),        # p = 1 with removals: inclusive 32-bit threshold 2^32 - 1
])
def test_update_parity_every_mcs(pkg, L, T, p, q, seed, n):
    """The tiled kernel (kpz_update_kernel, forced: small lattices would otherwise take the resident path)."""
    k = pkg.KPZ(L, p, q, T, seed)
    k.set_path("tiled")
    k.init_flat()
    o = Oracle(L, p, q, T, seed, threads=NTHREADS)
    o.init_flat()
    for t in range(n):
        k.run(1)
        o.run(1)
        _compare_full(k, o)
        _compare_scalars(k, [o])
        assert k.state_hash() == o.state_hash()


@pytest.mark.parametrize("path", ["resident", "auto"])
@pytest.mark.parametrize("L,T,p,q,seed,R,n", [
    (32, 4, 1.0, 0.0, 61, 1, 5),           # one word per row, 16 steps per tile: half a warp batch
    (32, 4, 0.75, 0.25, 62, 7, 4),
    (64, 8, 0.75, 0.25, 63, 3, 4),
    (64, 16, 0.5, 0.0, 64, 2, 4),          # a probability of exactly 0
    (128, 16, 1.0, 0.0, 4, 6, 5),          # config-4 shape
    (128, 32, 0.3, 0.9, 65, 1, 4),
    (128, 64, 0.0, 0.7, 66, 2, 3),         # a single tile per colour
    (256, 16, 1.0, 0.0, 1, 1, 6),          # config 1
    (256, 64, 0.75, 0.25, 3, 1, 3),
    (512, 16, 1.0, 0.0, 67, 1, 2),
    (512, 32, 0.6, 0.1, 68, 2, 2),
    (96, 16, 0.5, 0.5, 69, 3, 3),          # L not a power of two
    (384, 64, 1.0, 0.0, 70, 1, 2),
])
def test_resident_paths_parity(pkg, path, L, T, p, q, seed, R, n):
    """Lattice-resident kernel (kpz_resident_kernel: the packed lattices of a CTA's replicas in shared memory, all MCS
    of a call in one launch): state, sums, counters after every MCS, then n more MCS in ONE launch."""
    k = pkg.KPZ(L, p, q, T, seed, n_replicas=R)
    k.set_path(path)
    k.init_flat()
    os_ = [Oracle(L, p, q, T, seed, replica=r, threads=NTHREADS) for r in range(R)]
    for o in os_:
        o.init_flat()
    for t in range(n):
        l0 = k.launch_count()
        k.run(1)
        assert k.launch_count() - l0 == 1          # one launch per call, not four per MCS
        for o in os_:
            o.run(1)
        _compare_scalars(k, os_)
        for r in range(R):
            _compare_full(k, os_[r], replica=r)
    l0 = k.launch_count()
    k.run(n)
    assert k.launch_count() - l0 == 1
    for o in os_:
        o.run(n)
    _compare_scalars(k, os_)
    for r in range(R):
        assert k.state_hash(r) == os_[r].state_hash()
    # switching to the tiled kernel mid-run continues the same trajectory
    k.set_path("tiled")
    k.run(1)
    for o in os_:
        o.run(1)
    _compare_scalars(k, os_)
    _compare_full(k, os_[R - 1], replica=R - 1)


@pytest.mark.parametrize("L,T,p,q,K,R,seed", [
    (64, 8, 1.0, 0.0, 2, 3, 46),
    (128, 16, 1.0, 0.0, 4, 6, 47),             # config-4 shape with the knob that removes the S(k) peaks
    (128, 16, 0.75, 0.25, 32, 2, 48),          # one site call per tile and sub-sweep
    (256, 32, 0.6, 0.2, 8, 1, 49),
    (512, 64, 1.0, 0.0, 16, 1, 50),
])
def test_resident_path_sub_sweeps_parity(pkg, L, T, p, q, K, R, seed):
    """Schedule S6 through the lattice-resident kernel (every sub-sweep draws its own origin and colour order; all of
    them inside ONE launch): state, sums, counters against the oracle, and against the tiled kernel."""
    k = pkg.KPZ(L, p, q, T, seed, n_replicas=R)
    k.set_path("resident"); k.set_sub_sweeps(K)
    k.init_flat()
    os_ = [Oracle(L, p, q, T, seed, replica=r, threads=NTHREADS) for r in range(R)]
    for o in os_:
        o.set_sub_sweeps(K); o.init_flat()
    for n in (1, 3):
        l0 = k.launch_count()
        k.run(n)
        assert k.launch_count() - l0 == 1
        for o in os_:
            o.run(n)
        _compare_scalars(k, os_)
        for r in range(R):
            _compare_full(k, os_[r], replica=r)
    t = pkg.KPZ(L, p, q, T, seed, n_replicas=R)
    t.set_path("tiled"); t.set_sub_sweeps(K)
    t.init_flat(); t.run(4)
    assert [t.state_hash(r) for r in range(R)] == [k.state_hash(r) for r in range(R)]


def test_resident_path_is_refused_when_it_cannot_hold_the_lattice(pkg):
    for (L, T, path) in ((2048, 16, "resident"), (1024, 64, "resident")):
        k = pkg.KPZ(L, 1.0, 0.0, T, 1)
        k.set_path(path)
        k.init_flat()
        with pytest.raises(pkg.KpzError) as e:
            k.run(1)
        assert e.value.code == pkg.KPZ_EINVAL
        k.set_path("auto")
        k.run(1)
        o = Oracle(L, 1.0, 0.0, T, 1, threads=NTHREADS)
        o.init_flat(); o.run(1)
        assert k.state_hash() == o.state_hash()
    k = pkg.KPZ(128, 1.0, 0.0, 16, 1)
    k.set_path("resident")
    k.set_schedule("dead_border")
    k.init_flat()
    with pytest.raises(pkg.KpzError):
        k.run(1)                                   # the dead-border schedule runs on the tiled kernel only
    with pytest.raises(KeyError):
        k.set_path("nonsense")


def test_config1_full(pkg):
    """BASELINE config 1: L=256, T=16, p=1, q=0, seed 1, 64 MCS; state and sums after EVERY MCS."""
    L, T, seed = 256, 16, 1
    k = pkg.KPZ(L, 1.0, 0.0, T, seed)
    k.init_flat()
    o = Oracle(L, 1.0, 0.0, T, seed)
    o.init_flat()
    w2_series = {}
    for t in range(1, 65):
        k.run(1); o.run(1)
        _compare_full(k, o)
        _compare_scalars(k, [o])
        if t in (1, 2, 4, 8, 16, 32, 64):
            w2_series[t] = float(k.measure()[2][0])
    assert all(w2_series[a] < w2_series[b] for a, b in zip((1, 2, 4, 8, 16, 32), (2, 4, 8, 16, 32, 64)))
    assert w2_series[64] == o.measure()[2]    # every value above was compared with the oracle's, bit for bit


CONFIG2_TIMES = [1, 2, 3, 4, 5, 7, 9, 11, 14, 17, 22, 28, 36, 45, 57, 73, 92, 117, 149, 189, 240, 304, 386, 489,
                 621, 788, 1000]


def test_config2_prefix(pkg):
    """BASELINE config 2: L=4096, T=32, p=1, q=0, seed 7; the log-spaced sample times up to KPZ_CONFIG2_TMAX
    (default 1000 = the whole config, 27 samples, about 50 s of oracle time) with the full state compared at every sample."""
    tmax = int(os.environ.get("KPZ_CONFIG2_TMAX", "1000"))
    L, T, seed = 4096, 32, 7
    k = pkg.KPZ(L, 1.0, 0.0, T, seed)
    k.init_flat()
    o = Oracle(L, 1.0, 0.0, T, seed, threads=NTHREADS)
    o.init_flat()
    t = 0
    for ts in [x for x in CONFIG2_TIMES if x <= tmax]:
        k.run(ts - t); o.run(ts - t)
        t = ts
        _compare_scalars(k, [o])
        assert k.state_hash() == o.state_hash()
    _compare_full(k, o)


def test_replica_batch_parity(pkg):
    """Config-4 shape: independent replicas of L=128, T=16, p=1, q=0, seed 4 (replica id = Philox counter word)."""
    L, T, seed, R, n = 128, 16, 4, 48, 12
    k = pkg.KPZ(L, 1.0, 0.0, T, seed, n_replicas=R)
    k.init_flat()
    os_ = [Oracle(L, 1.0, 0.0, T, seed, replica=r) for r in range(R)]
    for o in os_:
        o.init_flat(); o.run(n)
    k.run(n)
    _compare_scalars(k, os_)
    for r in (0, 1, 17, R - 1):
        _compare_full(k, os_[r], replica=r)
        assert k.state_hash(r) == os_[r].state_hash()
    assert len({k.state_hash(r) for r in range(R)}) == R


def test_config4_replicas_2000_mcs_in_one_launch(pkg):
    """Config-4 shape over the run length S:8(d) asks for ("all replicas for the first 2 000 MCS"): 16 replicas of
    L = 128, T = 16, p = 1, q = 0, seed 4 advanced 2 000 MCS by ONE launch of the lattice-resident kernel (the MCS clock
    counts inside the kernel), then 7 more; sums, W^2, counters and hashes of every replica against the oracle."""
    L, T, seed, R = 128, 16, 4, 16
    k = pkg.KPZ(L, 1.0, 0.0, T, seed, n_replicas=R)
    k.init_flat()
    l0 = k.launch_count()
    k.run(2000)
    assert k.launch_count() - l0 == 1
    k.run(7)
    os_ = [Oracle(L, 1.0, 0.0, T, seed, replica=r) for r in range(R)]
    for o in os_:
        o.init_flat(); o.run(2007)
    _compare_scalars(k, os_)
    for r in range(R):
        assert k.state_hash(r) == os_[r].state_hash()
    _compare_full(k, os_[R - 1], replica=R - 1)


@pytest.mark.parametrize("L,T,R,n", [(128, 8, 64, 300), (256, 8, 12, 120), (128, 4, 16, 150), (512, 8, 3, 40)])
def test_replica_batch_small_tiles_resident_and_tiled(pkg, L, T, R, n):
    """Config 4 with the paper's own 8 x 8 cells (the configuration of profiles/r02_config4_fss_t8.md and of the 400 / 540
    Gupd/s figures) and with 4 x 4: n MCS in ONE launch of the lattice-resident kernel, then 3 more, every replica against
    the oracle; the tiled kernel on the same handle parameters must land on the same states."""
    seed = 4
    k = pkg.KPZ(L, 1.0, 0.0, T, seed, n_replicas=R)
    k.init_flat()
    l0 = k.launch_count()
    k.run(n)
    assert k.launch_count() - l0 == 1            # lattice-resident: one launch for the whole call
    k.run(3)
    os_ = [Oracle(L, 1.0, 0.0, T, seed, replica=r, threads=NTHREADS) for r in range(R)]
    for o in os_:
        o.init_flat(); o.run(n + 3)
    _compare_scalars(k, os_)
    for r in range(R):
        assert k.state_hash(r) == os_[r].state_hash()
        assert k.counters(r) == os_[r].counters()
    _compare_full(k, os_[R - 1], replica=R - 1)
    t = pkg.KPZ(L, 1.0, 0.0, T, seed, n_replicas=R)
    t.set_path("tiled")
    t.init_flat()
    t.run(n + 3)
    for r in range(R):
        assert t.state_hash(r) == os_[r].state_hash()
    k.close(); t.close()


def test_replica_batch_1024_general_pq(pkg):
    L, T, seed, R, n = 128, 16, 4, 1024, 3
    k = pkg.KPZ(L, 0.75, 0.25, T, seed, n_replicas=R)
    k.init_flat()
    k.run(n)
    s1, s2, w2 = k.measure()
    for r in (0, 5, 511, 1023):
        o = Oracle(L, 0.75, 0.25, T, seed, replica=r)
        o.init_flat(); o.run(n)
        assert (int(s1[r]), int(s2[r]), float(w2[r])) == o.measure()
        assert k.state_hash(r) == o.state_hash()
        assert k.counters(r) == o.counters()


def test_run_split_checkpoint_and_step_host(pkg):
    import torch
    L, T, seed = 512, 32, 77
    a = pkg.KPZ(L, 0.75, 0.25, T, seed)
    b = pkg.KPZ(L, 0.75, 0.25, T, seed)
    a.init_flat(); b.init_flat()
    a.run(7)
    b.run(3)
    host = torch.empty(b.lattice_bytes, dtype=torch.uint8).pin_memory()
    b.export_packed(host)
    h00 = np.array([b.counters()["h00"]], dtype=np.int64)
    c = pkg.KPZ(L, 0.75, 0.25, T, seed)
    s1, s2, w2 = c.step_host(host, h00, 3, 4)       # resume at MCS 3, run 4 more, through HOST buffers
    assert a.state_hash() == c.state_hash()
    assert (int(a.measure()[0][0]), int(a.measure()[1][0])) == (int(s1[0]), int(s2[0]))
    assert h00[0] == a.counters()["h00"]
    b.run(4)
    assert a.state_hash() == b.state_hash()
    host2 = torch.empty(b.lattice_bytes, dtype=torch.uint8).pin_memory()
    b.export_packed(host2)
    assert torch.equal(host, host2)                 # step_host wrote the advanced lattice back


@pytest.mark.parametrize("L,T,p,q,S,mcs,seed", [
    (2048, 16, 1.0, 0.0, 4, 3, 95),            # 4 slabs of 512 rows, 12 passes eat 204 rows per side
    (2048, 16, 0.75, 0.25, 2, 5, 96),
    (4096, 32, 1.0, 0.0, 4, 2, 97),
    (4096, 32, 0.6, 0.2, 8, 1, 98),            # slabs of 512 rows: just tall enough for 4 passes of T = 32
    (8192, 64, 1.0, 0.0, 4, 2, 99),
    (8192, 64, 0.75, 0.25, 2, 3, 100),
    (6144, 64, 1.0, 0.0, 3, 2, 101),           # L not a power of two, three slabs
])
def test_step_host_overlapped_matches_oracle_and_plain_step(pkg, L, T, p, q, S, mcs, seed):
    """kpz_step_host_overlapped: one lattice through pinned HOST memory with its copies overlapped slab by slab with the
    colour passes (a trapezoid of passes per slab, the wedges last).  Three steps in a row from the flat state: sums,
    W^2, h(0,0), counters and the host lattice itself against the oracle and against kpz_step_host."""
    import torch
    a = pkg.KPZ(L, p, q, T, seed)
    b = pkg.KPZ(L, p, q, T, seed)
    a.set_path("tiled"); b.set_path("tiled")
    a.init_flat()
    ha = torch.empty(a.lattice_bytes, dtype=torch.uint8).pin_memory()
    a.export_packed(ha)
    hb = ha.clone().pin_memory()
    h00a, h00b = np.zeros(1, dtype=np.int64), np.zeros(1, dtype=np.int64)
    o = Oracle(L, p, q, T, seed, threads=NTHREADS)
    o.init_flat()
    t = 0
    for step in range(3):
        l0 = a.launch_count()
        ra = a.step_host_overlapped(ha, h00a, t, mcs, S)
        assert a.launch_count() - l0 > 4 * mcs + 3          # the passes were really split over the slabs
        rb = b.step_host(hb, h00b, t, mcs)
        o.run(mcs)
        t += mcs
        want = o.measure()
        assert (int(ra[0][0]), int(ra[1][0]), float(ra[2][0])) == want == (int(rb[0][0]), int(rb[1][0]), float(rb[2][0]))
        assert int(h00a[0]) == int(h00b[0]) == o.counters()["h00"]
        assert torch.equal(ha, hb), "host lattices differ after step %d" % step
        assert a.state_hash() == o.state_hash()
        ca, oc = a.counters(), o.counters()
        assert (ca["deposits"], ca["removals"], ca["mcs"], ca["attempts"]) == (oc["deposits"], oc["removals"], oc["mcs"], oc["attempts"])


def test_step_host_overlapped_falls_back_when_it_cannot_overlap(pkg):
    """Too many passes for the slab height, several replicas, a resident-path lattice: the call IS kpz_step_host."""
    import torch
    for (L, T, R, S, mcs) in ((2048, 64, 1, 8, 4), (256, 16, 3, 2, 2), (128, 16, 1, 2, 1)):
        k = pkg.KPZ(L, 0.75, 0.25, T, 31, n_replicas=R)
        k.init_flat()
        host = torch.empty(k.lattice_bytes, dtype=torch.uint8).pin_memory()
        k.export_packed(host)
        h00 = np.zeros(R, dtype=np.int64)
        s1, s2, w2 = k.step_host_overlapped(host, h00, 0, mcs, S)
        for r in range(R):
            o = Oracle(L, 0.75, 0.25, T, 31, replica=r, threads=NTHREADS)
            o.init_flat(); o.run(mcs)
            assert (int(s1[r]), int(s2[r]), float(w2[r])) == o.measure() and int(h00[r]) == o.counters()["h00"]
            assert k.state_hash(r) == o.state_hash()


def _host_ram_gib():
    for line in open("/proc/meminfo"):
        if line.startswith("MemAvailable:"):
            return int(line.split()[1]) / 2**20
    return 0.0


class _WindowSet:
    """Light-cone window oracles (inner W x W exact for n_max MCS: margin M = 4 (T+1) n_max) advanced in
    lockstep with the GPU lattice and compared at the sampled times."""

    def __init__(self, L, T, p, q, seed, n_max, corners, W, schedule=None):
        self.L, self.W, self.M = L, W, 4 * (T + 1) * n_max
        full = W + 2 * self.M
        self.items = []
        for (wx0, wy0) in corners:
            o = Oracle(L, p, q, T, seed, window=((wx0 - self.M) % L, (wy0 - self.M) % L, full, full), threads=NTHREADS)
            if schedule:
                o.set_schedule(schedule)
            o.init_flat()
            self.items.append((wx0 % L, wy0 % L, o))

    def run(self, n):
        for _, _, o in self.items:
            o.run(n)

    def check(self, k):
        M, W = self.M, self.W
        for wx0, wy0, o in self.items:
            osx, osy = o.slopes()
            gx, gy = k.get_window(wx0, wy0, W, W)
            assert np.array_equal(gx, osx[M:M + W, M:M + W]), (wx0, wy0, o.counters()["mcs"])
            assert np.array_equal(gy, osy[M:M + W, M:M + W]), (wx0, wy0, o.counters()["mcs"])
            if wx0 + W > self.L and wy0 + W > self.L:       # the window holds site (0,0): its tracked height
                assert k.counters()["h00"] == o.counters()["h00"]


def _edge_windows(L, W):
    """>= 8 windows: the corner that holds (0,0), the four lattice edges (each wrapping), and interior ones."""
    h = W // 2
    return [(L - h, L - h), (L - h, L // 3), (L // 5, L - h), (L - h, 7 * (L // 8)), (3 * (L // 4) + 11, L - h),
            (50000 % L, 77777 % L), (L // 2 - 100, 3), (12345 % L, L // 2 + 4321)]


def test_config3_full_size_windows_and_invariants(pkg):
    """BASELINE config 3 at full size (L=2^17, T=64, p=1, q=0, seed 42), in the launch configuration bench.py
    times: eight 512^2 windows (the corner holding (0,0), all four lattice edges, interior) against the light-cone
    window oracle at t = 1, 2, 4, 8, plus the properties that hold at any size."""
    import torch
    torch.cuda.empty_cache()
    L, T, seed = 1 << 17, 64, 42
    k = pkg.KPZ(L, 1.0, 0.0, T, seed)
    k.init_flat()
    s1, s2, w2 = k.measure()
    assert (int(s1[0]), int(s2[0]), float(w2[0])) == (L * L // 2, L * L // 2, 0.25)       # P:88, exact at full size
    ws = _WindowSet(L, T, 1.0, 0.0, seed, 8, _edge_windows(L, 512), 512)
    t = 0
    for ts in (1, 2, 4, 8):
        k.run(ts - t); ws.run(ts - t)
        t = ts
        ws.check(k)
        s1, s2, w2 = k.measure()
        c = k.counters()
        assert c["removals"] == 0 and c["attempts"] == t * L * L and c["mcs"] == t
        assert int(s1[0]) - L * L // 2 == 2 * c["deposits"]            # +2 per accepted flip, exactly
    k.close()
    torch.cuda.empty_cache()


@pytest.mark.parametrize("L", [1 << 17, 1 << 19])
def test_flat_start_exact_sums_at_full_size(pkg, L):
    """kpz_init_flat + kpz_measure at the sizes of configs 3 and 5: sum h = sum h^2 = L^2/2, W^2 = 1/4 -- the
    exact pin of the measurement kernels (128 / 512 row chunks per column, word indices beyond 2^32 at 2^19) that
    needs no host array."""
    import torch
    torch.cuda.empty_cache()
    free_bytes, _ = torch.cuda.mem_get_info()
    need = pkg.workspace_bytes(L, 64, 1)
    if free_bytes < need[0] + need[1] + (2 << 30):
        pytest.skip("SKIPPED: GPU has %.0f GiB free, L=%d needs %.0f GiB" % (free_bytes / 2**30, L, sum(need) / 2**30))
    k = pkg.KPZ(L, 1.0, 0.0, 64, 1)
    k.init_flat()
    s1, s2, w2 = k.measure()
    assert int(s1[0]) == L * L // 2 and int(s2[0]) == L * L // 2 and float(w2[0]) == 0.25
    o = Oracle(L, 1.0, 0.0, 64, 1, window=(L - 64, L - 64, 128, 128))
    o.init_flat()
    gx, gy = k.get_window(L - 64, L - 64, 128, 128)
    osx, osy = o.slopes()
    assert np.array_equal(gx, osx) and np.array_equal(gy, osy)
    k.close()
    torch.cuda.empty_cache()


@pytest.mark.parametrize("p,q,seed", [(1.0, 0.0, 42), (0.75, 0.25, 3)])
def test_full_lattice_parity_2p16(pkg, p, q, seed):
    """full parity at L = 2^16, T = 64 with the parameters of config 3 (p=1, q=0, seed 42) and of
    config 5 (p=3/4, q=1/4, seed 3; option (i) of the config table): the FULL oracle (8 GiB of int8 slopes) for
    3 MCS; state hash, sum h, sum h^2, W^2 and all counters after every MCS, and the full lattice at the end on
    four quadrant-sized strips.  64 row chunks per column in the measurement kernels."""
    import torch
    L, T, n = 1 << 16, 64, 3
    if _host_ram_gib() < 14:
        print("SKIPPED test_full_lattice_parity_2p16: host RAM %.0f GiB < 14 GiB" % _host_ram_gib())
        pytest.skip("host RAM")
    torch.cuda.empty_cache()
    k = pkg.KPZ(L, p, q, T, seed)
    k.init_flat()
    o = Oracle(L, p, q, T, seed, threads=NTHREADS)
    o.init_flat()
    for t in range(n):
        k.run(1); o.run(1)
        _compare_scalars(k, [o])
        assert k.state_hash() == o.state_hash()
    osx, osy = o.slopes()
    for y0 in (0, L // 2 - 500, L - 1000):                   # full-width strips, element by element
        gx, gy = k.get_window(0, y0, L, 1000)
        assert np.array_equal(gx, osx[y0:y0 + 1000]) and np.array_equal(gy, osy[y0:y0 + 1000])
    k.close()
    torch.cuda.empty_cache()


def test_config3_full_oracle_2p17(pkg):
    """BASELINE config 3 itself against the FULL oracle (L = 2^17: 32 GiB of int8 slopes, about a minute per MCS on
    16 cores): state hash, sum h, sum h^2, W^2, counters after MCS 1 and 2.  Skipped, loudly, only when the host has
    less than 40 GiB of free RAM."""
    import torch
    L, T, seed, n = 1 << 17, 64, 42, 2
    if _host_ram_gib() < 40 or os.environ.get("KPZ_TEST_FULL_2P17", "1") != "1":
        print("SKIPPED test_config3_full_oracle_2p17: host RAM %.0f GiB < 40 GiB (or KPZ_TEST_FULL_2P17=0)" % _host_ram_gib())
        pytest.skip("host RAM")
    torch.cuda.empty_cache()
    k = pkg.KPZ(L, 1.0, 0.0, T, seed)
    k.init_flat()
    o = Oracle(L, 1.0, 0.0, T, seed, threads=NTHREADS)
    o.init_flat()
    for t in range(n):
        k.run(1); o.run(1)
        _compare_scalars(k, [o])
        assert k.state_hash() == o.state_hash()
    k.close()
    del o
    torch.cuda.empty_cache()


def test_blocked_lane_mapping_with_replicas(pkg):
    """The 8x4 lane blocking of tiles (HN % 8 == 0) together with n_replicas > 1 -- the launch shape of the config-4
    L = 2048 ensembles -- for T = 64 / general (p,q) and T = 16 / p = 1."""
    for (L, T, p, q, R, n) in ((1024, 64, 0.75, 0.25, 3, 2), (256, 16, 1.0, 0.0, 5, 3)):
        k = pkg.KPZ(L, p, q, T, 19, n_replicas=R)
        k.init_flat()
        os_ = [Oracle(L, p, q, T, 19, replica=r, threads=NTHREADS) for r in range(R)]
        for o in os_:
            o.init_flat()
            o.run(n)
        k.run(n)
        _compare_scalars(k, os_)
        for r in range(R):
            _compare_full(k, os_[r], replica=r)
            assert k.state_hash(r) == os_[r].state_hash()


def test_mcs_clock_near_2p32(pkg):
    """The MCS clock is Philox counter word c2 (S1): a trajectory started at clock 2^32 - 3 runs two
    more MCS bit-exactly and refuses the next one (KPZ_EINVAL), on both sides."""
    import torch
    L, T, seed, start = 256, 16, 5, 2**32 - 3
    k = pkg.KPZ(L, 0.75, 0.25, T, seed)
    k.init_flat()
    host = torch.empty(k.lattice_bytes, dtype=torch.uint8).pin_memory()
    k.export_packed(host)
    k.import_packed(host, np.zeros(1, dtype=np.int64), start)
    o = Oracle(L, 0.75, 0.25, T, seed)
    o.init_flat(); o.set_clock(start)
    k.run(2); o.run(2)
    _compare_full(k, o)
    _compare_scalars(k, [o])
    assert k.counters()["mcs"] == 2**32 - 1
    with pytest.raises(pkg.KpzError) as e:
        k.run(1)
    assert e.value.code == pkg.KPZ_EINVAL
    with pytest.raises(RuntimeError):
        o.run(1)
    assert k.state_hash() == o.state_hash()               # the refused call changed nothing
    with pytest.raises(pkg.KpzError):
        k.import_packed(host, np.zeros(1, dtype=np.int64), 2**32)


def test_config5_shape_general_pq(pkg):
    """BASELINE config 5 parameters (p=0.75, q=0.25, T=64, seed 3): full parity at L=8192, then the config itself
    (L=2^19, 64 GiB packed) with sampled windows vs the light-cone window oracle and the global invariants,
    whenever the GPU has the memory (KPZ_TEST_2P19=0 skips it)."""
    import torch
    L, T, seed = 8192, 64, 3
    k = pkg.KPZ(L, 0.75, 0.25, T, seed)
    k.init_flat()
    o = Oracle(L, 0.75, 0.25, T, seed, threads=NTHREADS)
    o.init_flat()
    for t in range(3):
        k.run(1); o.run(1)
        _compare_scalars(k, [o])
        assert k.state_hash() == o.state_hash()
    _compare_full(k, o)
    k.close()
    free_bytes, _ = torch.cuda.mem_get_info()
    if os.environ.get("KPZ_TEST_2P19", "1") == "1" and free_bytes > 72 * 2**30:
        torch.cuda.empty_cache()
        L = 1 << 19
        k = pkg.KPZ(L, 0.75, 0.25, T, seed)
        k.init_flat()
        ws = _WindowSet(L, T, 0.75, 0.25, seed, 4, _edge_windows(L, 512), 512)
        t = 0
        for ts in (1, 2, 4):
            k.run(ts - t); ws.run(ts - t)
            t = ts
            ws.check(k)
            s1, s2, w2 = k.measure()
            c = k.counters()
            assert int(s1[0]) - L * L // 2 == 2 * (c["deposits"] - c["removals"]) and c["attempts"] == t * L * L
        k.close()
        torch.cuda.empty_cache()


def _spectrum_bound(prof, S_ref_dir, L):
    """|S_gpu - S_oracle| allowed for one axis: both sides run an fp64 FFT whose
    output error is at most delta = 4 eps log2(L) sqrt(L) ||c||_2 per mode (c = mean-free integer profile), twice
    for the two sides; S = |X|^2 / L^2, so |dS| <= (2 |X| delta + delta^2) / L^2."""
    c = prof.astype(np.float64) - prof.mean()
    delta = 2 * 4 * np.finfo(np.float64).eps * np.log2(L) * np.sqrt(L) * np.linalg.norm(c)
    X = L * np.sqrt(S_ref_dir)
    return (2 * X * delta + delta * delta) / (L * L) + 1e-300


@pytest.mark.parametrize("L,kind", [(64, "tri8"), (256, "raised"), (128, "stair"), (1024, "stair"), (96, "raised"),
                                    (512, "evolved"), (2048, "evolved75")])
def test_profiles_and_power_spectrum_parity(pkg, L, kind):
    """kpz_profiles bit-exact against the oracle's height field; kpz_power_spectrum (1-D transforms of the two
    profiles on the device) against the oracle's definition (2-D transform of the height field, fp64)."""
    from oracle.spectrum import power_spectrum, profiles
    T = 16
    if kind in ("evolved", "evolved75"):
        p, q = (1.0, 0.0) if kind == "evolved" else (0.75, 0.25)
        k = pkg.KPZ(L, p, q, T, 21)
        k.init_flat(); k.run(12)
        o = Oracle(L, p, q, T, 21, threads=NTHREADS)
        o.init_flat(); o.run(12)
    else:
        h = {"tri8": lambda: gen.triangle_heights(L, 8), "raised": lambda: gen.raised_flat_heights(L, 11, 0.4) - 5,
             "stair": lambda: gen.staircase_heights(L, 3) + 1_000_000}[kind]()
        sx, sy = gen.heights_to_slopes(h)
        k = pkg.KPZ(L, 1.0, 0.0, T, 1)
        k.init_flat(); k.set_slopes(sx, sy, h00=int(h[0, 0]))
        o = Oracle(L, 1.0, 0.0, T, 1)
        o.set_slopes(sx, sy, h00=int(h[0, 0]))
    ho = o.heights().astype(np.int64)
    oc, orow = profiles(ho)
    gc, grow = k.profiles()
    assert np.array_equal(gc, oc) and np.array_equal(grow, orow)
    if L & (L - 1):
        with pytest.raises(pkg.KpzError) as e:
            k.power_spectrum()
        assert e.value.code == pkg.KPZ_EINVAL
        return
    S, Sx, Sy = k.power_spectrum()
    oS, oSx, oSy = power_spectrum(ho)
    bx, by = _spectrum_bound(oc, oSx, L), _spectrum_bound(orow, oSy, L)
    assert np.all(np.abs(Sx - oSx) <= bx), float(np.max(np.abs(Sx - oSx) / bx))
    assert np.all(np.abs(Sy - oSy) <= by), float(np.max(np.abs(Sy - oSy) / by))
    assert np.all(np.abs(S - oS) <= 0.5 * (bx + by))
    assert S[0] == 0.0
    if kind == "tri8":
        n = L // 16                       # first harmonic of the period-16 triangle wave
        assert abs(S[n] - (L / 16) ** 2 / np.sin(np.pi / 16) ** 4) < 1e-9 * S[n]
    # the lattice is untouched
    assert k.state_hash() == o.state_hash()


@pytest.mark.parametrize("L,T,p,q,seed,n", [
    (32, 4, 1.0, 0.0, 31, 5),
    (64, 8, 0.75, 0.25, 32, 5),
    (96, 16, 0.5, 0.5, 33, 4),
    (128, 32, 1.0, 0.0, 34, 5),
    (192, 32, 0.3, 0.9, 35, 4),
    (512, 64, 1.0, 0.0, 36, 4),
    (1024, 64, 0.75, 0.25, 37, 3),
    (1024, 64, 0.5, 0.0, 38, 2),
])
def test_dead_border_schedule_parity(pkg, L, T, p, q, seed, n):
    """Schedule S5: every tile in one launch, +x / +y edge sites dead; bit-exact state, sums, counters."""
    k = pkg.KPZ(L, p, q, T, seed)
    k.set_schedule("dead_border")
    k.init_flat()
    o = Oracle(L, p, q, T, seed, threads=NTHREADS)
    o.set_schedule("dead_border")
    o.init_flat()
    l0 = k.launch_count()
    for t in range(n):
        k.run(1)
        o.run(1)
        _compare_full(k, o)
        _compare_scalars(k, [o])
        assert k.state_hash() == o.state_hash()
    # switching back to the colour schedule mid-run keeps parity (the MCS clock and the streams are shared)
    k.set_schedule("colours"); o.set_schedule("colours")
    k.run(1); o.run(1)
    _compare_full(k, o)
    _compare_scalars(k, [o])


def test_dead_border_replicas_and_full_size_window(pkg):
    import torch
    L, T, R = 128, 16, 5
    k = pkg.KPZ(L, 0.75, 0.25, T, 4, n_replicas=R)
    k.set_schedule("dead_border")
    k.init_flat(); k.run(3)
    os_ = []
    for r in range(R):
        o = Oracle(L, 0.75, 0.25, T, 4, replica=r, threads=NTHREADS)
        o.set_schedule("dead_border")
        o.init_flat(); o.run(3)
        os_.append(o)
        _compare_full(k, o, replica=r)
    _compare_scalars(k, os_)
    k.close()
    torch.cuda.empty_cache()
    # L = 2^16 (1 GiB): one launch over 2^20 tiles; windows against the light-cone window oracle
    L, T, seed, n = 1 << 16, 64, 9, 2
    k = pkg.KPZ(L, 1.0, 0.0, T, seed)
    k.set_schedule("dead_border")
    k.init_flat(); k.run(n)
    s1, s2, w2 = k.measure()
    c = k.counters()
    assert int(s1[0]) - L * L // 2 == 2 * c["deposits"] and c["removals"] == 0
    for (wx0, wy0) in ((L - 200, L - 200), (12345, 54321)):
        W, M = 400, 4 * (T + 1) * n
        full = W + 2 * M
        o = Oracle(L, 1.0, 0.0, T, seed, window=((wx0 - M) % L, (wy0 - M) % L, full, full), threads=NTHREADS)
        o.set_schedule("dead_border")
        o.init_flat(); o.run(n)
        osx, osy = o.slopes()
        gx, gy = k.get_window(wx0, wy0, W, W)
        assert np.array_equal(gx, osx[M:M + W, M:M + W]) and np.array_equal(gy, osy[M:M + W, M:M + W])
    k.close()
    torch.cuda.empty_cache()


def test_steady_state_harness_against_oracle_ensemble(pkg):
    """The config-4 harness on a small ensemble: its per-sample W^2 values are the oracle's (bit-exact), and the
    reductions are analysis.py applied to them."""
    from paper_1110_6745_b200 import steady_state, analysis
    L, T, R, t_end, samples = 64, 16, 6, 40, 4
    out = steady_state.run(L, R, tile=T, seed=4, t_end=t_end, samples=samples, spectrum_replicas=2)
    os_ = [Oracle(L, 1.0, 0.0, T, 4, replica=r, threads=NTHREADS) for r in range(R)]
    for o in os_:
        o.init_flat(); o.run(t_end // 2)
    step = (t_end - t_end // 2) // samples
    w2 = []
    for _ in range(samples):
        for o in os_:
            o.run(step)
        w2.append([o.measure()[2] for o in os_])
    assert out["n_samples"] == R * samples
    assert out["cumulants"] == list(analysis.cumulants(np.array(w2)))
    from oracle.spectrum import power_spectrum
    S = np.mean([power_spectrum(o.heights().astype(np.int64))[0] for o in os_[:2]], axis=0)
    assert np.allclose(out["S_k"], S, rtol=1e-9, atol=1e-9 * S.max())


@pytest.mark.parametrize("L,T,p,q,K,sched,seed", [
    (64, 8, 1.0, 0.0, 2, "colours", 41),
    (96, 16, 0.75, 0.25, 8, "colours", 42),
    (128, 32, 1.0, 0.0, 4, "dead_border", 43),
    (512, 64, 1.0, 0.0, 16, "colours", 44),
    (512, 64, 0.6, 0.2, 512, "colours", 45),       # one site call per tile and sub-sweep
])
def test_sub_sweeps_parity(pkg, L, T, p, q, K, sched, seed):
    """Schedule S6 (bias-reduction knob): K sub-sweeps per MCS; bit-exact state, sums, counters."""
    k = pkg.KPZ(L, p, q, T, seed)
    k.set_schedule(sched); k.set_sub_sweeps(K)
    k.init_flat()
    o = Oracle(L, p, q, T, seed, threads=NTHREADS)
    o.set_schedule(sched); o.set_sub_sweeps(K)
    o.init_flat()
    for t in range(3):
        k.run(1); o.run(1)
        _compare_full(k, o)
        _compare_scalars(k, [o])
    with pytest.raises(pkg.KpzError):
        k.set_sub_sweeps(3)


def test_run_sampled_config1_times(pkg):
    """kpz_run_sampled on BASELINE config 1 (L=256, T=16, p=1, q=0, seed 1; t = 1,2,4,...,64): every sample equals the
    oracle's, and the call equals the run/measure sequence it stands for."""
    L, T, seed = 256, 16, 1
    times = [1, 2, 4, 8, 16, 32, 64]
    k = pkg.KPZ(L, 1.0, 0.0, T, seed)
    k.init_flat()
    s1, s2, w2 = k.run_sampled(times)
    o = Oracle(L, 1.0, 0.0, T, seed, threads=NTHREADS)
    o.init_flat()
    done = 0
    for i, t in enumerate(times):
        o.run(t - done); done = t
        os1, os2, ow2 = o.measure()
        assert (int(s1[i, 0]), int(s2[i, 0]), float(w2[i, 0])) == (os1, os2, ow2)
    assert k.counters()["mcs"] == 64 and k.state_hash() == o.state_hash()
    with pytest.raises(pkg.KpzError):
        k.run_sampled([10, 20])            # behind the MCS clock
    with pytest.raises(pkg.KpzError):
        k.run_sampled([70, 70])


def test_growth_exponent_loose_sanity(pkg):
    """Physics sanity, not parity (S:section 4): from the flat start W^2(t) - 1/4 ~ t^(2 beta) with beta_eff(t) =
    (1/2) log2[(W^2(t) - 1/4) / (W^2(t/2) - 1/4)] (eq. 11 with t/t' = 2 after subtracting 1/4) drifting
    up towards the paper's beta = 0.2415(15) once t > t_mic ~ 50.  One run at L = 2^14, T = 64, p = 1, q = 0;
    the schedule changes pre-factors, not exponents, so the band is loose."""
    import math
    L = 1 << 14
    k = pkg.KPZ(L, 1.0, 0.0, 64, 42)
    k.init_flat()
    times = [64, 128, 256, 512, 1024, 2048]
    _, _, w2 = k.run_sampled(times)
    w = w2[:, 0] - 0.25
    beta = [0.5 * math.log2(w[i] / w[i - 1]) for i in range(1, len(times))]
    assert all(0.225 < b < 0.255 for b in beta), beta
    assert all(w[i] > w[i - 1] for i in range(1, len(times)))
    k.close()


@pytest.mark.parametrize("L,T,p,q,K,sched,seed", [
    (64, 8, 1.0, 0.0, 1, "colours", 51),
    (96, 16, 0.75, 0.25, 4, "colours", 52),
    (128, 32, 1.0, 0.0, 2, "dead_border", 53),
    (512, 64, 1.0, 0.0, 1, "colours", 54),
    (512, 64, 0.6, 0.2, 16, "colours", 55),
])
def test_poissonised_counts_parity(pkg, L, T, p, q, K, sched, seed):
    """Schedule S7: Poissonised number of steps per tile and sub-sweep; bit-exact state, sums and counters
    (including the number of attempts really made)."""
    k = pkg.KPZ(L, p, q, T, seed)
    k.set_schedule(sched); k.set_sub_sweeps(K); k.set_poisson(True)
    k.init_flat()
    o = Oracle(L, p, q, T, seed, threads=NTHREADS)
    o.set_schedule(sched); o.set_sub_sweeps(K); o.set_poisson(True)
    o.init_flat()
    for t in range(3):
        k.run(1); o.run(1)
        _compare_full(k, o)
        _compare_scalars(k, [o])
    assert k.counters()["attempts"] != 3 * L * L or L <= 64
    # back to fixed counts: the attempts counter continues with exactly L*L per MCS
    k.set_poisson(False); o.set_poisson(False)
    a0 = k.counters()["attempts"]
    k.run(1); o.run(1)
    _compare_full(k, o)
    _compare_scalars(k, [o])
    assert k.counters()["attempts"] == a0 + L * L


@pytest.mark.parametrize("L,T,p,q,seed,t_max", [(256, 16, 1.0, 0.0, 1, 64), (256, 64, 0.75, 0.25, 3, 20)])
def test_growth_harness_against_oracle(pkg, L, T, p, q, seed, t_max):
    """growth_run (config 1 in full: the {1,2,5}*10^n and 2^i times up to 64; a T = 64 general-(p,q) case): every
    sample is the oracle's, bit for bit; beta_eff is eq. 11 applied to those samples; the invariant holds."""
    import math
    from paper_1110_6745_b200 import growth_run
    out = growth_run.run(L, T, p, q, seed, t_max)
    o = Oracle(L, p, q, T, seed, threads=NTHREADS)
    o.init_flat()
    t = 0
    for row in out["samples"]:
        o.run(row["t"] - t)
        t = row["t"]
        s1, s2, w2 = o.measure()
        assert (row["sum_h"], row["sum_h2"], row["W2"]) == (s1, s2, w2)
    assert out["invariant_sum_h"] and out["counters"]["attempts"] == t * L * L
    w = {r["t"]: r["W2"] - 0.25 for r in out["samples"]}
    for b in out["beta_eff"]:
        assert b["beta_eff"] == 0.5 * math.log2(w[b["t"]] / w[b["t"] // 2])


@pytest.mark.parametrize("L,T,p,q,R,lanes", [(256, 16, 1.0, 0.0, 1, 3), (512, 64, 0.75, 0.25, 1, 2),
                                              (128, 16, 0.75, 0.25, 3, 3), (2048, 32, 0.75, 0.25, 1, 1),
                                              (4096, 64, 1.0, 0.0, 1, 2)])
def test_pipeline_host_matches_oracle(pkg, L, T, p, q, R, lanes):
    """kpz_pipeline_host: 1-3 lanes at different MCS clocks, 3 rounds of 2 MCS through pinned HOST lattices with the
    copies overlapped; every batch's sums, every lane's final lattice and h(0,0) against the oracle, bit-exact."""
    import torch
    seed, mcs, rounds = 11, 2, 3
    k = pkg.KPZ(L, p, q, T, seed, n_replicas=R)
    k.init_flat()
    hosts, h00, start = [], np.zeros((lanes, R), dtype=np.int64), []
    for lane in range(lanes):                     # lane j starts from the state after 2j+1 MCS
        k.run(1 if lane == 0 else 2)
        t = torch.empty(k.lattice_bytes, dtype=torch.uint8).pin_memory()
        k.export_packed(t)
        hosts.append(t)
        start.append(2 * lane + 1)
        h00[lane] = [k.counters(r)["h00"] for r in range(R)]
    s1, s2, w2 = k.pipeline_host(hosts, h00, start, mcs, rounds)
    chk = pkg.KPZ(L, p, q, T, seed, n_replicas=R)
    for r in range(R):
        o = Oracle(L, p, q, T, seed, replica=r, threads=NTHREADS)
        o.init_flat()
        done = 0
        want = {}
        for t_end in sorted({start[lane] + mcs * (rd + 1) for lane in range(lanes) for rd in range(rounds)}):
            o.run(t_end - done)
            done = t_end
            want[t_end] = (o.measure(), o.state_hash(), o.counters()["h00"])
        for lane in range(lanes):
            for rd in range(rounds):
                t_end = start[lane] + mcs * (rd + 1)
                assert (int(s1[rd, lane, r]), int(s2[rd, lane, r]), float(w2[rd, lane, r])) == want[t_end][0]
            t_end = start[lane] + mcs * rounds
            chk.import_packed(hosts[lane], h00[lane], t_end)
            assert chk.state_hash(r) == want[t_end][1]
            assert int(h00[lane, r]) == want[t_end][2]
    # the handle works again after a re-import, and continues the trajectory of lane 0
    k.import_packed(hosts[0], h00[0], start[0] + mcs * rounds)
    k.run(1)
    o = Oracle(L, p, q, T, seed, replica=0)
    o.init_flat(); o.run(start[0] + mcs * rounds + 1)
    assert k.state_hash(0) == o.state_hash()


def test_pipeline_host_rejects_bad_arguments(pkg):
    import ctypes
    import torch
    k = pkg.KPZ(64, 1.0, 0.0, 16, 1)
    k.init_flat()
    t = torch.empty(k.lattice_bytes, dtype=torch.uint8).pin_memory()
    k.export_packed(t)
    h00 = np.zeros((1, 1), dtype=np.int64)
    with pytest.raises(pkg.KpzError):
        k.pipeline_host([t], h00, [0], 1, 0)                         # no rounds
    with pytest.raises(pkg.KpzError):
        k.pipeline_host([t[:-1]], h00, [0], 1, 1)                    # host lattice too short
    with pytest.raises(pkg.KpzError):
        k.pipeline_host([t], h00, [0xFFFFFFFF], 1, 1)                # MCS clock overflow
    k.init_flat()
    k.run(1)                                                         # the handle is intact after a rejected call
    o = Oracle(64, 1.0, 0.0, 16, 1)
    o.init_flat(); o.run(1)
    assert k.state_hash() == o.state_hash()


@pytest.mark.parametrize("L,T,p,q,seed,N,n", [
    (256, 16, 1.0, 0.0, 81, 1, 4),           # one slab: the ghost rows wrap onto the slab's own first rows
    (256, 16, 0.75, 0.25, 82, 2, 5),
    (512, 16, 1.0, 0.0, 83, 4, 4),
    (512, 32, 0.6, 0.1, 84, 2, 4),
    (1024, 64, 1.0, 0.0, 85, 2, 3),
    (2048, 64, 0.75, 0.25, 86, 4, 3),        # blocked lane mapping inside a slab (HN = 16, 4 tile rows per colour)
    (1024, 64, 1.0, 0.0, 87, 8, 3),          # one tile row of each parity per slab
])
def test_slabs_match_whole_lattice_and_oracle(pkg, L, T, p, q, seed, N, n):
    """One lattice as N slabs of rows (kpz_create_slab / kpz_slab_pass, paper_1110_6745_b200/slabs.py; all slabs on
    this GPU, run one after the other): packed state, sums, W^2 and counters after every MCS equal the oracle's and
    the single-handle lattice's, bit for bit."""
    import torch
    from paper_1110_6745_b200.slabs import SlabLattice
    sl = SlabLattice(L, p, q, T, seed, N)
    sl.init_flat()
    k = pkg.KPZ(L, p, q, T, seed)
    k.set_path("tiled")
    k.init_flat()
    o = Oracle(L, p, q, T, seed, threads=NTHREADS)
    o.init_flat()
    host = torch.empty(k.lattice_bytes, dtype=torch.uint8).pin_memory()
    assert sl.measure() == (L * L // 2, L * L // 2, 0.25)
    for t in range(n):
        sl.run(1); k.run(1); o.run(1)
        s1, s2, w2 = k.measure()
        assert sl.measure() == (int(s1[0]), int(s2[0]), float(w2[0])) == o.measure()
        k.export_packed(host)
        assert torch.equal(sl.packed_rows().reshape(-1), host), t
        assert sl.counters() == k.counters() == o.counters()
    sl.run(2); o.run(2)                                    # several MCS per call
    assert sl.measure() == o.measure()
    sl.close()


def test_slab_handles_validate_and_refuse_whole_lattice_calls(pkg):
    import ctypes
    from paper_1110_6745_b200.slabs import SlabHandle
    lib = pkg.load_library()
    a, b = ctypes.c_size_t(), ctypes.c_size_t()
    assert lib.kpz_slab_workspace_bytes(256, 16, 3, ctypes.addressof(a), ctypes.addressof(b)) == pkg.KPZ_EINVAL   # NT % (2 N)
    assert lib.kpz_slab_workspace_bytes(256, 16, 16, ctypes.addressof(a), ctypes.addressof(b)) == pkg.KPZ_EINVAL
    assert lib.kpz_slab_workspace_bytes(256, 16, 2, ctypes.addressof(a), ctypes.addressof(b)) == pkg.KPZ_OK
    assert a.value == 2 * (128 + 16 + 2) * 32
    h = SlabHandle(256, 1.0, 0.0, 16, 1, 2, 1)
    h.init_flat()
    out = ctypes.c_uint64()
    assert lib.kpz_state_hash(h._h, 0, ctypes.addressof(out)) == pkg.KPZ_ESTATE
    assert lib.kpz_run(h._h, 1) == pkg.KPZ_ESTATE
    assert lib.kpz_slab_pass(h._h, 4) == pkg.KPZ_EINVAL
    k = pkg.KPZ(256, 1.0, 0.0, 16, 1)
    assert lib.kpz_slab_pass(k._h, 0) == pkg.KPZ_ESTATE
    o = Oracle(256, 1.0, 0.0, 16, 1)
    for m in (0, 1, 17, 2**32 - 2):
        assert tuple(h.global_draw(m)) == tuple(o.global_draw(m))      # host evaluation of S2 = the oracle's
    h.close()


def test_dist_slab_single_rank_matches_oracle(pkg):
    """DistSlab (the one-process-per-GPU driver) with the real CUDA slab handle in a group of one rank: the ghost rows
    wrap onto the slab's own head; state sums and counters against the oracle.  (World sizes 2 and 4 of the same driver
    run on CPU with a stand-in handle: tests/test_slabs_gloo.py.)"""
    import socket
    import torch.distributed as dist
    from paper_1110_6745_b200.slabs import DistSlab, SlabHandle
    L, T, p, q, seed = 512, 32, 0.75, 0.25, 91
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK="0", WORLD_SIZE="1")
    dist.init_process_group("gloo", rank=0, world_size=1)
    try:
        d = DistSlab(SlabHandle(L, p, q, T, seed, 1, 0))
        d.init_flat()
        o = Oracle(L, p, q, T, seed, threads=NTHREADS)
        o.init_flat()
        for _ in range(3):
            d.run(2); o.run(2)
            assert d.measure() == o.measure()
            assert d.h.counters() == o.counters()
        d.h.close()
    finally:
        dist.destroy_process_group()


def test_pipe_peaks_and_layout_measurements_are_physical(pkg):
    """kpz_measure_peaks / kpz_measure_layouts (the figures the roofline and DESIGN.md section 7.1 quote) against what the
    hardware fixes: no integer pipe issues more than 16 lanes per scheduler and clock, a bank-conflict-free warp load
    moves at most 128 bytes per SM and clock, the dependent chain of a tile cannot beat the shared-memory latency, and the
    occupancies of the two tile layouts are the ones their shared-memory footprints give on a 228 KB SM."""
    pk = pkg.measure_peaks()
    sms, clk = pk["n_sms"], pk["sm_clock_hz"]
    assert sms >= 1 and 0.5e9 < clk < 4e9
    lane_cap = sms * 4 * 16 * clk
    for name in ("lop3_lane_ops", "shf_lane_ops", "imad_lane_ops"):
        assert 0.5 * lane_cap < pk[name] < 1.05 * lane_cap, (name, pk[name], lane_cap)
    assert pk["imad_wide_lane_ops"] < 0.6 * lane_cap
    assert 0.5 * sms * 128 * clk < pk["lds_bytes"] < 1.05 * sms * 128 * clk
    assert pk["attempt_mix"] * 5 * 4 * 32 / 32 <= 1.05 * pk["lds_bytes"]        # five 4-byte loads per attempt and lane
    assert 20 < pk["chain_cycles_w1"] < pk["chain_cycles_w2"] < 2 * pk["chain_cycles_w1"]
    ly = pkg.measure_layouts()
    assert ly["rows3_warps_per_sm"] == 9 and ly["pitch66_warps_per_sm"] == 12
    # an attempt of the present layout needs >= 9 ALU-pipe instructions + 2.4 of its share of a Philox call
    assert 0 < ly["rows3_attempts_per_s"] < lane_cap / 11.0
    assert 0 < ly["pitch66_attempts_per_s"] < lane_cap / 11.0
