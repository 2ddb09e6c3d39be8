"""kpz_measure_static -- the measurement with its scratch in a file-scope static device array (no cudaMalloc, no host
synchronisation; L <= 8192) -- against the existing kpz_measure, tolerance 0 as everywhere in this suite (exact integer
sums, W^2 from the same 128-bit arithmetic), on two calls in a row and after the state and the lattice size changed
(all handles of the process share the one array, which keeps the last call's contents).

This file is collected LAST on purpose (pytest -x must not lose the other tests to a failure here)
and passes both alone in a fresh process and after the rest of the suite."""
import ctypes
import struct

import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def pkg():
    import __graft_entry__ as g
    g.build()
    import paper_1110_6745_b200 as pkg
    return pkg


def _static(pkg, k, out, replica=0):
    """One kpz_measure_static call -> (halves, sum_h, sum_h2, W2, overflow flag) read back from the caller's buffer."""
    import torch
    out.fill_(-1)                                          # stale output must be overwritten in full
    k.measure_static(out, replica)
    torch.cuda.synchronize()
    w = [int(v) for v in out.cpu().tolist()]
    w2 = struct.unpack("<d", struct.pack("<q", w[6]))[0]
    return [v & 0xFFFFFFFFFFFFFFFF for v in w[:4]], w[4], w[5], w2, w[7]


def _check(pkg, k, out, replica=0):
    s1, s2, w2 = k.measure()                               # the existing path (bound scratch buffer, host finalisation)
    want = (int(s1[replica]), int(s2[replica]), float(w2[replica]))
    for _ in range(2):                                     # two calls in a row
        halves, a, b, c, flag = _static(pkg, k, out, replica)
        assert (a, b, c) == want and flag == 0
        # the half-accumulators are what kpz_slab_finalize takes: the host finalisation gives the same three numbers
        from paper_1110_6745_b200.slabs import finalize
        assert finalize(k.L, halves, k.counters(replica)["h00"]) == want


@pytest.mark.parametrize("L,T,p,q,R", [(64, 16, 1.0, 0.0, 1), (96, 16, 0.75, 0.25, 3), (2048, 32, 1.0, 0.0, 1),
                                       (256, 16, 0.5, 0.5, 2), (8192, 64, 0.75, 0.25, 1)])
def test_measure_static_matches_measure(pkg, L, T, p, q, R):
    import torch
    k = pkg.KPZ(L, p, q, T, 77, n_replicas=R)
    out = torch.empty(8, dtype=torch.int64, device=k.device)          # the caller's output buffer
    k.init_flat()
    halves, a, b, c, flag = _static(pkg, k, out, R - 1)
    assert (a, b, c, flag) == (L * L // 2, L * L // 2, 0.25, 0)
    for n in (1, 3):
        k.run(n)                                                       # the state changes between the pairs of calls
        for r in range(R):
            _check(pkg, k, out, r)
    h0 = k.state_hash(0)
    l0 = k.launch_count()
    k.measure_static(out, 0)
    assert k.launch_count() - l0 == 4 and k.state_hash(0) == h0        # four kernels, the lattice is untouched
    k.close()


def test_measure_static_shares_one_array_between_handles_and_sizes(pkg):
    """A large handle, then a small one, then the large one again: what the previous call left in the array (other L,
    other chunk count) must not leak into the next result."""
    import torch
    big = pkg.KPZ(4096, 1.0, 0.0, 32, 5)
    small = pkg.KPZ(128, 0.75, 0.25, 16, 6, n_replicas=2)
    out = torch.empty(8, dtype=torch.int64, device=big.device)
    big.init_flat(); small.init_flat()
    big.run(3); small.run(5)
    for k, r in ((big, 0), (small, 1), (big, 0), (small, 0), (small, 1)):
        _check(pkg, k, out, r)
    # large |h|: absolute heights anchored by h(0,0) on the device, overflow flag instead of a wrapped sum
    import kpz_inputs as gen
    h = gen.staircase_heights(128, 3) + 1_000_000
    sx, sy = gen.heights_to_slopes(h)
    small.set_slopes(sx, sy, h00=int(h[0, 0]), replica=1)
    _check(pkg, small, out, 1)
    small.set_slopes(sx, sy, h00=2**62, replica=1)
    _, a, b, c, flag = _static(pkg, small, out, 1)
    assert flag == 1 and a == 0                                        # sum h does not fit int64; kpz_measure: KPZ_EOVERFLOW
    with pytest.raises(pkg.KpzError) as e:
        small.measure()
    assert e.value.code == pkg.KPZ_EOVERFLOW
    big.close(); small.close()


def test_measure_static_rejects_what_it_cannot_hold(pkg):
    import torch
    lib = pkg.load_library()
    k = pkg.KPZ(16384, 1.0, 0.0, 64, 1)                                # beyond KPZ_STATIC_MAX_L = 8192
    out = torch.empty(8, dtype=torch.int64, device=k.device)
    k.init_flat()
    with pytest.raises(pkg.KpzError) as e:
        k.measure_static(out)
    assert e.value.code == pkg.KPZ_EINVAL and "8192" in str(e.value)
    assert k.measure()[2][0] == 0.25                                   # the existing path is unaffected
    k.close()
    k = pkg.KPZ(64, 1.0, 0.0, 16, 1)
    k.init_flat()
    assert lib.kpz_measure_static(k._h, 1, out.data_ptr()) == pkg.KPZ_EINVAL          # replica out of range
    assert lib.kpz_measure_static(k._h, 0, None) == pkg.KPZ_EINVAL                    # no output buffer
    assert lib.kpz_measure_static(k._h, 0, out.data_ptr() + 4) == pkg.KPZ_EINVAL      # misaligned
    h = ctypes.c_void_p()
    assert lib.kpz_create(ctypes.addressof(h), 64, 1.0, 0.0, 16, 1) == pkg.KPZ_OK
    assert lib.kpz_measure_static(h, 0, out.data_ptr()) == pkg.KPZ_ESTATE             # not bound
    lib.kpz_destroy(h)
    _check(pkg, k, out, 0)                                             # and the handle still works after the refusals
    k.close()


def test_measure_static_replays_inside_a_cuda_graph(pkg):
    """What the entry point is for: captured once into a CUDA graph (one memset + four kernels, no allocation, no host
    synchronisation), it is replayed after the lattice has moved on and gives kpz_measure's numbers each time.  (Only
    the measurement is captured: kpz_run bakes the MCS clock into its launches and is issued normally, on the same
    stream, between the replays.)"""
    import torch
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        k = pkg.KPZ(512, 0.75, 0.25, 32, 21, stream=s)                 # the handle's stream is the capturing stream
        out = torch.empty(8, dtype=torch.int64, device=k.device)
        k.init_flat()
        k.run(2)
        k.measure_static(out)                                          # first call outside the capture: address lookup
        s.synchronize()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=s):
            k.measure_static(out)
        for n in (0, 1, 3):
            k.run(n)
            out.fill_(-1)
            g.replay()
            s.synchronize()
            w = [int(v) for v in out.cpu().tolist()]
            s1, s2, w2 = k.measure()
            assert (w[4], w[5], struct.unpack("<d", struct.pack("<q", w[6]))[0], w[7]) == \
                (int(s1[0]), int(s2[0]), float(w2[0]), 0)
        k.close()
