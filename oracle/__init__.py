"""CPU oracle for the octahedron-KPZ hot path -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl reference`` legs
may import this package.  It never imports ``paper_1110_6745_b200`` and shares no code with it.

``oracle/kpz_oracle.cpp`` is the oracle proper (plain C++, unpacked int8 slopes, own Philox);
``oracle/kpz_twin.py`` is an independent pure-Python restatement used on tiny lattices to cross-check it.
This module only compiles the C++ file (g++) and marshals arguments through ctypes.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "kpz_oracle.cpp"
_LIB = _HERE / "libkpz_oracle.so"
_lib = None


def build(force: bool = False) -> Path:
    """Compile oracle/kpz_oracle.cpp -> oracle/libkpz_oracle.so (g++ -O2 -fopenmp)."""
    if force or not _LIB.exists() or _LIB.stat().st_mtime < _SRC.stat().st_mtime:
        tmp = _LIB.with_suffix(".so.tmp%d" % os.getpid())
        cmd = ["g++", "-O2", "-std=c++17", "-fopenmp", "-fPIC", "-shared", "-o", str(tmp), str(_SRC)]
        subprocess.check_call(cmd)
        os.replace(tmp, _LIB)
    return _LIB


def lib() -> ctypes.CDLL:
    global _lib
    if _lib is None:
        build()
        L = ctypes.CDLL(str(_LIB))
        vp, u32, u64, i64, dbl, ci = (ctypes.c_void_p, ctypes.c_uint32, ctypes.c_uint64, ctypes.c_int64,
                                      ctypes.c_double, ctypes.c_int)
        L.kpzo_create.restype = vp
        L.kpzo_create.argtypes = [u32, dbl, dbl, u32, u64, u32, u32, u32, u32, u32, ci]
        L.kpzo_destroy.argtypes = [vp]
        L.kpzo_set_threads.argtypes = [vp, ci]
        L.kpzo_get_threads.argtypes = [vp]
        L.kpzo_get_threads.restype = ci
        L.kpzo_init_flat.argtypes = [vp]
        L.kpzo_set_schedule.argtypes = [vp, ci]
        L.kpzo_set_schedule.restype = ci
        L.kpzo_set_sub_sweeps.argtypes = [vp, u32]
        L.kpzo_set_sub_sweeps.restype = ci
        L.kpzo_set_poisson.argtypes = [vp, ci]
        L.kpzo_set_poisson.restype = ci
        L.kpzo_poisson_table.argtypes = [vp, vp, vp]
        L.kpzo_poisson_table.restype = u32
        L.kpzo_run.argtypes = [vp, u64]
        L.kpzo_run.restype = ci
        L.kpzo_run_checked.argtypes = [vp, u64]
        L.kpzo_run_checked.restype = ci
        L.kpzo_run_rs.argtypes = [vp, u64]
        L.kpzo_run_rs.restype = ci
        L.kpzo_check.argtypes = [vp]
        L.kpzo_check.restype = ci
        L.kpzo_measure.argtypes = [vp, vp, vp, vp]
        L.kpzo_measure.restype = ci
        L.kpzo_heights.argtypes = [vp, vp]
        L.kpzo_heights.restype = ci
        L.kpzo_get_slopes.argtypes = [vp, vp, vp]
        L.kpzo_set_slopes.argtypes = [vp, vp, vp, i64]
        L.kpzo_set_slopes.restype = ci
        L.kpzo_get_shadow.argtypes = [vp, vp]
        L.kpzo_counters.argtypes = [vp, vp, vp, vp, vp, vp]
        L.kpzo_global_draw.argtypes = [vp, u32, vp, vp, vp]
        L.kpzo_set_clock.argtypes = [vp, u64]
        L.kpzo_set_clock.restype = ci
        L.kpzo_state_hash.argtypes = [vp]
        L.kpzo_state_hash.restype = u64
        L.kpzo_philox4x32_10.argtypes = [vp, vp, vp]
        L.kpzo_threshold.argtypes = [dbl]
        L.kpzo_threshold.restype = u64
        L.kpzo_openmp.restype = ci
        _lib = L
    return _lib


def philox4x32_10(ctr, key):
    c = np.asarray(ctr, dtype=np.uint32).copy()
    k = np.asarray(key, dtype=np.uint32).copy()
    out = np.zeros(4, dtype=np.uint32)
    lib().kpzo_philox4x32_10(c.ctypes.data, k.ctypes.data, out.ctypes.data)
    return out


def threshold(prob: float) -> int:
    return int(lib().kpzo_threshold(float(prob)))


def _to_int128(lohi) -> int:
    v = int(lohi[0]) | (int(lohi[1]) << 64)
    return v - (1 << 128) if v >= (1 << 127) else v


class Oracle:
    """One lattice (or one window of a lattice) advanced by the C++ oracle."""

    def __init__(self, L, p, q, T, seed, replica=0, window=None, shadow=False, threads=1):
        wx0, wy0, ww, wh = window if window is not None else (0, 0, 0, 0)
        self._h = lib().kpzo_create(L, float(p), float(q), T, seed, replica, wx0, wy0, ww, wh, int(shadow))
        if not self._h:
            raise ValueError("invalid oracle parameters")
        self.L, self.T, self.p, self.q, self.seed, self.replica = L, T, p, q, seed, replica
        self.shape = (wh, ww) if window is not None else (L, L)
        self.window = window
        self.shadow = shadow
        lib().kpzo_set_threads(self._h, threads)

    def __del__(self):
        if getattr(self, "_h", None):
            lib().kpzo_destroy(self._h)
            self._h = None

    @property
    def threads(self):
        return lib().kpzo_get_threads(self._h)

    def set_schedule(self, name):
        """'colours' (S4, default) or 'dead_border' (S5, the paper's own device-level scheme)."""
        if lib().kpzo_set_schedule(self._h, {"colours": 0, "dead_border": 1}[name]) != 0:
            raise ValueError(name)

    def set_sub_sweeps(self, K):
        """K sub-sweeps per MCS, each with its own origin shift and colour order (S6)."""
        if lib().kpzo_set_sub_sweeps(self._h, int(K)) != 0:
            raise ValueError("K must divide T*T")

    def set_poisson(self, on=True):
        """Poissonised number of steps per tile and sub-sweep (S7)."""
        if lib().kpzo_set_poisson(self._h, int(bool(on))) != 0:
            raise ValueError("tile*tile/K too large for the Poissonised schedule")

    def poisson_table(self):
        """(kmin, thresholds) of the S7 count table; thresholds[i] = floor(2^32 P(n <= kmin + i))."""
        kmin = ctypes.c_uint32()
        n = lib().kpzo_poisson_table(self._h, ctypes.addressof(kmin), None)
        thr = np.zeros(n, dtype=np.uint64)
        lib().kpzo_poisson_table(self._h, ctypes.addressof(kmin), thr.ctypes.data)
        return kmin.value, thr

    def init_flat(self):
        lib().kpzo_init_flat(self._h)

    def run(self, n_mcs):
        if lib().kpzo_run(self._h, n_mcs) != 0:
            raise RuntimeError("oracle run failed")

    def run_checked(self, n_mcs) -> int:
        return lib().kpzo_run_checked(self._h, n_mcs)

    def run_rs(self, n_mcs):
        if lib().kpzo_run_rs(self._h, n_mcs) != 0:
            raise RuntimeError("oracle rs run failed")

    def check(self) -> int:
        return lib().kpzo_check(self._h)

    def measure(self):
        """-> (sum_h, sum_h2) as Python ints, W2 as float."""
        a = np.zeros(2, dtype=np.uint64)
        b = np.zeros(2, dtype=np.uint64)
        w = ctypes.c_double()
        if lib().kpzo_measure(self._h, a.ctypes.data, b.ctypes.data, ctypes.addressof(w)) != 0:
            raise RuntimeError("measure needs the full lattice")
        return _to_int128(a), _to_int128(b), w.value

    def heights(self):
        out = np.zeros(self.shape, dtype=np.int32)
        if lib().kpzo_heights(self._h, out.ctypes.data) != 0:
            raise RuntimeError("heights needs the full lattice")
        return out

    def slopes(self):
        sx = np.zeros(self.shape, dtype=np.int8)
        sy = np.zeros(self.shape, dtype=np.int8)
        lib().kpzo_get_slopes(self._h, sx.ctypes.data, sy.ctypes.data)
        return sx, sy

    def set_slopes(self, sx, sy, h00=0):
        sx = np.ascontiguousarray(sx, dtype=np.int8)
        sy = np.ascontiguousarray(sy, dtype=np.int8)
        assert sx.shape == self.shape and sy.shape == self.shape
        if lib().kpzo_set_slopes(self._h, sx.ctypes.data, sy.ctypes.data, int(h00)) != 0:
            raise ValueError("slopes must be +-1")

    def shadow_heights(self):
        out = np.zeros(self.shape, dtype=np.int32)
        lib().kpzo_get_shadow(self._h, out.ctypes.data)
        return out

    def counters(self):
        a, d, r, m = (ctypes.c_uint64() for _ in range(4))
        h = ctypes.c_int64()
        lib().kpzo_counters(self._h, ctypes.addressof(a), ctypes.addressof(d), ctypes.addressof(r),
                            ctypes.addressof(h), ctypes.addressof(m))
        return {"attempts": a.value, "deposits": d.value, "removals": r.value, "h00": h.value, "mcs": m.value}

    def set_clock(self, mcs):
        """MCS clock := mcs (attempts := mcs * L*L); the lattice is untouched."""
        if lib().kpzo_set_clock(self._h, int(mcs)) != 0:
            raise ValueError("the MCS clock is a 32-bit counter word")

    def global_draw(self, m):
        ox, oy = ctypes.c_uint32(), ctypes.c_uint32()
        perm = np.zeros(4, dtype=np.uint32)
        lib().kpzo_global_draw(self._h, m, ctypes.addressof(ox), ctypes.addressof(oy), perm.ctypes.data)
        return ox.value, oy.value, [int(v) for v in perm]

    def state_hash(self) -> int:
        return int(lib().kpzo_state_hash(self._h))


def openmp_max_threads() -> int:
    return int(lib().kpzo_openmp())
