"""ctypes binding of include/kpz.h -- argument marshalling only; every step of the path runs in the CUDA kernels.

Names mirror the C ABI: KPZ.init_flat -> kpz_init_flat, KPZ.run -> kpz_run, KPZ.measure -> kpz_measure, ...
"""
from __future__ import annotations

import ctypes
from pathlib import Path

import numpy as np

KPZ_OK, KPZ_EINVAL, KPZ_ENOMEM, KPZ_ECUDA, KPZ_EOVERFLOW, KPZ_ESTATE = 0, -1, -2, -3, -4, -5
_CODES = {KPZ_EINVAL: "KPZ_EINVAL", KPZ_ENOMEM: "KPZ_ENOMEM", KPZ_ECUDA: "KPZ_ECUDA",
          KPZ_EOVERFLOW: "KPZ_EOVERFLOW", KPZ_ESTATE: "KPZ_ESTATE"}

_LIB_PATH = Path(__file__).resolve().parent / "libkpz_b200.so"
_lib = None

# every symbol include/kpz.h declares
exported_symbols = [
    "kpz_workspace_bytes", "kpz_create", "kpz_create_batch", "kpz_bind", "kpz_init_flat", "kpz_run", "kpz_measure",
    "kpz_destroy", "kpz_synchronize", "kpz_last_error", "kpz_get_slopes", "kpz_get_window", "kpz_set_slopes",
    "kpz_state_hash", "kpz_counters", "kpz_export_packed", "kpz_import_packed", "kpz_step_host", "kpz_pipeline_host",
    "kpz_launch_count", "kpz_philox_selftest", "kpz_profiles", "kpz_power_spectrum", "kpz_set_schedule", "kpz_set_sub_sweeps", "kpz_run_sampled", "kpz_set_poisson",
    "kpz_set_path", "kpz_measure_peaks", "kpz_measure_layouts", "kpz_overlap_plan",
    "kpz_slab_workspace_bytes", "kpz_create_slab", "kpz_slab_info", "kpz_global_draw", "kpz_slab_pass", "kpz_slab_end_mcs",
    "kpz_slab_measure_local", "kpz_slab_measure_finish", "kpz_slab_finalize", "kpz_measure_static",
    "kpz_step_host_overlapped",
]


class KpzError(RuntimeError):
    def __init__(self, code, msg=""):
        super().__init__("%s (%d)%s" % (_CODES.get(code, "KPZ_E?"), code, ": " + msg if msg else ""))
        self.code = code


def load_library() -> ctypes.CDLL:
    """Loads the compiled extension; fails loudly if it is missing (no fallback of any kind)."""
    global _lib
    if _lib is not None:
        return _lib
    if not _LIB_PATH.exists():
        raise ImportError("%s is missing: run `python -c 'import __graft_entry__ as g; g.build()'` "
                          "(nvcc, sm_100a) first -- there is no CPU fallback" % _LIB_PATH)
    L = ctypes.CDLL(str(_LIB_PATH))
    vp, u32, u64, i64, dbl, i32, sz = (ctypes.c_void_p, ctypes.c_uint32, ctypes.c_uint64, ctypes.c_int64,
                                       ctypes.c_double, ctypes.c_int32, ctypes.c_size_t)
    sig = {
        "kpz_workspace_bytes": [u32, u32, u32, vp, vp],
        "kpz_create": [vp, u32, dbl, dbl, u32, u64],
        "kpz_create_batch": [vp, u32, dbl, dbl, u32, u64, u32],
        "kpz_bind": [vp, vp, sz, vp, sz, vp],
        "kpz_init_flat": [vp],
        "kpz_run": [vp, u64],
        "kpz_measure": [vp, vp, vp, vp],
        "kpz_destroy": [vp],
        "kpz_synchronize": [vp],
        "kpz_get_slopes": [vp, u32, vp, vp],
        "kpz_get_window": [vp, u32, u32, u32, u32, u32, vp, vp],
        "kpz_set_slopes": [vp, u32, vp, vp, i64],
        "kpz_state_hash": [vp, u32, vp],
        "kpz_counters": [vp, u32, vp, vp, vp, vp, vp],
        "kpz_run_sampled": [vp, vp, u32, vp, vp, vp],
        "kpz_set_schedule": [vp, i32],
        "kpz_set_poisson": [vp, i32],
        "kpz_set_path": [vp, i32],
        "kpz_set_sub_sweeps": [vp, u32],
        "kpz_profiles": [vp, u32, vp, vp],
        "kpz_power_spectrum": [vp, u32, vp, vp, vp],
        "kpz_export_packed": [vp, vp, sz],
        "kpz_import_packed": [vp, vp, sz, vp, u64],
        "kpz_step_host": [vp, vp, sz, vp, u64, u64, vp, vp, vp],
        "kpz_pipeline_host": [vp, vp, sz, u32, vp, sz, vp, vp, u64, u32, vp, vp, vp],
        "kpz_launch_count": [vp, vp],
        "kpz_philox_selftest": [vp, vp, vp, u32],
        "kpz_measure_peaks": [vp, u32],
        "kpz_measure_layouts": [vp, u32],
        "kpz_overlap_plan": [u32, u32, u64, u32, u32, vp, vp, vp, vp, vp, vp, vp],
        "kpz_slab_workspace_bytes": [u32, u32, u32, vp, vp],
        "kpz_create_slab": [vp, u32, dbl, dbl, u32, u64, u32, u32],
        "kpz_slab_info": [vp, vp, vp, vp, vp, vp],
        "kpz_global_draw": [vp, u64, vp, vp, vp],
        "kpz_slab_pass": [vp, u32],
        "kpz_slab_end_mcs": [vp],
        "kpz_slab_measure_local": [vp],
        "kpz_slab_measure_finish": [vp, vp, vp, vp],
        "kpz_slab_finalize": [u32, vp, i64, vp, vp, vp],
        "kpz_measure_static": [vp, u32, vp],
        "kpz_step_host_overlapped": [vp, vp, sz, vp, u64, u64, u32, vp, vp, vp],
    }
    for name, args in sig.items():
        fn = getattr(L, name)
        fn.argtypes = args
        fn.restype = i32
    L.kpz_last_error.argtypes = [vp]
    L.kpz_last_error.restype = ctypes.c_char_p
    _lib = L
    return L


def workspace_bytes(L, tile, n_replicas=1):
    a, b = ctypes.c_size_t(), ctypes.c_size_t()
    rc = load_library().kpz_workspace_bytes(L, tile, n_replicas, ctypes.addressof(a), ctypes.addressof(b))
    if rc != KPZ_OK:
        raise KpzError(rc)
    return a.value, b.value


PEAK_NAMES = ("sm_clock_hz", "lop3_lane_ops", "shf_lane_ops", "imad_lane_ops", "imad_wide_lane_ops", "lds_bytes",
              "smem_xor_lane_ops", "attempt_mix", "n_sms", "chain_cycles_w1", "chain_cycles_w2")


def measure_peaks():
    """kpz_measure_peaks on the current device -> dict of its figures (see include/kpz.h)."""
    out = np.zeros(len(PEAK_NAMES), dtype=np.float64)
    rc = load_library().kpz_measure_peaks(out.ctypes.data, len(out))
    if rc != KPZ_OK:
        raise KpzError(rc, "kpz_measure_peaks")
    return dict(zip(PEAK_NAMES, out.tolist()))


def overlap_plan(L, tile, oy, n_slabs, wave_tiles=0):
    """kpz_overlap_plan (host only): the schedule of kpz_step_host_overlapped for a step of len(oy) MCS with y offsets oy.
    -> (boundaries, launches[n][4] = stage, pass, first, last tile row, copies[n][3] = stage, first, last row), or None
    when the shape does not allow the overlap."""
    oy = np.ascontiguousarray(oy, dtype=np.uint32)
    mcs = len(oy)
    bnd = np.zeros(n_slabs + 1, dtype=np.int64)
    lau = np.zeros((max(1, n_slabs) * 4 * mcs, 4), dtype=np.int64)
    cop = np.zeros((n_slabs + 1, 3), dtype=np.int64)
    ns, nl, nc = ctypes.c_uint32(), ctypes.c_uint32(), ctypes.c_uint32()
    rc = load_library().kpz_overlap_plan(L, tile, mcs, n_slabs, wave_tiles, oy.ctypes.data, bnd.ctypes.data, ctypes.addressof(ns),
                                         lau.ctypes.data, ctypes.addressof(nl), cop.ctypes.data, ctypes.addressof(nc))
    if rc != KPZ_OK:
        raise KpzError(rc, "kpz_overlap_plan")
    if ns.value == 0:
        return None
    return bnd[:ns.value + 1].copy(), lau[:nl.value].copy(), cop[:nc.value].copy()


LAYOUT_NAMES = ("rows3_attempts_per_s", "rows3_warps_per_sm", "pitch66_attempts_per_s", "pitch66_warps_per_sm")


def measure_layouts():
    """kpz_measure_layouts on the current device -> dict (the attempt loop alone in two tile layouts, include/kpz.h)."""
    out = np.zeros(len(LAYOUT_NAMES), dtype=np.float64)
    rc = load_library().kpz_measure_layouts(out.ctypes.data, len(out))
    if rc != KPZ_OK:
        raise KpzError(rc, "kpz_measure_layouts")
    return dict(zip(LAYOUT_NAMES, out.tolist()))


def philox_selftest(ctr, key):
    ctr = np.ascontiguousarray(ctr, dtype=np.uint32).reshape(-1, 4)
    key = np.ascontiguousarray(key, dtype=np.uint32).reshape(-1, 2)
    out = np.zeros_like(ctr)
    rc = load_library().kpz_philox_selftest(ctr.ctypes.data, key.ctypes.data, out.ctypes.data, len(ctr))
    if rc != KPZ_OK:
        raise KpzError(rc)
    return out


class KPZ:
    """One handle = n_replicas lattices of size L x L (kpz_create_batch + kpz_bind with torch-allocated buffers)."""

    def __init__(self, L, p, q, tile, seed, n_replicas=1, device="cuda:0", stream=None):
        import torch
        self._torch = torch
        self._lib = load_library()
        self._h = ctypes.c_void_p()
        self.L, self.p, self.q, self.tile, self.seed, self.n_replicas = L, p, q, tile, seed, n_replicas
        rc = self._lib.kpz_create_batch(ctypes.addressof(self._h), L, float(p), float(q), tile, seed, n_replicas)
        if rc != KPZ_OK:
            self._h = ctypes.c_void_p()
            raise KpzError(rc, "kpz_create_batch")
        self.lattice_bytes, self.scratch_bytes = workspace_bytes(L, tile, n_replicas)
        self.device = torch.device(device)
        with torch.cuda.device(self.device):
            self.lattice = torch.empty(self.lattice_bytes, dtype=torch.uint8, device=self.device)
            self.scratch = torch.empty(self.scratch_bytes, dtype=torch.uint8, device=self.device)
            self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
            self._check(self._lib.kpz_bind(self._h, self.lattice.data_ptr(), self.lattice_bytes,
                                           self.scratch.data_ptr(), self.scratch_bytes, self.stream.cuda_stream))

    def _check(self, rc, allow=()):
        if rc != KPZ_OK and rc not in allow:
            msg = self._lib.kpz_last_error(self._h)
            raise KpzError(rc, msg.decode() if msg else "")
        return rc

    def close(self):
        if getattr(self, "_h", None) and self._h.value:
            self._lib.kpz_destroy(self._h)
            self._h = ctypes.c_void_p()

    __del__ = close

    def init_flat(self):
        self._check(self._lib.kpz_init_flat(self._h))

    def run(self, mcs):
        self._check(self._lib.kpz_run(self._h, int(mcs)))

    def synchronize(self):
        self._check(self._lib.kpz_synchronize(self._h))

    def measure(self):
        """-> (sum_h, sum_h2, W2) numpy arrays of length n_replicas (int64, int64, float64)."""
        R = self.n_replicas
        s1 = np.zeros(R, dtype=np.int64)
        s2 = np.zeros(R, dtype=np.int64)
        w2 = np.zeros(R, dtype=np.float64)
        self._check(self._lib.kpz_measure(self._h, s1.ctypes.data, s2.ctypes.data, w2.ctypes.data))
        return s1, s2, w2

    def measure_static(self, out, replica=0):
        """kpz_measure_static: the measurement with its scratch in the library's static device array (no allocation, no
        host synchronisation; L <= 8192).  `out` is the CALLER's device tensor of 8 int64 words (see include/kpz.h);
        it is written asynchronously on the bound stream."""
        assert out.is_cuda and out.numel() * out.element_size() >= 64 and out.is_contiguous()
        self._check(self._lib.kpz_measure_static(self._h, replica, out.data_ptr()))

    def get_slopes(self, replica=0):
        sx = np.zeros((self.L, self.L), dtype=np.int8)
        sy = np.zeros((self.L, self.L), dtype=np.int8)
        self._check(self._lib.kpz_get_slopes(self._h, replica, sx.ctypes.data, sy.ctypes.data))
        return sx, sy

    def get_window(self, x0, y0, w, h, replica=0):
        sx = np.zeros((h, w), dtype=np.int8)
        sy = np.zeros((h, w), dtype=np.int8)
        self._check(self._lib.kpz_get_window(self._h, replica, x0, y0, w, h, sx.ctypes.data, sy.ctypes.data))
        return sx, sy

    def set_slopes(self, sx, sy, h00=0, replica=0):
        sx = np.ascontiguousarray(sx, dtype=np.int8)
        sy = np.ascontiguousarray(sy, dtype=np.int8)
        if sx.shape != (self.L, self.L) or sy.shape != (self.L, self.L):
            raise ValueError("slope arrays must be L x L")
        self._check(self._lib.kpz_set_slopes(self._h, replica, sx.ctypes.data, sy.ctypes.data, int(h00)))

    def run_sampled(self, times):
        """kpz_run_sampled: (sum_h, sum_h2, W2) arrays of shape [len(times), n_replicas] at the absolute MCS clocks."""
        t = np.ascontiguousarray(times, dtype=np.uint64)
        n = len(t)
        s1 = np.zeros((n, self.n_replicas), dtype=np.int64)
        s2 = np.zeros((n, self.n_replicas), dtype=np.int64)
        w2 = np.zeros((n, self.n_replicas), dtype=np.float64)
        self._check(self._lib.kpz_run_sampled(self._h, t.ctypes.data, n, s1.ctypes.data, s2.ctypes.data, w2.ctypes.data),
                    allow=(KPZ_EOVERFLOW,))
        return s1, s2, w2

    def set_schedule(self, name):
        """kpz_set_schedule: 'colours' (default) or 'dead_border' (the paper's own scheme)."""
        self._check(self._lib.kpz_set_schedule(self._h, {"colours": 0, "dead_border": 1}[name]))

    def set_path(self, name):
        """kpz_set_path: 'auto' (default), 'tiled' or 'resident' (lattice kept in shared memory, one launch per run
        call); the results are bit-identical."""
        self._check(self._lib.kpz_set_path(self._h, {"auto": 0, "tiled": 1, "resident": 2}[name]))

    def set_poisson(self, on=True):
        """kpz_set_poisson: Poissonised number of steps per tile and sub-sweep (S7)."""
        self._check(self._lib.kpz_set_poisson(self._h, int(bool(on))))

    def set_sub_sweeps(self, K):
        """kpz_set_sub_sweeps: K sub-sweeps per MCS, each with its own origin shift and colour order."""
        self._check(self._lib.kpz_set_sub_sweeps(self._h, int(K)))

    def profiles(self, replica=0):
        """kpz_profiles: exact (col_sums[x] = sum_y h, row_sums[y] = sum_x h), int64 arrays of length L."""
        c = np.empty(self.L, dtype=np.int64)
        r = np.empty(self.L, dtype=np.int64)
        self._check(self._lib.kpz_profiles(self._h, replica, c.ctypes.data, r.ctypes.data))
        return c, r

    def power_spectrum(self, replica=0):
        """kpz_power_spectrum: (S, Sx, Sy), float64 arrays of length L/2 + 1 (k = 2 pi n / L)."""
        n = self.L // 2 + 1
        S, Sx, Sy = (np.empty(n, dtype=np.float64) for _ in range(3))
        self._check(self._lib.kpz_power_spectrum(self._h, replica, S.ctypes.data, Sx.ctypes.data, Sy.ctypes.data))
        return S, Sx, Sy

    def state_hash(self, replica=0):
        out = ctypes.c_uint64()
        self._check(self._lib.kpz_state_hash(self._h, replica, ctypes.addressof(out)))
        return out.value

    def counters(self, replica=0):
        a, d, r, m = (ctypes.c_uint64() for _ in range(4))
        h = ctypes.c_int64()
        self._check(self._lib.kpz_counters(self._h, replica, ctypes.addressof(a), ctypes.addressof(d),
                                           ctypes.addressof(r), ctypes.addressof(h), ctypes.addressof(m)))
        return {"attempts": a.value, "deposits": d.value, "removals": r.value, "h00": h.value, "mcs": m.value}

    def export_packed(self, host_tensor):
        self._check(self._lib.kpz_export_packed(self._h, host_tensor.data_ptr(), host_tensor.numel()))

    def import_packed(self, host_tensor, h00=None, mcs=0):
        h = None if h00 is None else np.ascontiguousarray(h00, dtype=np.int64)
        self._check(self._lib.kpz_import_packed(self._h, host_tensor.data_ptr(), host_tensor.numel(),
                                                None if h is None else h.ctypes.data, int(mcs)))

    def step_host(self, host_tensor, h00, mcs_start, mcs):
        """kpz_step_host: H2D lattice + run + measure + D2H lattice.  h00 (int64 array) is updated in place."""
        R = self.n_replicas
        s1 = np.zeros(R, dtype=np.int64)
        s2 = np.zeros(R, dtype=np.int64)
        w2 = np.zeros(R, dtype=np.float64)
        self._check(self._lib.kpz_step_host(self._h, host_tensor.data_ptr(), host_tensor.numel(), h00.ctypes.data,
                                            int(mcs_start), int(mcs), s1.ctypes.data, s2.ctypes.data, w2.ctypes.data))
        return s1, s2, w2

    def step_host_overlapped(self, host_tensor, h00, mcs_start, mcs, n_slabs=4):
        """kpz_step_host_overlapped: kpz_step_host with the copies of ONE lattice overlapped with its kernels slab by slab."""
        R = self.n_replicas
        s1 = np.zeros(R, dtype=np.int64)
        s2 = np.zeros(R, dtype=np.int64)
        w2 = np.zeros(R, dtype=np.float64)
        self._check(self._lib.kpz_step_host_overlapped(self._h, host_tensor.data_ptr(), host_tensor.numel(), h00.ctypes.data,
                                                       int(mcs_start), int(mcs), int(n_slabs), s1.ctypes.data,
                                                       s2.ctypes.data, w2.ctypes.data))
        return s1, s2, w2

    def pipeline_host(self, host_tensors, h00, mcs_start, mcs, n_rounds=1):
        """kpz_pipeline_host: every pinned host lattice of `host_tensors` advanced by mcs MCS and measured, n_rounds
        times, copies overlapped with the kernels.  h00 (int64 [n_lanes, R]) is updated in place.  Returns sum_h,
        sum_h2, W2 of shape [n_rounds, n_lanes, R]."""
        torch = self._torch
        R, n = self.n_replicas, len(host_tensors)
        if getattr(self, "lattice2", None) is None:
            with torch.cuda.device(self.device):
                self.lattice2 = torch.empty(self.lattice_bytes, dtype=torch.uint8, device=self.device)
        ptrs = (ctypes.c_void_p * n)(*[t.data_ptr() for t in host_tensors])
        nbytes = min(t.numel() for t in host_tensors)
        start = np.ascontiguousarray(mcs_start, dtype=np.uint64)
        assert start.size == n and h00.dtype == np.int64 and h00.size == n * R and h00.flags.c_contiguous
        s1 = np.zeros((n_rounds, n, R), dtype=np.int64)
        s2 = np.zeros((n_rounds, n, R), dtype=np.int64)
        w2 = np.zeros((n_rounds, n, R), dtype=np.float64)
        self._check(self._lib.kpz_pipeline_host(self._h, self.lattice2.data_ptr(), self.lattice_bytes, n,
                                                ctypes.addressof(ptrs), nbytes, h00.ctypes.data, start.ctypes.data,
                                                int(mcs), int(n_rounds), s1.ctypes.data, s2.ctypes.data, w2.ctypes.data))
        return s1, s2, w2

    def launch_count(self):
        out = ctypes.c_uint64()
        self._check(self._lib.kpz_launch_count(self._h, ctypes.addressof(out)))
        return out.value
