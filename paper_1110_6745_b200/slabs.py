"""One lattice split into slabs of rows over several handles / GPUs (include/kpz.h "slabs").

Plumbing only: every step of the path runs in the kernels behind the C ABI (kpz_slab_pass, kpz_slab_measure_*); this
module moves the ghost rows between the slabs' device buffers and gathers the per-column totals of the measurement.

  * SlabHandle     one slab: kpz_create_slab + torch-allocated buffers, views of its first rows and of its ghost rows
  * SlabLattice    all slabs driven by ONE process (each slab on any visible device; copies are torch device copies)
  * DistSlab       one slab per rank of a torch.distributed group (NCCL on GPUs): the same exchange as point-to-point
                   sends between neighbouring ranks, the measurement through all_gather / broadcast / all_reduce

The exchange rule (the only host logic; `exchange_plan`): the tiles of a slab's last tile row reach oy + 1 rows into
the next slab and are active in the colour passes whose colour has bit 1 set (ty odd).  For such a pass every slab
first fetches rows [0, oy + 1) of the next slab into its ghost rows and afterwards writes them back.
"""
from __future__ import annotations

import ctypes

import numpy as np

from .binding import KPZ_OK, KPZ_EOVERFLOW, KpzError, load_library


def exchange_plan(oy: int, perm, slot: int):
    """(exchange?, n_rows) for colour pass `slot` of an MCS with y origin oy and colour order perm."""
    return bool(perm[slot] & 2), oy + 1


class SlabHandle:
    """Slab `slab` of `n_slabs` of an L x L lattice on `device` (kpz_create_slab + kpz_bind)."""

    def __init__(self, L, p, q, tile, seed, n_slabs, slab, device="cuda:0"):
        import torch
        self._torch = torch
        self._lib = load_library()
        self._h = ctypes.c_void_p()
        self.L, self.tile, self.n_slabs, self.slab = L, tile, n_slabs, slab
        rc = self._lib.kpz_create_slab(ctypes.addressof(self._h), L, float(p), float(q), tile, seed, n_slabs, slab)
        if rc != KPZ_OK:
            self._h = ctypes.c_void_p()
            raise KpzError(rc, "kpz_create_slab")
        a, b = ctypes.c_size_t(), ctypes.c_size_t()
        self._check(self._lib.kpz_slab_workspace_bytes(L, tile, n_slabs, ctypes.addressof(a), ctypes.addressof(b)))
        self.lattice_bytes, self.scratch_bytes = a.value, b.value
        self.device = torch.device(device)
        with torch.cuda.device(self.device):
            self.lattice = torch.empty(self.lattice_bytes, dtype=torch.uint8, device=self.device)
            self.scratch = torch.empty(self.scratch_bytes, dtype=torch.uint8, device=self.device)
            self.stream = torch.cuda.current_stream(self.device)
            self._check(self._lib.kpz_bind(self._h, self.lattice.data_ptr(), self.lattice_bytes, self.scratch.data_ptr(),
                                           self.scratch_bytes, self.stream.cuda_stream))
        ro, rs = ctypes.c_uint32(), ctypes.c_uint32()
        rb, bo, to = ctypes.c_size_t(), ctypes.c_size_t(), ctypes.c_size_t()
        self._check(self._lib.kpz_slab_info(self._h, ctypes.addressof(ro), ctypes.addressof(rs), ctypes.addressof(rb),
                                            ctypes.addressof(bo), ctypes.addressof(to)))
        self.rows_own, self.rows, self.row_bytes = ro.value, rs.value, rb.value
        self.planes = self.lattice.view(2, self.rows, self.row_bytes)            # [plane X / Y][row][byte]
        self.base0 = self.scratch[bo.value:bo.value + 4 * L].view(torch.int32)   # row-0 prefix (slab 0)
        self.totals = self.scratch[to.value:to.value + 4 * L].view(torch.int32)  # per-column step totals of this slab

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

    def head(self, n):
        """First n owned rows of both planes (what the previous slab's last tile row reaches into)."""
        return self.planes[:, 0:n]

    def ghost(self, n):
        """First n ghost rows of both planes (the copy of the next slab's head)."""
        return self.planes[:, self.rows_own:self.rows_own + n]

    def owned(self):
        return self.planes[:, 0:self.rows_own]

    def init_flat(self):
        self._check(self._lib.kpz_init_flat(self._h))

    def global_draw(self, m):
        ox, oy = ctypes.c_uint32(), ctypes.c_uint32()
        perm = (ctypes.c_uint32 * 4)()
        self._check(self._lib.kpz_global_draw(self._h, int(m), ctypes.addressof(ox), ctypes.addressof(oy), ctypes.addressof(perm)))
        return ox.value, oy.value, list(perm)

    def pass_(self, slot):
        self._check(self._lib.kpz_slab_pass(self._h, slot))

    def end_mcs(self):
        self._check(self._lib.kpz_slab_end_mcs(self._h))

    def counters(self):
        a, d, r, m = (ctypes.c_uint64() for _ in range(4))
        h = ctypes.c_int64()
        self._check(self._lib.kpz_counters(self._h, 0, ctypes.addressof(a), ctypes.addressof(d), ctypes.addressof(r),
                                           ctypes.addressof(h), ctypes.addressof(m)))
        return {"attempts": a.value, "deposits": d.value, "removals": r.value, "h00": h.value, "mcs": m.value}

    def measure_local(self):
        self._check(self._lib.kpz_slab_measure_local(self._h))

    def measure_finish(self, base0, totals_all):
        """base0: int32 [L] and totals_all: int32 [n_slabs, L] tensors on this slab's device -> four Python ints."""
        out = (ctypes.c_uint64 * 4)()
        assert base0.is_contiguous() and totals_all.is_contiguous() and base0.device == self.device
        self._check(self._lib.kpz_slab_measure_finish(self._h, base0.data_ptr(), totals_all.data_ptr(), ctypes.addressof(out)))
        return [int(v) for v in out]


def finalize(L, halves, h00):
    """kpz_slab_finalize: (sum_h, sum_h2, W2) from the half-accumulators summed mod 2^64 over the slabs."""
    arr = (ctypes.c_uint64 * 4)(*[v & 0xFFFFFFFFFFFFFFFF for v in halves])
    s1, s2, w2 = ctypes.c_int64(), ctypes.c_int64(), ctypes.c_double()
    rc = load_library().kpz_slab_finalize(L, ctypes.addressof(arr), int(h00), ctypes.addressof(s1), ctypes.addressof(s2),
                                          ctypes.addressof(w2))
    if rc not in (KPZ_OK, KPZ_EOVERFLOW):
        raise KpzError(rc, "kpz_slab_finalize")
    return s1.value, s2.value, w2.value


class SlabLattice:
    """An L x L lattice as n_slabs slabs driven by one process; devices[s] holds slab s (all on one GPU is allowed:
    the slabs then simply run one after the other, which is how the single-GPU parity tests exercise the path)."""

    def __init__(self, L, p, q, tile, seed, n_slabs, devices=None):
        devices = list(devices) if devices is not None else ["cuda:0"] * n_slabs
        assert len(devices) == n_slabs
        self.L, self.n_slabs = L, n_slabs
        self.slabs = [SlabHandle(L, p, q, tile, seed, n_slabs, s, devices[s]) for s in range(n_slabs)]
        self._multi = len({str(s.device) for s in self.slabs}) > 1
        self.mcs = 0

    def close(self):
        for s in self.slabs:
            s.close()

    def _sync(self):
        # one device: every copy and kernel is ordered by the one stream; several: wait for all of them at each phase
        if self._multi:
            for s in self.slabs:
                self.slabs[0]._torch.cuda.synchronize(s.device)

    def init_flat(self):
        for s in self.slabs:
            s.init_flat()
        self.mcs = 0
        self._sync()

    def run(self, n_mcs):
        N = self.n_slabs
        for _ in range(int(n_mcs)):
            _, oy, perm = self.slabs[0].global_draw(self.mcs)
            for slot in range(4):
                exch, n = exchange_plan(oy, perm, slot)
                if exch:
                    for s in range(N):
                        self.slabs[s].ghost(n).copy_(self.slabs[(s + 1) % N].head(n))
                    self._sync()
                for s in self.slabs:
                    s.pass_(slot)
                self._sync()
                if exch:
                    for s in range(N):
                        self.slabs[(s + 1) % N].head(n).copy_(self.slabs[s].ghost(n))
                    self._sync()
            for s in self.slabs:
                s.end_mcs()
            self.mcs += 1

    def counters(self):
        cs = [s.counters() for s in self.slabs]
        out = {k: sum(c[k] for c in cs) for k in ("attempts", "deposits", "removals", "h00")}
        out["mcs"] = cs[0]["mcs"]
        return out

    def measure(self):
        torch = self.slabs[0]._torch
        for s in self.slabs:
            s.measure_local()
        self._sync()
        halves = [0, 0, 0, 0]
        for s in self.slabs:
            base0 = self.slabs[0].base0.to(s.device).contiguous()
            totals = torch.stack([t.totals.to(s.device) for t in self.slabs]).contiguous()
            halves = [(a + b) & 0xFFFFFFFFFFFFFFFF for a, b in zip(halves, s.measure_finish(base0, totals))]
        return finalize(self.L, halves, self.counters()["h00"])

    def packed_rows(self):
        """The whole lattice in the device layout of a single handle (uint8 [2][L][L/8], on the CPU): for parity tests."""
        torch = self.slabs[0]._torch
        return torch.cat([s.owned().cpu() for s in self.slabs], dim=1).contiguous()


class DistSlab:
    """This rank's slab of a lattice spread over a torch.distributed group (one process per GPU, NCCL): rank r holds
    slab r.  The ghost rows travel point to point between neighbouring ranks; the measurement needs one all_gather of
    [L] int32 per rank, one broadcast and one all_reduce of four 64-bit words.  `handle` may be any object with the
    SlabHandle interface (the gloo CPU tests pass a stand-in)."""

    def __init__(self, handle, group=None):
        import torch.distributed as dist
        self.h, self.dist, self.group = handle, dist, group
        self.rank, self.world = dist.get_rank(group), dist.get_world_size(group)
        assert self.world == handle.n_slabs and self.rank == handle.slab
        self.mcs = 0

    def _shift(self, send_view, recv_view, to_rank, from_rank):
        """send_view -> to_rank, recv_view <- from_rank, plane by plane (each plane's rows are one contiguous block)."""
        dist = self.dist
        if self.world == 1:
            recv_view.copy_(send_view)
            return
        ops = []
        for pl in range(send_view.shape[0]):
            ops.append(dist.P2POp(dist.isend, send_view[pl].contiguous(), to_rank, self.group))
        bufs = [recv_view[pl].contiguous() for pl in range(recv_view.shape[0])]
        for pl in range(recv_view.shape[0]):
            ops.append(dist.P2POp(dist.irecv, bufs[pl], from_rank, self.group))
        for w in dist.batch_isend_irecv(ops):
            w.wait()
        for pl in range(recv_view.shape[0]):
            if bufs[pl].data_ptr() != recv_view[pl].data_ptr():
                recv_view[pl].copy_(bufs[pl])

    def init_flat(self):
        self.h.init_flat()
        self.mcs = 0

    def run(self, n_mcs):
        nxt, prv = (self.rank + 1) % self.world, (self.rank - 1) % self.world
        for _ in range(int(n_mcs)):
            _, oy, perm = self.h.global_draw(self.mcs)
            for slot in range(4):
                exch, n = exchange_plan(oy, perm, slot)
                if exch:       # my head goes to the previous rank's ghost rows, my ghost rows come from the next rank's head
                    self._shift(self.h.head(n), self.h.ghost(n), prv, nxt)
                self.h.pass_(slot)
                if exch:       # and back: my ghost rows overwrite the next rank's head, my head comes from the previous rank
                    self._shift(self.h.ghost(n), self.h.head(n), nxt, prv)
            self.h.end_mcs()
            self.mcs += 1

    def measure(self):
        """(sum_h, sum_h2, W2) of the whole lattice, the same on every rank."""
        import torch
        dist = self.dist
        self.h.measure_local()
        tot = self.h.totals.contiguous()
        gathered = [torch.empty_like(tot) for _ in range(self.world)]
        base0 = self.h.base0.clone()
        if self.world > 1:
            dist.all_gather(gathered, tot, group=self.group)
            dist.broadcast(base0, src=dist.get_global_rank(self.group, 0) if self.group is not None else 0, group=self.group)
        else:
            gathered = [tot]
        halves = self.h.measure_finish(base0, torch.stack(gathered).contiguous())
        c = self.h.counters()
        # 64-bit words that wrap: int64 tensors add mod 2^64
        acc = torch.tensor([v - (1 << 64) if v >= (1 << 63) else v for v in halves] + [c["h00"]], dtype=torch.int64,
                           device=tot.device)
        if self.world > 1:
            dist.all_reduce(acc, op=dist.ReduceOp.SUM, group=self.group)
        vals = [int(v) for v in acc.tolist()]
        return finalize(self.h.L, vals[:4], vals[4])
