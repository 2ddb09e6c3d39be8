"""Host logic of the slab decomposition (paper_1110_6745_b200/slabs.py) on CPU: two gloo ranks run DistSlab with a
stand-in for the CUDA slab handle whose "kernel" only stamps the rows its active tile rows cover.  The final stamps on
every rank's owned rows must be those of the same stamping on one whole lattice: this holds exactly when the right
rows travel to the right neighbour before and after the right colour passes (include/kpz.h "slabs")."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1110_6745_b200 import slabs

L, T = 256, 16
NT = L // T


def _draw(m):
    """A deterministic stand-in for the global draw: y origin (multiple of 4 below T) and colour order of MCS m."""
    rng = np.random.default_rng(1000 + m)
    return 0, int(4 * rng.integers(0, T // 4)), [int(v) for v in rng.permutation(4)]


def _stamp_rows(rows, ty_first, ty_count, oy, colour, stamp, local_base):
    """Active tile rows (global index parity = colour >> 1) stamp the rows they cover, halo row included."""
    for tyl in range(ty_count):
        if ((ty_first + tyl) & 1) == (colour >> 1):
            y0 = oy + tyl * T - local_base
            rows[:, y0:y0 + T + 1] = stamp


class FakeSlab:
    """SlabHandle interface on CPU tensors: planes [2][rows][1] of int64 stamps."""

    def __init__(self, n_slabs, slab):
        self.L, self.n_slabs, self.slab = L, n_slabs, slab
        self.rows_own = L // n_slabs
        self.rows = self.rows_own + T + 2
        self.planes = torch.zeros(2, self.rows, 1, dtype=torch.int64)
        self.mcs = 0

    def head(self, n):
        return self.planes[:, 0:n]

    def ghost(self, n):
        return self.planes[:, self.rows_own:self.rows_own + n]

    def init_flat(self):
        self.planes.zero_()
        self.mcs = 0

    def global_draw(self, m):
        return _draw(m)

    def pass_(self, slot):
        _, oy, perm = _draw(self.mcs)
        _stamp_rows(self.planes[:, :, 0], self.slab * (NT // self.n_slabs), NT // self.n_slabs, oy, perm[slot],
                    4 * self.mcs + slot + 1, 0)

    def end_mcs(self):
        self.mcs += 1


def _whole_lattice(n_mcs):
    rows = torch.zeros(2, L + T + 2, dtype=torch.int64)      # rows beyond L wrap onto rows 0..
    for m in range(n_mcs):
        _, oy, perm = _draw(m)
        for slot in range(4):
            stamp = 4 * m + slot + 1
            for ty in range(NT):
                if (ty & 1) == (perm[slot] >> 1):
                    ys = (oy + ty * T + np.arange(T + 1)) % L
                    rows[:, ys] = stamp
    return rows[:, :L]


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def _worker(rank, world, port, n_mcs, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        d = slabs.DistSlab(FakeSlab(world, rank))
        d.init_flat()
        d.run(n_mcs)
        q.put((rank, d.h.planes[:, :d.h.rows_own, 0].clone().numpy()))
        dist.barrier()
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world", [2, 4])
def test_distributed_exchange_moves_the_right_rows(world):
    n_mcs, port = 6, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, n_mcs, q)) for r in range(world)]
    for p in procs:
        p.start()
    got = dict(q.get(timeout=180) for _ in range(world))
    for p in procs:
        p.join(timeout=180)
        assert p.exitcode == 0
    want = _whole_lattice(n_mcs).numpy()
    own = L // world
    for r in range(world):
        assert np.array_equal(got[r], want[:, r * own:(r + 1) * own]), r
    assert any(_draw(m)[1] > 0 for m in range(n_mcs))          # the test did move ghost rows with a non-zero origin


def test_exchange_plan_and_single_rank_group():
    assert slabs.exchange_plan(12, [0, 2, 1, 3], 0) == (False, 13)
    assert slabs.exchange_plan(12, [0, 2, 1, 3], 1) == (True, 13)
    assert slabs.exchange_plan(0, [3, 1, 0, 2], 0) == (True, 1)
    # one rank: the ghost rows wrap onto the slab's own head, no communication
    port = _free_port()
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK="0", WORLD_SIZE="1")
    dist.init_process_group("gloo", rank=0, world_size=1)
    try:
        d = slabs.DistSlab(FakeSlab(1, 0))
        d.init_flat()
        d.run(5)
        assert np.array_equal(d.h.planes[:, :L, 0].numpy(), _whole_lattice(5).numpy())
    finally:
        dist.destroy_process_group()
