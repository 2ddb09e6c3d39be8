"""N > 1 host logic on CPU: two gloo processes exercise the rank sharding and the whole-job aggregation that
bench.py --gpus N uses (replicas only, no data-path collective)."""
import os
import socket

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1110_6745_b200 import shard


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world),
                      LOCAL_RANK=str(rank))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        r, w, lr = shard.rank_world()
        lo, hi = shard.replica_slice(1024 + 1, r, w)
        # rank 1 is "slower" and processes a different number of units: the job rate is sum(units) / max(seconds)
        units, secs, rate = shard.aggregate(100.0 * (hi - lo), 2.0 + rank)
        q.put((r, w, lr, shard.rank_seed(42, r), lo, hi, units, secs, rate))
        dist.barrier()
    finally:
        dist.destroy_process_group()


def test_two_rank_sharding_and_aggregation():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=120)
        assert p.exitcode == 0
    (r0, w0, _, s0, lo0, hi0, u0, t0, rate0), (r1, w1, _, s1, lo1, hi1, u1, t1, rate1) = res
    assert (r0, r1, w0, w1) == (0, 1, 2, 2)
    assert s0 == 42 and s1 == 43                              # distinct Philox keys per rank
    assert (lo0, hi0, lo1, hi1) == (0, 513, 513, 1025)        # contiguous cover, remainder to the first ranks
    assert u0 == u1 == 100.0 * 1025 and t0 == t1 == 3.0       # sum of units, max of seconds, same on every rank
    assert rate0 == rate1 == pytest.approx(102500.0 / 3.0)


def test_single_process_defaults_and_slices():
    assert shard.aggregate(10.0, 2.0) == (10.0, 2.0, 5.0)
    assert shard.rank_seed(2**64 - 1, 1) == 0
    for n, w in ((1024, 8), (7, 3), (2, 4)):
        parts = [shard.replica_slice(n, r, w) for r in range(w)]
        assert parts[0][0] == 0 and parts[-1][1] == n
        assert all(a[1] == b[0] for a, b in zip(parts, parts[1:]))
        assert max(h - l for l, h in parts) - min(h - l for l, h in parts) <= 1
    with pytest.raises(ValueError):
        shard.replica_slice(4, 4, 4)


def test_bench_gpus_2_starts_two_ranks_itself():
    """`python bench.py --gpus 2` with no torchrun environment (the way the driver calls it for N = 1, and what a
    user types for N > 1) must start the two ranks itself: the launcher self-test joins a gloo group of world size
    2 through that path and reports n_gpus = 2; a WORLD_SIZE that contradicts --gpus is refused."""
    import json
    import subprocess
    import sys
    from pathlib import Path
    root = Path(__file__).resolve().parent.parent
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT")}
    out = subprocess.run([sys.executable, str(root / "bench.py"), "--gpus", "2", "--launcher-selftest"],
                         capture_output=True, text=True, timeout=300, cwd=str(root), env=env)
    assert out.returncode == 0, out.stderr[-800:]
    lines = [l for l in out.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["n_gpus"] == 2 and d["units"] == 300.0 and d["seconds"] == 2.0 and d["seeds"] == [42, 43]
    env["WORLD_SIZE"] = "1"
    bad = subprocess.run([sys.executable, str(root / "bench.py"), "--gpus", "2", "--launcher-selftest"],
                         capture_output=True, text=True, timeout=300, cwd=str(root), env=env)
    assert bad.returncode != 0 and "WORLD_SIZE" in (bad.stderr + bad.stdout)
