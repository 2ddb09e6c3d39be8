"""Host-side sharding of the path over ranks (replicas only, no data-path collective).

The path partitions into independent lattices ("independent runs"): rank r of N advances its own lattice(s) with
its own Philox seed; nothing is exchanged while the lattices run.  The only collectives are the barrier and the
reduction of the timing (max over ranks) and of the processed units (sum over ranks) -- both go through
torch.distributed (NCCL on GPUs, gloo in the CPU tests) on small host- or device-side scalars.
"""
from __future__ import annotations

import os


def rank_world():
    """(rank, world_size, local_rank) from the torchrun environment; (0, 1, 0) when launched directly."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1")),
            int(os.environ.get("LOCAL_RANK", "0")))


def rank_seed(seed: int, rank: int) -> int:
    """Seed (64-bit Philox key) of the lattice rank `rank` advances: distinct keys give independent streams."""
    return (int(seed) + int(rank)) & 0xFFFFFFFFFFFFFFFF


def replica_slice(n_replicas: int, rank: int, world: int):
    """Contiguous block of replica ids [lo, hi) of rank `rank` when an ensemble of n_replicas lattices is sharded
    (first n_replicas % world ranks get one more)."""
    if not (0 <= rank < world):
        raise ValueError("rank out of range")
    q, r = divmod(int(n_replicas), int(world))
    lo = rank * q + min(rank, r)
    return lo, lo + q + (1 if rank < r else 0)


def aggregate(units_local: float, seconds_local: float, device=None):
    """Whole-job throughput: (sum over ranks of units) / (max over ranks of seconds).  Returns (units, seconds, rate).
    Works with any initialised torch.distributed backend; without one it is the local values."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return units_local, seconds_local, units_local / seconds_local
    t = torch.tensor([float(seconds_local)], dtype=torch.float64, device=device)
    u = torch.tensor([float(units_local)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(u.item()), float(t.item()), float(u.item()) / float(t.item())
