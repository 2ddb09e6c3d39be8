#!/usr/bin/env python
"""bench.py -- throughput of the octahedron-KPZ hot path on B200 (BASELINE.json metric: attempted site updates/s).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 1..5] [--peaks]

One "step" = one pass of the whole hot path over one batch: MCS_PER_STEP Monte-Carlo steps of the lattice
(kpz_run: global draw, tile staging, in-kernel Philox, sequential updates, write-back, bookkeeping) followed by one
sampling-time measurement (kpz_measure: height reconstruction, sum h, sum h^2, W^2).  Default: BASELINE config 3
(L = 2^17, T = 64, p = 1, q = 0, seed 42, flat start), K = 10 steps of 10 MCS = its 100 timed MCS.
`--config N` times another BASELINE config the same way (parity-test cases otherwise).

Prints ONE JSON line (rank 0).  See DESIGN.md "Measurement" for every field.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time
from pathlib import Path

ROOT = Path(__file__).resolve().parent
sys.path.insert(0, str(ROOT))

METRIC = "attempted site updates/s"
UNIT = "Gupd/s"

# BASELINE.json configs: lattice, tile, probabilities, seed, replicas, MCS per step, default steps
CONFIGS = {
    1: dict(name="config1: L=2^8 flat start, p=1 q=0, tile 16, seed 1, 64 MCS", L=1 << 8, tile=16, p=1.0, q=0.0, seed=1,
            replicas=1, mcs_per_step=8, steps=8),
    2: dict(name="config2: L=2^12 flat start, p=1 q=0, tile 32, seed 7, 1000 MCS", L=1 << 12, tile=32, p=1.0, q=0.0, seed=7,
            replicas=1, mcs_per_step=100, steps=10),
    3: dict(name="config3: L=2^17 flat start, p=1 q=0, tile 64, seed 42", L=1 << 17, tile=64, p=1.0, q=0.0, seed=42,
            replicas=1, mcs_per_step=10, steps=10),
    4: dict(name="config4: 1024 replicas x L=2^7, p=1 q=0, tile 16, seed 4 (steady-state batch)", L=1 << 7, tile=16, p=1.0,
            q=0.0, seed=4, replicas=1024, mcs_per_step=500, steps=10),
    5: dict(name="config5: L=2^19 flat start, p=0.75 q=0.25, tile 64, seed 3, 50 MCS", L=1 << 19, tile=64, p=0.75, q=0.25,
            seed=3, replicas=1, mcs_per_step=1, steps=50),
}
WORKLOAD = {k: CONFIGS[3][k] for k in ("L", "tile", "p", "q", "seed")}
MCS_PER_STEP = CONFIGS[3]["mcs_per_step"]

# ---- algorithmic work per attempted update (SASS listing: profiles/r02_update_T64_mode0.md) ----
# ALU pipe (LOP3 / SHF / LEA; 16 lanes per clock and scheduler), p = 1, q = 0:
#   1/8 Philox4x32-10 call = 2.5 three-input XORs (its 2.5 32x32->64 multiplies run on the FMA pipe)
#   + 9 for the attempt: row index, word index, site index, site bit, 2 neighbour alignments, 2 neighbour tests, mask.
# General p, q adds the accept stream (1/4 call per attempt: 5 XORs, 5 multiplies), the two maximum tests, two compares
# and two selects, one OR: 11.5 + 5 + 2 + 2 + 2 + 1 = 23.5.
ALG_ALU_OPS_PER_UPDATE = 11.5
ALG_ALU_OPS_PER_UPDATE_GENERAL = 23.5
ALG_MUL_OPS_PER_UPDATE = 2.5
ALG_SMEM_BYTES_PER_UPDATE = 24.0      # five 32-bit shared-memory loads and one 32-bit XOR reduction
ALG_BYTES_PER_UPDATE = 0.5            # HBM: each site (2 bits) read once and written once per MCS
ALG_BYTES_PER_SITE_MEASURE = 0.125    # kpz_measure reads plane Y once (one bit per site)
# dram__bytes_read.sum + dram__bytes_write.sum of one update launch at L = 2^17 (ncu --set full)
TRAFFIC_BYTES_PER_LAUNCH = 6.26e9
TRAFFIC_SOURCE = "profiles/r02_ncu_full.md (ncu --set full on the final tree of round 2, launch 48: 4.154 GB read + 2.104 GB written)"


def _peaks():
    f = ROOT / "MEASURED_PEAKS.json"
    if f.exists():
        d = json.loads(f.read_text())
        return d.get("hbm_gbs", 6650.0), d.get("sm_max_mhz", 1965.0), "measured"
    return 6650.0, 1965.0, "fallback"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.proc, self.lines = index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            parts = [p.strip() for p in ln.split(",")]
            if len(parts) < 7:
                continue
            try:
                sm.append(float(parts[0])); mx.append(float(parts[1]))
            except ValueError:
                continue
            for n, v in zip(names, parts[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


def _event_ms(torch, fn, reps=1):
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record()
    for _ in range(reps):
        fn()
    b.record()
    torch.cuda.synchronize()
    return a.elapsed_time(b) / reps


def run_ours(args):
    import numpy as np
    import torch
    import paper_1110_6745_b200 as pkg

    from paper_1110_6745_b200 import shard
    rank, world, local = shard.rank_world()
    if world != args.gpus:       # the reported n_gpus can never disagree with the request
        raise SystemExit("bench.py: --gpus %d but WORLD_SIZE=%d (launch with torchrun --nproc-per-node %d, or let "
                         "bench.py start the ranks itself by leaving WORLD_SIZE unset)" % (args.gpus, world, args.gpus))
    if torch.cuda.device_count() <= local:
        raise SystemExit("bench.py: rank %d needs cuda:%d but only %d device(s) are visible" % (rank, local, torch.cuda.device_count()))
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)

    cfg = dict(CONFIGS[args.config])
    if args.L:
        cfg["L"] = args.L
    if args.tile:
        cfg["tile"] = args.tile
        cfg["name"] += " [tile overridden: %d]" % args.tile
    L, T, R, mcs_per_step = cfg["L"], cfg["tile"], cfg["replicas"], cfg["mcs_per_step"]
    general = not (cfg["p"] >= 1.0 and cfg["q"] <= 0.0)
    # weak scaling: every rank advances its own independent lattice(s) (its own Philox key)
    k = pkg.KPZ(L, cfg["p"], cfg["q"], T, shard.rank_seed(cfg["seed"], rank), n_replicas=R, device=dev)
    k.init_flat()
    att_per_step = mcs_per_step * R * L * L

    for _ in range(args.warmup):
        k.run(mcs_per_step)
        k.measure()

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    sampler = ClockSampler(local)
    launches0 = k.launch_count()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True))
          for _ in range(args.steps)]
    barrier()
    sampler.start()
    t0 = torch.cuda.Event(enable_timing=True); t1 = torch.cuda.Event(enable_timing=True)
    t0.record()
    last = None
    for i in range(args.steps):
        ev[i][0].record()
        k.run(mcs_per_step)
        ev[i][1].record()
        last = k.measure()
        ev[i][2].record()
    t1.record()
    barrier()
    clocks = sampler.stop()
    ms_total = t0.elapsed_time(t1)
    launches = k.launch_count() - launches0
    upd_ms = sum(a.elapsed_time(b) for a, b, _ in ev)
    meas_ms = sum(b.elapsed_time(c) for _, b, c in ev)
    # whole job: units of all ranks / max over ranks of the device time
    _, sec_total, rate = shard.aggregate(args.steps * att_per_step, ms_total * 1e-3, device=dev)
    ms_total = sec_total * 1e3
    value = rate / 1e9

    # ---- end to end through the C ABI with HOST buffers, copies inside the timed region ----
    # "value": ONE pinned host lattice through kpz_step_host_overlapped (a step's output is the next step's input, so steps
    # cannot overlap, but the copies of a step overlap its own colour passes slab by slab: DESIGN.md 8.2);
    # "sequential_value": the same through kpz_step_host (H2D, kpz_run, kpz_measure, D2H in sequence).
    # "two_lane_value": two INDEPENDENT pinned host lattices through kpz_pipeline_host, the copies of one overlapping the
    # kernels of the other.
    # Local timings first; the reductions over ranks come after the try block, so that a rank whose pinned
    # allocation fails still takes part in them (a leg that failed on any rank is reported as unavailable).
    serial = (0.0, float("inf"))
    overl = (0.0, float("inf"))
    piped = (0.0, float("inf"))
    n_e2e = max(1, min(args.steps, 3))
    n_rounds = max(3, (args.steps + 1) // 2)      # at least 6 pipelined steps, so that fill and drain do not dominate
    e2e_err = None
    try:
        host = torch.empty(k.lattice_bytes, dtype=torch.uint8).pin_memory()
        k.export_packed(host)
        h00 = np.array([k.counters(r)["h00"] for r in range(R)], dtype=np.int64)
        mcs_now = k.counters()["mcs"]
        k.step_host(host, h00, mcs_now, mcs_per_step)       # warm-up of the pinned path
        mcs_now += mcs_per_step
        torch.cuda.synchronize()
        w0 = time.perf_counter()
        for _ in range(n_e2e):
            k.step_host(host, h00, mcs_now, mcs_per_step)
            mcs_now += mcs_per_step
        torch.cuda.synchronize()
        serial = (n_e2e * att_per_step, time.perf_counter() - w0)
        # the same steps with the copies of the ONE lattice overlapped with its kernels slab by slab
        k.step_host_overlapped(host, h00, mcs_now, mcs_per_step, args.e2e_slabs)       # warm-up
        mcs_now += mcs_per_step
        torch.cuda.synchronize()
        w0 = time.perf_counter()
        for _ in range(n_e2e):
            k.step_host_overlapped(host, h00, mcs_now, mcs_per_step, args.e2e_slabs)
            mcs_now += mcs_per_step
        torch.cuda.synchronize()
        overl = (n_e2e * att_per_step, time.perf_counter() - w0)
        if args.config == 3 or args.pipeline:
            # lane 1: a genuinely different lattice -- grown under another Philox key, then advanced (like lane 0) under
            # the handle's key; the lane clocks differ as well
            k2 = pkg.KPZ(L, cfg["p"], cfg["q"], T, shard.rank_seed(cfg["seed"], rank) + 1000003, n_replicas=R, device=dev)
            k2.init_flat()
            k2.run(3 * mcs_per_step)
            host2 = torch.empty(k.lattice_bytes, dtype=torch.uint8).pin_memory()
            k2.export_packed(host2)
            h00_l = np.stack([h00, np.array([k2.counters(r)["h00"] for r in range(R)], dtype=np.int64)])
            k2.close()
            del k2
            torch.cuda.empty_cache()
            clock = [mcs_now, 3 * mcs_per_step]
            k.pipeline_host([host, host2], h00_l, clock, mcs_per_step, 1)   # warm-up of the pipelined path
            clock = [t + mcs_per_step for t in clock]
            torch.cuda.synchronize()
            w0 = time.perf_counter()
            k.pipeline_host([host, host2], h00_l, clock, mcs_per_step, n_rounds)
            torch.cuda.synchronize()
            piped = (2 * n_rounds * att_per_step, time.perf_counter() - w0)
    except Exception as exc:   # e.g. not enough pinned host memory on the box
        e2e_err = str(exc)[:200]
    _, serial_s, serial_rate = shard.aggregate(serial[0], serial[1], device=dev)
    _, overl_s, overl_rate = shard.aggregate(overl[0], overl[1], device=dev)
    _, piped_s, piped_rate = shard.aggregate(piped[0], piped[1], device=dev)
    e2e = {"value": None, "unit": UNIT,
           "h2d_bytes_per_step": k.lattice_bytes + 8 * R, "d2h_bytes_per_step": k.lattice_bytes + (3 * 8 + 32) * R}
    if serial_s != float("inf"):
        e2e.update({"value": serial_rate / 1e9, "steps": n_e2e,
                    "api": "kpz_step_host: ONE pinned host lattice copied in, advanced, measured and copied out per step"})
    if overl_s != float("inf"):
        e2e.update({"value": overl_rate / 1e9, "steps": n_e2e, "sequential_value": serial_rate / 1e9,
                    "api": "kpz_step_host_overlapped (%d slabs): ONE pinned host lattice copied in, advanced, measured and "
                           "copied out per step, the copies overlapped with the colour passes slab by slab; "
                           "sequential_value = the same through kpz_step_host (copy, kernels, copy in sequence)" % args.e2e_slabs})
    if piped_s != float("inf"):
        e2e.update({"two_lane_value": piped_rate / 1e9, "two_lane_steps": 2 * n_rounds,
                    "two_lane_api": "kpz_pipeline_host: two independent pinned host lattices; the copies of step b-1 / "
                                    "b+1 overlap the kernels of step b"})
    if e2e_err is not None:
        e2e["error"] = e2e_err

    if rank != 0:
        return
    hbm_peak, sm_max, src = _peaks()
    pk = pkg.measure_peaks()                       # integer / shared-memory pipe peaks measured on this box, now
    # ---- roofline of the dominant kernel: the update kernel(s) behind kpz_run, timed by CUDA events around kpz_run ----
    tiled = launches >= args.steps * mcs_per_step * 4          # 4 launches per MCS (tiled) or 1 per call (resident)
    n_upd_launch = args.steps * mcs_per_step * 4 if tiled else args.steps
    upd_launch_ms = upd_ms / n_upd_launch
    upd_per_launch = R * L * L / 4 if tiled else R * L * L * mcs_per_step
    upd_rate = upd_per_launch / (upd_launch_ms * 1e-3)
    alu_ops = ALG_ALU_OPS_PER_UPDATE_GENERAL if general else ALG_ALU_OPS_PER_UPDATE
    alu_peak_derived = pk["n_sms"] * 4 * 16 * sm_max * 1e6
    mode = 0 if not general else (1 if (cfg["p"] > 0 and cfg["q"] > 0) else 2)
    nthr = {64: 96, 32: 64}.get(T, 128)
    roofline = {
        "bound": "alu", "achieved": upd_rate * alu_ops / 1e12, "peak": pk["lop3_lane_ops"] / 1e12,
        "unit": "Tops/s (ALU-pipe lane-ops)", "frac": upd_rate * alu_ops / pk["lop3_lane_ops"],
        "traffic": TRAFFIC_BYTES_PER_LAUNCH if (L == (1 << 17) and not general) else None,
        "traffic_source": TRAFFIC_SOURCE if (L == (1 << 17) and not general) else None,
        "kernel": ("kpz_update_kernel<%d,%d,%d>" % (T, nthr, mode)) if tiled else ("kpz_resident_kernel<%d,..,%d>" % (T, mode)),
        "alg_alu_ops_per_update": alu_ops, "alg_mul_ops_per_update": ALG_MUL_OPS_PER_UPDATE * (3 if general else 1),
        "launch_ms": upd_launch_ms, "updates_per_launch": upd_per_launch,
        "peak_source": "kpz_measure_peaks on this box in this run: LOP3 lane-ops/s with every warp slot of every SM busy "
                       "(SM clock %.0f MHz while it ran)" % (pk["sm_clock_hz"] / 1e6),
        "peak_derived": alu_peak_derived / 1e12,
        "peak_derived_source": "%d SM x 4 schedulers x 16 ALU lanes/clk x clocks.max.sm (%s MEASURED_PEAKS.json)" % (pk["n_sms"], src),
        "frac_of_derived": upd_rate * alu_ops / alu_peak_derived,
        "measured_peaks": {kk: (v / 1e12 if kk.endswith("ops") or kk == "lds_bytes" else v) for kk, v in pk.items()},
        "measured_peaks_units": "T lane-ops/s (lop3, shf, imad, imad_wide, smem_xor), TB/s (lds_bytes), attempts/s (attempt_mix), Hz, count, "
                                "SM clocks per attempt and warp of one tile's dependent chain at 1 and 2 warps per scheduler (chain_cycles_*)",
        # the shared-memory data pipe is the other co-limit: 5 loads + 1 XOR reduction of 4 bytes per update
        "lsu": {"bound": "shared-memory data pipe", "achieved": upd_rate * ALG_SMEM_BYTES_PER_UPDATE / 1e12,
                "peak": pk["lds_bytes"] / 1e12, "unit": "TB/s", "frac": upd_rate * ALG_SMEM_BYTES_PER_UPDATE / pk["lds_bytes"],
                "alg_bytes_per_update": ALG_SMEM_BYTES_PER_UPDATE},
        # the same instruction mix issued without the dependent chain of a tile (perfect latency hiding)
        "attempt_mix": {"achieved": upd_rate / 1e9, "peak": pk["attempt_mix"] / 1e9, "unit": UNIT,
                        "frac": upd_rate / pk["attempt_mix"]},
        "hbm": {"achieved": upd_rate * ALG_BYTES_PER_UPDATE / 1e9, "peak": hbm_peak, "unit": "GB/s",
                "peak_source": src + " MEASURED_PEAKS.json", "frac": upd_rate * ALG_BYTES_PER_UPDATE / 1e9 / hbm_peak},
    }
    kernels = [{"kernel": roofline["kernel"], "unit": "attempted update", "bound": "alu", "launch_ms": upd_launch_ms,
                "units_per_launch": upd_per_launch, "alg_ops_per_unit": alu_ops, "alg_hbm_bytes_per_unit": ALG_BYTES_PER_UPDATE,
                "gupds": upd_rate / 1e9, "frac": roofline["frac"]}]
    # kpz_measure = kpz_row0_prefix_kernel + kpz_column_chunk_kernel + kpz_combine_kernel (+ one 64-byte copy and a sync)
    m_ms = meas_ms / args.steps
    m_bytes = R * L * L * ALG_BYTES_PER_SITE_MEASURE
    kernels.append({"kernel": "kpz_measure: kpz_row0_prefix_kernel + kpz_column_chunk_kernel + kpz_combine_kernel",
                    "unit": "site", "bound": "hbm", "launch_ms": m_ms, "units_per_launch": R * L * L,
                    "alg_hbm_bytes_per_unit": ALG_BYTES_PER_SITE_MEASURE, "achieved_gbs": m_bytes / (m_ms * 1e-3) / 1e9,
                    "peak_gbs": hbm_peak, "frac": m_bytes / (m_ms * 1e-3) / 1e9 / hbm_peak,
                    "hbm_floor_ms": m_bytes / (hbm_peak * 1e9) * 1e3})
    lattice_bytes = k.lattice_bytes
    if args.config == 3 and not args.L and world == 1:
        # the general-(p,q) kernel (MODE 1) on config 5's parameters at L = 2^17: 10 MCS from the flat start after 10
        k.close()
        torch.cuda.empty_cache()
        c5 = CONFIGS[5]
        kg = pkg.KPZ(L, c5["p"], c5["q"], T, c5["seed"], device=dev)
        kg.init_flat()
        kg.run(10)
        g_ms = _event_ms(torch, lambda: kg.run(10)) / 40.0
        kg.close()
        g_rate = (L * L / 4) / (g_ms * 1e-3)
        kernels.append({"kernel": "kpz_update_kernel<64,96,1> (general p, q: config 5 parameters p=0.75 q=0.25 seed 3 at L=2^17)",
                        "unit": "attempted update", "bound": "alu", "launch_ms": g_ms, "units_per_launch": L * L / 4,
                        "alg_ops_per_unit": ALG_ALU_OPS_PER_UPDATE_GENERAL, "alg_hbm_bytes_per_unit": ALG_BYTES_PER_UPDATE,
                        "gupds": g_rate / 1e9, "frac": g_rate * ALG_ALU_OPS_PER_UPDATE_GENERAL / pk["lop3_lane_ops"]})
    roofline["kernels"] = kernels
    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        cpu = cpu_baseline_sample()
    out = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
           "ms_per_step": ms_total / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
           "dtype": "u32 bit-logic + Philox4x32 (int32/int64 sums)", "data": "synthetic",
           "config": {"workload": cfg["name"] if not args.L else "L=%d" % L,
                      "L": L, "tile": T, "p": cfg["p"], "q": cfg["q"], "seed": cfg["seed"], "replicas": R,
                      "mcs_per_step": mcs_per_step, "step": "kpz_run(%d) + kpz_measure" % mcs_per_step,
                      "path": "tiled (4 launches per MCS)" if tiled else "lattice-resident (1 launch per kpz_run)",
                      "l2": ("lattice %.1f GiB >> 126 MB L2, no flush needed" % (lattice_bytes / 2**30)) if lattice_bytes > (1 << 28)
                            else "lattice %.1f MiB: smaller than L2 by construction of the config" % (lattice_bytes / 2**20),
                      "parallelism": "independent lattice per GPU" if world > 1 else "1 GPU"},
           "update_only_gupds": args.steps * att_per_step / (upd_ms * 1e-3) / 1e9,
           "measure_ms": m_ms, "W2_last": float(last[2][0]),
           "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches), "roofline": roofline, "cpu_baseline": cpu}
    print(json.dumps(out))


def run_slabs(args):
    """--slabs: the config's ONE lattice as N slabs of rows, rank r holding slab r (paper_1110_6745_b200/slabs.py:
    ghost rows point to point between neighbouring ranks twice per MCS, the measurement through one all_gather, one
    broadcast and one all_reduce).  Strong scaling: the total work is fixed as N grows."""
    import torch
    import torch.distributed as dist
    from paper_1110_6745_b200 import shard
    from paper_1110_6745_b200.slabs import DistSlab, SlabHandle
    rank, world, local = shard.rank_world()
    if world != args.gpus:
        raise SystemExit("bench.py: --gpus %d but WORLD_SIZE=%d" % (args.gpus, world))
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    else:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29531")
        dist.init_process_group("gloo", rank=0, world_size=1)
    cfg = CONFIGS[args.config]
    L, T, mcs_per_step = cfg["L"], cfg["tile"], cfg["mcs_per_step"]
    d = DistSlab(SlabHandle(L, cfg["p"], cfg["q"], T, cfg["seed"], world, rank, device=dev))
    d.init_flat()
    for _ in range(args.warmup):
        d.run(mcs_per_step)
        d.measure()
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    sampler = ClockSampler(local)
    sampler.start()
    t0 = torch.cuda.Event(enable_timing=True); t1 = torch.cuda.Event(enable_timing=True)
    t0.record()
    last = None
    for _ in range(args.steps):
        d.run(mcs_per_step)
        last = d.measure()
    t1.record()
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    clocks = sampler.stop()
    sec = torch.tensor([t0.elapsed_time(t1) * 1e-3], dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(sec, op=dist.ReduceOp.MAX)
    sec = float(sec.item())
    if rank == 0:
        units = args.steps * mcs_per_step * L * L
        print(json.dumps({"metric": METRIC, "value": units / sec / 1e9, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                          "warmup": args.warmup, "ms_per_step": sec / args.steps * 1e3, "higher_is_better": True,
                          "scaling": "strong", "vs_baseline": None, "dtype": "u32 bit-logic + Philox4x32 (int32/int64 sums)",
                          "data": "synthetic",
                          "config": {"workload": cfg["name"], "L": L, "tile": T, "p": cfg["p"], "q": cfg["q"], "seed": cfg["seed"],
                                     "mcs_per_step": mcs_per_step, "parallelism": "one lattice as %d slabs of rows" % world,
                                     "step": "4 colour passes per MCS with ghost-row exchange + slab measurement"},
                          "W2_last": last[2], "clocks": clocks, "e2e": None, "gpu_launches": None, "roofline": None,
                          "cpu_baseline": None}))
    dist.destroy_process_group()


def _cpu_model():
    try:
        for line in open("/proc/cpuinfo"):
            if line.startswith("model name"):
                return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


REF_WINDOW = 4096      # both oracle legs time the same sample: a 4096^2 window of the config-3 lattice


def _oracle_window_rate(threads, n_mcs, window=REF_WINDOW):
    from oracle import Oracle
    w = WORKLOAD
    o = Oracle(w["L"], w["p"], w["q"], w["tile"], w["seed"], window=(0, 0, window, window), threads=threads)
    o.init_flat()
    o.run(1)
    t0 = time.perf_counter()
    o.run(n_mcs)
    return n_mcs * window * window / (time.perf_counter() - t0) / 1e9, o.threads


def _oracle_full_rate(L, T, threads, n_mcs):
    from oracle import Oracle
    w = WORKLOAD
    o = Oracle(L, w["p"], w["q"], T, w["seed"], threads=threads)
    o.init_flat()
    o.run(1)
    t0 = time.perf_counter()
    o.run(n_mcs)
    return n_mcs * L * L / (time.perf_counter() - t0) / 1e9


def cpu_baseline_sample():
    """The oracle, as it stands, on the host cores (SURVEY 8(d) "Timing the oracle beside it"): all cores and one
    thread (the paper's comparison was one core), on a window of the SAME workload (L=2^17 tile ids, offsets and
    Philox streams; out of cache as a whole lattice would be) and on a whole in-cache L=2^12 lattice (the paper's L3
    remark).  Bounded to roughly 15-25 s of CPU work."""
    cores = os.cpu_count() or 1
    v_all, thr = _oracle_window_rate(cores, 3)
    v_one, _ = _oracle_window_rate(1, 1)
    return {"value": v_all, "unit": UNIT, "cores": thr, "kind": "oracle", "cpu_model": _cpu_model(),
            "sample": "window %dx%d of the L=2^17 config-3 lattice, 3 MCS after 1 warm-up MCS from the flat start, OpenMP over "
                      "the tiles of a colour (tiles touching the window run all T*T attempts; attempts leaving the window "
                      "are skipped and not counted; every pass scans the 2^20 tile slots of the colour for window hits)"
                      % (REF_WINDOW, REF_WINDOW),
            "one_thread": {"value": v_one, "cores": 1, "sample": "same window, 1 MCS after 1 warm-up MCS"},
            "in_cache_L4096": {"value": _oracle_full_rate(4096, 32, cores, 3), "cores": thr,
                               "one_thread_value": _oracle_full_rate(4096, 32, 1, 1),
                               "sample": "whole L=2^12, T=32 lattice (32 MiB of int8 slopes), 3 MCS (1 MCS for one thread) "
                                         "after 1 warm-up MCS"},
            "note": "unoptimised oracle (int8 slopes, a modulo per neighbour): a reported baseline, not a tuned CPU code"}


def run_reference(args):
    """--impl reference: the oracle timed as the reference arm (rank 0 only)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    from oracle import Oracle
    w = WORKLOAD
    window = REF_WINDOW
    threads = os.cpu_count() or 1
    o = Oracle(w["L"], w["p"], w["q"], w["tile"], w["seed"], window=(0, 0, window, window), threads=threads)
    o.init_flat()
    for _ in range(args.warmup):
        o.run(MCS_PER_STEP)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        o.run(MCS_PER_STEP)
    dt = time.perf_counter() - t0
    value = args.steps * MCS_PER_STEP * window * window / dt / 1e9
    sample = ("each step = %d MCS of a %dx%d window of the L=2^17 config-3 lattice (same tile ids, offsets, Philox "
              "streams; the window of bench.py's cpu_baseline); measurement excluded (the windowed oracle has no global "
              "height walk)" % (MCS_PER_STEP, window, window))
    out = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": int(os.environ.get("WORLD_SIZE", "1")),
           "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3, "higher_is_better": True,
           "scaling": "weak", "vs_baseline": None, "dtype": "int8 slopes + Philox4x32", "data": "synthetic",
           "config": {"workload": CONFIGS[3]["name"], "sample": sample},
           "cpu_baseline": {"value": value, "unit": UNIT, "cores": o.threads, "kind": "oracle", "sample": sample,
                            "cpu_model": _cpu_model()},
           "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(out))


def relaunch_under_torchrun(args):
    """`python bench.py --gpus N` with N > 1 and no torchrun environment: start the N ranks ourselves (one process
    per GPU, the driver's own command line) and pass their output through.  Returns the exit code."""
    import socket
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(args.gpus),
           "--master-addr", "127.0.0.1", "--master-port", str(port), str(Path(__file__).resolve())] + sys.argv[1:]
    return subprocess.call(cmd)


def launcher_selftest(args):
    """Host logic of the multi-rank launch without any kernel (tests/test_shard_gloo.py): every rank joins a gloo
    group, takes the barrier and the two reductions of shard.aggregate; rank 0 prints the world it saw."""
    import torch.distributed as dist
    from paper_1110_6745_b200 import shard
    rank, world, _ = shard.rank_world()
    if world != args.gpus:
        raise SystemExit("bench.py: --gpus %d but WORLD_SIZE=%d" % (args.gpus, world))
    if world > 1:
        dist.init_process_group("gloo")
        dist.barrier()
    units, seconds, rate = shard.aggregate(100.0 * (rank + 1), 1.0 + rank)
    if rank == 0:
        print(json.dumps({"launcher_selftest": True, "n_gpus": world, "units": units, "seconds": seconds, "rate": rate,
                          "seeds": [shard.rank_seed(WORKLOAD["seed"], r) for r in range(world)]}))
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=0, help="timed steps (default: the config's own, 10 for config 3)")
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=3, choices=sorted(CONFIGS), help="BASELINE config to time (default 3)")
    ap.add_argument("--L", type=int, default=0, help="override the lattice size (debugging only)")
    ap.add_argument("--tile", type=int, default=0, help="override the tile edge (config 4 does not fix it: --config 4 --tile 8 "
                                                        "runs the paper's own 8 x 8 cells)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--pipeline", action="store_true", help="also time kpz_pipeline_host for configs other than 3")
    ap.add_argument("--e2e-slabs", type=int, default=5, help="row slabs of kpz_step_host_overlapped in the e2e leg")
    ap.add_argument("--peaks", action="store_true", help="print the pipe micro-benchmarks (kpz_measure_peaks) and exit")
    ap.add_argument("--layouts", action="store_true", help="print the tile-layout experiment (kpz_measure_layouts) and exit")
    ap.add_argument("--slabs", action="store_true", help="ONE lattice of the config split into slabs of rows over the N ranks "
                                                         "(strong scaling; DESIGN.md Multi-GPU) instead of one lattice per rank")
    ap.add_argument("--launcher-selftest", action="store_true", help="multi-rank launch + reductions only (gloo, no GPU)")
    args = ap.parse_args()
    args.steps = args.steps or CONFIGS[args.config]["steps"]
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "reference":
        run_reference(args)
        return
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        sys.exit(relaunch_under_torchrun(args))
    if args.launcher_selftest:
        launcher_selftest(args)
        return
    if args.slabs:
        run_slabs(args)
        return
    if args.peaks:
        import paper_1110_6745_b200 as pkg
        print(json.dumps({"peaks": pkg.measure_peaks(), "units": "per second; see include/kpz.h kpz_measure_peaks"}))
        return
    if args.layouts:
        import paper_1110_6745_b200 as pkg
        print(json.dumps({"layouts": pkg.measure_layouts(), "units": "attempts/s of the T = 64 attempt loop alone, resident warps "
                          "per SM; see include/kpz.h kpz_measure_layouts"}))
        return
    run_ours(args)


if __name__ == "__main__":
    main()
