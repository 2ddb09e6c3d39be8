#!/usr/bin/env python
"""bench.py -- throughput of the octahedron-KPZ hot path on B200 (BASELINE.json metric: attempted site updates/s).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]

One "step" = one pass of the whole hot path over one batch: MCS_PER_STEP Monte-Carlo steps of the lattice
(kpz_run: global draw, tile staging, in-kernel Philox, sequential updates, write-back, bookkeeping) followed by one
sampling-time measurement (kpz_measure: height reconstruction, sum h, sum h^2, W^2).  Default K = 10 steps of 10
MCS = the 100 timed MCS of BASELINE config 3 (L = 2^17, T = 64, p = 1, q = 0, seed 42, flat start).

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
MCS_PER_STEP = 10
WORKLOAD = dict(L=1 << 17, tile=64, p=1.0, q=0.0, seed=42)

# Algorithmic work per attempted update on the binding pipe, for p = 1, q = 0:
# ALU-pipe operations (LOP3 / SHF / LEA; 16 lanes per clock per scheduler):
#   1/8 Philox4x32-10 call = 2.5 three-input XORs  (its 2.5 32x32->64 multiplies run on the FMA pipe)
#   + 9 for the attempt: row index, word index, site index, site bit, 2 neighbour alignments, 2 neighbour tests, mask
#   (the parity-free tile encoding needs no parity word; the address multiply-add and the deposit count run on
#   the FMA pipe).  Hand count of the minimal sequence for this data layout; the SASS executes 11.4.
ALG_ALU_OPS_PER_UPDATE = 11.5
ALG_MUL_OPS_PER_UPDATE = 2.5
ALG_BYTES_PER_UPDATE = 0.5          # each site (2 bits) read once and written once per MCS
# dram__bytes_read.sum + dram__bytes_write.sum of one update launch at L = 2^17 (profiles/, ncu --set full)
TRAFFIC_BYTES_PER_LAUNCH = 6.27e9


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

    w = dict(WORKLOAD)
    if args.L:
        w["L"] = args.L
    L, T = w["L"], w["tile"]
    # weak scaling: every rank advances its own independent lattice (replica id = rank in the Philox counter)
    k = pkg.KPZ(L, w["p"], w["q"], T, shard.rank_seed(w["seed"], rank), device=dev)
    k.init_flat()
    att_per_step = MCS_PER_STEP * L * L

    def step():
        k.run(MCS_PER_STEP)
        return k.measure()

    for _ in range(args.warmup):
        step()

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
        k.run(MCS_PER_STEP)
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

    # ---- end to end through the C ABI with HOST buffers (kpz_step_host, then kpz_pipeline_host), copies inside the
    # timed region ----
    # Local timings first; the reductions over ranks come after the try block, so that a rank whose pinned
    # allocation fails still takes part in them (a leg that failed on any rank is reported as unavailable).
    serial = (0.0, float("inf"))
    piped = (0.0, float("inf"))
    n_e2e = max(1, min(args.steps, 3))
    n_rounds = max(3, (args.steps + 1) // 2)      # at least 6 pipelined steps, so that fill and drain do not dominate
    e2e_err = None
    try:
        host = torch.empty(k.lattice_bytes, dtype=torch.uint8).pin_memory()
        k.export_packed(host)
        c = k.counters()
        h00 = np.array([c["h00"]], dtype=np.int64)
        mcs_now = c["mcs"]
        k.step_host(host, h00, mcs_now, MCS_PER_STEP)       # warm-up of the pinned path
        mcs_now += MCS_PER_STEP
        torch.cuda.synchronize()
        w0 = time.perf_counter()
        for _ in range(n_e2e):
            k.step_host(host, h00, mcs_now, MCS_PER_STEP)
            mcs_now += MCS_PER_STEP
        torch.cuda.synchronize()
        serial = (n_e2e * att_per_step, time.perf_counter() - w0)
        # the same steps through kpz_pipeline_host: two independent pinned host lattices (lanes) at different MCS
        # clocks, each batch = one kpz_step_host (H2D + 10 MCS + measurement + D2H), copies overlapped with kernels
        host2 = torch.empty(k.lattice_bytes, dtype=torch.uint8).pin_memory()
        host2.copy_(host)
        h00_l = np.array([[h00[0]], [h00[0]]], dtype=np.int64)
        k.step_host(host2, h00_l[1], mcs_now, MCS_PER_STEP)  # lane 1 runs one step ahead of lane 0
        clock = [mcs_now, mcs_now + MCS_PER_STEP]
        k.pipeline_host([host, host2], h00_l, clock, MCS_PER_STEP, 1)   # warm-up of the pipelined path
        clock = [t + MCS_PER_STEP for t in clock]
        torch.cuda.synchronize()
        w0 = time.perf_counter()
        k.pipeline_host([host, host2], h00_l, clock, MCS_PER_STEP, n_rounds)
        torch.cuda.synchronize()
        piped = (2 * n_rounds * att_per_step, time.perf_counter() - w0)
    except Exception as exc:   # e.g. not enough pinned host memory on the box
        e2e_err = str(exc)[:200]
    _, serial_s, serial_rate = shard.aggregate(serial[0], serial[1], device=dev)
    _, piped_s, piped_rate = shard.aggregate(piped[0], piped[1], device=dev)
    e2e = {"value": None, "unit": UNIT,
           "h2d_bytes_per_step": k.lattice_bytes + 8, "d2h_bytes_per_step": k.lattice_bytes + 3 * 8 + 32}
    if serial_s != float("inf"):
        e2e.update({"value": serial_rate / 1e9, "steps": n_e2e,
                    "api": "kpz_step_host (one pinned host lattice in/out, no overlap)"})
    if piped_s != float("inf"):
        e2e.update({"value": piped_rate / 1e9, "steps": 2 * n_rounds,
                    "api": "kpz_pipeline_host (2 pinned host lattices in/out, copies of step b-1 / b+1 overlap the "
                           "kernels of step b)",
                    "serial_value": serial_rate / 1e9, "serial_api": "kpz_step_host (one pinned host lattice, no overlap)"})
    if e2e_err is not None:
        e2e["error"] = e2e_err

    if rank != 0:
        return
    hbm_peak, sm_max, src = _peaks()
    # dominant kernel: kpz_update_kernel, 4 launches per MCS; duration from CUDA events around kpz_run
    n_upd_launch = args.steps * MCS_PER_STEP * 4
    upd_launch_ms = upd_ms / n_upd_launch
    upd_per_launch = L * L / 4
    sm_mhz = clocks.get("sm_mhz") or sm_max
    # ALU-pipe peak: 148 SMs x 4 schedulers x 16 lanes/clk at the maximum SM clock
    alu_peak_tops = 148 * 4 * 16 * sm_max * 1e6 / 1e12
    achieved_tops = upd_per_launch * ALG_ALU_OPS_PER_UPDATE / (upd_launch_ms * 1e-3) / 1e12
    general = not (w["p"] >= 1.0 and w["q"] <= 0.0)
    roofline = {"bound": "alu", "achieved": achieved_tops, "peak": alu_peak_tops, "unit": "Tops/s (ALU-pipe lane-ops)",
                "frac": achieved_tops / alu_peak_tops, "traffic": TRAFFIC_BYTES_PER_LAUNCH if L == (1 << 17) else None,
                "kernel": "kpz_update_kernel<%d,%d,%d>" % (T, 96 if T == 64 else 64, 1 if general else 0),
                "alg_alu_ops_per_update": ALG_ALU_OPS_PER_UPDATE, "alg_mul_ops_per_update": ALG_MUL_OPS_PER_UPDATE,
                "launch_ms": upd_launch_ms, "updates_per_launch": upd_per_launch,
                "peak_source": "148 SM x 4 schedulers x 16 ALU lanes/clk x clocks.max.sm from MEASURED_PEAKS.json "
                               "(%s); LOP3 issue interval of 2 clk per scheduler confirmed by microbenchmark (DESIGN.md)" % src,
                "hbm": {"achieved": upd_per_launch * ALG_BYTES_PER_UPDATE / (upd_launch_ms * 1e-3) / 1e9,
                        "peak": hbm_peak, "unit": "GB/s", "peak_source": src + " MEASURED_PEAKS.json",
                        "frac": upd_per_launch * ALG_BYTES_PER_UPDATE / (upd_launch_ms * 1e-3) / 1e9 / hbm_peak}}
    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        cpu = cpu_baseline_sample()
    out = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
           "ms_per_step": ms_total / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
           "dtype": "u32 bit-logic + Philox4x32 (int32/int64 sums)", "data": "synthetic",
           "config": {"workload": "config3: L=2^17 flat start, p=1 q=0, tile 64, seed 42" if L == (1 << 17) else "L=%d" % L,
                      "L": L, "tile": T, "p": w["p"], "q": w["q"], "seed": w["seed"], "mcs_per_step": MCS_PER_STEP,
                      "step": "kpz_run(%d) + kpz_measure" % MCS_PER_STEP,
                      "l2": "lattice %.1f GiB >> 126 MB L2, no flush needed" % (k.lattice_bytes / 2**30),
                      "parallelism": "independent lattice per GPU" if world > 1 else "1 GPU"},
           "update_only_gupds": args.steps * att_per_step / (upd_ms * 1e-3) / 1e9,
           "measure_ms": meas_ms / args.steps, "W2_last": float(last[2][0]),
           "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches), "roofline": roofline, "cpu_baseline": cpu}
    print(json.dumps(out))


def cpu_baseline_sample(threads=None, window=4096, n_mcs=3):
    """The oracle, as it stands, on the host cores: a window of the SAME workload (L=2^17 tile ids, offsets and
    Philox streams) advanced from the flat start.  Bounded to roughly 10-30 s of CPU work."""
    from oracle import Oracle
    w = WORKLOAD
    threads = threads or (os.cpu_count() or 1)
    o = Oracle(w["L"], w["p"], w["q"], w["tile"], w["seed"], window=(0, 0, window, window), threads=threads)
    o.init_flat()
    o.run(1)
    t0 = time.perf_counter()
    o.run(n_mcs)
    dt = time.perf_counter() - t0
    # tiles touching the window all execute their full T*T attempts (attempts leaving the window are skipped)
    att = n_mcs * window * window
    return {"value": att / dt / 1e9, "unit": UNIT, "cores": o.threads, "kind": "oracle",
            "sample": "window %dx%d of the L=2^17 config-3 lattice, %d MCS after 1 warm-up MCS, OpenMP over tiles"
                      % (window, window, n_mcs)}


def run_reference(args):
    """--impl reference: the oracle timed as the reference arm (rank 0 only)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    from oracle import Oracle
    w = WORKLOAD
    window = 2048
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
              "streams); measurement excluded (the windowed oracle has no global height walk)" % (MCS_PER_STEP, window, window))
    out = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": int(os.environ.get("WORLD_SIZE", "1")),
           "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3, "higher_is_better": True,
           "scaling": "weak", "vs_baseline": None, "dtype": "int8 slopes + Philox4x32", "data": "synthetic",
           "config": {"workload": "config3: L=2^17 flat start, p=1 q=0, tile 64, seed 42", "sample": sample},
           "cpu_baseline": {"value": value, "unit": UNIT, "cores": o.threads, "kind": "oracle", "sample": sample},
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
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--L", type=int, default=0, help="override the lattice size (debugging only)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--launcher-selftest", action="store_true", help="multi-rank launch + reductions only (gloo, no GPU)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "reference":
        run_reference(args)
        return
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        sys.exit(relaunch_under_torchrun(args))
    if args.launcher_selftest:
        launcher_selftest(args)
        return
    run_ours(args)


if __name__ == "__main__":
    main()
