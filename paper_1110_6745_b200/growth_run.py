"""Growth-regime harness (BASELINE configs 1-3, 5): one lattice from the flat state, W^2 and the mean height
at the sampling times of the configuration through `kpz_run_sampled`, the effective exponent
beta_eff(t) = (1/2) log2[(W^2(t) - 1/4) / (W^2(t/2) - 1/4)] (eq. 11, t/t' = 2 after subtracting W^2(0) = 1/4)
and the exact invariant sum_h(t) = L^2/2 + 2 (deposits - removals).  Everything heavy runs in the kernels.

    python -m paper_1110_6745_b200.growth_run --L 131072 --tile 64 --seed 42 --t-max 10000
    python -m paper_1110_6745_b200.growth_run --L 524288 --tile 64 --p 0.75 --q 0.25 --seed 3 --t-max 50 --every
"""
from __future__ import annotations

import argparse
import json
import math
import time

from . import analysis
from .binding import KPZ


T_MIC = 50      # "we disregarded the initial time region t < t_mic ~ 50"


def sampling_times(t_max):
    """{1,2,5}*10^n (reading R15 for config 3) merged with the powers of two that beta_eff needs."""
    ts = {m * 10 ** n for n in range(0, 12) for m in (1, 2, 5)} | {2 ** i for i in range(0, 40)}
    ts |= {25 * 10 ** n for n in range(0, 12)}       # the t/2 partners of 5 * 10^(n+1): every decade time has one
    return sorted(t for t in ts if t <= t_max)


def run(L, tile, p=1.0, q=0.0, seed=42, t_max=10000, device="cuda:0", every=False):
    k = KPZ(L, p, q, tile, seed, device=device)
    try:
        k.init_flat()
        times = list(range(1, t_max + 1)) if every else sampling_times(t_max)      # config 5: t = 1..50
        t0 = time.time()
        s1, s2, w2 = k.run_sampled(times)
        k.synchronize()
        wall = time.time() - t0
        c = {kk: int(v) for kk, v in k.counters().items()}
        rows = [{"t": t, "sum_h": int(s1[i, 0]), "sum_h2": int(s2[i, 0]), "W2": float(w2[i, 0]),
                 "mean_h": int(s1[i, 0]) / (L * L)} for i, t in enumerate(times)]
        w = {r["t"]: r["W2"] - 0.25 for r in rows}
        beta = [{"t": t, "beta_eff": 0.5 * math.log2(w[t] / w[t // 2])} for t in times
                if t >= 4 and (t & (t - 1)) == 0 and w[t // 2] > 0]
        # eq. 11 on every sampled pair (t, t/2), and the correction fit of eq. 12 beyond t_mic ~ 50
        slopes = [(t, b) for t, b in analysis.beta_eff(times, [r["W2"] for r in rows]) if t > T_MIC]
        fit = None
        if len(slopes) >= 4:
            f = analysis.fit_correction([t for t, _ in slopes], [b for _, b in slopes])
            fit = {"beta": f["asymptote"], "b1": f["amplitude"], "phi1": f["exponent"], "rss": f["rss"],
                   "correction_resolved": not f["at_bound"], "n_points": len(slopes), "t_min": slopes[0][0]}
        n = L * L
        return {"L": L, "tile": tile, "p": p, "q": q, "seed": seed, "samples": rows, "beta_eff": beta, "eq12_fit": fit,
                "counters": c,
                "invariant_sum_h": int(s1[-1, 0]) == n // 2 + 2 * (c["deposits"] - c["removals"]),
                "wall_s": wall, "gupds_incl_measurements": n * times[-1] / wall / 1e9}
    finally:
        k.close()


def main():
    ap = argparse.ArgumentParser(description=__doc__.splitlines()[0])
    ap.add_argument("--L", type=int, default=1 << 12)
    ap.add_argument("--tile", type=int, default=32)
    ap.add_argument("--p", type=float, default=1.0)
    ap.add_argument("--q", type=float, default=0.0)
    ap.add_argument("--seed", type=int, default=7)
    ap.add_argument("--t-max", type=int, default=1000)
    ap.add_argument("--every", action="store_true", help="sample after every MCS (config 5) instead of the log-spaced times")
    a = ap.parse_args()
    print(json.dumps(run(a.L, a.tile, a.p, a.q, a.seed, a.t_max, every=a.every)))


if __name__ == "__main__":
    main()
