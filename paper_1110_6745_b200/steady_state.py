"""Steady-state ensemble harness (BASELINE config 4): R independent replicas of an L x L lattice
are advanced together by the CUDA library; per-replica W^2 is sampled in the second half of the run and reduced to
the cumulants kappa_1..kappa_4 (eq. 18), the width distribution Psi_L(x) and the replica-averaged power spectrum S(k)
(eq. 15-16).  Everything heavy runs in the kernels; this file only drives them and applies analysis.py.

    python -m paper_1110_6745_b200.steady_state --L 128 --replicas 1024 [--t-end N] [--samples 100] [--tile 16]
                                                  [--sub-sweeps K] [--spectrum-replicas 8] [--peaks]
    python -m paper_1110_6745_b200.steady_state --sizes 128,256,512,1024 --replicas 1024,256,256,256
        (finite-size scaling over several sizes: alpha_eff(L) of eq. 13, the power laws of eq. 19 for kappa_1..kappa_4)
    python -m paper_1110_6745_b200.steady_state --pool batch1.json batch2.json ... [--fss-with runs.json]
        (no GPU: pools the cumulants of several independent batches of ONE size -- outputs of this program, e.g. config
        4's 256 replicas of L = 2048 run as four batches of 64 under different Philox keys -- and, with --fss-with, adds
        the pooled size to the runs of a --sizes output and repeats the finite-size scaling)
"""
from __future__ import annotations

import argparse
import json

import numpy as np

from . import analysis
from .binding import KPZ


def run(L, replicas, tile=16, p=1.0, q=0.0, seed=4, t_end=None, samples=100, spectrum_replicas=8, device="cuda:0",
        sub_sweeps=1):
    t_end = analysis.steady_state_t_end(L) if t_end is None else int(t_end)
    k = KPZ(L, p, q, tile, seed, n_replicas=replicas, device=device)
    try:
        k.init_flat()
        if sub_sweeps > 1:
            k.set_sub_sweeps(sub_sweeps)      # schedule S6
        t_half = t_end // 2
        k.run(t_half)
        step = max(1, (t_end - t_half) // max(1, samples))
        w2 = []
        t = t_half
        while t + step <= t_end:
            k.run(step)
            t += step
            w2.append(k.measure()[2].copy())
        if t < t_end:
            k.run(t_end - t)
        w2 = np.array(w2) if w2 else k.measure()[2][None, :]
        out = {"L": L, "replicas": replicas, "tile": tile, "p": p, "q": q, "seed": seed, "t_end": t_end,
               "sub_sweeps": sub_sweeps,
               "n_samples": int(w2.size), "cumulants": list(analysis.cumulants(w2)),
               "W2_final_mean": float(k.measure()[2].mean())}
        x, psi = analysis.width_distribution(w2)
        out["psi_x"], out["psi"] = x.tolist(), psi.tolist()
        if L & (L - 1) == 0 and spectrum_replicas > 0:
            n = min(replicas, spectrum_replicas)
            S = np.mean([k.power_spectrum(r)[0] for r in range(n)], axis=0)
            out["spectrum_replicas"] = n
            out["S_k"] = S.tolist()
            # the schedule's imprint on S(k) (R18): the affected modes, each beside its neighbourhood
            out["schedule_peaks"] = schedule_peaks(S, L, tile) if L >= 8 * tile else []
        return out
    finally:
        k.close()


def finite_size_scaling(results):
    """Finite-size scaling of a list of run() outputs of different L: alpha_eff(L) of eq. (13)
    between sizes L and L/2 from kappa_1 = <W^2> -- with the intrinsic 1/4 of the zig-zag start subtracted and
    without --, the power-law exponents of eq. (19) as alpha_n = s_n / (2 n) for the cumulants that are positive at
    every size, and the fit of eq. (14) when at least four local slopes exist (three parameters)."""
    results = sorted(results, key=lambda r: r["L"])
    sizes = [r["L"] for r in results]
    k1 = [r["cumulants"][0] for r in results]
    out = {"sizes": sizes, "W2_mean": k1,
           "alpha_eff": [{"L": L, "alpha_eff": a} for L, a in analysis.alpha_eff(sizes, k1)],
           "alpha_eff_raw": [{"L": L, "alpha_eff": a} for L, a in analysis.alpha_eff(sizes, k1, intrinsic=0.0)],
           "cumulant_power_laws": []}
    for n in range(1, 5):
        kn = [r["cumulants"][n - 1] for r in results]
        if len(sizes) >= 2 and all(v > 0 for v in kn):
            c, sl = analysis.fit_power_law(sizes, kn)
            out["cumulant_power_laws"].append({"n": n, "prefactor": c, "exponent": sl, "alpha_n": sl / (2 * n)})
    if len(out["alpha_eff"]) >= 4:
        f = analysis.fit_correction([a["L"] for a in out["alpha_eff"]], [a["alpha_eff"] for a in out["alpha_eff"]])
        out["eq14_fit"] = {"alpha": f["asymptote"], "a1": f["amplitude"], "omega1": f["exponent"], "rss": f["rss"],
                           "correction_resolved": not f["at_bound"]}
        vals = [a["alpha_eff"] for a in out["alpha_eff"]]
        out["alpha_eff_mean"] = float(np.mean(vals))
        out["alpha_eff_spread"] = float(np.std(vals, ddof=1))
    return out


def pool_batches(batches):
    """Several run() outputs (or {"L", "replicas", "n_samples", "cumulants"} records) of ONE lattice size -> one record
    with the cumulants of the union of their samples (analysis.pool_cumulants)."""
    sizes = {b["L"] for b in batches}
    if len(sizes) != 1:
        raise ValueError("batches of different lattice sizes cannot be pooled")
    return {"L": sizes.pop(), "replicas": sum(b["replicas"] for b in batches),
            "n_samples": sum(b["n_samples"] for b in batches), "seeds": [b.get("seed") for b in batches],
            "t_end": batches[0].get("t_end"),
            "cumulants": list(analysis.pool_cumulants([(b["n_samples"], b["cumulants"]) for b in batches]))}


def schedule_peaks(S, L, tile):
    """S(k) at the mode numbers where the four-colour schedule leaves its imprint (odd multiples of L / (2 tile), and
    L / 4), each beside the median of its 12 neighbouring modes (profiles/r01_config4_steady.md, addendum)."""
    S = np.asarray(S)
    n0 = L // (2 * tile)
    modes = [n0 * j for j in range(5, tile, 2) if 6 <= n0 * j < len(S) - 6] + [L // 4]
    return [{"n": n, "S": float(S[n]), "background": float(np.median(np.r_[S[n - 6:n], S[n + 1:n + 7]]))}
            for n in modes]


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--L", type=int, default=128)
    ap.add_argument("--replicas", type=str, default="1024", help="replicas (one number, or one per entry of --sizes)")
    ap.add_argument("--tile", type=int, default=16)
    ap.add_argument("--p", type=float, default=1.0)
    ap.add_argument("--q", type=float, default=0.0)
    ap.add_argument("--seed", type=int, default=4)
    ap.add_argument("--t-end", type=int, default=None, help="default: 20 L^1.61 (BASELINE config 4)")
    ap.add_argument("--samples", type=int, default=100)
    ap.add_argument("--sub-sweeps", type=int, default=1, help="K sub-sweeps per MCS (schedule S6)")
    ap.add_argument("--spectrum-replicas", type=int, default=8)
    ap.add_argument("--peaks", action="store_true", help="print only S(k) at the schedule's peak modes")
    ap.add_argument("--sizes", type=str, default=None, help="comma-separated L: run every size, then finite_size_scaling")
    ap.add_argument("--pool", nargs="+", default=None, help="JSON outputs of batches of one size: pool them (no GPU)")
    ap.add_argument("--fss-with", type=str, default=None, help="with --pool: a --sizes output whose runs join the pooled size")
    args = ap.parse_args()
    if args.pool:
        pooled = pool_batches([json.load(open(f)) for f in args.pool])
        out = {"pooled": pooled}
        if args.fss_with:
            runs = [r for r in json.load(open(args.fss_with))["runs"] if r["L"] != pooled["L"]] + [pooled]
            out["fss"] = finite_size_scaling(runs)
        print(json.dumps(out))
        return
    if args.sizes:
        sizes = [int(v) for v in args.sizes.split(",")]
        reps = [int(v) for v in str(args.replicas).split(",")] if isinstance(args.replicas, str) else [args.replicas]
        reps = reps * len(sizes) if len(reps) == 1 else reps
        res = []
        for L, R in zip(sizes, reps):
            r = run(L, R, args.tile, args.p, args.q, args.seed, args.t_end, args.samples, spectrum_replicas=0,
                    sub_sweeps=args.sub_sweeps)
            res.append({k: r[k] for k in ("L", "replicas", "tile", "t_end", "n_samples", "cumulants", "W2_final_mean")})
        print(json.dumps({"runs": res, "fss": finite_size_scaling(res)}))
        return
    args.replicas = int(args.replicas)
    out = run(args.L, args.replicas, args.tile, args.p, args.q, args.seed, args.t_end, args.samples,
              spectrum_replicas=args.spectrum_replicas, sub_sweeps=args.sub_sweeps)
    if args.peaks:
        out = {"L": out["L"], "tile": out["tile"], "replicas": out["spectrum_replicas"], "t_end": out["t_end"],
               "sub_sweeps": out["sub_sweeps"], "peaks": schedule_peaks(out["S_k"], out["L"], out["tile"])}
    print(json.dumps(out))


if __name__ == "__main__":
    main()
