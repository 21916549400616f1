"""Ensemble of independent quenches in batches: the L=256 x 1000-run domain-size
histogram of Supp. Fig. 3 (01-cycle checkerboard, rescaled time 4000 MCS = 4000/1.75 =
2286 sweeps by Table I, mean domain size 19.9), with the paper's estimator (FFT + radial average,
`ising3d_measure_radial`) and the axis-averaged one side by side.

    python -m paper_2305_12161_b200.ensemble                      # 1000 x L=256, 2286 sweeps
    python -m paper_2305_12161_b200.ensemble --replicas 64 --L 128 --sweeps 1000

Prints one JSON line.  Every replica is an independent lattice of one batch handle (one launch sweeps
the whole batch); seeds are first_seed, first_seed+1, ...
"""
from __future__ import annotations

import argparse
import json
import sys
import time

import numpy as np


def main(argv=None):
    ap = argparse.ArgumentParser()
    ap.add_argument("--L", type=int, default=256)
    ap.add_argument("--replicas", type=int, default=1000)
    ap.add_argument("--sweeps", type=int, default=2286)
    ap.add_argument("--chunk", type=int, default=250, help="replicas per batch handle")
    ap.add_argument("--first-seed", type=int, default=5000)
    args = ap.parse_args(argv)
    from . import binding, build
    build.build()
    N = args.L ** 3
    ell_r, ell_a, m = [], [], []
    t0 = time.perf_counter()
    for lo in range(0, args.replicas, args.chunk):
        seeds = list(range(args.first_seed + lo, args.first_seed + min(lo + args.chunk, args.replicas)))
        sim = binding.Ising3D(args.L, seeds)
        sim.sweep(args.sweeps)
        r, a = sim.measure_radial(), sim.measure()
        ell_r += [float(x) for x in r["ell"]]
        ell_a += [float(x) for x in a["ell"]]
        m += [float(2.0 * int(u) - N) / N for u in a["n_up"]]
        sim.free()
    wall = time.perf_counter() - t0
    er, ea = np.array(ell_r), np.array(ell_a)
    ok = ~np.isnan(er)
    lo_edge = np.floor(er[ok].min()) if ok.any() else 0.0
    hi_edge = np.floor(er[ok].max()) + 1.0 if ok.any() else 1.0
    hist, edges = np.histogram(er[ok], bins=np.arange(lo_edge, hi_edge + 0.5, 1.0))
    line = {
        "L": args.L, "replicas": args.replicas, "sweeps": args.sweeps, "seeds": [args.first_seed, args.first_seed + args.replicas - 1],
        "ell_radial_mean": float(np.nanmean(er)), "ell_radial_sd": float(np.nanstd(er, ddof=1)),
        "ell_radial_sem": float(np.nanstd(er, ddof=1) / np.sqrt(ok.sum())),
        "ell_axis_mean": float(np.nanmean(ea)), "ell_axis_sd": float(np.nanstd(ea, ddof=1)),
        "ell_nan": int((~ok).sum()), "abs_m_mean": float(np.mean(np.abs(m))),
        "hist_radial": {"left_edges": [float(e) for e in edges[:-1]], "counts": [int(c) for c in hist]},
        "site_updates": float(N) * args.replicas * args.sweeps, "wall_s": wall,
    }
    print(json.dumps(line))
    return 0


if __name__ == "__main__":
    sys.exit(main())
