#!/usr/bin/env python
"""Run the five BASELINE.json workloads through the C-ABI library and report, per workload,
the trajectory of the measured quantities and the throughput in site-updates/ns.

  python -m paper_2305_12161_b200.run_configs [--configs config1_L64,config5_L2048]
         [--max-sweeps N] [--radial] [--variant V] [--cycle 01|mixed|dcb|dcb_mixed] [--temperature T]
         [--out results.jsonl]

Per workload: ising3d_init(_batch) from the workload's seeds, then for
each measurement time T(n) (S12): ising3d_sweep(dt), ising3d_measure().  Reported:
  * one JSON line per checkpoint (sweep, m, n_broken, ell, ms of the sweeps since the last one),
  * one summary line: site-updates/ns over the sweeps only and over sweeps + measurements,
    both from CUDA events on the handle's stream.
Only argument marshalling and printing happen here; every step of the path runs in the kernels
of libising3d.so.  The ensemble lines of config 3 (D9: mean over replicas in ascending seed
order of C_rep(r) and ell_rep, NaNs skipped and counted; ell of the mean C) are host fp64
post-processing of the returned per-replica values.
"""
from __future__ import annotations

import argparse
import json
import sys

import numpy as np

from . import inputs


def ell_from_C(C: np.ndarray, c: float = 0.5) -> float:
    """First crossing of C(r) with c, linear interpolation (D9)."""
    for r in range(len(C) - 1):
        if C[r] >= c and C[r + 1] < c:
            return r + (C[r] - c) / (C[r] - C[r + 1])
    return float("nan")


def run_workload(name: str, max_sweeps: int | None, emit, variant: str = "auto", radial: bool = False,
                 cycle: str = "01", temperature: float = 0.0):
    import torch
    from . import binding

    w = inputs.WORKLOADS[name]
    L, seeds = w["L"], w["seeds"]
    n_total = w["sweeps"] if max_sweeps is None else min(w["sweeps"], max_sweeps)
    times = [t for t in w["times"] if t <= n_total]
    if not times or times[-1] != n_total:
        times.append(n_total)
    sim = binding.Ising3D(L, seeds, variant={"auto": binding.VARIANT_AUTO, "generic": binding.VARIANT_GENERIC,
                                             "fused": binding.VARIANT_FUSED, "fused2": binding.VARIANT_FUSED2,
                                             "fused3": binding.VARIANT_FUSED3, "active": binding.VARIANT_ACTIVE,
                                             "resident": binding.VARIANT_RESIDENT}[variant])
    if cycle != "01":
        sim.set_cycle({"mixed": binding.CYCLE_MIXED, "dcb": binding.CYCLE_DOUBLE_CB,
                       "dcb_mixed": binding.CYCLE_DOUBLE_CB_MIXED}[cycle])
    if temperature > 0.0:
        sim.set_temperature(temperature)
    N = L ** 3 * len(seeds)
    ev = lambda: torch.cuda.Event(enable_timing=True)
    t_sweeps = t_meas = t_rad = 0.0
    t = 0
    e_all0 = ev(); e_all0.record()
    for cp in times:
        e0, e1, e2 = ev(), ev(), ev()
        e0.record()
        sim.sweep(cp - t)
        e1.record()
        m = sim.measure()
        e2.record()
        torch.cuda.synchronize()
        ms_s, ms_m = e0.elapsed_time(e1), e1.elapsed_time(e2)
        t_sweeps += ms_s
        t_meas += ms_m
        n_up = m["n_up"].astype(np.float64)
        mag = (2.0 * n_up - L ** 3) / L ** 3
        line = {"workload": name, "sweep": cp, "ms_sweeps": ms_s, "ms_measure": ms_m,
                "m": float(mag.mean()), "n_broken_mean": float(m["n_broken"].mean()),
                "ell_mean": float(np.nanmean(m["ell"])) if np.isfinite(m["ell"]).any() else None,
                "ell_nan": int(np.isnan(m["ell"]).sum())}
        if len(seeds) > 1:
            line["ell_of_mean_C"] = ell_from_C(m["C"].mean(axis=0))
        line["kernel"] = sim.variant_name
        if L >= 256 and (L & (L - 1)) == 0:
            line["awake_group_fraction"] = sim.activity()[1]     # groups holding a Delta E <= 0 site
        if radial:      # the paper's estimator (eq. 7 + radial average), outside the timed totals
            e3, e4 = ev(), ev()
            e3.record()
            r = sim.measure_radial()
            e4.record()
            torch.cuda.synchronize()
            line["ell_radial_mean"] = float(np.nanmean(r["ell"])) if np.isfinite(r["ell"]).any() else None
            line["ms_measure_radial"] = e3.elapsed_time(e4)
            t_rad += line["ms_measure_radial"]
        emit(line)
        t = cp
    e_all1 = ev(); e_all1.record(); torch.cuda.synchronize()
    total_ms = e_all0.elapsed_time(e_all1) - t_rad
    summary = {"workload": name, "summary": True, "L": L, "replicas": len(seeds), "sweeps": n_total,
               "checkpoints": len(times), "kernel": sim.variant_name, "cluster_size": sim.cluster_size,
               "site_updates_per_ns_sweeps": N * n_total / (t_sweeps * 1e6),
               "site_updates_per_ns_total": N * n_total / (total_ms * 1e6),
               "ms_sweeps": t_sweeps, "ms_measure": t_meas, "ms_total": total_ms,
               "ms_per_sweep": t_sweeps / n_total, "ms_per_measure": t_meas / len(times),
               "gpu_launches": sim.launch_count}
    emit(summary)
    sim.free()
    return summary


def main(argv=None):
    ap = argparse.ArgumentParser()
    ap.add_argument("--configs", default=",".join(inputs.WORKLOADS))
    ap.add_argument("--max-sweeps", type=int, default=None,
                    help="truncate each workload to this many sweeps (default: the full run)")
    ap.add_argument("--variant", default="auto",
                    choices=["auto", "generic", "fused", "fused2", "fused3", "resident", "active"],
                    help="sweep kernel (default: the library's choice)")
    ap.add_argument("--cycle", default="01", choices=["01", "mixed", "dcb", "dcb_mixed"],
                    help="update order (ising3d_set_cycle)")
    ap.add_argument("--temperature", type=float, default=0.0, help="T > 0: Glauber dynamics, eq. (5)")
    ap.add_argument("--radial", action="store_true",
                    help="also call ising3d_measure_radial (FFT + radial average) at every checkpoint")
    ap.add_argument("--out", default=None, help="also append the JSON lines to this file")
    args = ap.parse_args(argv)
    from . import build
    build.build()
    fh = open(args.out, "a") if args.out else None

    def emit(line):
        s = json.dumps(line)
        print(s, flush=True)
        if fh:
            fh.write(s + "\n")
            fh.flush()

    for name in args.configs.split(","):
        run_workload(name.strip(), args.max_sweeps, emit, args.variant, args.radial, args.cycle, args.temperature)
    return 0


if __name__ == "__main__":
    sys.exit(main())
