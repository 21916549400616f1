#!/usr/bin/env python
"""Benchmark of the hot path: site-updates/ns of the zero-temperature
checkerboard sweep at L = 2048 on one B200, against the HBM / integer-ALU roofline, with
the CPU oracle timed beside it.

One "step" = one pass of the whole hot path over config 5 of BASELINE.json:
  ising3d_reset (a1: T = infinity start from Philox) -> ising3d_sweep(1000) (a2-a5: the
  throughput window, sweeps 0..999) -> ising3d_measure (a6-a9: N_up, A_mu(r) for r <= 1024,
  C(r), ell).
`value` counts the L^3 * 1000 site-updates of the step over the device time of the whole
step.  The lattice (1 GiB, ping-pong 2 GiB) is far larger than the 126 MB L2, so no L2
flush is needed between steps.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
N > 1 (torchrun): the path does not shard (one lattice per GPU) -> N
independent replicas with different seeds, no data-path collective ("replicas only").
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "site_updates_per_ns"
UNIT = "site-updates/ns"
ALGO_BYTES_PER_SITE_UPDATE = 0.375      # 3 N/8 bytes per sweep


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--L", type=int, default=2048)
    ap.add_argument("--sweeps", type=int, default=1000, help="sweeps per step (throughput window)")
    ap.add_argument("--variant", default="auto", choices=["auto", "generic", "fused", "fused2"])
    ap.add_argument("--ref-L", type=int, default=512, help="--impl reference: lattice size of the CPU sample")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-measure", action="store_true", help="step = reset + sweeps only")
    ap.add_argument("--no-late-windows", action="store_true",
                    help="skip the sweeps-only windows at t = 10^4 and 10^5 of the full run (about 40 s)")
    ap.add_argument("--profile-sweeps", type=int, default=0,
                    help="after each sweeps-only window run this many extra sweeps between cudaProfilerStart/Stop "
                         "(for `ncu --profile-from-start off`; outside every timed region)")
    ap.add_argument("--cpu-sizes", default="256x20,1024x2,2048x1",
                    help="extra oracle timings LxSWEEPS (SURVEY.md 8(d)); empty to skip")
    return ap.parse_args()


# ----------------------------------------------------------------------------- clocks
class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons during the timed region (NVML)."""

    def __init__(self, index: int, period_s: float = 0.05):
        super().__init__(daemon=True)
        self.index, self.period = index, period_s
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._stop_evt = threading.Event()
        self.ok = False
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
            self.ok = True
        except Exception:
            self.ok = False

    def run(self):
        if not self.ok:
            return
        nv = self.nv
        names = {
            getattr(nv, "nvmlClocksEventReasonHwSlowdown", 0x8): "hw_slowdown",
            getattr(nv, "nvmlClocksEventReasonHwThermalSlowdown", 0x40): "hw_thermal_slowdown",
            getattr(nv, "nvmlClocksEventReasonSwThermalSlowdown", 0x20): "sw_thermal_slowdown",
            getattr(nv, "nvmlClocksEventReasonSwPowerCap", 0x4): "sw_power_cap",
        }
        while not self._stop_evt.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                try:
                    r = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                except Exception:
                    r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for bit, name in names.items():
                    if r & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            self._stop_evt.wait(self.period)

    def stop(self):
        self._stop_evt.set()
        if self.is_alive():
            self.join(timeout=2)
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": []}
        s = sorted(self.samples)
        return {"sm_mhz": float(s[len(s) // 2]), "sm_max_mhz": float(self.max_mhz),
                "reasons": sorted(self.reasons), "samples": len(s)}


def physical_gpu_index(local_index: int) -> int:
    vis = os.environ.get("CUDA_VISIBLE_DEVICES")
    if vis:
        try:
            return int(vis.split(",")[local_index])
        except Exception:
            return local_index
    return local_index


# ----------------------------------------------------------------------------- CPU oracle legs
def oracle_rate(L: int, n_sweeps: int, seed: int):
    """The oracle as it stands, timed on this box's host cores: site-updates/ns."""
    from oracle import oracle as orc
    o = orc.Oracle(L, seed)                      # T = infinity start (not timed)
    t0 = time.perf_counter()
    o.sweep(n_sweeps)
    dt = time.perf_counter() - t0
    return (L ** 3) * n_sweeps / dt / 1e9, dt, orc.num_threads()


def oracle_sizes(spec: str):
    """the oracle timed at L=256 x 20, L=1024 x 2, L=2048 x 1 sweeps (the last one
    only with >= 16 GiB of free host RAM), plus its single-thread rate (L=256 x 4)."""
    from oracle import oracle as orc
    out = []
    try:
        import psutil
        free_gib = psutil.virtual_memory().available / 2 ** 30
    except Exception:
        free_gib = 0.0
    for item in [x for x in spec.split(",") if x]:
        L, n = (int(v) for v in item.split("x"))
        if L ** 3 / 2 ** 30 * 1.5 > free_gib or (L >= 2048 and free_gib < 16):
            out.append({"L": L, "sweeps": n, "skipped": "%.0f GiB of host RAM free" % free_gib})
            continue
        rate, dt, cores = oracle_rate(L, n, 4)
        out.append({"L": L, "sweeps": n, "value": rate, "unit": UNIT, "cores": cores, "seconds": dt})
    cores = orc.num_threads()
    orc.set_num_threads(1)
    try:
        rate, dt, _ = oracle_rate(256, 4, 4)
    finally:
        orc.set_num_threads(cores)
    single = {"L": 256, "sweeps": 4, "value": rate, "unit": UNIT, "cores": 1, "seconds": dt}
    return out, single


def run_reference(args):
    """--impl reference: the CPU oracle on the same metric; each step a bounded sample."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    from oracle import oracle as orc
    L, n_sw, seed = args.ref_L, 20, 4
    sample = ("L=%d (config-5 start rule: iid p=1/2 from seed %d), sweeps 0..%d per step; "
              "the oracle cannot hold 1000 sweeps of L=2048 in minutes" % (L, seed, n_sw - 1))
    for _ in range(args.warmup):
        oracle_rate(L, 2, seed)
    t_all, units = 0.0, 0
    for _ in range(args.steps):
        rate, dt, cores = oracle_rate(L, n_sw, seed)
        t_all += dt
        units += L ** 3 * n_sw
    value = units / t_all / 1e9
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT,
        "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": 1e3 * t_all / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "int8", "data": "synthetic",
        "config": {"workload": "config5_L2048 throughput window (bounded CPU sample)", "sample": sample},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))
    return 0


# ----------------------------------------------------------------------------- replicas only
# The path does not shard (one lattice per GPU): N ranks = N independent lattices,
# no data-path collective.  What the ranks share is the timing protocol below (covered on CPU by
# the world_size-2 gloo test in tests/test_bench_host.py).
def rank_seed(rank: int) -> int:
    """Config 5 uses seed 4; replica r of an N-GPU run uses seed 4 + r."""
    return 4 + rank


def max_over_ranks(ms: float, world: int, device) -> float:
    """Device time of the slowest rank (the contract's max over ranks)."""
    import torch
    import torch.distributed as dist
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_rate(world: int, n_sites: int, sweeps: int, steps: int, ms_max: float) -> float:
    """site-updates/ns of the whole job: every rank did n_sites * sweeps * steps proposals."""
    return world * n_sites * sweeps * steps / (ms_max * 1e6)


# ----------------------------------------------------------------------------- ours
def measured_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        d = json.load(open(p))
        return float(d["hbm_gbs"]), "MEASURED_PEAKS.json hbm_gbs (of measured)", d
    except Exception:
        return 6650.0, "B200_PROFILING.md fallback 6.65 TB/s (of fallback)", {}


def ncu_row(kernel: str, L: int, t0: int = 0):
    """The row of profiles/roofline_traffic.csv for (kernel, L, t0): numbers of one launch of that kernel
    from a committed `ncu --set full` capture -- dram__bytes_read.sum + dram__bytes_write.sum, and
    smsp__inst_executed.sum over the launch's warp-steps (stated in the capture's .md).  t0 = the sweep index the capture was taken near (the activity-driven
    kernel's traffic depends on how far the quench is).  None if not captured."""
    p = os.path.join(ROOT, "profiles", "roofline_traffic.csv")
    try:
        for line in open(p).read().splitlines()[1:]:
            k, l, t, b, inst, cap = line.split(",")
            if k == kernel and int(l) == L and int(t) == t0:
                return {"dram_bytes": float(b), "instr_per_step": float(inst) if inst else None, "capture": cap}
    except Exception:
        pass
    return None


def run_ours(args):
    import numpy as np
    import torch
    import torch.distributed as dist

    from paper_2305_12161_b200 import binding, build
    build.build()

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the CUDA path has no CPU fallback)")
    torch.cuda.set_device(local)
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    L, S = args.L, args.sweeps
    seed = rank_seed(rank)
    variant = {"auto": binding.VARIANT_AUTO, "generic": binding.VARIANT_GENERIC,
               "fused": binding.VARIANT_FUSED, "fused2": binding.VARIANT_FUSED2}[args.variant]
    sim = binding.Ising3D(L, [seed], variant=variant)
    N = L ** 3
    n_words = N // 32

    def step(timers=None):
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(4)] if timers is not None else None
        if ev: ev[0].record()
        sim.reset()
        if ev: ev[1].record()
        sim.sweep(S)
        if ev: ev[2].record()
        out = None if args.no_measure else sim.measure()
        if ev:
            ev[3].record()
            timers.append(ev)
        return out

    # ---------------- device-resident timing ----------------
    for _ in range(args.warmup):
        step()
    barrier()
    sampler = ClockSampler(physical_gpu_index(local))
    sampler.start()
    launches0 = sim.launch_count
    timers = []
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    last = None
    for _ in range(args.steps):
        last = step(timers)
    e1.record()
    barrier()
    clocks = sampler.stop()
    launches = sim.launch_count - launches0
    timed_kernel = sim.variant_name            # the sweep kernel of the timed steps
    total_ms = e0.elapsed_time(e1)
    init_ms = sum(t[0].elapsed_time(t[1]) for t in timers) / args.steps
    sweep_ms = sum(t[1].elapsed_time(t[2]) for t in timers) / args.steps
    meas_ms = sum(t[2].elapsed_time(t[3]) for t in timers) / args.steps
    total_ms_max = max_over_ranks(total_ms, world, "cuda")
    value = whole_job_rate(world, N, S, args.steps, total_ms_max)

    # ---------------- end to end through the C ABI with HOST buffers ----------------
    e2e = None
    if not args.no_e2e:
        sim.reset()
        host = torch.empty(n_words, dtype=torch.int32).pin_memory()
        sim.sync()
        binding._check(binding.load().ising3d_get_state(sim._h, host.data_ptr(), n_words, None))
        d2h_bytes = (1 + 3 * (L // 2 + 1)) * 8
        for _ in range(1):
            sim.set_state_ptr(host.data_ptr(), n_words, 0)
            sim.sweep(S)
            sim.measure()
        barrier()
        k_e2e = args.steps
        t0 = torch.cuda.Event(enable_timing=True)
        t1 = torch.cuda.Event(enable_timing=True)
        t0.record()
        for _ in range(k_e2e):
            sim.set_state_ptr(host.data_ptr(), n_words, 0)     # H2D of the step's input (pinned)
            sim.sweep(S)
            r = sim.measure()                                   # D2H of the step's result
        t1.record()
        barrier()
        ems = max_over_ranks(t0.elapsed_time(t1), world, "cuda")
        e2e = {"value": whole_job_rate(world, N, S, k_e2e, ems), "unit": UNIT,
               "h2d_bytes_per_step": n_words * 4, "d2h_bytes_per_step": d2h_bytes,
               "ms_per_step": ems / k_e2e,
               "note": "set_state(pinned host, 1 GiB at L=2048) + sweep + measure(host counts) per step"}

    def profile_sweeps(h, k):
        torch.cuda.synchronize()
        torch.cuda.profiler.start()
        h.sweep(k)
        torch.cuda.synchronize()
        torch.cuda.profiler.stop()

    if args.profile_sweeps and world == 1:
        profile_sweeps(sim, args.profile_sweeps)          # the state after the last step: t = S, still all awake

    # ---------------- sweeps-only windows of the full run ----------------
    # t = 0 is the headline window above; the lattice is then taken on to t = 10^4 and 10^5 (AUTO policy:
    # fused2, handing over to the activity-driven kernel once few groups can still change) and `wS` sweeps
    # are timed at each, with the fraction of 128-spin groups that hold a Delta E <= 0 site.
    windows = [{"t0": 0, "sweeps": S, "ms_per_sweep": sweep_ms / S, "kernel": timed_kernel,
                "site_updates_per_ns": N / (sweep_ms / S * 1e6), "awake_group_fraction": 1.0 if L >= 256 else None}]
    if not args.no_late_windows and world == 1:
        sim.reset()
        wS = 200
        for t0 in (10_000, 100_000):
            sim.sweep(t0 - sim.sweep_count)
            try:
                frac = sim.activity()[1]
            except Exception:
                frac = None
            sim.sync()
            w0, w1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            w0.record()
            sim.sweep(wS)
            w1.record()
            torch.cuda.synchronize()
            ms = w0.elapsed_time(w1) / wS
            windows.append({"t0": t0, "sweeps": wS, "ms_per_sweep": ms, "kernel": sim.variant_name,
                            "site_updates_per_ns": N / (ms * 1e6), "awake_group_fraction": frac})
            if args.profile_sweeps:
                profile_sweeps(sim, args.profile_sweeps)
        # per window: the bytes its kernel moved per sweep in the committed ncu capture taken at that t0
        # (profiles/roofline_traffic.csv), and the fraction of the copy bandwidth that is at this window's speed
        peak_w = measured_peak()[0]
        for w in windows:
            kname, per_sweep = {"fused2": ("fused2_sweep_kernel", 1), "active": ("active_halfsweep_kernel", 2)}.get(
                w["kernel"], (None, 0))
            row = ncu_row(kname, L, w["t0"]) if kname else None
            w["traffic_bytes_per_sweep"] = row["dram_bytes"] * per_sweep if row else None
            w["frac_on_bytes_moved"] = (row["dram_bytes"] * per_sweep / (w["ms_per_sweep"] * 1e-3) / 1e9 / peak_w
                                        if row else None)
            w["traffic_capture"] = row["capture"] if row else None

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return 0

    # ---------------- roofline of the dominant kernel (the sweep kernel) ----------------
    peak, peak_src, peaks = measured_peak()
    kernel = {"fused": "fused_sweep_kernel", "fused2": "fused2_sweep_kernel"}.get(timed_kernel, "halfsweep_generic_kernel")
    launches_per_sweep = {"fused": 1, "fused2": 1}.get(timed_kernel, 2)
    avg_launch_ms = sweep_ms / (S * launches_per_sweep)
    algo_bytes_per_launch = ALGO_BYTES_PER_SITE_UPDATE * N / launches_per_sweep
    achieved = algo_bytes_per_launch / (avg_launch_ms * 1e-3) / 1e9
    sm_mhz = clocks.get("sm_mhz") or 1965.0
    # Integer issue roofline: the 16-lane integer instructions (LOP3, SHF, IMAD.WIDE)
    # issue at 0.5 warp-instructions/clk/SMSP = 64 thread-instructions/clk/SM whatever their pipe
    # (profiles/r1c, r1h); the rule + Philox need 51 + 18 = 69 of them per 128 sites and colour;
    # 148 SMs at the SM clock seen during the run
    alu_ops_per_site = 69.0 / 128.0
    alu_bound = 148 * 64 * sm_mhz * 1e6 / alu_ops_per_site / 1e9
    hbm_bound = peak / ALGO_BYTES_PER_SITE_UPDATE
    sweep_rate = N * S / (sweep_ms * 1e6)
    row = ncu_row(kernel, L)
    traffic = row["dram_bytes"] if row else None
    # as compiled: warp-instructions per thread-step of 4 groups = 512 sites = smsp__inst_executed.sum of the
    # committed capture over the launch's warp-steps (profiles/roofline_traffic.csv, derived in the capture's
    # .md; 337.9 in r2); 60 of 64 tile rows and 256 of 260 planes stored
    compiled_instr = row["instr_per_step"] if (row and row["instr_per_step"]) else 337.9
    compiled_per_site = compiled_instr / 512.0 * (64.0 / 60.0) * (260.0 / 256.0)
    compiled_bound = 148 * 64 * sm_mhz * 1e6 / compiled_per_site / 1e9
    roofline = {
        "bound": "hbm", "kernel": kernel, "achieved": achieved, "peak": peak, "unit": "GB/s",
        "frac": achieved / peak, "traffic": traffic,
        "frac_algorithmic_3N8": achieved / peak,      # the same number under the name of its byte model
        # what binds the kernel is the issue rate of its integer instructions, not HBM:
        "binding_limit": "issue",
        "issue_frac": sweep_rate / alu_bound,
        "issue_frac_as_compiled": sweep_rate / compiled_bound if kernel == "fused2_sweep_kernel" else None,
        "issue_model": {"thread_instr_per_clk_per_sm": 64, "sms": 148, "sm_mhz": sm_mhz,
                        "min_instr_per_128_sites_per_colour": 69,
                        "compiled_warp_instr_per_thread_step_of_512_sites": compiled_instr,
                        "source": "microbench/pipe_rates.cu, microbench/sweep_ceiling.cu; profiles/r1c, r1h, r1i"},
        # on the bytes the kernel really moves (ncu dram__bytes_read + write per launch)
        "frac_on_bytes_moved": (traffic / (avg_launch_ms * 1e-3) / 1e9) / peak if traffic else None,
        "algorithmic_bytes_per_launch": algo_bytes_per_launch, "avg_launch_ms": avg_launch_ms,
        "peak_source": peak_src,
        "sweep_only_site_updates_per_ns": sweep_rate,
        "hbm_bound_site_updates_per_ns": hbm_bound,
        "alu_bound_site_updates_per_ns": alu_bound,
        "frac_of_min_roofline": sweep_rate / min(hbm_bound, alu_bound),
        # the stricter view: the N/4 bytes per sweep a fused black+white pass cannot avoid moving
        "frac_on_fused_floor_bytes": (0.25 * N / launches_per_sweep / (avg_launch_ms * 1e-3) / 1e9) / peak
        if launches_per_sweep <= 1 else None,
        "note": "algorithmic bytes = 3N/8 per sweep (two half-sweeps each read both colours' "
                "share and write one); the fused kernel moves ~N/4 + halo, so frac can pass 1",
    }

    cpu = None
    if not args.no_cpu_baseline and world == 1:
        Lc, nsw = 1024, 16                          # ~1.7e10 site-updates: 10-30 s on 8-16 cores
        rate, dt, cores = oracle_rate(Lc, nsw, 4)
        cpu = {"value": rate, "unit": UNIT, "cores": cores, "kind": "oracle",
               "sample": "L=%d, iid p=1/2 start from seed 4, sweeps 0..%d (%.1f s of CPU work); "
                         "same rule and RNG as config 5, smaller box" % (Lc, nsw - 1, dt)}
        if args.cpu_sizes:
            cpu["other_sizes"], cpu["single_thread"] = oracle_sizes(args.cpu_sizes)

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": total_ms_max / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "u32", "data": "synthetic",
        "config": {"workload": "config5_L2048: L=%d periodic cube, iid p=1/2 start from seed %d, "
                               "step = reset + %d zero-T checkerboard sweeps + measure(r<=%d)" % (
                                   L, seed, S, L // 2),
                   "L": L, "sweeps_per_step": S, "replicas_per_gpu": 1, "kernel": timed_kernel,
                   "l2": "inputs larger than L2 (%.0f MiB packed lattice, ping-pong; L2 126 MB)" % (
                       N / 8 / 2 ** 20),
                   "parallelism": "replicas only" if world > 1 else "single GPU"},
        "breakdown_ms": {"init": init_ms, "sweeps": sweep_ms, "measure": meas_ms},
        "windows": windows,
        "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches),
        "roofline": roofline, "cpu_baseline": cpu,
        "result": None if last is None else {"sweep": last["sweep"], "n_up": int(last["n_up"][0]),
                                             "n_broken": int(last["n_broken"][0]),
                                             "ell": float(last["ell"][0])},
    }
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


def main():
    args = parse()
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
