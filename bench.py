#!/usr/bin/env python
"""bench.py — throughput of the Arnold-web hot path on B200 (metric: BASELINE.json).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--scaling weak|strong]
                    [--config 3] [--order 4] [--horizon STEPS] [--no-e2e] [--no-cpu-baseline]

One "step" = one pass of the whole hot path over one batch of synthetic input:
aw_init_shell (a1) -> aw_integrate over the config's full horizon (a2 + a3 + a4, chained launches)
-> aw_indicator FLI image (a5) -> aw_density histogram (a6) [-> NCCL all-reduce of the histogram and gather of the
image strips, N > 1].  Workload at N = 1: BASELINE.json configs[3] (2048 x 2048 scan, eps = 3e-2, dt = 0.005, 2e5
steps, FLI), the configuration the metric's target is quoted on.

N > 1: one rank per GPU.  Launched by torchrun (RANK / WORLD_SIZE in the environment) or, if `--gpus N` is given
without them, bench.py starts the N ranks itself (torch.distributed.run --standalone); it refuses to run when fewer
than N devices are visible or when WORLD_SIZE and --gpus disagree.  `--scaling weak` (default): every rank scans
its own 2048 x 2048 block of a 2048 x (2048 N) image of the same action square; `--scaling strong`: the 2048 x 2048
image is split by rows.  Either way a rank holds a slice [k0, k0 + n) of ONE seeded ensemble (aw_grid.k0), so the
sharded result is bit-identical to the single-GPU one; no data-path collective except the histogram sum and the
image gather.

value   = live trajectory-steps / s, whole job, inputs resident in HBM (device-timed, max over ranks)
e2e     = same metric through aw_map_host: host (pinned) state in, image + histogram out, copies timed
roofline= fp64 ALU bound: min(nominal 498 flop / traj-step for order 4 with tangent; fp64
          flops the step loop's SASS executes) per integrate launch / its CUDA-event duration, against
          148 SM x 64 DFMA/clk x 2 x 1.965 GHz
cpu_baseline = the oracle (oracle/aw_oracle.cpp, as it stands) on all host cores and on one core, bounded sample
--impl reference = the oracle as the reference arm (rank 0 only).
"""
import argparse
import csv
import json
import math
import os
import socket
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
for p in (ROOT, os.path.join(ROOT, "tests")):          # tests/: aw_probe (measurement support: DFMA peak probe)
    if p not in sys.path:
        sys.path.insert(0, p)

METRIC = "trajectory-steps/s (fp64, with tangent map)"
UNIT = "traj-steps/s"
HIST_SCRATCH = lambda g: (g * g * 4 + 7) // 8 * 8 + 8   # AW_HIST_SCRATCH_BYTES (include/aw.h)


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=2)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--scaling", default="weak", choices=["weak", "strong"])
    ap.add_argument("--config", type=int, default=3)
    ap.add_argument("--order", type=int, default=0, help="0 = the config's (4); 6 = the paper's scheme")
    ap.add_argument("--horizon", type=int, default=0, help="integration steps per pass (0 = the config's)")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cpu-seconds", type=float, default=15.0)
    ap.add_argument("--density-bench", action="store_true",
                    help="only time aw_density / aw_init_shell / aw_indicator alone (HBM-bound kernels, DESIGN.md 6.3-6.4)")
    ap.add_argument("--dfma-shapes", action="store_true",
                    help="only run the fp64 operand-shape probe (tests/aw_probe.h) and print its JSON line")
    return ap.parse_args()


# ------------------------------------------------------------------------------------------- clocks

class ClockSampler:
    """Samples SM clock and throttle reasons with NVML while the timed region runs."""

    def __init__(self, index):
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._stop = threading.Event()
        self._thread = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self.nv = None

    def _run(self):
        nv = self.nv
        names = {"hw_slowdown": nv.nvmlClocksThrottleReasonHwSlowdown,
                 "hw_thermal_slowdown": nv.nvmlClocksThrottleReasonHwThermalSlowdown,
                 "sw_thermal_slowdown": nv.nvmlClocksThrottleReasonSwThermalSlowdown,
                 "sw_power_cap": nv.nvmlClocksThrottleReasonSwPowerCap}
        while not self._stop.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for k, bit in names.items():
                    if r & bit:
                        self.reasons.add(k)
            except Exception:
                pass
            self._stop.wait(0.2)

    def start(self):
        if self.nv:
            self._thread = threading.Thread(target=self._run, daemon=True)
            self._thread.start()

    def stop(self):
        self._stop.set()
        if self._thread:
            self._thread.join()
        s = sorted(self.samples)
        return {"sm_mhz": s[len(s) // 2] if s else None, "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(s)}


# ------------------------------------------------------------------------------------------- workload description

def workload_config(cfg, order, tangent, horizon, world, scaling, live_all):
    """The `config` object of the JSON line; both arms print the same keys and, for the same flags, the same values."""
    from paper_1107_4107_b200 import parallel
    gx, gy_total, _, n_rank = parallel.slice_of(cfg["gx"], cfg["gy"], world, 0, scaling)
    dens_mode = cfg.get("density_mode", 0)
    out = {"workload": cfg["name"], "grid": [gx, gy_total],
           "trajectories_per_gpu": n_rank if scaling == "weak" else (gx * gy_total + world - 1) // world,
           "live_trajectories": live_all, "eps": cfg["eps"], "E": cfg["E"], "dt": cfg["dt"],
           "steps_per_pass": horizon, "stride": cfg["stride"], "order": order, "tangent": tangent,
           "outputs": ("FLI image fp64" if tangent else "max|dH| image fp64") + " + 1024x1024 uint32 density"
                      + (" of the projected averaged velocity (mode %d)" % dens_mode if dens_mode else ""),
           "parallelism": "dp%d (%s scaling: %s)" % (world, scaling, "one gx x gy block of the image per rank"
                                                     if scaling == "weak" else "image rows split over the ranks"),
           "l2": "state planes %.0f MB per rank per pass > 126 MB L2 (no flush needed)"
                 % (n_rank * (16 * 8 + 12 + 1) / 1e6) if n_rank * 141 > 126e6 else
                 "state planes %.1f MB per rank; a 256 MB buffer is written between timed passes to flush L2"
                 % (n_rank * (16 * 8 + 12 + 1) / 1e6)}
    if cfg.get("survive"):
        out["survivors"] = ("survivor filter on the launch square (P:99): live_trajectories counts the survivors at the end; "
                            "trajectories that left stopped being integrated, so `value` undercounts the work done")
    if cfg.get("window"):
        out["window_steps"] = cfg["window"]
    if cfg.get("density_every"):
        out["density_every"] = cfg["density_every"]
    return out


def effective_horizon(args, cfg):
    horizon = args.horizon or cfg["steps"]
    unit = cfg.get("window") or cfg["stride"]
    return max(unit, horizon // unit * unit)


# ------------------------------------------------------------------------------------------- oracle arm

def oracle_rate(cfg, order, tangent, seconds, cores=None):
    """Time the oracle, as it stands, on `cores` host threads (default: all) on a bounded sample of the workload:
    a 64 x 64 sub-lattice of the config's ensemble (same eps, dt, stride, order, tangent), for a prefix of the
    horizon sized to ~`seconds` of wall time.  Returns (traj-steps/s, cores, description, work, elapsed)."""
    import numpy as np
    import oracle
    oracle.build()
    cores = cores or os.cpu_count() or 1
    sub = 64                                     # 64 x 64 = 4096-trajectory sub-lattice of the grid
    st = oracle.State(sub * sub, tangent=tangent, wind=True)
    st.order = order
    g = oracle.make_grid(sub, sub, cfg["lo"], cfg["hi"], cfg["angle_mode"], cfg["shape"], cfg["cx"],
                         cfg["cy"], cfg["r"], resample=cfg.get("resample", 0))
    oracle.init_shell(st, g, cfg["E"], cfg["eps"], cfg["seed"])
    live = int((st.status == 1).sum())

    def run(steps):
        edges = np.linspace(0, st.n, cores + 1).astype(int)
        ts = [threading.Thread(target=oracle.integrate, args=(st, steps, cfg["dt"], cfg["stride"]),
                               kwargs=dict(k0=int(a), k1=int(b), advance_clock=False))
              for a, b in zip(edges[:-1], edges[1:]) if b > a]
        t0 = time.perf_counter()
        [t.start() for t in ts]
        [t.join() for t in ts]
        return time.perf_counter() - t0

    dt_cal = run(cfg["stride"])                                       # calibration: one stride
    rate_cal = live * cfg["stride"] / max(dt_cal, 1e-6)
    steps = int(seconds * rate_cal / max(live, 1)) // cfg["stride"] * cfg["stride"]
    steps = max(cfg["stride"], min(steps, cfg["steps"]))
    el = run(steps)
    desc = ("%dx%d sub-lattice of the %dx%d ensemble (%d live), first %d of %d steps, order %d, tangent=%s, "
            "stride %d, %d thread%s over disjoint trajectory ranges"
            % (sub, sub, cfg["gx"], cfg["gy"], live, steps, cfg["steps"], order, tangent, cfg["stride"], cores,
               "" if cores == 1 else "s"))
    return live * steps / el, cores, desc, live * steps, el


def oracle_live_count(cfg, world, scaling):
    """Live trajectories of the whole job's ensemble (the oracle's generator; the reference arm's `config`)."""
    import oracle
    from paper_1107_4107_b200 import parallel
    gx, gy_total, _, _ = parallel.slice_of(cfg["gx"], cfg["gy"], world, 0, scaling)
    st = oracle.State(gx * gy_total, tangent=False, wind=False)
    g = oracle.make_grid(gx, gy_total, cfg["lo"], cfg["hi"], cfg["angle_mode"], cfg["shape"], cfg["cx"], cfg["cy"],
                         cfg["r"], resample=cfg.get("resample", 0))
    oracle.init_shell(st, g, cfg["E"], cfg["eps"], cfg["seed"])
    return int((st.status == 1).sum())


def run_reference(args, cfg, order, tangent):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    horizon = effective_horizon(args, cfg)
    per = max(2.0, min(args.cpu_seconds, 120.0 / max(1, args.steps + args.warmup)))
    for _ in range(args.warmup):
        oracle_rate(cfg, order, tangent, min(per, 2.0))
    work, el = 0, 0.0
    desc, cores = "", 0
    for _ in range(args.steps):
        _, cores, desc, w, e = oracle_rate(cfg, order, tangent, per)
        work += w
        el += e
    value = work / el
    config = workload_config(cfg, order, tangent, horizon, args.gpus, args.scaling,
                             oracle_live_count(cfg, args.gpus, args.scaling))
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * el / max(1, args.steps),
            "higher_is_better": True, "scaling": args.scaling, "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "gpu_launches": 0, "config": config,
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------------------- our arm

def measured_traffic(build_hash, kernel, config, steps_per_launch):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch from the ncu --set full capture of THIS build
    (profiles/traffic_by_build.csv, keyed by the hash of the library's sources and flags); None for any other build
    or launch shape — a typed-in figure would go stale with the next kernel edit."""
    path = os.path.join(ROOT, "profiles", "traffic_by_build.csv")
    try:
        for row in csv.DictReader(open(path)):
            if (row["build_hash"] == build_hash and row["kernel"] == kernel and int(row["config"]) == config
                    and int(row["steps_per_launch"]) == steps_per_launch):
                return int(row["dram_read_bytes"]) + int(row["dram_write_bytes"]), row["source"]
    except (OSError, KeyError, ValueError):
        pass
    return None, None


def ptxas_report(kernel_tag):
    """(registers per thread, spill bytes) ptxas printed for the kernel when libaw.so was built (build/ptxas.log)."""
    import re
    try:
        log = open(os.path.join(ROOT, "paper_1107_4107_b200", "build", "ptxas.log")).read()
    except OSError:
        return None, None
    m = re.search(re.escape(kernel_tag) + r".*?\n.*?(\d+) bytes spill stores, (\d+) bytes spill loads\n.*?Used (\d+) registers",
                  log, re.S)
    return (int(m.group(3)), int(m.group(1)) + int(m.group(2))) if m else (None, None)


def run_ours(args, cfg, order, tangent):
    import torch
    import torch.distributed as dist

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world != args.gpus:
        raise SystemExit("bench.py: --gpus %d but WORLD_SIZE=%d (launch with torchrun --nproc-per-node %d, or "
                         "without torchrun and let bench.py start the ranks)" % (args.gpus, world, args.gpus))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product has no CPU fallback)")
    if torch.cuda.device_count() <= local:
        raise SystemExit("bench.py: rank %d needs cuda:%d but only %d device(s) are visible"
                         % (rank, local, torch.cuda.device_count()))
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        if rank == 0:
            # the communicator lines (ncclCommInitRank ... nranks N) go to stderr: stdout carries the one JSON line
            os.environ.setdefault("NCCL_DEBUG", "INFO")
            os.environ.setdefault("NCCL_DEBUG_SUBSYS", "INIT")
            os.environ.setdefault("NCCL_DEBUG_FILE", "/dev/stderr")
        dist.init_process_group("nccl", device_id=dev)

    from paper_1107_4107_b200 import build as awbuild
    awbuild.build()
    import paper_1107_4107_b200 as aw
    from paper_1107_4107_b200 import parallel
    from paper_1107_4107_b200.configs import (FP64_PEAK_TFLOPS_NOMINAL, HIST_G, HIST_HI, HIST_LO,
                                               NOMINAL_FLOPS)

    # this rank's slice [k0, k0 + n) of the whole job's ensemble
    gx, gy_total, k0, n = parallel.slice_of(cfg["gx"], cfg["gy"], world, rank, args.scaling)
    counts = [parallel.slice_of(cfg["gx"], cfg["gy"], world, r, args.scaling)[3] for r in range(world)]
    horizon = effective_horizon(args, cfg)
    grid = aw.make_grid(gx, gy_total, cfg["lo"], cfg["hi"], cfg["angle_mode"], cfg["shape"], cfg["cx"], cfg["cy"],
                        cfg["r"], 1, 0, k0=k0, resample=cfg.get("resample", 0))
    dens_mode = cfg.get("density_mode", 0)          # 0: instantaneous actions; 1-3: the paper's averaged velocity
    window = cfg.get("window", 0)                   # > 0: consecutive averaging windows, density accumulated (Fig. 4)
    every = cfg.get("density_every", 0)             # > 0: instantaneous density binned every `every` steps (configs[4])
    hist_lo, hist_hi = cfg.get("hist_lo", HIST_LO), cfg.get("hist_hi", HIST_HI)
    ens = aw.Ensemble(n, tangent=tangent, wind=True, order=order, device=dev, ref=dens_mode != 0)
    image = torch.empty(max(n, 1), dtype=torch.float64, device=dev)
    hist = torch.zeros((HIST_G, HIST_G), dtype=torch.int32, device=dev)
    dropped = torch.zeros(1, dtype=torch.int64, device=dev)
    stream = torch.cuda.current_stream()
    kind = aw.AW_IND_FLI if tangent else aw.AW_IND_DH
    flush = None if n * 141 > 126e6 else torch.empty(256 << 20, dtype=torch.uint8, device=dev)   # > 126 MB L2

    # calls of aw_integrate per pass and steps per call
    if window:
        calls = [window] * (horizon // window)
    elif every and horizon > every:
        calls = [every] * (horizon // every) + ([horizon % every] if horizon % every else [])
    else:
        calls = [horizon]
    integ_events = []

    def one_pass(record):
        if flush is not None:
            flush.fill_(1)
        aw.aw_init_shell(ens, grid, cfg["E"], cfg["eps"], cfg["seed"])
        hist.zero_()
        dropped.zero_()
        if cfg.get("survive"):                       # only trajectories that stay inside the launch square
            ens.set_survivors((cfg["lo"], cfg["hi"], cfg["lo"], cfg["hi"]))
        if dens_mode and not window:
            aw.aw_mark(ens)                          # X(t) of the averaging window
        if record:
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
        for steps in calls:
            # Fig. 4: consecutive windows, each with its own snapshot, the density accumulated over all of
            # them; configs[4]: bin the instantaneous actions every `every` steps.  The mark / binning launches sit
            # inside the integrate events' bracket (< 0.1 % of it).
            if window:
                aw.aw_mark(ens)
            aw.aw_integrate(ens, n, steps, cfg["dt"], cfg["stride"])
            if window or (every and horizon > every and steps == every):
                aw.aw_density(ens, hist, hist_lo, hist_hi, dens_mode, dropped)
        if record:
            e1.record(stream)
            integ_events.append((e0, e1))
        aw.aw_indicator(ens, kind, 0.0, out=image)
        if len(calls) == 1 and not window:
            aw.aw_density(ens, hist, hist_lo, hist_hi, dens_mode, dropped)
        if world > 1:
            parallel.allreduce_hist(hist)
            parallel.gather_image(image[:n], counts)

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        one_pass(False)
    barrier()
    live = int((ens.status[:n] == 1).sum().item())
    clocks = ClockSampler(local)
    launches0 = aw.aw_launch_count()
    t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    clocks.start()
    t0.record(stream)
    for _ in range(args.steps):
        one_pass(True)
    t1.record(stream)
    barrier()
    clk = clocks.stop()
    launches = aw.aw_launch_count() - launches0
    ms = torch.tensor([t0.elapsed_time(t1)], dtype=torch.float64, device=dev)
    livet = torch.tensor([live], dtype=torch.int64, device=dev)
    if world > 1:
        dist.all_reduce(ms, op=dist.ReduceOp.MAX)
        dist.all_reduce(livet, op=dist.ReduceOp.SUM)
    total_ms = ms.item()
    live_all = int(livet.item())
    value = live_all * horizon * args.steps / (total_ms * 1e-3)

    # dominant kernel: integrate_kernel — average launch duration from CUDA events on its stream.
    # flops per trajectory-step = min(nominal accounting figure, fp64 flops the SASS of the step loop
    # executes) so neither a fat nor a lean sincos can inflate the fraction.
    import sass_count
    integ_ms = sum(a.elapsed_time(b) for a, b in integ_events)
    max_launch = 20000 // cfg["stride"] * cfg["stride"]                  # AW_MAX_STEPS_PER_LAUNCH (include/aw.h)
    n_integ_launches = args.steps * sum(math.ceil(c / max_launch) for c in calls)
    level = aw.aw_trig_level(ens, cfg["dt"])
    schedule = aw.aw_kernel_schedule(ens, cfg["dt"])      # 1: throughput flavour, 0: latency flavour (small ensembles)
    mix = sass_count.integrate_step_mix(order, tangent, level, schedule=schedule)
    flops_nominal = NOMINAL_FLOPS[(order, tangent)]
    flops_per_step = min(flops_nominal, mix["flops"])
    launch_ms = integ_ms / n_integ_launches
    steps_per_launch = horizon * args.steps / n_integ_launches
    kernel_rate = live * steps_per_launch / (launch_ms * 1e-3)          # traj-steps/s inside the kernel
    achieved = kernel_rate * flops_per_step / 1e12
    sms = torch.cuda.get_device_properties(dev).multi_processor_count
    fp64_slots = sms * 64 * 1.965e9                                      # fp64 thread-instructions / s
    kernel_name = "integrate_kernel<%d,%s,%d,%d>" % (3 if order == 4 else 7, str(tangent).lower(), level, schedule)
    build_hash = awbuild.source_hash()
    traffic, traffic_src = (None, None) if world > 1 else measured_traffic(
        build_hash, kernel_name, args.config, int(steps_per_launch))
    regs, spill = ptxas_report("integrate_kernelILi%dELb%dELi%dELi%dE" % (3 if order == 4 else 7, int(tangent), level,
                                                                          schedule))
    roofline = {"bound": "alu", "kernel": kernel_name, "registers_per_thread": regs, "spill_bytes": spill,
                "achieved": achieved, "peak": FP64_PEAK_TFLOPS_NOMINAL, "unit": "TFLOP/s",
                "frac": achieved / FP64_PEAK_TFLOPS_NOMINAL, "traffic": traffic, "traffic_source": traffic_src,
                "build_hash": build_hash,
                "peak_source": "derived: 148 SM x 64 DFMA/clk/SM x 2 flop x 1.965 GHz (DESIGN.md §6.1); "
                               "MEASURED_PEAKS.json has no fp64 entry",
                # SURVEY 8(d) reporting rule: the smaller of the nominal accounting figure and the executed flops;
                # at the nominal figure the same run would read achieved_at_nominal_flops (can exceed the peak:
                # the kernel does the step's work in fewer flops than the accounting convention assumes)
                "achieved_at_nominal_flops": kernel_rate * flops_nominal / 1e12,
                "flops_per_traj_step": flops_per_step, "flops_per_traj_step_nominal": flops_nominal,
                "flops_per_traj_step_executed": mix["flops"],
                "sass_per_step": {k: mix[k] for k in ("dfma", "dmul", "dadd", "other")},
                "fp64_pipe_busy_est": kernel_rate * (mix["dfma"] + mix["dmul"] + mix["dadd"]) / fp64_slots,
                # register-operand model (sass_count.py): 2 issue cycles per fp64 instruction, 3 for a DFMA that
                # reads three distinct registers without the reuse cache -> the ceiling this SASS can reach
                "fp64_issue_cycles_per_step_model": mix["issue_cycles"],
                "three_register_fp64_per_step": mix["three_register_fp64"],
                "fp64_pipe_busy_ceiling_model": 2.0 * (mix["dfma"] + mix["dmul"] + mix["dadd"]) / mix["issue_cycles"],
                "trig_level": level, "block_threads": aw.aw_block_size(ens, cfg["dt"]),
                "launch_ms": launch_ms, "launches_timed": n_integ_launches,
                "kernel_share_of_step": integ_ms / total_ms}

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": total_ms / args.steps, "higher_is_better": True,
            "scaling": args.scaling, "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": workload_config(cfg, order, tangent, horizon, world, args.scaling, live_all),
            "clocks": clk, "gpu_launches": int(launches), "roofline": roofline}

    # measured DFMA peak beside the derived one (rank 0; independent chains, all SMs; tests/aw_probe.h)
    if rank == 0:
        try:
            import aw_probe
            best = 0.0
            for chains in (8, 16):
                msd, cnt = aw_probe.dfma_peak(sms * 8, 256, chains, 1 << 16, device=dev)
                best = max(best, 2.0 * cnt / (msd * 1e-3) / 1e12)
            roofline["peak_measured_dfma_tflops"] = best
            roofline["frac_of_measured_dfma"] = achieved / best
        except Exception as e:  # the probe is evidence, not the product
            roofline["peak_measured_dfma_tflops"] = None
            roofline["peak_probe_error"] = str(e)

    # e2e: host (pinned) state -> aw_map_host / aw_velocity_map_host -> image + histogram on the host, copies timed
    if not args.no_e2e:
        aw.aw_init_shell(ens, grid, cfg["E"], cfg["eps"], cfg["seed"])
        torch.cuda.synchronize()
        host_in = dict(q=ens.q.cpu().pin_memory(), acc=ens.acc.cpu().pin_memory(),
                       wind=ens.wind.cpu().pin_memory(), status=ens.status[:n].cpu().pin_memory())
        if tangent:
            host_in["w"] = ens.w.cpu().pin_memory()
        out = dict(hist=torch.empty((HIST_G, HIST_G), dtype=torch.int32).pin_memory(),
                   dropped=torch.zeros(1, dtype=torch.int64).pin_memory())
        if not dens_mode:
            out["image"] = torch.empty(max(n, 1), dtype=torch.float64).pin_memory()
        hist_dev = torch.empty(HIST_SCRATCH(HIST_G) // 4, dtype=torch.int32, device=dev)
        h2d = sum(t.numel() * t.element_size() for t in host_in.values())
        d2h = sum(t.numel() * t.element_size() for t in out.values())
        e2e_steps = window or horizon                # the velocity pipeline's call is one averaging window

        def call(steps):
            if dens_mode:
                # the paper's pipeline: upload, mark, integrate one window, sphere density, download
                aw.aw_velocity_map_host(ens, host_in, steps, cfg["dt"], cfg["stride"], dens_mode, (HIST_G, HIST_G),
                                        hist_lo, hist_hi, hist_dev, out)
            else:
                aw.aw_map_host(ens, host_in, steps, cfg["dt"], cfg["stride"], kind, 0.0, (HIST_G, HIST_G),
                               HIST_LO, HIST_HI, image, hist_dev, out)

        call(cfg["stride"])                          # warm the path once with a short horizon
        barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        w0 = time.perf_counter()
        e0.record(stream)
        call(e2e_steps)
        if world > 1:
            parallel.allreduce_hist(hist_dev[:HIST_G * HIST_G])
        e1.record(stream)
        torch.cuda.synchronize()
        wall = time.perf_counter() - w0
        ems = torch.tensor([max(e0.elapsed_time(e1), wall * 1e3)], dtype=torch.float64, device=dev)
        if world > 1:
            dist.all_reduce(ems, op=dist.ReduceOp.MAX)
        line["e2e"] = {"value": live_all * e2e_steps / (ems.item() * 1e-3), "unit": UNIT,
                       "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h), "ms": ems.item(),
                       "steps": e2e_steps,
                       "api": "aw_velocity_map_host (pinned host state in; sphere density of the averaged velocity out)"
                              if dens_mode else "aw_map_host (pinned host state in; FLI image + histogram out)"}

    if rank == 0 and not args.no_cpu_baseline and world == 1:
        v, cores, desc, _, _ = oracle_rate(cfg, order, tangent, args.cpu_seconds)
        v1, _, desc1, _, _ = oracle_rate(cfg, order, tangent, min(8.0, args.cpu_seconds), cores=1)
        line["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc,
                                "one_core": {"value": v1, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": desc1}}

    if rank == 0:
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def run_dfma_shapes():
    """fp64 issue rate by operand shape on this GPU (tests/aw_probe.h, awp_dfma_shape)."""
    import torch
    import aw_probe
    sms = torch.cuda.get_device_properties(0).multi_processor_count
    names = ["fma(v,u0,w0) shared operands (reuse)", "fma(v,u_c,w_c) three distinct registers",
             "fma(v,u_c,imm) two registers + immediate", "fma(v,v,w_c) three operands, two distinct",
             "v*u_c DMUL two registers", "fma(u_c,w_c',v) accumulate, three distinct registers"]
    out = {}
    for shape, name in enumerate(names):
        ms, cnt = aw_probe.dfma_shape(sms * 8, 256, shape, 1 << 15)
        rate = cnt / (ms * 1e-3)
        out[name] = {"ms": ms, "fp64_inst_per_s": rate, "frac_of_sm_x_64_x_1.965GHz": rate / (sms * 64 * 1.965e9)}
    print(json.dumps({"probe": "awp_dfma_shape", "sms": sms, "shapes": out}), flush=True)


def run_density_bench():
    """The HBM-bound kernels alone (the histogram on clustered and on spread input, 2^20 and 2^22 points;
    init_shell; indicator), CUDA events over 20 back-to-back launches each, against the measured HBM copy bandwidth."""
    import torch
    from paper_1107_4107_b200 import build as awbuild
    awbuild.build()
    import paper_1107_4107_b200 as aw
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        pass
    hbm = peaks.get("hbm_gbs")
    stream = torch.cuda.current_stream()

    def timed(fn, reps=20):
        fn()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(reps):
            fn()
        e1.record(stream)
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) * 1e-3 / reps

    rows = []
    for logn in (20, 22):
        g = 1 << (logn // 2)
        n = g * g
        ens = aw.Ensemble(n, tangent=True, wind=True, ref=True)
        hist = torch.zeros((1024, 1024), dtype=torch.int32, device="cuda")
        dropped = torch.zeros(1, dtype=torch.int64, device="cuda")
        image = torch.empty(n, dtype=torch.float64, device="cuda")
        for label, grid, eps in (("clustered: disk r = 1e-3 at (0,0), <= 4 bins", aw.make_grid(g, g, -1.0, 1.0, 1, 1, 0.0, 0.0, 1e-3), 1e-3),
                                 ("spread: cell-centred grid over [-1,1]^2", aw.make_grid(g, g, -1.0, 1.0, 0, 0), 3e-2)):
            t_init = timed(lambda: aw.aw_init_shell(ens, grid, 1.0, eps, 0))
            aw.aw_mark(ens)
            aw.aw_integrate(ens, n, 100, 0.005, 100)
            t_act = timed(lambda: aw.aw_density(ens, hist, -1.0, 1.0, 0, dropped))
            t_vel = timed(lambda: aw.aw_density(ens, hist, -1.5, 1.5, 3, dropped))
            t_ind = timed(lambda: aw.aw_indicator(ens, aw.AW_IND_FLI, 0.0, out=image))
            b_init = n * (48 + 48 + 32 + 12 + 1)            # bytes written per trajectory
            rows.append({"n": n, "input": label,
                         "init_shell_us": t_init * 1e6, "init_shell_GBs": b_init / t_init / 1e9,
                         "density_action_us": t_act * 1e6, "density_action_GBs": n * 17 / t_act / 1e9,
                         "density_velocity_us": t_vel * 1e6, "density_velocity_GBs": n * 73 / t_vel / 1e9,
                         "indicator_us": t_ind * 1e6, "indicator_GBs": n * 17 / t_ind / 1e9})
    print(json.dumps({"probe": "hbm_bound_kernels", "hbm_copy_peak_GBs": hbm,
                      "bytes_per_trajectory": {"init_shell": 141, "density_action": 17, "density_velocity": 73,
                                               "indicator": 17}, "rows": rows}), flush=True)


def spawn_ranks(args):
    """`python bench.py --gpus N` without torchrun: start the N ranks here (one per GPU, NCCL over NVLink), after
    checking that N devices exist — never silently benchmark fewer GPUs than asked for."""
    import torch
    have = torch.cuda.device_count() if torch.cuda.is_available() else 0
    if have < args.gpus:
        raise SystemExit("bench.py: --gpus %d but only %d CUDA device(s) are visible" % (args.gpus, have))
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(args.gpus),
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    raise SystemExit(subprocess.call(cmd))


def main():
    args = parse()
    if args.dfma_shapes:
        return run_dfma_shapes()
    if args.density_bench:
        return run_density_bench()
    if args.gpus < 1:
        raise SystemExit("bench.py: --gpus must be >= 1")
    from paper_1107_4107_b200.configs import CONFIGS
    cfg = dict(CONFIGS[args.config])
    order = args.order or cfg["order"]
    tangent = cfg["tangent"]
    if args.impl == "reference":
        return run_reference(args, cfg, order, tangent)
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        return spawn_ranks(args)
    run_ours(args, cfg, order, tangent)


if __name__ == "__main__":
    main()
