#!/usr/bin/env python
"""bench.py -- SU(3) Landau overrelaxation throughput on B200 (BASELINE.json metric, configs[3]).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload NAME]
                    [--gauge landau|coulomb] [--series-order N] [--sa-temperature T] [--micro] [--variant V]

A STEP is one full overrelaxation sweep (black half-sweep + white half-sweep = V site updates,
PAPER.md L54) of the resident field; every --check-every steps the timed region also computes
theta and F, as the paper's driver loop does.  Default workload: cfg3_fp32 = 32^4 SU(3), fp32
12-parameter storage, omega = 1.7, near-identity (eps 0.8) gauge-scrambled seeded input -- the
configuration the paper's Fig. 1 and BASELINE.json's metric are quoted on.

value       site-updates/s over all ranks, inputs resident in HBM, CUDA events, max over ranks.
e2e         the same through culgt_fix_host: pinned HOST canonical field -> H2D -> pack -> K
            sweeps -> theta, F -> unpack -> D2H, all inside the timed region (one job of K steps;
            the byte counts are per step = job bytes / K).
roofline    dominant kernel = the half-sweep; `achieved` = ALGORITHMIC bytes per launch (2 * field
            bytes: every link read once and written once) / the average
            launch duration measured live with CUDA events on the launching stream.  Part of
            those bytes is served by the L2 (the white half-sweep walks the lattice backwards):
            `dram_achieved` = the DRAM bytes per launch of the committed steady-state ncu capture
            (profiles/roofline_traffic.csv, stamped with the kernel it was taken on) / the same
            duration is what HBM itself moves.
kernels     the other kernels of the path at the same workload: theta+F, pack, unpack, gauge transform.
extra_workloads   the second half of BASELINE.json configs[3] (fp64 18-parameter) and configs[4]
            (48^3 x 96 fp32-12, 64^4 fp64-18), a few steps each, and the driver loop
            (culgt_landau_fix) on the latency-bound configs[0..2].
cpu_baseline the oracle (oracle/, as it stands) timed on this host's cores on a bounded sample.
--impl reference  times the oracle itself (rank 0 only), same metric / config / unit.

Multi-GPU: by default replicas only (BASELINE.json north_star): each rank fixes its own
independent configuration; value = total site-updates / max-over-ranks time; scaling "weak".
--sharded instead cuts ONE lattice (default cfg4_fp64, 64^4 fp64-18, 9.7 GB) into --gpus time slabs,
one per rank, with one halo message each way per boundary and half-sweep over NCCL and theta/F from
all-gathered per-slab sums; value = V * steps / max-over-ranks time; scaling "strong".
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import lattice_inputs as li  # noqa: E402

METRIC = "su3_landau_or_site_updates_per_s"
UNIT = "site-updates/s"
FALLBACK_HBM_GBS = 6650.0   # /opt/skills/guides/B200_PROFILING.md fallback


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=500)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default=None, choices=sorted(li.CONFIGS),
                    help="default: cfg3_fp32 (BASELINE.json configs[3], the headline); with --sharded: cfg4_fp64")
    ap.add_argument("--sharded", action="store_true",
                    help="strong scaling: ONE lattice cut into --gpus time slabs, one per rank, halo messages over "
                         "NCCL (include/culgt_b200.h 'Time-slab decomposition'); default is replicas (north_star)")
    ap.add_argument("--check-every", type=int, default=50)
    ap.add_argument("--variant", type=int, default=0, help="sweep kernel variant (0 = default)")
    ap.add_argument("--gauge", default="landau", choices=["landau", "coulomb"],
                    help="coulomb: K(x) from the spatial links, per-slice theta_t/F_t (DESIGN.md C-22)")
    ap.add_argument("--series-order", type=int, default=0,
                    help="> 0: truncated-series g^omega of that order instead of the exact power (DESIGN.md C-24)")
    ap.add_argument("--micro", action="store_true",
                    help="microcanonical sweeps (reflection g^2, DESIGN.md C-26) instead of overrelaxation")
    ap.add_argument("--sa-temperature", type=float, default=0.0,
                    help="> 0: time simulated-annealing sweeps at this temperature instead of overrelaxation (DESIGN.md C-25)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-extra", action="store_true",
                    help="skip the extra_workloads / kernels blocks (they only run for the default workload, N = 1)")
    ap.add_argument("--extra-steps", type=int, default=10, help="timed sweeps of each extra workload")
    ap.add_argument("--extra-workloads", default=None,
                    help="comma-separated workloads for the extra_workloads block (default: cfg3_fp64,cfg4_fp32,"
                         "cfg4_fp64 when the main workload is cfg3_fp32, none otherwise)")
    args = ap.parse_args()
    if args.workload is None:
        args.workload = "cfg4_fp64" if args.sharded else "cfg3_fp32"
    return args


def measured_peak():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


def committed_traffic(workload: str, capture: str, kernel: str):
    """DRAM bytes (read + write) per half-sweep launch from the committed ncu captures
    (profiles/roofline_traffic.csv: workload, capture, read, write, commit, kernel, source).  They
    cannot be measured live without ncu attached, so every row names the commit and the kernel
    (culgt_sweep_kernel_name) it was captured on; a row taken on another kernel than the one this
    run launches is reported as stale instead of being used.  Returns (bytes or None, info dict)."""
    try:
        with open(os.path.join(ROOT, "profiles", "roofline_traffic.csv")) as f:
            for line in f:
                p = [x.strip() for x in line.strip().split(";")]
                if len(p) >= 7 and p[0] == workload and p[1] == capture:
                    info = {"commit": p[4], "kernel": p[5], "source": p[6]}
                    if p[5] != kernel:
                        info["stale"] = f"captured on another kernel than this run's ({kernel})"
                        return None, info
                    return int(p[2]) + int(p[3]), info
    except Exception as e:      # pragma: no cover
        return None, {"stale": f"profiles/roofline_traffic.csv unreadable: {e}"}
    return None, {"stale": "no capture committed for this workload"}


class ClockSampler:
    """Samples SM clock and throttle reasons with NVML while the timed region runs."""
    REASONS = {0x4: "sw_power_cap", 0x8: "hw_slowdown", 0x20: "sw_thermal_slowdown",
               0x40: "hw_thermal_slowdown", 0x80: "hw_power_brake_slowdown"}

    def __init__(self, index: int):
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self.t0 = None
        self._stop = threading.Event()
        self._thread = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
            pynvml.nvmlDeviceGetClockInfo(self.h, pynvml.NVML_CLOCK_SM)          # warm the query path (slow the first time)
            pynvml.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
        except Exception:
            self.nv = None

    def _run(self):
        nv = self.nv
        while not self._stop.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                mask = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for bit, name in self.REASONS.items():
                    if mask & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            time.sleep(0.004)

    def start(self):
        self.t0 = time.perf_counter()
        if self.nv is not None:
            self._thread = threading.Thread(target=self._run, daemon=True)
            self._thread.start()

    def stop(self):
        if self._thread is not None:
            self._stop.set()
            self._thread.join()
        med = float(np.median(self.samples)) if self.samples else None
        return {"sm_mhz": med, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(self.samples),
                "window_ms": 1e3 * (time.perf_counter() - self.t0) if self.t0 else None}


def time_oracle(dims, group, ur, omega, max_sweeps, budget_s, threads, gauge="landau"):
    """Full oracle sweeps until budget_s or max_sweeps; returns (site-updates/s, sweeps)."""
    import oracle
    oracle.set_threads(threads)
    sweep = oracle.full_sweep_coulomb if gauge == "coulomb" else oracle.full_sweep
    V = li.volume(dims)
    t0 = time.perf_counter()
    n = 0
    while n < max_sweeps:
        sweep(dims, ur, omega)
        n += 1
        if time.perf_counter() - t0 > budget_s:
            break
    dt = time.perf_counter() - t0
    return V * n / dt, n


def run_reference(args):
    """--impl reference: the oracle as it stands, on the host cores, rank 0 only."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    cfg = li.CONFIGS[args.workload]
    total = args.steps + args.warmup
    dims = cfg["dims"]
    sample = "whole lattice, one full sweep per step"
    if li.volume(dims) * total > 32 ** 4 * 600:
        dims = (16, 16, 16, 16)
        sample = "16^4 sub-volume with the same recipe (periodic), one full sweep per step"
    threads = min(oracle.max_threads(), os.cpu_count() or 1)
    oracle.set_threads(threads)
    u = li.make_config(dims, cfg["group"], cfg["kind"], cfg["seed"], eps=cfg["eps"], scramble=cfg["scramble"])
    if cfg["precision"] == 32:
        u = li.round_to_fp32(u)
    ur = li.to_real(u)
    sweep = oracle.full_sweep_coulomb if args.gauge == "coulomb" else oracle.full_sweep
    for _ in range(args.warmup):
        sweep(dims, ur, cfg["omega"])
    t0 = time.perf_counter()
    for _ in range(args.steps):
        sweep(dims, ur, cfg["omega"])
    dt = time.perf_counter() - t0
    V = li.volume(dims)
    value = V * args.steps / dt
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic", "config": workload_config(args, cfg),
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gflops": value * flops_per_site(cfg, args.gauge) / 1e9,
    }
    print(json.dumps(line), flush=True)


def max_over_ranks(value: float, world: int, device="cpu") -> float:
    """MAX over the ranks of a per-rank scalar (the only cross-rank data dependency of the
    bench: the path itself has no exchange step).  Works on any backend."""
    if world <= 1:
        return float(value)
    import torch
    import torch.distributed as dist
    t = torch.tensor([value], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(world: int, volume: int, steps: int, elapsed_max_s: float) -> float:
    """Replicas only: every rank sweeps its own lattice; units of all ranks / slowest rank's time."""
    return world * volume * steps / elapsed_max_s


def rank_seed(base_seed: int, rank: int) -> int:
    """One independent seeded configuration per rank."""
    return base_seed + 7919 * rank


def flops_per_site(cfg, gauge="landau"):
    """Fixed algorithmic counts: Coulomb gauge gathers 6 links instead of 8 into K."""
    if gauge == "coulomb":
        return 2304 - 36 if cfg["group"] == 3 else 278 - 8
    return 2304 if cfg["group"] == 3 else 278


def workload_config(args, cfg):
    return {
        "gauge": args.gauge, "power": ("microcanonical g^2" if args.micro else
                                       f"heat bath at T={args.sa_temperature}" if args.sa_temperature > 0 else
                                       f"series order {args.series_order}" if args.series_order > 0 else "exact"),
        "workload": f"{args.workload}: {'x'.join(str(d) for d in cfg['dims'])} SU({cfg['group']}) "
                    f"fp{cfg['precision']} {cfg['params']}-parameter, omega={cfg['omega']}, "
                    f"{cfg['kind']} eps={cfg['eps']} scramble={cfg['scramble']} seed={cfg['seed']}",
        "step": "one full sweep (black+white half-sweep) = V site updates; theta and F every "
                f"{args.check_every} steps inside the timed region",
        "l2": "no flush between steps: the field (201 MB ... 9.7 GB at 32^4 and above) is larger than the "
              "126 MB L2; the white half-sweep walks the lattice backwards, so the L2 carries the last "
              "lines of one half-sweep into the next (15 % of the traffic at 32^4 fp32-12, "
              "roofline.traffic_steady_state) -- part of the method's steady state, reported, not hidden",
        "parallelism": "replicas only (one independent configuration per GPU)",
    }


class Field:
    """One seeded configuration resident on the GPU: pinned host canonical field, device canonical
    scratch, internal links, workspace."""

    def __init__(self, culgt, torch, name, rank):
        cfg = li.CONFIGS[name]
        self.name, self.cfg = name, cfg
        self.dims, self.omega = cfg["dims"], cfg["omega"]
        self.V = li.volume(self.dims)
        self.lat = culgt.Lattice(tuple(self.dims), cfg["group"], cfg["precision"], cfg["params"])
        u = li.make_config(self.dims, cfg["group"], cfg["kind"], rank_seed(cfg["seed"], rank), eps=cfg["eps"],
                           scramble=cfg["scramble"])
        np_dt = np.float32 if cfg["precision"] == 32 else np.float64
        self.host = torch.from_numpy(li.to_real(u, np_dt)).pin_memory()
        del u
        self.can_dev = torch.empty_like(self.host, device="cuda")
        self.links = culgt.alloc_links(self.lat)
        self.ws = culgt.alloc_workspace(self.lat)
        self.can_dev.copy_(self.host)
        culgt.culgt_pack(self.lat, self.can_dev, self.links)
        torch.cuda.synchronize()
        # algorithmic bytes: the stored parameters (fp32-18 keeps 2 pad floats per link that are not counted)
        self.field_bytes = 4 * self.V * cfg["params"] * (cfg["precision"] // 8)


def time_sweep_loop(torch, field, sweeps, check, steps, warmup, check_every, barrier, sampler=None, window_ms=60.0):
    """W warm-up sweeps, then K timed sweeps with a check every check_every; CUDA events on the current
    stream.  With a sampler: when the timed window is shorter than window_ms, untimed sweeps before and
    after it keep the GPU under the same load until NVML has been sampled for that long, so that the
    clocks record never rests on one sample (a 20-step run at 32^4 is 2 ms of work)."""
    stream = torch.cuda.current_stream()
    sweeps(max(warmup, 3))
    check()
    barrier()

    def roll_until(t_end, min_samples, t_cap):
        # keep the GPU under the same load until the time has passed AND NVML has answered often enough
        # (the first NVML queries of a process on a fresh box can take tens of milliseconds each)
        while (time.perf_counter() < t_end or len(sampler.samples) < min_samples) and time.perf_counter() < t_cap:
            sweeps(8)
            torch.cuda.synchronize()

    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    checks = []
    t_start = time.perf_counter()
    if sampler is not None:
        sampler.start()
        roll_until(t_start + 0.4e-3 * window_ms, 2 if sampler.nv is not None else 0, t_start + 1.5)
    ev0.record(stream)
    done = 0
    while done < steps:
        n = min(check_every, steps - done)
        sweeps(n)
        done += n
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(stream)
        check()
        b.record(stream)
        checks.append((a, b))
    ev1.record(stream)
    if sampler is not None:
        torch.cuda.synchronize()
        roll_until(t_start + 1e-3 * window_ms, 6 if sampler.nv is not None else 0, t_start + 4.0)
    barrier()
    clocks = sampler.stop() if sampler is not None else None
    elapsed_ms = ev0.elapsed_time(ev1)
    check_ms = sum(a.elapsed_time(b) for a, b in checks)
    return {"elapsed_ms": elapsed_ms, "check_ms": check_ms, "n_checks": len(checks), "clocks": clocks,
            "launch_ms": (elapsed_ms - check_ms) / (2 * steps)}


def time_kernel(torch, fn, reps=20, warm=3):
    """Average device time of fn() in microseconds (CUDA events on the current stream)."""
    stream = torch.cuda.current_stream()
    for _ in range(warm):
        fn()
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record(stream)
    for _ in range(reps):
        fn()
    b.record(stream)
    torch.cuda.synchronize()
    return 1e3 * a.elapsed_time(b) / reps


def other_kernels(culgt, torch, f, peak):
    """theta+F, pack, unpack, gauge transform at the workload of `f`: us per call, algorithmic GB/s
    (bytes the call must move once), fraction of the measured copy peak."""
    scal = torch.zeros(2, dtype=torch.float64, device="cuda")
    cbytes = culgt.culgt_canonical_bytes(f.lat)
    g = li.haar_su3(f.V, f.cfg["seed"] + 500) if f.cfg["group"] == 3 else li.haar_su2(f.V, f.cfg["seed"] + 500)
    gt = torch.from_numpy(li.to_real(g, np.float32 if f.cfg["precision"] == 32 else np.float64)).cuda()
    del g
    spec = {
        "theta_F": (lambda: culgt.culgt_gauge_precision_functional(f.lat, f.links, f.ws, scal[0:1], scal[1:2]),
                    f.field_bytes, "one read of the field"),
        "pack": (lambda: culgt.culgt_pack(f.lat, f.can_dev, f.links), cbytes + f.field_bytes,
                 "canonical read + internal write"),
        "unpack": (lambda: culgt.culgt_unpack(f.lat, f.links, f.can_dev), cbytes + f.field_bytes,
                   "internal read + canonical write"),
        "gauge_transform": (lambda: culgt.culgt_gauge_transform(f.lat, f.links, gt),
                            2 * f.field_bytes + gt.numel() * gt.element_size(), "links read + written, g once"),
    }
    out = {}
    culgt.culgt_unpack(f.lat, f.links, f.can_dev)      # pack/unpack round-trip on the current field
    for name, (fn, nbytes, what) in spec.items():
        us = time_kernel(torch, fn)
        gbs = nbytes / (us * 1e-6) / 1e9
        out[name] = {"us": us, "bytes": nbytes, "what": what, "gbs": gbs, "frac": gbs / peak}
    return out


def sweep_variants(culgt, torch, f, peak, steps):
    """The widening steps of the path at the workload of `f`: us per half-sweep of the
    Coulomb-gauge, truncated-series, microcanonical and simulated-annealing sweeps (same loads, stores and
    link products as the overrelaxation sweep; only the per-subgroup update differs), algorithmic GB/s."""
    lat, links, omega = f.lat, f.links, f.omega
    runs = {
        "coulomb": lambda n: culgt.culgt_or_sweeps_coulomb(lat, links, n, omega),
        "series_order_4": lambda n: culgt.culgt_or_sweeps_series(lat, links, n, omega, 4),
        "microcanonical": lambda n: culgt.culgt_micro_sweeps(lat, links, n),
        "annealing_T_0.1": lambda n: culgt.culgt_sa_anneal(lat, links, 0.1, 0.1, n, 2024),
        "annealing_T_2": lambda n: culgt.culgt_sa_anneal(lat, links, 2.0, 2.0, n, 2024),
    }
    out = {}
    stream = torch.cuda.current_stream()
    for name, run in runs.items():
        culgt.culgt_pack(lat, f.can_dev, links)           # every variant starts from the same stored field
        run(3)
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(stream)
        run(steps)
        b.record(stream)
        torch.cuda.synchronize()
        us = 1e3 * a.elapsed_time(b) / (2 * steps)
        gbs = 2 * f.field_bytes / (us * 1e-6) / 1e9
        out[name] = {"half_sweep_us": us, "value": f.V * steps / (a.elapsed_time(b) * 1e-3), "gbs": gbs, "frac": gbs / peak}
    return out


def driver_loop_times(culgt, torch, rank):
    """The paper's driver loop on the latency-bound BASELINE.json configs[0..2]: wall time of
    culgt_landau_fix (stopping decision on the device, one host synchronisation per batch of checks)
    next to the same loop driven from the host with a synchronisation at every check."""
    runs = {"cfg0": (1e-20, 5000, 1), "cfg1": (0.0, 200, 10), "cfg2": (0.0, 1000, 10)}
    out = {}
    for name, (target, max_sweeps, every) in runs.items():
        f = Field(culgt, torch, name, rank)
        scal = torch.zeros(2, dtype=torch.float64, device="cuda")

        def host_loop():
            culgt.culgt_gauge_precision_functional(f.lat, f.links, f.ws, scal[0:1], scal[1:2])
            theta, done = float(scal[0].item()), 0
            while not (theta < target) and done < max_sweeps:
                n = min(every, max_sweeps - done)
                culgt.culgt_or_sweeps(f.lat, f.links, n, f.omega)
                done += n
                culgt.culgt_gauge_precision_functional(f.lat, f.links, f.ws, scal[0:1], scal[1:2])
                theta = float(scal[0].item())
            return done, theta

        def fix(variant):
            # variant 34 = the production kernels launched per half-sweep (no L2 hints: irrelevant at this
            # size), stop word on the device; variant 0 additionally takes the one-kernel loop where it applies
            def run():
                culgt.culgt_set_sweep_variant(variant)
                try:
                    return culgt.culgt_landau_fix(f.lat, f.links, f.ws, f.omega, target, max_sweeps, every)[:2]
                finally:
                    culgt.culgt_set_sweep_variant(0)
            return run

        res = {}
        for label, loop in (("host_sync_every_check", host_loop), ("device_stop_flag_launch_per_half_sweep", fix(34)),
                            ("device_stop_flag", fix(0))):
            best = None
            for _ in range(3):
                culgt.culgt_pack(f.lat, f.can_dev, f.links)
                torch.cuda.synchronize()
                t0 = time.perf_counter()
                done, theta = loop()
                torch.cuda.synchronize()
                dt = time.perf_counter() - t0
                best = dt if best is None else min(best, dt)
            res[label] = {"wall_ms": 1e3 * best, "sweeps": done, "theta": theta,
                          "us_per_sweep": 1e6 * best / max(done, 1), "value": f.V * done / best}
        res["speedup"] = res["host_sync_every_check"]["wall_ms"] / res["device_stop_flag"]["wall_ms"]
        res["workload"] = f"{name}: {'x'.join(map(str, f.dims))} SU({f.cfg['group']}) fp{f.cfg['precision']}, " \
                          f"theta checked every {every} sweep(s), target {target:g}, at most {max_sweeps} sweeps"
        out[name] = res
    return out


def run_sharded(args):
    """--sharded: the time-slab decomposition, one slab per rank (csrc/slab.cu)."""
    import torch
    import torch.distributed as dist
    import paper_1412_3655_b200 as culgt

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (there is no CPU fallback)")
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    cfg = li.CONFIGS[args.workload]
    dims, omega = cfg["dims"], cfg["omega"]
    V = li.volume(dims)
    lat = culgt.Lattice(tuple(dims), cfg["group"], cfg["precision"], cfg["params"])
    local = culgt.culgt_slab_lattice(lat, world)          # raises unless N3 / world is an even number of slices
    T = local.dims[3]
    # my slab of the ONE seeded configuration, made without making the rest
    u = li.make_config(dims, cfg["group"], cfg["kind"], cfg["seed"], eps=cfg["eps"], scramble=cfg["scramble"],
                       t_range=(rank * T, (rank + 1) * T))
    np_dt = np.float32 if cfg["precision"] == 32 else np.float64
    host = torch.from_numpy(li.to_real(u, np_dt)).pin_memory()
    del u
    can_dev = torch.empty_like(host, device="cuda")
    links = culgt.alloc_slab_links(local)
    ws = culgt.alloc_workspace(local)
    sums = torch.zeros(2 * world + 2, dtype=torch.float64, device="cuda")
    scal = torch.zeros(2, dtype=torch.float64, device="cuda")
    if os.environ.get("NCCL_DEBUG", "").upper() in ("", "VERSION", "WARN"):
        os.environ["NCCL_DEBUG"] = "NONE"               # at VERSION and WARN NCCL prints a banner on stdout: one JSON line only
    uid = [culgt.culgt_slab_comm_unique_id() if rank == 0 else None]
    if world > 1:
        dist.broadcast_object_list(uid, src=0)
    comm = culgt.culgt_slab_comm_create(uid[0], rank, world)
    comm_stream = torch.cuda.Stream()                     # halo messages travel here while the interior is swept

    def load():
        can_dev.copy_(host, non_blocking=True)
        culgt.culgt_slab_pack(local, can_dev, links)
        culgt.culgt_slab_exchange_all_nccl(comm, local, links)

    def sweeps(n):
        culgt.culgt_slab_or_sweeps_nccl(comm, local, links, n, omega, comm_stream)

    def check():
        culgt.culgt_slab_theta_F_nccl(comm, lat, local, links, ws, sums, scal[0:1], scal[1:2])

    load()
    t = time_sweep_loop(torch, None, sweeps, check, args.steps, args.warmup, args.check_every, barrier,
                        ClockSampler(local_rank))
    theta, F = (float(x) for x in scal.cpu())
    elapsed_max_ms = max_over_ranks(t["elapsed_ms"], world, "cuda")
    value = V * args.steps / (elapsed_max_ms * 1e-3)
    slab_bytes = 4 * (V // world) * cfg["params"] * (cfg["precision"] // 8)
    halo = culgt.culgt_slab_halo_bytes(local)
    peak, peak_src = measured_peak()
    gbs = 2 * slab_bytes / (t["launch_ms"] * 1e-3) / 1e9

    e2e = None
    if not args.no_e2e:
        def host_job(n):
            load()
            sweeps(n)
            check()
            culgt.culgt_slab_unpack(local, links, can_dev)
            host.copy_(can_dev, non_blocking=True)
            return tuple(float(x) for x in scal.cpu())
        host_job(2)
        barrier()
        t0 = time.perf_counter()
        th_e, F_e = host_job(args.steps)
        torch.cuda.synchronize()
        dt_max = max_over_ranks(time.perf_counter() - t0, world, "cuda")
        cbytes = host.numel() * host.element_size()
        e2e = {"value": V * args.steps / dt_max, "unit": UNIT, "h2d_bytes_per_step": world * cbytes / args.steps,
               "d2h_bytes_per_step": world * (cbytes + 16) / args.steps,
               "job": f"every rank: H2D of its slab ({cbytes} B) + pack + halo exchange + {args.steps} sweeps + "
                      f"theta,F + unpack + D2H", "theta": th_e, "F": F_e}
    culgt.culgt_slab_comm_destroy(comm)
    if rank == 0:
        conf = workload_config(args, cfg)
        conf["parallelism"] = (f"time-slab split: {world} slab(s) of {T} time-slices, one per GPU; per half-sweep one "
                               f"ncclSend/ncclRecv halo message of {halo} B each way per boundary, boundary slices swept "
                               f"first; theta/F from all-gathered per-slab sums")
        print(json.dumps({
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": elapsed_max_ms / args.steps, "higher_is_better": True,
            "scaling": "strong", "vs_baseline": None, "dtype": "f32" if cfg["precision"] == 32 else "f64",
            "data": "synthetic", "config": conf, "gflops": value * flops_per_site(cfg) / 1e9,
            "algorithmic_gbs": value * 16 * (cfg["params"] * cfg["precision"] // 8) / 1e9,
            "gpu_launches": 2 * args.steps * (3 if T > 2 else 2) + 3 * t["n_checks"],
            "halo_bytes_per_step_per_rank": 4 * halo, "e2e": e2e,
            "roofline": {"bound": "hbm", "achieved": gbs, "peak": peak, "unit": "GB/s", "frac": gbs / peak,
                         "traffic": None, "kernel": culgt.culgt_sweep_kernel_name(lat) + " on one slab (windowed)",
                         "bytes_per_launch": 2 * slab_bytes, "launch_us": 1e3 * t["launch_ms"], "peak_source": peak_src,
                         "note": "per rank: a half-sweep of ONE slab (its three window launches), algorithmic bytes"},
            "cpu_baseline": None, "clocks": t["clocks"], "final": {"theta": theta, "F": F},
            "check_ms_total": t["check_ms"],
        }), flush=True)
    if world > 1:
        dist.destroy_process_group()


def main():
    args = parse_args()
    if args.impl == "reference":
        run_reference(args)
        return
    if args.sharded:
        run_sharded(args)
        return

    import torch
    import torch.distributed as dist
    import paper_1412_3655_b200 as culgt

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (there is no CPU fallback)")
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    culgt.culgt_set_sweep_variant(args.variant)
    f = Field(culgt, torch, args.workload, rank)      # seeded synthetic input, one independent configuration per rank
    cfg, lat, links, ws, V, omega = f.cfg, f.lat, f.links, f.ws, f.V, f.omega
    peak, peak_src = measured_peak()

    coulomb = args.gauge == "coulomb"
    n3 = int(f.dims[3])
    scal = torch.zeros(2 * n3 if coulomb else 2, dtype=torch.float64, device="cuda")   # Coulomb: theta_t, F_t per slice
    with_ws = hasattr(culgt.lib(), "culgt_or_sweeps_ws")     # measurement library: variant 60 needs the workspace
    if coulomb:
        sweeps = lambda n: culgt.culgt_or_sweeps_coulomb(lat, links, n, omega)  # noqa: E731
    elif with_ws:
        sweeps = lambda n: culgt.culgt_or_sweeps_ws(lat, links, ws, n, omega)  # noqa: E731
    else:
        sweeps = lambda n: culgt.culgt_or_sweeps(lat, links, n, omega)  # noqa: E731
    if args.sa_temperature > 0:
        if coulomb or args.series_order > 0:
            raise SystemExit("--sa-temperature applies to Landau gauge and excludes --series-order")
        sweeps = lambda n: culgt.culgt_sa_anneal(lat, links, args.sa_temperature, args.sa_temperature, n, 2024)  # noqa: E731
    if args.micro:
        if coulomb or args.series_order > 0 or args.sa_temperature > 0:
            raise SystemExit("--micro applies to Landau gauge and excludes --series-order / --sa-temperature")
        sweeps = lambda n: culgt.culgt_micro_sweeps(lat, links, n)  # noqa: E731
    if args.series_order > 0:
        if coulomb:
            raise SystemExit("--series-order applies to Landau gauge")
        sweeps = lambda n: culgt.culgt_or_sweeps_series(lat, links, n, omega, args.series_order)  # noqa: E731

    def check():
        if coulomb:
            culgt.culgt_coulomb_precision_functional(lat, links, ws, scal[:n3], scal[n3:])
        else:
            culgt.culgt_gauge_precision_functional(lat, links, ws, scal[0:1], scal[1:2])

    # ---- the timed region: K steps, theta/F every check_every steps
    t = time_sweep_loop(torch, f, sweeps, check, args.steps, args.warmup, args.check_every, barrier,
                        ClockSampler(local_rank))
    elapsed_ms, check_ms, n_checks, clocks, launch_ms = (t["elapsed_ms"], t["check_ms"], t["n_checks"], t["clocks"],
                                                         t["launch_ms"])
    res = scal.cpu()
    theta, F = (float(res[:n3].max()), float(res[n3:].mean())) if coulomb else (float(res[0]), float(res[1]))

    elapsed_max_ms = max_over_ranks(elapsed_ms, world, "cuda")
    value = whole_job_value(world, V, args.steps, elapsed_max_ms * 1e-3)

    sweep_launches = 2 * args.steps
    gpu_launches = sweep_launches + n_checks * 2        # fused theta+F: partial + final kernel
    alg_bytes_per_launch = 2 * f.field_bytes
    achieved_gbs = alg_bytes_per_launch / (launch_ms * 1e-3) / 1e9
    kernel_name = culgt.culgt_sweep_kernel_name(lat)
    traffic, traffic_info = committed_traffic(args.workload, "ncu_set_full_cold_cache", kernel_name)
    steady, steady_info = committed_traffic(args.workload, "steady_state", kernel_name)
    plain_or = not (coulomb or args.micro or args.series_order > 0 or args.sa_temperature > 0 or args.variant != 0)
    if not plain_or:
        traffic = steady = None
        traffic_info = steady_info = {"stale": "captures exist for the default overrelaxation sweep only"}

    # ---- end to end through the host-buffer entry point
    e2e = None
    if not args.no_e2e:
        host, can_dev = f.host, f.can_dev

        def host_job(n):
            if not coulomb:
                return culgt.culgt_fix_host(lat, host, can_dev, links, ws, n, omega)
            # Coulomb: the same job assembled from the C-ABI calls (H2D, pack, sweeps, theta_t/F_t,
            # unpack, D2H of the field and of the 2*N3 scalars)
            can_dev.copy_(host, non_blocking=True)
            culgt.culgt_pack(lat, can_dev, links)
            sweeps(n)
            check()
            culgt.culgt_unpack(lat, links, can_dev)
            host.copy_(can_dev, non_blocking=True)
            r = scal.cpu()
            return float(r[:n3].max()), float(r[n3:].mean())

        host_job(2)                                                         # warm the path
        barrier()
        t0 = time.perf_counter()
        th_e, F_e = host_job(args.steps)
        torch.cuda.synchronize()
        dt = time.perf_counter() - t0
        dt_max = max_over_ranks(dt, world, "cuda")
        cbytes = culgt.culgt_canonical_bytes(lat)
        e2e = {"value": whole_job_value(world, V, args.steps, dt_max), "unit": UNIT,
               "h2d_bytes_per_step": cbytes / args.steps, "d2h_bytes_per_step": (cbytes + 16) / args.steps,
               "job": f"one {'culgt_fix_host call' if not coulomb else 'host job (pack, sweeps, theta_t/F_t, unpack)'} = H2D {cbytes} B + pack + {args.steps} sweeps + theta,F + unpack + D2H {cbytes} B",
               "theta": th_e, "F": F_e}

    # ---- the other kernels of the path at this workload; the other BASELINE.json workloads; the driver loop
    kernels = extra = loops = variants = None
    extra_names = (args.extra_workloads.split(",") if args.extra_workloads
                   else ["cfg3_fp64", "cfg4_fp32", "cfg4_fp64"] if args.workload == "cfg3_fp32" else [])
    if world == 1 and not args.no_extra and plain_or and extra_names:
        culgt.culgt_unpack(lat, links, f.can_dev)        # the gauge-fixed field, as the canonical input of what follows
        variants = sweep_variants(culgt, torch, f, peak, max(args.extra_steps, 10))
        kernels = other_kernels(culgt, torch, f, peak)
        del f, links, ws
        torch.cuda.empty_cache()
        extra = []
        for name in extra_names:
            fx = Field(culgt, torch, name, rank)
            sx = torch.zeros(2, dtype=torch.float64, device="cuda")
            tx = time_sweep_loop(
                torch, fx, lambda n: culgt.culgt_or_sweeps(fx.lat, fx.links, n, fx.omega),
                lambda: culgt.culgt_gauge_precision_functional(fx.lat, fx.links, fx.ws, sx[0:1], sx[1:2]),
                args.extra_steps, 3, args.extra_steps, barrier, ClockSampler(local_rank))
            gbs = 2 * fx.field_bytes / (tx["launch_ms"] * 1e-3) / 1e9
            chk_us = 1e3 * tx["check_ms"] / tx["n_checks"]
            extra.append({
                "workload": workload_config(argparse.Namespace(**{**vars(args), "workload": name}), fx.cfg)["workload"],
                "steps": args.extra_steps, "value": fx.V * args.extra_steps / (tx["elapsed_ms"] * 1e-3), "unit": UNIT,
                "ms_per_step": tx["elapsed_ms"] / args.extra_steps, "launch_us": 1e3 * tx["launch_ms"],
                "roofline": {"bound": "hbm", "achieved": gbs, "peak": peak, "unit": "GB/s", "frac": gbs / peak,
                             "bytes_per_launch": 2 * fx.field_bytes},
                "theta_F": {"us": chk_us, "gbs": fx.field_bytes / (chk_us * 1e-6) / 1e9,
                            "frac": fx.field_bytes / (chk_us * 1e-6) / 1e9 / peak},
                "clocks": tx["clocks"], "final": {"theta": float(sx[0].item()), "F": float(sx[1].item())},
                "kernels": other_kernels(culgt, torch, fx, peak) if fx.V <= 32 ** 4 else None,
            })
            del fx, sx
            torch.cuda.empty_cache()
        loops = driver_loop_times(culgt, torch, rank)

    # ---- CPU baseline: the oracle on this host's cores (rank 0, N=1 only)
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        import oracle
        threads = min(oracle.max_threads(), os.cpu_count() or 1)
        dims = cfg["dims"]
        u0 = li.make_config(dims, cfg["group"], cfg["kind"], cfg["seed"], eps=cfg["eps"], scramble=cfg["scramble"])
        if cfg["precision"] == 32:
            u0 = li.round_to_fp32(u0)
        ur = li.to_real(u0)
        del u0
        v_all, n_all = time_oracle(dims, cfg["group"], ur, omega, 40, 12.0, threads, args.gauge)
        v_one, n_one = time_oracle(dims, cfg["group"], ur, omega, 3, 6.0, 1, args.gauge)
        cpu = {"value": v_all, "unit": UNIT, "cores": threads, "kind": "oracle",
               "sample": f"{n_all} full sweeps of the same {'x'.join(map(str, dims))} lattice on {threads} threads "
                         f"(fp64, canonical layout); one core: {v_one:.4g} site-updates/s over {n_one} sweep(s)",
               "one_core_value": v_one}

    if rank == 0:
        roofline = {"bound": "hbm", "achieved": achieved_gbs, "peak": peak, "unit": "GB/s",
                    "frac": achieved_gbs / peak, "traffic": traffic, "traffic_steady_state": steady,
                    "traffic_capture": traffic_info, "traffic_steady_state_capture": steady_info,
                    "kernel": kernel_name, "bytes_per_launch": alg_bytes_per_launch,
                    "launch_us": launch_ms * 1e3, "peak_source": peak_src,
                    "note": "achieved / frac count ALGORITHMIC bytes (the contract); the L2 serves part of them, "
                            "so frac can exceed 1 -- dram_achieved / dram_frac is what HBM itself moves",
                    "algorithmic_frac_of_8TBs_nominal": achieved_gbs / 8000.0}
        if steady is not None:
            dram_gbs = steady / (launch_ms * 1e-3) / 1e9
            roofline.update({"dram_achieved": dram_gbs, "dram_frac": dram_gbs / peak,
                             "dram_frac_of_8TBs_nominal": dram_gbs / 8000.0})
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": elapsed_max_ms / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32" if cfg["precision"] == 32 else "f64", "data": "synthetic",
            "config": workload_config(args, cfg),
            "gflops": value * flops_per_site(cfg, args.gauge) / 1e9,
            "algorithmic_gbs": value * 16 * (cfg["params"] * cfg["precision"] // 8) / 1e9,
            "gpu_launches": gpu_launches,
            "e2e": e2e,
            "roofline": roofline,
            "cpu_baseline": cpu,
            "clocks": clocks,
            "final": {"theta": theta, "F": F},
            "check_ms_total": check_ms, "variant": args.variant,
            "kernels": kernels, "sweep_variants": variants, "extra_workloads": extra, "driver_loop": loops,
            "context": {"paper": "470 GFlops at 80% of peak bandwidth on a GeForce GTX 580 (PAPER.md L7), context only"},
        }
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
