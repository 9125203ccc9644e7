#!/usr/bin/env python
"""bench.py -- lattice site-steps/s of the fused second-order Trotter-Suzuki step on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C4] [--impl reference]

A "step" is one ts_evolve call with the workload's full step count (C4: 16384^2 fp32 periodic,
200 second-order steps) on a state already resident in HBM.  Timed with CUDA events on the
launch stream, barrier + synchronize on both sides, max over ranks.  The path does not shard
("replicas only"): with N GPUs every rank evolves its own lattice and the value
is the sum ("weak").  One JSON line is printed by rank 0.

`--impl reference` times the CPU oracle (oracle/ts_oracle.c, as it stands) on a bounded sample
of the same workload on the host cores; it is the only other place that executes oracle/.
"""
from __future__ import annotations

import argparse
import json
import math
import os
import subprocess
import sys
import threading
import time
from pathlib import Path

ROOT = Path(__file__).resolve().parent
sys.path.insert(0, str(ROOT))

METRIC = "lattice site-steps/sec"
UNIT = "site-steps/s"


def load_peaks():
    p = ROOT / "MEASURED_PEAKS.json"
    if p.exists():
        d = json.loads(p.read_text())
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


# Plain-ALU peak: 148 SMs x 4 sub-partitions x 32 fp32 FMA lanes (16 fp64) x 2 flop at
# the 1965 MHz maximum SM clock of the profiling guide -- derived, not measured.
SM_COUNT, SM_MAX_MHZ = 148, 1965.0
ALU_PEAK_TFLOPS = {"f32": SM_COUNT * 128 * 2 * SM_MAX_MHZ * 1e6 / 1e12,
                   "f64": SM_COUNT * 64 * 2 * SM_MAX_MHZ * 1e6 / 1e12}


def cpu_model():
    try:
        for ln in open("/proc/cpuinfo"):
            if ln.startswith("model name"):
                return ln.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (profiling recipe line)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                 "--format=csv,noheader,nounits", "-lms", "25"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except OSError:
            self.proc = None

    def _read(self):
        for ln in self.proc.stdout:
            self.rows.append((time.time(), ln.strip()))

    def stop(self, t0, t1):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        sm, smax, reasons = [], None, set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        rows = [r for (t, r) in self.rows if t0 - 0.05 <= t <= t1 + 0.15] or [r for _, r in self.rows]
        for r in rows:
            f = [x.strip() for x in r.split(",")]
            try:
                sm.append(float(f[0])); smax = float(f[1])
            except (ValueError, IndexError):
                continue
            for n, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": smax,
                "reasons": sorted(reasons), "samples": len(sm)}


def host_ram_bytes():
    try:
        for ln in open("/proc/meminfo"):
            if ln.startswith("MemAvailable"):
                return int(ln.split()[1]) * 1024
    except OSError:
        pass
    return 0


def oracle_sample(cfg_name, budget_site_steps, full_ok=False):
    """(config, steps) of the bounded oracle sample: the workload's own lattice when the budget and
    the host memory allow whole steps of it (C1-C3; C4: 2 steps of 16384^2, 4.3 GB of float64
    state, only when full_ok), else the workload's recipe on a 2048^2 lattice (the cost is linear
    in sites x steps)."""
    from paper_1208_2407_b200 import inputs
    cfg = inputs.CONFIGS[cfg_name]
    need = cfg.sites * 8 * (2 + (2 if cfg.has_pot else 0)) * 2.5      # float64 planes + generation
    ram = host_ram_bytes()
    if cfg.sites <= 2 ** 24 and cfg.sites <= budget_site_steps:                      # C1 - C3
        return cfg, max(1, min(cfg.n_steps, int(budget_site_steps // cfg.sites)))
    if full_ok and cfg.sites <= 2 ** 28 and 2 * cfg.sites <= budget_site_steps and need < 0.5 * ram:
        return cfg, 2                                                                # C4: 2 steps
    n = min(cfg.nx, 2048)
    small = inputs.scaled(cfg, n, n)
    steps = max(1, min(cfg.n_steps, int(budget_site_steps // small.sites)))
    return small, steps


def time_oracle(cfg_name, budget_site_steps, full_ok=False):
    """Times oracle.evolve as it stands on ONE thread and on all host cores; returns a dict."""
    import numpy as np
    import oracle
    from paper_1208_2407_b200 import inputs
    small, steps = oracle_sample(cfg_name, budget_site_steps, full_ok)
    re, im, _ = inputs.full_state(small)
    pot = inputs.full_pot(small)
    re = re.astype(np.float64); im = im.astype(np.float64)
    potd = None if pot is None else (pot[0].astype(np.float64), pot[1].astype(np.float64))
    c = small.coeffs()
    cores = oracle.num_threads()
    oracle.evolve(re, im, *c, pot=potd, periodic=small.periodic, n_steps=1)  # warm
    t = time.perf_counter()
    oracle.evolve(re, im, *c, pot=potd, periodic=small.periodic, n_steps=steps)
    dt_all = time.perf_counter() - t
    # one thread: a quarter of the steps (at least one); on a lattice of more than 2^24 sites one
    # step on its first 2048 rows (a contiguous slab: same row length, same cost per site)
    steps1 = max(1, steps // 4) if cores > 1 else steps
    re1, im1, pot1 = re, im, potd
    if small.sites > 2 ** 24:
        rows = 2048
        re1, im1 = re[:rows], im[:rows]
        pot1 = None if potd is None else (potd[0][:rows], potd[1][:rows])
        steps1 = 1
    oracle.set_num_threads(1)
    t = time.perf_counter()
    oracle.evolve(re1, im1, *c, pot=pot1, periodic=small.periodic, n_steps=steps1)
    dt_one = time.perf_counter() - t
    oracle.set_num_threads(cores)
    sites1 = re1.shape[0] * re1.shape[1]
    sample = (f"{small.nx}x{small.ny} {'(the full lattice)' if small.nx == inputs.CONFIGS[cfg_name].nx else 'sub-lattice'}"
              f" of the {cfg_name} recipe ({small.boundary}, "
              f"{'potential' if small.has_pot else 'no potential'}, float64), {steps} steps on "
              f"{cores} threads, {steps1} on one"
              + (" (first 2048 rows)" if sites1 != small.sites else ""))
    return {"value": small.sites * steps / dt_all, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": sample, "seconds": dt_all, "value_1thread": sites1 * steps1 / dt_one,
            "nproc": os.cpu_count(), "cpu_model": cpu_model()}


def run_reference(args):
    """The oracle as the reference arm: K timed 'steps', each a bounded sample of the workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    from paper_1208_2407_b200 import inputs
    import numpy as np
    import oracle
    cfg = inputs.CONFIGS[args.config]
    small, steps = oracle_sample(args.config, 6e7)
    re, im, _ = inputs.full_state(small)
    pot = inputs.full_pot(small)
    re = re.astype(np.float64); im = im.astype(np.float64)
    potd = None if pot is None else (pot[0].astype(np.float64), pot[1].astype(np.float64))
    c = small.coeffs()
    for _ in range(args.warmup):
        oracle.evolve(re, im, *c, pot=potd, periodic=small.periodic, n_steps=steps)
    t = time.perf_counter()
    for _ in range(args.steps):
        oracle.evolve(re, im, *c, pot=potd, periodic=small.periodic, n_steps=steps)
    dt = time.perf_counter() - t
    value = small.sites * steps * args.steps / dt
    sample = (f"{small.nx}x{small.ny} sub-lattice of the {cfg.name} recipe ({small.boundary}, "
              f"float64), {steps} second-order steps per bench step")
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic",
        "config": {"workload": workload_text(cfg), "sample": sample},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": oracle.num_threads(),
                         "kind": "oracle", "sample": sample, "nproc": os.cpu_count(),
                         "cpu_model": cpu_model()},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)
    return 0


def work_of(kind, cfg, sep, info, eb):
    """Algorithmic (bytes, flops) of ONE launch of a kernel kind.
    Bytes: every plane the launch must read and write once.  Flops: 2 FMAs = 4 flops per site and
    pair sweep in the scaled form; without a potential a sub-step is 2 sweeps per axis (adjacent
    half sweeps merged), with one it is 7 sweeps + the phase (2 FMA + 2 MUL) = 34 flops."""
    sites = cfg.sites
    state = 4 * eb * sites                       # read + write of both planes
    S = max(1, info["fuse_steps"])
    if kind in (2, 3):                           # fused / stream pass: S whole sub-steps
        planes = cfg.has_pot and not sep
        by = state + (2 * eb * sites if planes else 0)
        fl = sites * S * (34 if cfg.has_pot else 16)
        return by, fl
    if kind in (5, 6, 11):                       # resident lines: all sub-steps of one axis
        return state, sites * cfg.n_steps * 8
    if kind == 7:
        return state, sites * max(1, info["chain_x"]) * 8
    if kind == 8:
        return state, sites * max(1, info["chain_y"]) * 8
    if kind == 9:
        return state, 0
    if kind == 4:                                # whole evolution on chip
        return state, sites * cfg.n_steps * (34 if cfg.has_pot else 16)
    if kind == 1:                                # per-sweep kernels of the whole call
        sweeps = 9 if cfg.has_pot else 7
        return state * sweeps * cfg.n_steps, sites * cfg.n_steps * (34 if cfg.has_pot else 28)
    return state, 0


def roofline_of(cfg, sep, info, per_kind, calls, hbm_peak, peak_src, call_ms):
    """The roofline object of the bench line: the kernel kind with the largest share of the call,
    its own average event time, and whichever of HBM and plain ALU binds it."""
    from paper_1208_2407_b200.binding import LAUNCH_KINDS
    eb = 4 if cfg.dtype == "f32" else 8
    alu_peak = ALU_PEAK_TFLOPS[cfg.dtype]
    if not per_kind:
        return {"bound": "hbm", "achieved": None, "peak": hbm_peak, "unit": "GB/s", "frac": None,
                "traffic": None, "note": "no launch times recorded"}
    shares = {k: sum(v) / calls for k, v in per_kind.items()}
    total = sum(shares.values())
    floor_ms = 0.0
    kernels = []
    for k, v in sorted(per_kind.items(), key=lambda kv: -sum(kv[1])):
        by, fl = work_of(k, cfg, sep, info, eb)
        avg = sum(v) / len(v)
        t_hbm = by / (hbm_peak * 1e9) * 1e3
        t_alu = fl / (alu_peak * 1e12) * 1e3
        floor_ms += max(t_hbm, t_alu) * len(v) / calls
        kernels.append({"kernel": LAUNCH_KINDS.get(k, str(k)), "launches_per_call": len(v) // calls,
                        "avg_ms": avg, "share": shares[k] / total,
                        "hbm_frac": t_hbm / avg, "alu_frac": t_alu / avg,
                        "GB/s": by / avg / 1e6, "TFLOP/s": fl / avg / 1e9})
    top = kernels[0]
    kind = max(shares, key=shares.get)
    by, fl = work_of(kind, cfg, sep, info, eb)
    bound = "alu" if top["alu_frac"] > top["hbm_frac"] else "hbm"
    traffic = tsrc = None
    tp = ROOT / "profiles" / "traffic.json"
    key = f"{cfg.name}:{top['kernel']}"
    if tp.exists():
        try:
            traffic = json.loads(tp.read_text()).get(key)
            tsrc = f"profiles/traffic.json[{key}]: one ncu --set full capture of this kernel, not this run"
        except (ValueError, OSError):
            traffic = None
    chain = {5: cfg.n_steps, 6: cfg.n_steps, 7: info["chain_x"], 8: info["chain_y"]}.get(
        kind, max(1, info["fuse_steps"]))
    roof = {
        "bound": bound,
        "achieved": top["TFLOP/s"] if bound == "alu" else top["GB/s"],
        "peak": alu_peak if bound == "alu" else hbm_peak,
        "unit": "TFLOP/s" if bound == "alu" else "GB/s",
        "frac": top["alu_frac"] if bound == "alu" else top["hbm_frac"],
        "traffic": traffic, "traffic_source": tsrc,
        "kernel": f"{top['kernel']}<{cfg.dtype}>, {chain} sub-steps per launch",
        "launch_ms": top["avg_ms"], "launches_per_call": top["launches_per_call"],
        "share_of_call": top["share"],
        "bytes_per_launch": by, "flops_per_launch": fl,
        "peak_source": (f"HBM: {peak_src}; ALU: derived, {SM_COUNT} SMs x "
                        f"{128 if cfg.dtype == 'f32' else 64} FMA lanes x 2 x {SM_MAX_MHZ:.0f} MHz"),
        "hbm": {"achieved": top["GB/s"], "peak": hbm_peak, "frac": top["hbm_frac"],
                "frac_of_8TBs_nominal": top["GB/s"] / 8000.0},
        "alu": {"achieved": top["TFLOP/s"], "peak": alu_peak, "frac": top["alu_frac"]},
        "kernels": kernels,
        # the whole call against the sum over its launches of max(HBM time, ALU time)
        "call": {"event_ms_sum": total, "call_ms": call_ms, "roofline_ms": floor_ms,
                 "frac": floor_ms / call_ms},
    }
    return roof


def workload_text(cfg):
    return (f"{cfg.name}: {cfg.nx}x{cfg.ny} {cfg.dtype} {cfg.boundary}, "
            f"{'harmonic potential' if cfg.has_pot else 'no potential'}, theta={cfg.theta}, "
            f"{cfg.n_steps} second-order steps per ts_evolve call")


def run_gpu(args):
    import torch
    from paper_1208_2407_b200 import inputs
    from paper_1208_2407_b200.binding import Plan
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)

    cfg = inputs.CONFIGS[args.config]
    if args.scale:
        # the config's recipe on an N x N lattice (not one of BASELINE.json's workloads: a size
        # sweep of the same path; cpu_baseline then uses its bounded sample)
        cfg = inputs.scaled(cfg, args.scale, args.scale)
    tdt = torch.float32 if cfg.dtype == "f32" else torch.float64
    eb = 4 if cfg.dtype == "f32" else 8
    re, im, _ = inputs.device_state(cfg, dev)
    pot = inputs.device_pot(cfg, dev)
    sep = None
    if args.sep:
        if not cfg.has_pot:
            raise SystemExit("--sep needs a config with a potential (C3, C5)")
        sx, sy = inputs.sep_pot(cfg)
        sep = (torch.from_numpy(sx).to(dev), torch.from_numpy(sy).to(dev))
        pot = None
    plan = Plan(cfg.nx, cfg.ny, tdt, cfg.boundary)
    if args.fuse_steps:
        plan.set_option("fuse_steps", args.fuse_steps)
    if args.seg_rows:
        plan.set_option("seg_rows", args.seg_rows)
    if args.chain:
        plan.set_option("chain", args.chain)
    if args.variant:
        plan.set_option("variant", args.variant)
    if args.ring_slots:
        plan.set_option("ring_slots", args.ring_slots)
    c = cfg.coeffs()
    stream = torch.cuda.current_stream()

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    def evolve_once():
        if sep is not None:
            plan.evolve_sep(re, im, *c, sep[0], sep[1], n_steps=cfg.n_steps, stream=stream)
        else:
            plan.evolve(re, im, *c, pot_phase=pot, n_steps=cfg.n_steps, stream=stream)

    n0 = plan.norm(re, im)
    for _ in range(args.warmup):
        evolve_once()
    barrier()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
        time.sleep(0.25)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    t0 = time.time()
    e0.record(stream)
    for _ in range(args.steps):
        evolve_once()
    e1.record(stream)
    barrier()
    t1 = time.time()
    ms = e0.elapsed_time(e1)
    clocks = sampler.stop(t0, t1) if rank == 0 else None
    if dist is not None:
        t = torch.tensor([ms], device=dev, dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms = float(t.item())
    n1 = plan.norm(re, im)
    info = {k: plan.info(k) for k in ("fused", "fuse_steps", "passes", "launches", "seg_rows",
                                     "variant", "chain_x", "chain_y")}
    value = world * cfg.sites * cfg.n_steps * args.steps / (ms * 1e-3)

    # per-kernel device times of the same call: the library brackets every launch with CUDA events
    # on the launch stream (plan option "timing"); a few calls right after the timed region,
    # same clocks and thermal state.  The timed region above runs without them.
    plan.set_option("timing", 1)
    per_kind = {}
    timing_calls = max(1, min(args.steps, 3))
    for _ in range(timing_calls):
        evolve_once()
        torch.cuda.synchronize()
        for kind, kms in plan.launch_times():
            per_kind.setdefault(kind, []).append(kms)
    plan.set_option("timing", 0)

    # end to end through ts_evolve_host: pinned host planes, H2D + D2H inside the timed region
    hre = torch.empty((cfg.ny, cfg.nx), dtype=tdt, pin_memory=True)
    him = torch.empty((cfg.ny, cfg.nx), dtype=tdt, pin_memory=True)
    hre.copy_(re); him.copy_(im)
    hpot = None
    if pot is not None:
        hpot = torch.empty(pot.shape, dtype=tdt, pin_memory=True)
        hpot.copy_(pot)
    e2e_reps = max(1, min(args.steps, 3))
    if sep is None:
        del re, im
        torch.cuda.empty_cache()
        e2e_call = lambda: plan.evolve_host(hre, him, *c, pot_phase=hpot, n_steps=cfg.n_steps)
        e2e_api = "ts_evolve_host (pinned host planes)"
    else:
        # separable entry: the state and the two phase vectors go up, the state comes back
        hsx = sep[0].cpu().pin_memory(); hsy = sep[1].cpu().pin_memory()

        def e2e_call():
            re.copy_(hre, non_blocking=True); im.copy_(him, non_blocking=True)
            sep[0].copy_(hsx, non_blocking=True); sep[1].copy_(hsy, non_blocking=True)
            plan.evolve_sep(re, im, *c, sep[0], sep[1], n_steps=cfg.n_steps, stream=stream)
            hre.copy_(re, non_blocking=True); him.copy_(im, non_blocking=True)
            torch.cuda.synchronize()
        e2e_api = "Plan.evolve_sep between pinned-host copies of the state and the phase vectors"
    e2e_call()    # warm (allocations)
    barrier()
    t = time.perf_counter()
    for _ in range(e2e_reps):
        e2e_call()
    barrier()
    e2e_s = (time.perf_counter() - t) / e2e_reps
    if dist is not None:
        tt = torch.tensor([e2e_s], device=dev, dtype=torch.float64)
        dist.all_reduce(tt, op=dist.ReduceOp.MAX)
        e2e_s = float(tt.item())
    e2e_val = world * cfg.sites * cfg.n_steps / e2e_s
    h2d = (2 + (2 if pot is not None else 0)) * cfg.sites * eb
    if sep is not None:
        h2d += 2 * (cfg.nx + cfg.ny) * eb
    d2h = 2 * cfg.sites * eb

    if rank != 0:
        return 0
    peak, peak_src = load_peaks()
    S = max(1, info["fuse_steps"])
    passes = max(1, info["passes"])
    roof = roofline_of(cfg, sep is not None, info, per_kind, timing_calls, peak, peak_src,
                       ms / args.steps)
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": cfg.dtype, "data": "synthetic",
        "config": {"workload": workload_text(cfg) + (" (separable factors, ts_evolve_sep)"
                                                     if sep is not None else ""),
                   "variant": {0: "per-sweep kernels", 1: "fused_kernel", 2: "stream_kernel",
                               3: "tiny_kernel", 4: "axis-split"}.get(info["variant"]),
                   "fuse_steps": S, "passes_per_call": passes,
                   "chain_x": info["chain_x"], "chain_y": info["chain_y"],
                   "seg_rows": info["seg_rows"], "fused": info["fused"],
                   "parallelism": "replicas only (no sharding of one lattice)",
                   "l2": ("state (2 planes x 2 buffers) far larger than the 126 MB L2; no flush"
                          if cfg.sites * eb * 4 > 2 * 126e6 else
                          "state fits the 126 MB L2 (the workload IS the L2-resident case; no flush)"),
                   "norm2_before": n0, "norm_drift": n1 / n0 - 1},
        "clocks": clocks,
        "e2e": {"value": e2e_val, "unit": UNIT, "h2d_bytes_per_step": h2d,
                "d2h_bytes_per_step": d2h, "ms_per_step": e2e_s * 1e3,
                "api": e2e_api,
                "note": "PCIe-bound: without a potential the planes go up in 8 row pieces and the row chain of a piece runs under the upload of the next; the column passes and the download are serial"},
        "gpu_launches": info["launches"] * args.steps,
        "roofline": roof,
        "cpu_baseline": time_oracle(args.config, args.cpu_budget, full_ok=True),
    }
    print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()
    return 0


def run_gpu_3d(args):
    """--lattice3d N: an N^3 fp32 lattice (the 3-D extension), periodic, seeded
    uniform state as in C4, theta = 0.02, 100 second-order steps per ts_evolve_3d call; with
    --pot3d a seeded random phase field.  Not one of BASELINE.json's configs: a bench line for the
    SURVEY 8(f) NEXT-4 row, same metric."""
    import torch
    from paper_1208_2407_b200.binding import Plan3D, LAUNCH_KINDS
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback")
    dev = torch.device("cuda", int(os.environ.get("LOCAL_RANK", "0")))
    torch.cuda.set_device(dev)
    n, n_steps, theta = args.lattice3d, 100, 0.02
    if args.pot3d:
        n_steps = 20
    g = torch.Generator(device=dev); g.manual_seed(12082407)
    re = torch.rand((n, n, n), device=dev, generator=g) * 2 - 1
    im = torch.rand((n, n, n), device=dev, generator=g) * 2 - 1
    nrm = float(torch.sqrt((re.double() ** 2 + im.double() ** 2).sum()))
    re /= nrm; im /= nrm
    pot = None
    if args.pot3d:
        V = torch.rand((n, n, n), device=dev, generator=g, dtype=torch.float64) * 6.28
        pot = torch.stack([torch.cos(V), -torch.sin(V)]).float().contiguous()
        del V
    plan = Plan3D(n, n, n, torch.float32, "periodic")
    c = (math.cos(theta / 2), math.sin(theta / 2), math.cos(theta), math.sin(theta))
    stream = torch.cuda.current_stream()
    call = lambda: plan.evolve(re, im, *c, pot_phase=pot, n_steps=n_steps, stream=stream)
    n0 = plan.norm(re, im)
    for _ in range(args.warmup):
        call()
    torch.cuda.synchronize()
    sampler = ClockSampler(dev.index or 0)
    sampler.start(); time.sleep(0.25)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t0 = time.time()
    e0.record(stream)
    for _ in range(args.steps):
        call()
    e1.record(stream)
    torch.cuda.synchronize()
    t1 = time.time()
    ms = e0.elapsed_time(e1)
    clocks = sampler.stop(t0, t1)
    n1 = plan.norm(re, im)
    plan.set_option("timing", 1)
    call(); torch.cuda.synchronize()
    per_kind = {}
    for kind, kms in plan.launch_times():
        per_kind.setdefault(kind, []).append(kms)
    plan.set_option("timing", 0)
    sites = n ** 3
    peak, peak_src = load_peaks()
    alu = ALU_PEAK_TFLOPS["f32"]
    kernels = []
    for k, v in sorted(per_kind.items(), key=lambda kv: -sum(kv[1])):
        by = sites * (16 + (8 if (pot is not None and k == 11) else 0))
        fl = sites * 8 * n_steps if pot is None else sites * (12 + (6 if k == 11 else 0))
        avg = sum(v) / len(v)
        kernels.append({"kernel": LAUNCH_KINDS.get(k, str(k)), "launches_per_call": len(v),
                        "avg_ms": avg, "hbm_frac": by / (peak * 1e9) * 1e3 / avg,
                        "alu_frac": fl / (alu * 1e12) * 1e3 / avg})
    top = kernels[0]
    bound = "alu" if top["alu_frac"] > top["hbm_frac"] else "hbm"
    line = {
        "metric": METRIC, "value": sites * n_steps * args.steps / (ms * 1e-3), "unit": UNIT,
        "n_gpus": 1, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
        "data": "synthetic",
        "config": {"workload": f"3-D {n}^3 f32 periodic, {'random phase field' if pot is not None else 'no potential'}, "
                               f"theta={theta}, {n_steps} second-order steps per ts_evolve_3d call",
                   "variant": plan.info("variant"), "launches_per_call": plan.info("launches"),
                   "norm2_before": n0, "norm_drift": n1 / n0 - 1,
                   "l2": "state far larger than the 126 MB L2; no flush" if sites * 8 > 2.5e8 else
                         "state comparable to the 126 MB L2"},
        "clocks": clocks, "gpu_launches": plan.info("launches") * args.steps,
        "roofline": {"bound": bound, "frac": top["alu_frac"] if bound == "alu" else top["hbm_frac"],
                     "peak": alu if bound == "alu" else peak,
                     "unit": "TFLOP/s" if bound == "alu" else "GB/s",
                     "achieved": (top["alu_frac"] * alu) if bound == "alu" else top["hbm_frac"] * peak,
                     "traffic": None, "kernel": top["kernel"], "kernels": kernels,
                     "peak_source": peak_src},
    }
    print(json.dumps(line), flush=True)
    return 0


def run_gpu_slab(args):
    """ONE lattice cut into row slabs (paper_1208_2407_b200/slab.py): with N > 1 ranks the global
    lattice is nx x (ny * N) (weak scaling: every rank owns a slab of the config's size) and halos
    travel over NCCL; with --slabs R on one GPU the config's lattice is cut into R slabs stepped in
    turn (measures the cost of the decomposition itself: halo recomputation + exchange copies)."""
    import torch
    from paper_1208_2407_b200 import inputs, slab
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    dist = None
    if world > 1:
        # the communicator lines (ranks, rings / NVLS, peer access) go to stderr, so that a scaling
        # run can be checked; stdout stays the one JSON line
        os.environ.setdefault("NCCL_DEBUG", "INFO")
        os.environ.setdefault("NCCL_DEBUG_SUBSYS", "INIT")
        os.environ.setdefault("NCCL_DEBUG_FILE", "/dev/stderr")
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)
    cfg = inputs.CONFIGS[args.config]
    tdt = torch.float32 if cfg.dtype == "f32" else torch.float64
    eb = 4 if cfg.dtype == "f32" else 8
    re, im, _ = inputs.device_state(cfg, dev)
    pot = inputs.device_pot(cfg, dev)
    k = args.exchange_every or slab.default_steps_per_exchange(tdt, pot is not None)
    c = cfg.coeffs()
    fused_halo = args.slab_mode == "peer"
    sep = None
    if fused_halo and pot is not None:
        # ts_slab_pass takes the potential as separable factors (the harmonic trap is separable)
        stacked = inputs.scaled(cfg, cfg.nx, cfg.ny * world) if world > 1 else cfg
        sx, sy = inputs.sep_pot(stacked)
        sep = (torch.from_numpy(sx).to(dev), torch.from_numpy(sy).to(dev))
        pot = None
    if fused_halo and world > 1:
        # one process per GPU, buffers in symmetric memory, halos read over NVLink in the kernel
        obj = slab.PeerRank(cfg.nx, cfg.ny * world, tdt, cfg.boundary)
        obj.slab.set_state(re, im)
        if sep is not None:
            obj.set_separable_potential(*sep)
        evolve = lambda: obj.evolve(c, cfg.n_steps)
        norm = obj.norm
        plans = [obj.slab.plan]
        n_slabs, halo, k = world, 2 * obj.S, obj.S
    elif fused_halo:
        obj = slab.PeerGroup(cfg.nx, cfg.ny, tdt, cfg.boundary, max(1, args.slabs), dev)
        if sep is not None:
            obj.scatter(re, im, *sep)
        else:
            obj.scatter(re, im)
        evolve = lambda: obj.evolve(c, cfg.n_steps)
        norm = obj.norm
        plans = [s.plan for s in obj.slabs]
        n_slabs, halo, k = len(obj.slabs), 2 * obj.S, obj.S
    elif world > 1:
        comm = slab.DistComm()
        obj = slab.Slab(cfg.nx, cfg.ny * world, tdt, cfg.boundary, rank, world, k, device=dev)
        obj.set_state(re, im)
        if pot is not None:
            obj.set_potential(pot, comm)
        evolve = lambda: obj.evolve(c, cfg.n_steps, comm)
        norm = lambda: obj.norm(comm)
        plans = [obj.plan]
        n_slabs, halo = world, obj.H
    else:
        obj = slab.LocalGroup(cfg.nx, cfg.ny, tdt, cfg.boundary, max(1, args.slabs), k, device=dev)
        obj.scatter(re, im, pot)
        evolve = lambda: obj.evolve(c, cfg.n_steps)
        norm = obj.norm
        plans = [s.plan for s in obj.slabs]
        n_slabs, halo = len(obj.slabs), obj.slabs[0].H
    del re, im, pot
    torch.cuda.empty_cache()

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    n0 = norm()
    for _ in range(args.warmup):
        evolve()
    barrier()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
        time.sleep(0.25)
    stream = torch.cuda.current_stream()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    t0 = time.time()
    e0.record(stream)
    for _ in range(args.steps):
        evolve()
    e1.record(stream)
    barrier()
    t1 = time.time()
    ms = e0.elapsed_time(e1)
    clocks = sampler.stop(t0, t1) if rank == 0 else None
    if dist is not None:
        t = torch.tensor([ms], device=dev, dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms = float(t.item())
    n1 = norm()
    S = obj.S if fused_halo else max(1, plans[0].info("fuse_steps"))
    periods = -(-cfg.n_steps // k)
    launches = sum(p.info("launches") for p in plans) * periods      # last period may be shorter
    sites = cfg.sites * world
    value = sites * cfg.n_steps * args.steps / (ms * 1e-3)
    if rank != 0:
        return 0
    peak, peak_src = load_peaks()
    bytes_per_site_step = (4 * eb + (2 * eb if (cfg.has_pot and not fused_halo) else 0)) / S
    achieved = value / world * bytes_per_site_step / 1e9
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": cfg.dtype, "data": "synthetic",
        "config": {"workload": workload_text(cfg) + (f", stacked {world}x in y" if world > 1 else ""),
                   "parallelism": (f"row slabs x{n_slabs}, halo {halo} rows "
                                   + ("read from the neighbours inside the kernel (ts_slab_pass) "
                                      f"every pass of {k} steps" if fused_halo else
                                      f"exchanged every {k} steps")
                                   + ((" over NVLink peer memory" if fused_halo else " over NCCL")
                                      if world > 1 else " (one GPU, slabs stepped in turn)")),
                   "fuse_steps": S, "norm2_before": n0, "norm_drift": n1 / n0 - 1,
                   "l2": "state far larger than the 126 MB L2; no flush",
                   "note": ("N > 1 had NOT RUN on hardware when this was written (rounds 1-2 had "
                            "one-GPU boxes only): NCCL halo exchange / symmetric-memory peer halos "
                            "are covered by gloo and one-device tests, DESIGN.md 8") if world > 1
                   else "one GPU: all slabs stepped in turn"},
        "clocks": clocks, "gpu_launches": launches * args.steps,
        "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s",
                     "frac": achieved / peak, "traffic": None,
                     "kernel": f"stream_kernel<{cfg.dtype}, S={S}> on slabs (per GPU, whole call "
                               "incl. halo exchange)", "peak_source": peak_src},
    }
    print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="C4", choices=["C1", "C2", "C3", "C4", "C5"])
    ap.add_argument("--fuse-steps", type=int, default=0)
    ap.add_argument("--seg-rows", type=int, default=0)
    ap.add_argument("--lattice3d", type=int, default=0, help="bench an N^3 fp32 lattice (ts_evolve_3d)")
    ap.add_argument("--pot3d", action="store_true", help="with --lattice3d: a phase field")
    ap.add_argument("--chain", type=int, default=0, help="axis-split path: sub-steps per pass")
    ap.add_argument("--variant", type=int, default=0, help="plan option variant (0 = default path)")
    ap.add_argument("--ring-slots", type=int, default=0, help="TMA ring: state row-pair slots per warp")
    ap.add_argument("--scale", type=int, default=0,
                    help="run the config's recipe on an N x N lattice instead (size sweeps)")
    ap.add_argument("--decomp", default="replicas", choices=["replicas", "slab"],
                    help="N > 1: independent lattices per GPU (default, north_star) or one lattice "
                         "cut into row slabs with NCCL halo exchange")
    ap.add_argument("--slabs", type=int, default=0,
                    help="N = 1: cut the lattice into this many slabs on the one GPU")
    ap.add_argument("--slab-mode", default="exchange", choices=["exchange", "peer"],
                    help="slabs: halo exchange step + ts_evolve, or ts_slab_pass reading the "
                         "neighbours' rows inside the kernel (no potential)")
    ap.add_argument("--exchange-every", type=int, default=0, help="steps between halo exchanges")
    ap.add_argument("--sep", action="store_true",
                    help="C3/C5: pass the harmonic potential as separable factors (ts_evolve_sep)")
    ap.add_argument("--cpu-budget", type=float, default=1.5e9,
                    help="site-steps of oracle work in the cpu_baseline leg")
    args = ap.parse_args()
    if args.warmup < 3:
        args.warmup = 3
    if args.impl == "reference":
        return run_reference(args)
    if args.lattice3d:
        return run_gpu_3d(args)
    if args.decomp == "slab" or args.slabs > 1 or args.slab_mode == "peer":
        return run_gpu_slab(args)
    return run_gpu(args)


if __name__ == "__main__":
    sys.exit(main())
