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


def oracle_sample(cfg_name, budget_site_steps):
    """(config, steps) of the bounded oracle sample: the workload's recipe on a smaller lattice."""
    from paper_1208_2407_b200 import inputs
    cfg = inputs.CONFIGS[cfg_name]
    n = min(cfg.nx, 2048)
    small = inputs.scaled(cfg, n, n)
    steps = max(1, min(cfg.n_steps, int(budget_site_steps // small.sites)))
    return small, steps


def time_oracle(cfg_name, budget_site_steps, repeats=1):
    """Times oracle.evolve as it stands on all host cores; returns (rate, cores, sample text, s)."""
    import numpy as np
    import oracle
    from paper_1208_2407_b200 import inputs
    small, steps = oracle_sample(cfg_name, budget_site_steps)
    re, im, _ = inputs.full_state(small)
    pot = inputs.full_pot(small)
    re = re.astype(np.float64); im = im.astype(np.float64)
    potd = None if pot is None else (pot[0].astype(np.float64), pot[1].astype(np.float64))
    oracle.evolve(re, im, *small.coeffs(), pot=potd, periodic=small.periodic, n_steps=1)  # warm
    best = None
    for _ in range(repeats):
        t = time.perf_counter()
        oracle.evolve(re, im, *small.coeffs(), pot=potd, periodic=small.periodic, n_steps=steps)
        dt = time.perf_counter() - t
        best = dt if best is None else min(best, dt)
    rate = small.sites * steps / best
    sample = (f"{small.nx}x{small.ny} sub-lattice of the {cfg_name} recipe ({small.boundary}, "
              f"{'potential' if small.has_pot else 'no potential'}, float64), {steps} steps")
    return rate, oracle.num_threads(), sample, best


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
                         "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)
    return 0


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
                                     "variant")}
    value = world * cfg.sites * cfg.n_steps * args.steps / (ms * 1e-3)

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
    # algorithmic bytes of one fused launch: read + write both planes once (+ phase planes once)
    bytes_per_launch = cfg.sites * (4 * eb + (2 * eb if (cfg.has_pot and sep is None) else 0))
    launch_ms = ms / (args.steps * passes)
    achieved = bytes_per_launch / (launch_ms * 1e-3) / 1e9
    traffic = None
    tp = ROOT / "profiles" / "traffic.json"
    if tp.exists():
        try:
            traffic = json.loads(tp.read_text()).get(f"{cfg.name}_S{S}")
        except (ValueError, OSError):
            traffic = None
    cpu_rate, cores, sample, cpu_s = time_oracle(args.config, args.cpu_budget)
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": cfg.dtype, "data": "synthetic",
        "config": {"workload": workload_text(cfg) + (" (separable factors, ts_evolve_sep)"
                                                     if sep is not None else ""),
                   "fuse_steps": S, "passes_per_call": passes,
                   "seg_rows": info["seg_rows"], "fused": info["fused"],
                   "parallelism": "replicas only (no sharding of one lattice)",
                   "l2": "state (2 planes x 2 buffers) far larger than the 126 MB L2; no flush",
                   "norm2_before": n0, "norm_drift": n1 / n0 - 1},
        "clocks": clocks,
        "e2e": {"value": e2e_val, "unit": UNIT, "h2d_bytes_per_step": h2d,
                "d2h_bytes_per_step": d2h, "ms_per_step": e2e_s * 1e3,
                "api": e2e_api},
        "gpu_launches": info["launches"] * args.steps,
        "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s",
                     "frac": achieved / peak, "traffic": traffic,
                     "kernel": f"{'stream_kernel' if info['variant'] == 2 else 'fused_kernel'}"
                               f"<{cfg.dtype}, S={S}>",
                     "bytes_per_launch": bytes_per_launch, "launch_ms": launch_ms,
                     "peak_source": peak_src,
                     "site_step_roofline": peak * 1e9 / (bytes_per_launch / cfg.sites / S),
                     "frac_of_8TBs_nominal": achieved / 8000.0},
        "cpu_baseline": {"value": cpu_rate, "unit": UNIT, "cores": cores, "kind": "oracle",
                         "sample": sample, "seconds": cpu_s},
    }
    print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()
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
                   "l2": "state far larger than the 126 MB L2; no flush"},
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
    if args.decomp == "slab" or args.slabs > 1 or args.slab_mode == "peer":
        return run_gpu_slab(args)
    return run_gpu(args)


if __name__ == "__main__":
    sys.exit(main())
