"""Timing probe for tuning the plan options (the sweeps under profiles/*_probe.txt).

    python -m paper_1208_2407_b200.probe [--u4] SPEC [SPEC ...]

    SPEC = nx,dtype,boundary,pot,S,seg,slots[,steps[,ny]]
           dtype f32|f64; boundary closed|periodic; pot 0 none, 1 phase planes, 2 separable;
           S = fuse_steps, seg = seg_rows, slots = ring_slots (0 = the library's default);
           steps per ts_evolve call (default 6 passes' worth); ny defaults to nx.

Each line times one ts_evolve call (2 warm-up calls, then best and mean of 5, CUDA events on the
current stream) on seeded uniform random planes and prints the rate, the algorithmic bytes moved
per second (16 / 24 B per site and pass in fp32, twice that in fp64) and the norm drift.
--u4 times ts_evolve_u4 instead (rate in fourth-order steps).  Needs a GPU; argument marshalling
and timing only -- the arithmetic is in libts.so.
"""
from __future__ import annotations

import math
import sys


def _inputs(torch, dev, nx, ny, dt, pot):
    g = torch.Generator(device=dev)
    g.manual_seed(1)
    re = torch.rand((ny, nx), device=dev, dtype=dt, generator=g) * 2 - 1
    im = torch.rand((ny, nx), device=dev, dtype=dt, generator=g) * 2 - 1
    ph = None
    if pot == 2:
        vx = torch.rand((nx,), device=dev, dtype=torch.float64, generator=g) * 6
        vy = torch.rand((ny,), device=dev, dtype=torch.float64, generator=g) * 6
        ph = (torch.stack([torch.cos(vx), -torch.sin(vx)]).to(dt).contiguous(),
              torch.stack([torch.cos(vy), -torch.sin(vy)]).to(dt).contiguous())
    elif pot == 1:
        v = torch.rand((ny, nx), device=dev, dtype=torch.float64, generator=g) * 6
        ph = torch.stack([torch.cos(v), -torch.sin(v)]).to(dt).contiguous()
    return re, im, ph


def run(spec: str, u4: bool, cache: dict) -> str:
    import torch
    from .binding import Plan
    dev = torch.device("cuda:0")
    f = spec.split(",")
    nx = int(f[0])
    dt = torch.float32 if f[1] == "f32" else torch.float64
    bnd, pot, S, seg, slots = f[2], int(f[3]), int(f[4]), int(f[5]), int(f[6])
    steps = int(f[7]) if len(f) > 7 else 0
    ny = int(f[8]) if len(f) > 8 else nx
    key = (nx, ny, dt, pot)
    if key not in cache:
        cache.clear()
        torch.cuda.empty_cache()
        cache[key] = _inputs(torch, dev, nx, ny, dt, pot)
    re, im, ph = cache[key]
    plan = Plan(nx, ny, dt, bnd)
    plan.set_option("fuse_steps", S)
    plan.set_option("seg_rows", seg)
    plan.set_option("ring_slots", slots)
    theta = 0.02
    c = (math.cos(theta / 2), math.sin(theta / 2), math.cos(theta), math.sin(theta))
    if steps == 0:
        steps = max(S, 1) * 6 if S else 24

    def call():
        if u4:
            plan.evolve_u4(re, im, theta, None, None, n_steps=steps)
        elif pot == 2:
            plan.evolve_sep(re, im, *c, ph[0], ph[1], n_steps=steps)
        else:
            plan.evolve(re, im, *c, pot_phase=ph, n_steps=steps)

    n0 = plan.norm(re, im)
    for _ in range(2):
        call()
    torch.cuda.synchronize()
    best, tot, reps = 1e30, 0.0, 5
    for _ in range(reps):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        call()
        e1.record()
        torch.cuda.synchronize()
        t = e0.elapsed_time(e1)
        best, tot = min(best, t), tot + t
    n1 = plan.norm(re, im)
    passes = plan.info("passes")
    el = 4 if dt == torch.float32 else 8
    bytes_pass = nx * ny * el * (4 + (2 if pot == 1 else 0))
    line = (f"{spec:40s} S={plan.info('fuse_steps')} seg={plan.info('seg_rows')} passes={passes} "
            f"best {best:8.3f} ms avg {tot / reps:8.3f} ms {nx * ny * steps / best * 1e3:.3e} "
            f"site-steps/s  alg {bytes_pass * passes / best / 1e6:7.1f} GB/s  drift {n1 / n0 - 1:+.2e}")
    plan.destroy()
    return line


def main(argv) -> int:
    u4 = "--u4" in argv
    specs = [a for a in argv if not a.startswith("--")]
    if not specs:
        print(__doc__)
        return 2
    cache: dict = {}
    for spec in specs:
        try:
            print(run(spec, u4, cache), flush=True)
        except Exception as ex:          # keep sweeping: one bad spec must not lose the others
            print(spec, "FAILED", ex, flush=True)
    return 0


if __name__ == "__main__":
    sys.exit(main(sys.argv[1:]))
