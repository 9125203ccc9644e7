#!/usr/bin/env python
"""Quick start: evolve a Gaussian wavepacket in a harmonic trap on one B200 and watch it move.

    python examples/quickstart.py

Everything numerical runs inside libts.so (include/ts.h); torch only owns the device memory.
"""
import math
import sys
from pathlib import Path

import torch

sys.path.insert(0, str(Path(__file__).resolve().parents[1]))
from paper_1208_2407_b200.binding import Plan      # noqa: E402

nx = ny = 2048
dev = torch.device("cuda:0")
x = torch.arange(nx, dtype=torch.float64, device=dev)[None, :]
y = torch.arange(ny, dtype=torch.float64, device=dev)[:, None]

# psi ~ exp(-r^2 / 4 sigma^2) exp(i k x), normalised
sigma, kx = 48.0, 0.4
env = torch.exp(-((x - 700) ** 2 + (y - 1024) ** 2) / (4 * sigma ** 2))
re, im = env * torch.cos(kx * x), env * torch.sin(kx * x)
norm = math.sqrt(float((re * re + im * im).sum()))
re, im = (re / norm).float().contiguous(), (im / norm).float().contiguous()

# harmonic trap V = w^2 r^2 / 2, passed as separable phase factors exp(-i V dt) = px(x) py(y)
w, dt = 2e-3, 1.0
vx = 0.5 * w * w * (x[0] - 1024) ** 2 * dt
vy = 0.5 * w * w * (y[:, 0] - 1024) ** 2 * dt
px = torch.stack([torch.cos(vx), -torch.sin(vx)]).float().contiguous()
py = torch.stack([torch.cos(vy), -torch.sin(vy)]).float().contiguous()

theta = 0.05                      # dt * |V_tunnel| / hbar
c = (math.cos(theta / 2), math.sin(theta / 2), math.cos(theta), math.sin(theta))
plan = Plan(nx, ny, torch.float32, "closed")
for k in range(5):
    prob = re * re + im * im
    print(f"step {200 * k:5d}  norm^2 {plan.norm(re, im):.9f}  <x> {float((prob * x).sum()):8.2f}"
          f"  <y> {float((prob * y).sum()):8.2f}")
    plan.evolve_sep(re, im, *c, px, py, n_steps=200)
torch.cuda.synchronize()
print("fused kernel used:", bool(plan.info("fused")), " steps per pass:", plan.info("fuse_steps"))
