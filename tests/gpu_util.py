"""Helpers for the -m gpu parity tests: run the CUDA path through the C ABI, run the oracle on the
same (already cast) inputs, compare element by element."""
from __future__ import annotations

import numpy as np

import oracle
from paper_1208_2407_b200 import inputs


def torch_dtype(cfg):
    import torch
    return torch.float32 if cfg.dtype == "f32" else torch.float64


def gpu_evolve(cfg, re_np, im_np, pot_np=None, n_steps=None, path=0, fuse=0, seg_rows=0,
               coeffs=None, variant=0, ring_slots=0, chain=0):
    """Upload, ts_evolve, download.  Returns (re, im, info dict)."""
    import torch
    from paper_1208_2407_b200.binding import Plan
    dev = torch.device("cuda:0")
    plan = Plan(cfg.nx, cfg.ny, torch_dtype(cfg), cfg.boundary)
    plan.set_option("path", path)
    plan.set_option("fuse_steps", fuse)
    plan.set_option("seg_rows", seg_rows)
    plan.set_option("variant", variant)
    plan.set_option("ring_slots", ring_slots)
    plan.set_option("chain", chain)
    re = torch.from_numpy(np.ascontiguousarray(re_np)).to(dev)
    im = torch.from_numpy(np.ascontiguousarray(im_np)).to(dev)
    pot = None if pot_np is None else torch.from_numpy(np.ascontiguousarray(pot_np)).to(dev)
    n = cfg.n_steps if n_steps is None else n_steps
    c = cfg.coeffs() if coeffs is None else coeffs
    n2_before = plan.norm(re, im)
    plan.evolve(re, im, *c, pot_phase=pot, n_steps=n)
    torch.cuda.synchronize()
    n2_after = plan.norm(re, im)
    info = {k: plan.info(k) for k in ("fused", "fuse_steps", "passes", "launches", "seg_rows",
                                     "variant", "chain_x", "chain_y")}
    info["norm2_before"], info["norm2_after"] = n2_before, n2_after
    out = re.cpu().numpy(), im.cpu().numpy()
    plan.destroy()
    return out[0], out[1], info


def oracle_evolve(cfg, re_np, im_np, pot_np=None, n_steps=None, coeffs=None):
    """Oracle on the same cast inputs, promoted to float64."""
    re = np.array(re_np, dtype=np.float64, order="C")
    im = np.array(im_np, dtype=np.float64, order="C")
    pot = None if pot_np is None else (np.asarray(pot_np[0], dtype=np.float64),
                                       np.asarray(pot_np[1], dtype=np.float64))
    n = cfg.n_steps if n_steps is None else n_steps
    c = cfg.coeffs() if coeffs is None else coeffs
    oracle.evolve(re, im, *c, pot=pot, periodic=cfg.periodic, n_steps=n)
    return re, im


def tol(cfg):
    """north_star: max-abs amplitude error 1e-4 (fp32), 1e-11 (fp64)."""
    return 1e-4 if cfg.dtype == "f32" else 1e-11


def errors(cfg, got_re, got_im, want_re, want_im):
    d = max(np.abs(got_re.astype(np.float64) - want_re).max(),
            np.abs(got_im.astype(np.float64) - want_im).max())
    scale = max(np.abs(want_re).max(), np.abs(want_im).max(), 1e-300)
    return d, d / scale


def random_inputs(nx, ny, dtype, seed, with_pot):
    """O(1) un-normalised amplitudes so that the absolute tolerance bites."""
    rng = np.random.default_rng(seed)
    dt = np.float32 if dtype == "f32" else np.float64
    re = rng.uniform(-1, 1, (ny, nx)).astype(dt)
    im = rng.uniform(-1, 1, (ny, nx)).astype(dt)
    pot = None
    if with_pot:
        V = rng.uniform(-10, 10, (ny, nx))
        pot = np.stack([np.cos(V), -np.sin(V)]).astype(dt)
    return re, im, pot


def make_cfg(nx, ny, dtype, boundary, theta, n_steps):
    return inputs.Config("adhoc", nx, ny, dtype, boundary, theta, n_steps, "random")
