"""-m gpu parity of ts_evolve_u4 (fourth-order step, Eq. 4) against
oracle.evolve_u4, element by element, through the C ABI: every path the five-sub-step pattern can
take (TMA ring kernel with per-sub-step angle tables, register-prefetch kernel, generic sweeps),
with and without the two potential-phase arrays."""
from __future__ import annotations

import math

import numpy as np
import pytest

import gpu_util as G
import oracle

pytestmark = pytest.mark.gpu

TIGHT = {"f32": 2e-5, "f64": 5e-14}


def run_u4(cfg, re, im, pp, pq, theta, n_steps, **opts):
    import torch
    from paper_1208_2407_b200.binding import Plan
    dev = torch.device("cuda:0")
    plan = Plan(cfg.nx, cfg.ny, G.torch_dtype(cfg), cfg.boundary)
    for k, v in opts.items():
        plan.set_option(k, v)
    dre = torch.from_numpy(np.ascontiguousarray(re)).to(dev)
    dim = torch.from_numpy(np.ascontiguousarray(im)).to(dev)
    dpp = None if pp is None else torch.from_numpy(np.ascontiguousarray(pp)).to(dev)
    dpq = None if pq is None else torch.from_numpy(np.ascontiguousarray(pq)).to(dev)
    n0 = plan.norm(dre, dim)
    plan.evolve_u4(dre, dim, theta, dpp, dpq, n_steps=n_steps)
    torch.cuda.synchronize()
    n1 = plan.norm(dre, dim)
    info = {k: plan.info(k) for k in ("fused", "fuse_steps", "passes", "launches", "variant")}
    info["drift"] = n1 / n0 - 1
    out = dre.cpu().numpy(), dim.cpu().numpy()
    plan.destroy()
    return out[0], out[1], info


def inputs_u4(nx, ny, dtype, seed, with_pot, dt=1.0):
    re, im, _ = G.random_inputs(nx, ny, dtype, seed, False)
    if not with_pot:
        return re, im, None, None
    rng = np.random.default_rng(seed + 1)
    V = rng.uniform(-3, 3, (ny, nx))
    p = oracle.U4_P
    q = 1 - 4 * p
    npdt = np.float32 if dtype == "f32" else np.float64
    pp = np.stack([np.cos(V * p * dt), -np.sin(V * p * dt)]).astype(npdt)
    pq = np.stack([np.cos(V * q * dt), -np.sin(V * q * dt)]).astype(npdt)
    return re, im, pp, pq


def check(cfg, theta, n_steps, with_pot, seed, **opts):
    re, im, pp, pq = inputs_u4(cfg.nx, cfg.ny, cfg.dtype, seed, with_pot)
    got_re, got_im, info = run_u4(cfg, re, im, pp, pq, theta, n_steps, **opts)
    wre = np.array(re, dtype=np.float64); wim = np.array(im, dtype=np.float64)
    f64 = lambda P: None if P is None else (P[0].astype(np.float64), P[1].astype(np.float64))
    oracle.evolve_u4(wre, wim, theta, pot_p=f64(pp), pot_q=f64(pq), periodic=cfg.periodic,
                     n_steps=n_steps)
    err, rel = G.errors(cfg, got_re, got_im, wre, wim)
    assert err <= G.tol(cfg), (err, info)
    assert err <= TIGHT[cfg.dtype] * max(1, n_steps), (err, rel, info)
    assert abs(info["drift"]) < (1e-4 if cfg.dtype == "f32" else 1e-12), info
    return info


@pytest.mark.parametrize("nx,ny", [(128, 40), (252, 66), (380, 130)])
@pytest.mark.parametrize("boundary", ["closed", "periodic"])
@pytest.mark.parametrize("with_pot", [False, True])
@pytest.mark.parametrize("dtype", ["f32", "f64"])
@pytest.mark.parametrize("fuse", [0, 1, 2, 3, 4])
def test_u4_stream_kernel(nx, ny, boundary, with_pot, dtype, fuse):
    cfg = G.make_cfg(nx, ny, dtype, boundary, 0.3, 3)
    info = check(cfg, 0.3, 3, with_pot, nx + ny + fuse, path=2, variant=2, fuse_steps=fuse,
                 seg_rows=32)
    assert info["fused"] == 1 and info["variant"] == 2
    S = info["fuse_steps"]
    if not with_pot:
        assert info["passes"] == math.ceil(15 / S)      # 15 sub-steps chained across U4 steps
    else:
        assert info["passes"] >= math.ceil(15 / S)      # runs break where the phase array changes


@pytest.mark.parametrize("fuse", [5, 6])
@pytest.mark.parametrize("boundary", ["closed", "periodic"])
def test_u4_deep_fusion_f32(fuse, boundary):
    # S = 5: exactly one fourth-order step per pass; S = 6: passes straddle U4 steps
    cfg = G.make_cfg(380, 130, "f32", boundary, 0.3, 4)
    info = check(cfg, 0.3, 4, False, 77 + fuse, path=2, variant=2, fuse_steps=fuse, seg_rows=32)
    assert info["passes"] == math.ceil(20 / fuse)


@pytest.mark.parametrize("nx,ny", [(64, 64), (124, 34)])
@pytest.mark.parametrize("with_pot", [False, True])
@pytest.mark.parametrize("dtype", ["f32", "f64"])
def test_u4_register_prefetch_kernel_and_generic(nx, ny, with_pot, dtype):
    cfg = G.make_cfg(nx, ny, dtype, "closed", 0.3, 2)
    info = check(cfg, 0.3, 2, with_pot, 5 * nx + ny, path=2, variant=1)
    assert info["fused"] == 1 and info["variant"] == 1
    info = check(cfg, 0.3, 2, with_pot, 5 * nx + ny, path=1)
    assert info["fused"] == 0


def test_u4_negative_theta_reverses_the_step():
    import torch
    from paper_1208_2407_b200.binding import Plan
    dev = torch.device("cuda:0")
    nx, ny = 256, 64
    re0, im0, _ = G.random_inputs(nx, ny, "f64", 9, False)
    plan = Plan(nx, ny, torch.float64, "periodic")
    re = torch.from_numpy(re0).to(dev); im = torch.from_numpy(im0).to(dev)
    plan.evolve_u4(re, im, 0.25, n_steps=7)
    plan.evolve_u4(re, im, -0.25, n_steps=7)
    torch.cuda.synchronize()
    assert np.abs(re.cpu().numpy() - re0).max() < 1e-12
    assert np.abs(im.cpu().numpy() - im0).max() < 1e-12
    plan.destroy()


def test_u4_argument_errors():
    import torch
    from paper_1208_2407_b200.binding import Plan, TsError, TS_EINVAL
    dev = torch.device("cuda:0")
    plan = Plan(128, 8, torch.float32, "closed")
    re = torch.zeros((8, 128), device=dev); im = torch.zeros((8, 128), device=dev)
    pot = torch.ones((2, 8, 128), device=dev)
    with pytest.raises(TsError) as e:
        plan.evolve_u4(re, im, 0.1, pot, None)
    assert e.value.code == TS_EINVAL
    with pytest.raises(TsError):
        plan.evolve_u4(re, im, float("nan"))
    plan.evolve_u4(re, im, 0.1, n_steps=0)
    plan.destroy()
