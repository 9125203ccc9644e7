"""-m gpu parity of the three-dimensional step (ts_plan_create_3d / ts_evolve_3d)
against the 3-D oracle (oracle/ts_oracle3d.c, pinned in tests/test_oracle_3d.py), element by
element: the per-sweep kernels (any extents), the three-chain path without a potential (every line
resident in registers, one launch per axis), the sweep-program path with a potential (O E O per
axis between two applications of the phase), closed / periodic / mixed boundaries, fp32 / fp64, and
a 256^3 lattice."""
from __future__ import annotations

import math

import numpy as np
import pytest

import oracle
from paper_1208_2407_b200.binding import TS_EINVAL, TS_EUNSUPPORTED, TsError

pytestmark = pytest.mark.gpu

TIGHT = {"f32": 2e-5, "f64": 5e-14}
GATE = {"f32": 1e-4, "f64": 1e-11}          # north_star's max-abs tolerance


def coeffs(theta):
    return (math.cos(theta / 2), math.sin(theta / 2), math.cos(theta), math.sin(theta))


def inputs3(shape, dtype, seed, with_pot):
    """O(1) un-normalised amplitudes so that the absolute tolerance bites."""
    rng = np.random.default_rng(seed)
    dt = np.float32 if dtype == "f32" else np.float64
    re = rng.uniform(-1, 1, shape).astype(dt)
    im = rng.uniform(-1, 1, shape).astype(dt)
    pot = None
    if with_pot:
        V = rng.uniform(-10, 10, shape)
        pot = np.stack([np.cos(V), -np.sin(V)]).astype(dt)
    return re, im, pot


def run(dims, dtype, boundary, theta, n_steps, with_pot, seed, **opts):
    import torch
    from paper_1208_2407_b200.binding import Plan3D
    nx, ny, nz = dims
    re, im, pot = inputs3((nz, ny, nx), dtype, seed, with_pot)
    dev = torch.device("cuda:0")
    tdt = torch.float32 if dtype == "f32" else torch.float64
    plan = Plan3D(nx, ny, nz, tdt, boundary)
    for k, v in opts.items():
        plan.set_option(k, v)
    dre, dim = torch.from_numpy(re).to(dev), torch.from_numpy(im).to(dev)
    dpot = None if pot is None else torch.from_numpy(pot).to(dev)
    n0 = plan.norm(dre, dim)
    plan.evolve(dre, dim, *coeffs(theta), pot_phase=dpot, n_steps=n_steps)
    torch.cuda.synchronize()
    n1 = plan.norm(dre, dim)
    info = {k: plan.info(k) for k in ("fused", "passes", "launches", "variant")}
    wre, wim = re.astype(np.float64), im.astype(np.float64)
    p64 = None if pot is None else (pot[0].astype(np.float64), pot[1].astype(np.float64))
    per = (boundary,) * 3 if isinstance(boundary, str) else boundary
    oracle.evolve3(wre, wim, *coeffs(theta), pot=p64, periodic=tuple(b == "periodic" for b in per),
                   n_steps=n_steps)
    err = max(np.abs(dre.cpu().numpy() - wre).max(), np.abs(dim.cpu().numpy() - wim).max())
    assert abs(n0 - oracle.norm2_3d(re.astype(np.float64), im.astype(np.float64))) < 1e-6 * n0
    plan.destroy()
    return err, n1 / n0 - 1, info


FUSED_SHAPES = [(8, 6, 4), (64, 64, 64), (100, 36, 24), (128, 16, 2), (32, 1024, 8), (2048, 4, 6),
                (16, 8, 1152)]
BOUNDARIES = ["closed", "periodic", ("periodic", "closed", "periodic"), ("closed", "periodic", "closed")]


@pytest.mark.parametrize("dtype", ["f32", "f64"])
@pytest.mark.parametrize("boundary", BOUNDARIES)
@pytest.mark.parametrize("dims", FUSED_SHAPES)
@pytest.mark.parametrize("with_pot", [False, True])
def test_fused_paths_match_the_oracle(dims, boundary, dtype, with_pot):
    if dtype == "f64" and max(dims) > 1024:
        dims = tuple(min(d, 1024) for d in dims)
    n_steps = 7
    err, drift, info = run(dims, dtype, boundary, 0.3, n_steps, with_pot,
                           seed=sum(dims) + with_pot, path=2)
    assert info["fused"] == 1 and info["variant"] == 4, info
    # without a potential: one launch per axis for all steps; with one: three per step (+ three)
    assert info["launches"] == (3 * n_steps + 3 if with_pot else 3), info
    assert err <= GATE[dtype] and err <= TIGHT[dtype] * 2, (err, info)
    assert abs(drift) < (1e-4 if dtype == "f32" else 1e-12), drift


@pytest.mark.parametrize("dtype", ["f32", "f64"])
@pytest.mark.parametrize("boundary", ["closed", "periodic", ("periodic", "closed", "closed")])
@pytest.mark.parametrize("dims", [(5, 3, 7), (6, 4, 2), (1, 8, 6), (12, 1, 1), (33, 20, 9), (64, 64, 64)])
@pytest.mark.parametrize("with_pot", [False, True])
def test_per_sweep_kernels_match_the_oracle(dims, boundary, dtype, with_pot):
    per = (boundary,) * 3 if isinstance(boundary, str) else boundary
    if any(b == "periodic" and d % 2 for b, d in zip(per, dims)):
        pytest.skip("a periodic axis needs an even extent")
    n_steps = 5
    err, drift, info = run(dims, dtype, boundary, 0.3, n_steps, with_pot, seed=3 * sum(dims), path=1)
    assert info["fused"] == 0 and info["variant"] == 0
    assert err <= GATE[dtype] and err <= TIGHT[dtype] * 2, (err, info)
    assert abs(drift) < (1e-4 if dtype == "f32" else 1e-12), drift


def test_default_path_choice_and_large_angles():
    # even extents that fit a block: the fused path by default; an odd extent or cos <= 0.25: the
    # per-sweep kernels; "path" = 2 then refuses
    _, _, info = run((16, 8, 4), "f32", "closed", 0.3, 2, False, 1)
    assert info["variant"] == 4
    err, _, info = run((15, 8, 4), "f32", "closed", 0.3, 2, True, 2)
    assert info["variant"] == 0 and err < 1e-5
    err, _, info = run((16, 8, 4), "f64", "periodic", 2.8, 3, True, 3)
    assert info["variant"] == 0 and err < 1e-12
    with pytest.raises(TsError) as e:
        run((15, 8, 4), "f32", "closed", 0.3, 2, False, 4, path=2)
    assert e.value.code == TS_EUNSUPPORTED


def test_2d_entry_points_refuse_a_3d_plan_and_bad_arguments():
    import torch
    from paper_1208_2407_b200.binding import Plan3D, lib
    import ctypes
    with pytest.raises(TsError):
        Plan3D(8, 8, 5, torch.float32, "periodic")          # odd periodic axis
    plan = Plan3D(8, 8, 4, torch.float32, "closed")
    re = torch.zeros((4, 8, 8), device="cuda:0"); im = torch.zeros_like(re)
    rc = lib().ts_evolve(plan._h, ctypes.c_void_p(re.data_ptr()), ctypes.c_void_p(im.data_ptr()),
                         1.0, 0.0, 1.0, 0.0, None, 1, None)
    assert rc == TS_EINVAL
    with pytest.raises(TsError):
        plan.evolve(re, im, 0.9, 0.9, 1.0, 0.0)              # a^2 + b^2 != 1
    plan.destroy()


@pytest.mark.parametrize("dtype,boundary,with_pot,n_steps",
                         [("f32", "periodic", False, 12), ("f32", "closed", True, 4),
                          ("f64", ("periodic", "periodic", "closed"), False, 6)])
def test_256_cubed_full_lattice(dtype, boundary, with_pot, n_steps):
    """256^3 (16.8 M sites), every element against the oracle."""
    err, drift, info = run((256, 256, 256), dtype, boundary, 0.05, n_steps, with_pot, 77)
    print(f"\n[256^3 {dtype} {boundary} pot={with_pot} {n_steps} steps] max-abs err {err:.3e} "
          f"norm drift {drift:.3e} {info}")
    assert info["fused"] == 1 and info["variant"] == 4
    assert err <= GATE[dtype] and err <= TIGHT[dtype] * 2, err
    assert abs(drift) < (1e-5 if dtype == "f32" else 1e-12)


def test_periodic_eigenstate_at_512_cubed():
    """512^3 fp32 (134 M sites): the +-1 checkerboard states are exact eigenstates of every sweep
    (closed form at any size; pinned on the oracle in tests/test_oracle_3d.py)."""
    import torch
    from paper_1208_2407_b200.binding import Plan3D
    n = 512
    dev = torch.device("cuda:0")
    ix = torch.arange(n, device=dev)
    sx, sy, sz = 1, 0, 1
    sign = ((-1.0) ** (sx * ix))[None, None, :] * ((-1.0) ** (sy * ix))[None, :, None] \
        * ((-1.0) ** (sz * ix))[:, None, None]
    amp = 1.0 / math.sqrt(float(n) ** 3)
    re = (sign * amp).to(torch.float32).contiguous()
    im = torch.zeros_like(re)
    plan = Plan3D(n, n, n, torch.float32, "periodic")
    n_steps, theta = 20, 0.02
    plan.evolve(re, im, *coeffs(theta), n_steps=n_steps)
    torch.cuda.synchronize()
    assert plan.info("variant") == 4 and plan.info("launches") == 3
    phi = 2 * n_steps * theta * ((1 - 2 * sx) + (1 - 2 * sy) + (1 - 2 * sz))
    want_re = sign * (amp * math.cos(phi)); want_im = sign * (amp * math.sin(phi))
    err = max(float((re - want_re).abs().max()), float((im - want_im).abs().max()))
    assert err < 2e-5 * amp, (err, amp)
    assert abs(plan.norm(re, im) - 1.0) < 1e-5
    plan.destroy()
