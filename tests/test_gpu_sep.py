"""-m gpu parity of ts_evolve_sep (separable potential phase, px(x) * py(y)) against
oracle.evolve_sep: the TMA ring kernel's phase mode 2 for every S, boundary and dtype, and the
write-out-as-planes route of the other paths."""
from __future__ import annotations

import math

import numpy as np
import pytest

import gpu_util as G
import oracle

pytestmark = pytest.mark.gpu

TIGHT = {"f32": 2e-5, "f64": 5e-14}


def coeffs(theta):
    return (math.cos(theta / 2), math.sin(theta / 2), math.cos(theta), math.sin(theta))


def run(nx, ny, dtype, boundary, n, seed, **opts):
    import torch
    from paper_1208_2407_b200.binding import Plan
    dev = torch.device("cuda:0")
    re, im, _ = G.random_inputs(nx, ny, dtype, seed, False)
    rng = np.random.default_rng(seed + 7)
    npdt = np.float32 if dtype == "f32" else np.float64
    Vx, Vy = rng.uniform(-6, 6, nx), rng.uniform(-6, 6, ny)
    px = np.stack([np.cos(Vx), -np.sin(Vx)]).astype(npdt)
    py = np.stack([np.cos(Vy), -np.sin(Vy)]).astype(npdt)
    tdt = torch.float32 if dtype == "f32" else torch.float64
    plan = Plan(nx, ny, tdt, boundary)
    for k, v in opts.items():
        plan.set_option(k, v)
    dre, dim = torch.from_numpy(re).to(dev), torch.from_numpy(im).to(dev)
    n0 = plan.norm(dre, dim)
    plan.evolve_sep(dre, dim, *coeffs(0.3), torch.from_numpy(px).to(dev),
                    torch.from_numpy(py).to(dev), n_steps=n)
    torch.cuda.synchronize()
    drift = plan.norm(dre, dim) / n0 - 1
    info = {k: plan.info(k) for k in ("fused", "fuse_steps", "passes", "variant")}
    wre, wim = re.astype(np.float64), im.astype(np.float64)
    oracle.evolve_sep(wre, wim, *coeffs(0.3), px.astype(np.float64), py.astype(np.float64),
                      periodic=boundary == "periodic", n_steps=n)
    err = max(np.abs(dre.cpu().numpy() - wre).max(), np.abs(dim.cpu().numpy() - wim).max())
    plan.destroy()
    assert err <= TIGHT[dtype] * max(1, n / 8), (err, info)
    assert abs(drift) < (1e-4 if dtype == "f32" else 1e-12), drift
    return info


@pytest.mark.parametrize("nx,ny", [(128, 40), (252, 66), (380, 130)])
@pytest.mark.parametrize("boundary", ["closed", "periodic"])
@pytest.mark.parametrize("dtype", ["f32", "f64"])
@pytest.mark.parametrize("fuse", [0, 1, 2, 3, 4])
def test_sep_stream_kernel(nx, ny, boundary, dtype, fuse):
    info = run(nx, ny, dtype, boundary, 9, nx + 3 * ny + fuse, path=2, variant=2,
               fuse_steps=fuse, seg_rows=16)
    assert info["fused"] == 1 and info["variant"] == 2
    if fuse:
        assert info["passes"] == math.ceil(9 / fuse)


@pytest.mark.parametrize("nx,ny", [(256, 2), (256, 4), (128, 6), (256, 10)])
@pytest.mark.parametrize("dtype", ["f32", "f64"])
@pytest.mark.parametrize("fuse", [0, 1, 2, 3, 4])
def test_sep_periodic_rings_shorter_than_the_warm_up(nx, ny, dtype, fuse):
    # the warm-up rows of the pipeline start 2S rows above row 0: on a periodic lattice with
    # ny < 2S + 2 they wrap around the ring more than once, and py must be indexed accordingly
    info = run(nx, ny, dtype, "periodic", 9, nx + 5 * ny + fuse, path=2, variant=2, fuse_steps=fuse)
    assert info["fused"] == 1 and info["variant"] == 2


@pytest.mark.parametrize("nx,ny,opts", [(64, 64, dict(path=2, variant=1)), (124, 34, dict(path=2, variant=1)),
                                        (129, 67, dict()), (256, 30, dict(path=1))])
@pytest.mark.parametrize("dtype", ["f32", "f64"])
def test_sep_other_paths_write_the_product_out(nx, ny, opts, dtype):
    info = run(nx, ny, dtype, "closed", 5, nx + ny, **opts)
    assert info["variant"] != 2


@pytest.mark.parametrize("nx,ny,opts", [(252, 66, dict(path=2, variant=2)), (64, 64, dict()),
                                        (129, 67, dict())])
@pytest.mark.parametrize("boundary", ["closed", "periodic"])
@pytest.mark.parametrize("dtype", ["f32", "f64"])
def test_time_dependent_potential(nx, ny, opts, boundary, dtype):
    # ts_evolve_tdep: a new phase array per step, with a repeated array (fused into one pass) and a
    # step without potential in between
    import torch
    from paper_1208_2407_b200.binding import Plan
    if boundary == "periodic" and (nx % 2 or ny % 2):
        pytest.skip("periodic needs even sizes")
    dev = torch.device("cuda:0")
    re, im, _ = G.random_inputs(nx, ny, dtype, nx + ny, False)
    rng = np.random.default_rng(11)
    npdt = np.float32 if dtype == "f32" else np.float64
    tdt = torch.float32 if dtype == "f32" else torch.float64
    arrays = []
    for _ in range(3):
        V = rng.uniform(-5, 5, (ny, nx))
        arrays.append(np.stack([np.cos(V), -np.sin(V)]).astype(npdt))
    order = [0, 1, 1, None, 2, 0, 0, 0]
    dpots = [torch.from_numpy(a).to(dev) for a in arrays]
    plan = Plan(nx, ny, tdt, boundary)
    for k, v in opts.items():
        plan.set_option(k, v)
    dre, dim = torch.from_numpy(re).to(dev), torch.from_numpy(im).to(dev)
    plan.evolve_tdep(dre, dim, *coeffs(0.3), [None if k is None else dpots[k] for k in order])
    torch.cuda.synchronize()
    wre, wim = re.astype(np.float64), im.astype(np.float64)
    opots = [None if k is None else (arrays[k][0].astype(np.float64), arrays[k][1].astype(np.float64))
             for k in order]
    oracle.evolve_tdep(wre, wim, *coeffs(0.3), opots, periodic=boundary == "periodic")
    err = max(np.abs(dre.cpu().numpy() - wre).max(), np.abs(dim.cpu().numpy() - wim).max())
    assert err <= TIGHT[dtype] * 2, err
    if opts.get("variant") == 2:
        assert plan.info("passes") == 5          # runs: 0 | 1 1 | none | 2 | 0 0 0
    plan.evolve_tdep(dre, dim, *coeffs(0.3), [])   # no steps: a no-op
    plan.destroy()
