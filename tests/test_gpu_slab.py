"""-m gpu: (1) the stream kernel with one boundary type per axis (ts_plan_create_xy) against
oracle.evolve_xy; (2) the row-slab decomposition (slab.LocalGroup: all ranks stepped in turn on
cuda:0, halos exchanged by copies) with the real kernels against the undivided oracle."""
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


@pytest.mark.parametrize("nx,ny", [(128, 40), (380, 130)])
@pytest.mark.parametrize("dtype", ["f32", "f64"])
@pytest.mark.parametrize("with_pot", [False, True])
@pytest.mark.parametrize("fuse", [1, 3, 4, 6])
@pytest.mark.parametrize("bx,by", [("periodic", "closed"), ("closed", "periodic")])
def test_per_axis_boundaries(nx, ny, dtype, with_pot, fuse, bx, by):
    import torch
    from paper_1208_2407_b200.binding import Plan
    if fuse > 4 and (with_pot or dtype == "f64"):
        pytest.skip("S = 5, 6 exist only for fp32 without a potential")
    dev = torch.device("cuda:0")
    re, im, pot = G.random_inputs(nx, ny, dtype, 31 * nx + ny + fuse, with_pot)
    tdt = torch.float32 if dtype == "f32" else torch.float64
    plan = Plan(nx, ny, tdt, bx, by)
    # (closed x, periodic y): the axis-split path without a potential (each axis has its own
    # boundary there), the per-sweep kernels with one
    stream_path = bx == "periodic"
    if stream_path:
        plan.set_option("path", 2); plan.set_option("variant", 2)
        plan.set_option("fuse_steps", fuse); plan.set_option("seg_rows", 16)
    dre, dim = torch.from_numpy(re).to(dev), torch.from_numpy(im).to(dev)
    dpot = None if pot is None else torch.from_numpy(pot).to(dev)
    n = 9
    plan.evolve(dre, dim, *coeffs(0.3), pot_phase=dpot, n_steps=n)
    torch.cuda.synchronize()
    # 128 sites are a resident line of the axis-split path; 380 are neither that nor long enough
    # for windowed rows
    axis_path = not stream_path and not with_pot and nx == 128
    assert plan.info("fused") == (1 if stream_path or axis_path else 0)
    assert plan.info("variant") == (2 if stream_path else (4 if axis_path else 0))
    wre, wim = re.astype(np.float64), im.astype(np.float64)
    p64 = None if pot is None else (pot[0].astype(np.float64), pot[1].astype(np.float64))
    oracle.evolve_xy(wre, wim, *coeffs(0.3), pot=p64, periodic_x=bx == "periodic",
                     periodic_y=by == "periodic", n_steps=n)
    err = max(np.abs(dre.cpu().numpy() - wre).max(), np.abs(dim.cpu().numpy() - wim).max())
    assert err <= TIGHT[dtype] * 2, err
    plan.destroy()


@pytest.mark.parametrize("world", [2, 3])
@pytest.mark.parametrize("boundary", ["closed", "periodic"])
@pytest.mark.parametrize("with_pot", [False, True])
@pytest.mark.parametrize("dtype", ["f32", "f64"])
def test_slab_decomposition_matches_undivided_oracle(world, boundary, with_pot, dtype):
    import torch
    from paper_1208_2407_b200 import slab
    dev = torch.device("cuda:0")
    nx, ny, k, n = 380, 132, 6, 20          # exchange every 6 steps (halo 12 rows), 4 periods
    re, im, pot = G.random_inputs(nx, ny, dtype, 99 + world, with_pot)
    tdt = torch.float32 if dtype == "f32" else torch.float64
    g = slab.LocalGroup(nx, ny, tdt, boundary, world, k, device=dev)
    g.scatter(torch.from_numpy(re).to(dev), torch.from_numpy(im).to(dev),
              None if pot is None else torch.from_numpy(pot).to(dev))
    n0 = g.norm()
    g.evolve(coeffs(0.3), n)
    out_re = torch.empty((ny, nx), dtype=tdt, device=dev); out_im = torch.empty_like(out_re)
    g.gather(out_re, out_im)
    torch.cuda.synchronize()
    n1 = g.norm()
    wre, wim = re.astype(np.float64), im.astype(np.float64)
    p64 = None if pot is None else (pot[0].astype(np.float64), pot[1].astype(np.float64))
    oracle.evolve(wre, wim, *coeffs(0.3), pot=p64, periodic=boundary == "periodic", n_steps=n)
    err = max(np.abs(out_re.cpu().numpy() - wre).max(), np.abs(out_im.cpu().numpy() - wim).max())
    assert err <= TIGHT[dtype] * 3, err
    assert abs(n0 / oracle.norm2(re.astype(np.float64), im.astype(np.float64)) - 1) < 1e-6
    assert abs(n1 / n0 - 1) < (1e-4 if dtype == "f32" else 1e-12)
    g.destroy()


@pytest.mark.parametrize("world", [1, 2, 3])
@pytest.mark.parametrize("boundary", ["closed", "periodic"])
@pytest.mark.parametrize("dtype", ["f32", "f64"])
def test_fused_peer_halo_path_matches_undivided_oracle(world, boundary, dtype):
    # ts_slab_pass: no halo storage, no exchange step -- the kernel reads the neighbours' rows
    import torch
    from paper_1208_2407_b200 import slab
    dev = torch.device("cuda:0")
    nx, ny, n = 380, 132, 17                # 17 steps = passes of 6, 6, 5 (fp32) / 4, 4, 4, 4, 1
    re, im, _ = G.random_inputs(nx, ny, dtype, 500 + world, False)
    tdt = torch.float32 if dtype == "f32" else torch.float64
    g = slab.PeerGroup(nx, ny, tdt, boundary, world, dev)
    g.scatter(torch.from_numpy(re).to(dev), torch.from_numpy(im).to(dev))
    n0 = g.norm()
    g.evolve(coeffs(0.3), n)
    out_re = torch.empty((ny, nx), dtype=tdt, device=dev); out_im = torch.empty_like(out_re)
    g.gather(out_re, out_im)
    torch.cuda.synchronize()
    n1 = g.norm()
    wre, wim = re.astype(np.float64), im.astype(np.float64)
    oracle.evolve(wre, wim, *coeffs(0.3), periodic=boundary == "periodic", n_steps=n)
    err = max(np.abs(out_re.cpu().numpy() - wre).max(), np.abs(out_im.cpu().numpy() - wim).max())
    assert err <= TIGHT[dtype] * 3, err
    assert abs(n1 / n0 - 1) < (1e-4 if dtype == "f32" else 1e-12)
    g.destroy()


@pytest.mark.parametrize("world", [1, 3])
@pytest.mark.parametrize("boundary", ["closed", "periodic"])
@pytest.mark.parametrize("dtype", ["f32", "f64"])
@pytest.mark.parametrize("what", ["u4", "sep"])
def test_fused_peer_halo_path_u4_and_separable_potential(world, boundary, dtype, what):
    import torch
    from paper_1208_2407_b200 import slab
    dev = torch.device("cuda:0")
    nx, ny = 252, 96
    re, im, _ = G.random_inputs(nx, ny, dtype, 700 + world, False)
    tdt = torch.float32 if dtype == "f32" else torch.float64
    npdt = np.float32 if dtype == "f32" else np.float64
    g = slab.PeerGroup(nx, ny, tdt, boundary, world, dev)
    wre, wim = re.astype(np.float64), im.astype(np.float64)
    d_re, d_im = torch.from_numpy(re).to(dev), torch.from_numpy(im).to(dev)
    if what == "u4":
        g.scatter(d_re, d_im)
        g.evolve_u4(0.3, 4)                 # 20 sub-steps in passes of 6 (fp32) / 4 (fp64)
        oracle.evolve_u4(wre, wim, 0.3, periodic=boundary == "periodic", n_steps=4)
        scale = 4
    else:
        rng = np.random.default_rng(5)
        Vx, Vy = rng.uniform(-6, 6, nx), rng.uniform(-6, 6, ny)
        px = np.stack([np.cos(Vx), -np.sin(Vx)]).astype(npdt)
        py = np.stack([np.cos(Vy), -np.sin(Vy)]).astype(npdt)
        g.scatter(d_re, d_im, torch.from_numpy(px).to(dev), torch.from_numpy(py).to(dev))
        g.evolve(coeffs(0.3), 11)
        oracle.evolve_sep(wre, wim, *coeffs(0.3), px.astype(np.float64), py.astype(np.float64),
                          periodic=boundary == "periodic", n_steps=11)
        scale = 2
    out_re = torch.empty((ny, nx), dtype=tdt, device=dev); out_im = torch.empty_like(out_re)
    g.gather(out_re, out_im)
    torch.cuda.synchronize()
    err = max(np.abs(out_re.cpu().numpy() - wre).max(), np.abs(out_im.cpu().numpy() - wim).max())
    assert err <= TIGHT[dtype] * scale, err
    g.destroy()


def test_slab_pass_argument_errors():
    import torch
    from paper_1208_2407_b200.binding import Plan, TsError
    dev = torch.device("cuda:0")
    plan = Plan(128, 16, torch.float32, "periodic", "closed")
    a = (torch.zeros((16, 128), device=dev), torch.zeros((16, 128), device=dev))
    b = (torch.zeros((16, 128), device=dev), torch.zeros((16, 128), device=dev))
    short = (torch.zeros((4, 128), device=dev), torch.zeros((4, 128), device=dev))
    c = coeffs(0.1)
    with pytest.raises(TsError):
        plan.slab_pass(a, a, None, None, [c] * 2)            # in place
    with pytest.raises(TsError):
        plan.slab_pass(a, b, short, None, [c] * 3)           # neighbour shorter than the halo
    with pytest.raises(TsError):
        plan.slab_pass(a, b, None, None, [c] * 7)            # deeper than the kernel goes
    plan.slab_pass(a, b, short, short, [c] * 2)
    plan.destroy()
    per = Plan(128, 16, torch.float32, "periodic")
    with pytest.raises(TsError):
        per.slab_pass(a, b, None, None, [c])                 # slab plans are closed in y
    per.destroy()


@pytest.mark.parametrize("bx,by,nx,ny,dtype,with_pot", [
    ("closed", "closed", 700, 20000, "f32", True),       # S = 3: x-edge strips and y-edge segments short
    ("closed", "closed", 700, 20000, "f32", False),      # S = 6 on the tile kernel (variant 2)
    ("periodic", "closed", 512, 24000, "f32", True),     # no x-edge strips, y-edge segments short
    ("closed", "closed", 100, 60000, "f32", True),       # one strip: every warp is an edge warp
    ("closed", "closed", 200, 30000, "f32", True),       # two strips, both x-edge
    ("closed", "closed", 600, 12000, "f64", True),       # two blocks per SM
    ("periodic", "periodic", 512, 24000, "f32", True),   # nothing closed: equal segments
])
def test_default_segments_on_tall_lattices(bx, by, nx, ny, dtype, with_pot):
    """DEFAULT segment heights of the tile kernel on lattices tall enough that the warps at a
    closed edge get shorter segments than the others (ts_stream.cu: stream_default_seg; the
    other tests force equal segments with the seg_rows option or are too small for the split):
    every element against the oracle."""
    import torch
    from paper_1208_2407_b200.binding import Plan
    dev = torch.device("cuda:0")
    re, im, pot = G.random_inputs(nx, ny, dtype, 7 * nx + ny, with_pot)
    tdt = torch.float32 if dtype == "f32" else torch.float64
    plan = Plan(nx, ny, tdt, bx, by)
    plan.set_option("path", 2); plan.set_option("variant", 2)
    dre, dim = torch.from_numpy(re).to(dev), torch.from_numpy(im).to(dev)
    dpot = None if pot is None else torch.from_numpy(pot).to(dev)
    n = 7
    n0 = plan.norm(dre, dim)
    plan.evolve(dre, dim, *coeffs(0.3), pot_phase=dpot, n_steps=n)
    torch.cuda.synchronize()
    n1 = plan.norm(dre, dim)
    assert plan.info("fused") == 1 and plan.info("variant") == 2
    assert plan.info("seg_rows") >= 32, plan.info("seg_rows")
    wre, wim = re.astype(np.float64), im.astype(np.float64)
    p64 = None if pot is None else (pot[0].astype(np.float64), pot[1].astype(np.float64))
    oracle.evolve_xy(wre, wim, *coeffs(0.3), pot=p64, periodic_x=bx == "periodic",
                     periodic_y=by == "periodic", n_steps=n)
    err = max(np.abs(dre.cpu().numpy() - wre).max(), np.abs(dim.cpu().numpy() - wim).max())
    assert err <= TIGHT[dtype] * 2, err
    assert abs(n1 / n0 - 1) < (1e-5 if dtype == "f32" else 1e-12)
    plan.destroy()
