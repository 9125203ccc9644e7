"""-m gpu parity of the axis-split path (csrc/ts_axis.cu, plan option variant = 4): steps without
a potential evolved as a row chain followed by a column chain -- against the oracle's literal stage
order, element by element, for every regime of both axes (lines resident in a warp's registers,
windowed rows, pipelined columns), closed / periodic, fp32 / fp64, several chain lengths, and the
fourth-order pattern."""
from __future__ import annotations

import math

import numpy as np
import pytest

import gpu_util as G
import oracle

pytestmark = pytest.mark.gpu

TIGHT = {"f32": 2e-5, "f64": 5e-14}


def check(cfg, n_steps, seed, **opts):
    re, im, _ = G.random_inputs(cfg.nx, cfg.ny, cfg.dtype, seed, False)
    got_re, got_im, info = G.gpu_evolve(cfg, re, im, None, n_steps=n_steps, variant=4, **opts)
    want_re, want_im = G.oracle_evolve(cfg, re, im, None, n_steps=n_steps)
    err, rel = G.errors(cfg, got_re, got_im, want_re, want_im)
    assert info["fused"] == 1 and info["variant"] == 4, info
    assert err <= G.tol(cfg), (err, info)
    assert err <= TIGHT[cfg.dtype] * max(1, n_steps / 8), (err, rel, info)
    drift = info["norm2_after"] / info["norm2_before"] - 1
    assert abs(drift) < (1e-4 if cfg.dtype == "f32" else 1e-12), drift
    return info


# lines of both axes resident in registers: one launch per axis whatever the step count
RESIDENT = {"f32": [(8, 6), (64, 64), (100, 36), (128, 128), (256, 24), (512, 200), (1024, 64),
                    (32, 1024)],
            "f64": [(8, 6), (64, 64), (100, 36), (256, 24), (512, 200), (16, 512)]}


@pytest.mark.parametrize("dtype", ["f32", "f64"])
@pytest.mark.parametrize("boundary", ["closed", "periodic"])
@pytest.mark.parametrize("idx", range(8))
@pytest.mark.parametrize("n_steps", [1, 23])
def test_resident_lines(dtype, boundary, idx, n_steps):
    if idx >= len(RESIDENT[dtype]):
        pytest.skip("no such shape for this dtype")
    nx, ny = RESIDENT[dtype][idx]
    cfg = G.make_cfg(nx, ny, dtype, boundary, 0.3, n_steps)
    info = check(cfg, n_steps, 31 * nx + ny)
    assert info["passes"] == 2 and info["launches"] == 2
    assert info["chain_x"] == n_steps and info["chain_y"] == n_steps


# lines shared by several warps of a block (2048 = 2 x 32 x 32, 1152 = 9 x 32 x 4, 4096 / 8192 in
# fp32 = 2 / 4 warps of 64 sites per lane, 16384 = 16 warps of 32, ...), rows that
# fit no block and are cut into windows with a halo (1056 = 33 x 32, 20480, 528, 12288), columns
# that are pipelined (130, 1100, 66 rows: no lane layout divides them)
LONG = {"f32": [(2048, 128), (1152, 200), (64, 2048), (1280, 130), (3072, 1100), (4096, 66),
                (1056, 200), (20480, 66), (16384, 16), (8192, 12)],
        "f64": [(1024, 128), (576, 200), (64, 1024), (640, 130), (1536, 1100), (528, 200),
                (12288, 66), (8192, 16)]}


@pytest.mark.parametrize("dtype", ["f32", "f64"])
@pytest.mark.parametrize("boundary", ["closed", "periodic"])
@pytest.mark.parametrize("idx", range(10))
@pytest.mark.parametrize("chain", [0, 4, 7, 16, 24])
def test_multi_warp_lines_windowed_rows_and_pipelined_columns(dtype, boundary, idx, chain):
    if idx >= len(LONG[dtype]):
        pytest.skip("no such shape for this dtype")
    if dtype == "f64" and chain > 12:
        pytest.skip("fp64 chains are at most 12 deep")
    nx, ny = LONG[dtype][idx]
    n_steps = 19
    cfg = G.make_cfg(nx, ny, dtype, boundary, 0.3, n_steps)
    info = check(cfg, n_steps, 17 * nx + ny + chain, chain=chain)
    assert info["passes"] >= 2
    if nx in (1056, 20480, 528, 12288):          # windowed rows: passes of `chain` sub-steps
        assert info["chain_x"] < n_steps or chain in (0, 24)


@pytest.mark.parametrize("seg_rows", [16, 34, 64, 1024])
@pytest.mark.parametrize("boundary", ["closed", "periodic"])
@pytest.mark.parametrize("slots", [0, 2, 3, 5, 64])
def test_column_segments_and_ring_depths(seg_rows, boundary, slots):
    # segments shorter than the warm-up, ragged last segment, one segment for the whole column;
    # any ring depth (clamped to [3, what shared memory holds]) gives the same result
    if slots and seg_rows != 34:
        pytest.skip("ring depths are swept at one segment size")
    cfg = G.make_cfg(200, 300, "f32", boundary, 0.3, 9)
    check(cfg, 9, 5 + seg_rows, chain=8, seg_rows=seg_rows, ring_slots=slots)


@pytest.mark.parametrize("boundary", ["closed", "periodic"])
def test_full_angle_coefficients_are_the_middle_sweep_only(boundary):
    # ts.h: (a_full, b_full) belong to the middle (vertical-odd) sweep; every merged angle must be
    # composed from the half-angle coefficients
    c = (math.cos(0.15), math.sin(0.15), math.cos(0.47), math.sin(0.47))
    for nx, ny in [(256, 64), (2048, 2048)]:
        cfg = G.make_cfg(nx, ny, "f64", boundary, 0.3, 7)
        re, im, _ = G.random_inputs(nx, ny, "f64", 321, False)
        got_re, got_im, info = G.gpu_evolve(cfg, re, im, None, n_steps=7, variant=4, coeffs=c)
        want_re, want_im = G.oracle_evolve(cfg, re, im, None, n_steps=7, coeffs=c)
        err, _ = G.errors(cfg, got_re, got_im, want_re, want_im)
        assert info["variant"] == 4 and err < 1e-13, (err, info)


@pytest.mark.parametrize("nx,ny", [(128, 64), (1024, 1024), (2048, 1536)])
@pytest.mark.parametrize("boundary", ["closed", "periodic"])
@pytest.mark.parametrize("dtype", ["f32", "f64"])
def test_fourth_order_pattern(nx, ny, boundary, dtype):
    import torch
    from paper_1208_2407_b200.binding import Plan
    if dtype == "f64" and nx > 1024:
        nx //= 2
    dev = torch.device("cuda:0")
    cfg = G.make_cfg(nx, ny, dtype, boundary, 0.3, 3)
    re, im, _ = G.random_inputs(nx, ny, dtype, nx + ny, False)
    plan = Plan(nx, ny, G.torch_dtype(cfg), boundary)
    plan.set_option("variant", 4)
    dre = torch.from_numpy(re).to(dev); dim = torch.from_numpy(im).to(dev)
    plan.evolve_u4(dre, dim, 0.3, n_steps=3)
    torch.cuda.synchronize()
    assert plan.info("variant") == 4
    wre = np.array(re, dtype=np.float64); wim = np.array(im, dtype=np.float64)
    oracle.evolve_u4(wre, wim, 0.3, periodic=cfg.periodic, n_steps=3)
    err, rel = G.errors(cfg, dre.cpu().numpy(), dim.cpu().numpy(), wre, wim)
    assert err <= TIGHT[dtype] * 3, (err, rel)
    plan.destroy()


def test_long_evolution_against_the_oracle():
    # all 2000 steps in one launch per axis; the deferred cosines are multiplied in on the way, or
    # the scaled amplitudes would leave the fp32 range (cos(0.45)^-4 per step)
    for dtype, theta, tol in (("f32", 0.9, 2e-3), ("f64", 0.9, 1e-10)):
        cfg = G.make_cfg(64, 32, dtype, "periodic", theta, 2000)
        re, im, _ = G.random_inputs(64, 32, dtype, 1, False)
        got_re, got_im, info = G.gpu_evolve(cfg, re, im, None, n_steps=2000, variant=4)
        want_re, want_im = G.oracle_evolve(cfg, re, im, None, n_steps=2000)
        err, rel = G.errors(cfg, got_re, got_im, want_re, want_im)
        assert info["launches"] == 2
        assert err < tol, (dtype, err, rel)
        assert abs(info["norm2_after"] / info["norm2_before"] - 1) < (2e-3 if dtype == "f32" else 1e-11)


def test_it_is_the_default_without_a_potential_and_only_then():
    cfg = G.make_cfg(1024, 1024, "f32", "closed", 0.01, 5)
    re, im, pot = G.random_inputs(1024, 1024, "f32", 3, True)
    _, _, info = G.gpu_evolve(cfg, re, im, None, n_steps=5)
    assert info["variant"] == 4
    _, _, info = G.gpu_evolve(cfg, re, im, pot, n_steps=5)
    assert info["variant"] == 2
    from paper_1208_2407_b200.binding import TsError, TS_EUNSUPPORTED
    with pytest.raises(TsError) as e:
        G.gpu_evolve(cfg, re, im, pot, n_steps=5, variant=4)
    assert e.value.code == TS_EUNSUPPORTED
    # a row length no lane layout divides: the 2-D streaming kernel takes it
    cfg = G.make_cfg(1000, 64, "f32", "closed", 0.01, 5)
    re, im, _ = G.random_inputs(1000, 64, "f32", 3, False)
    _, _, info = G.gpu_evolve(cfg, re, im, None, n_steps=5)
    assert info["variant"] == 2


@pytest.mark.parametrize("sx,sy", [(0, 0), (1, 0), (0, 1), (1, 1)])
def test_periodic_eigenstates(sx, sy):
    nx, ny, theta, n = 2048, 1200, 0.21, 40
    cfg = G.make_cfg(nx, ny, "f64", "periodic", theta, n)
    y, x = np.mgrid[0:ny, 0:nx]
    psi0 = ((-1.0) ** (sx * x + sy * y)) / math.sqrt(nx * ny)
    got_re, got_im, info = G.gpu_evolve(cfg, psi0, np.zeros_like(psi0), None, n_steps=n, variant=4)
    ph = np.exp(1j * 2 * n * theta * ((1 - 2 * sx) + (1 - 2 * sy)))
    assert np.abs((got_re + 1j * got_im) - ph * psi0).max() < 1e-15 * 200


@pytest.mark.parametrize("dtype", ["f32", "f64"])
@pytest.mark.parametrize("boundary", ["closed", "periodic"])
@pytest.mark.parametrize("seg_rows,chain", [(260, 8), (300, 12), (514, 4)])
def test_short_edge_segments_of_the_column_pipeline(dtype, boundary, seg_rows, chain):
    # closed lattices: the first and last 128 rows are segments of their own (they run the edge
    # variant of the loop), the interior is cut into seg_rows; 2050 rows fit no lane layout, so the
    # columns are pipelined
    cfg = G.make_cfg(128, 2050, dtype, boundary, 0.3, 13)
    info = check(cfg, 13, 5 * seg_rows + chain, chain=chain, seg_rows=seg_rows)
    assert info["seg_rows"] == seg_rows and info["chain_y"] <= chain
