"""-m gpu parity: CUDA path (through the C ABI) vs the CPU oracle, element by element, on small
lattices that still span several strips (128 sites), several y-segments and ragged tails, for
every template variant of the fused kernel (S = 1..4, potential or not, closed or periodic,
fp32 / fp64) and for the generic per-sweep path."""
from __future__ import annotations

import math

import numpy as np
import pytest

import gpu_util as G

pytestmark = pytest.mark.gpu

# tight bounds for short runs on O(1) amplitudes (rounding only): the north_star gate (1e-4 /
# 1e-11 after the config's step count) is asserted too, but a wrong coefficient or a wrong edge
# rule gives errors of order theta^2 ~ 1e-2, far above either.
TIGHT = {"f32": 2e-5, "f64": 5e-14}

# (nx, ny): single strip; strip tail; several strips + ragged tail; tall (several segments)
SHAPES = [(4, 2), (8, 6), (64, 64), (120, 30), (124, 34), (128, 128), (252, 66), (380, 130)]


def check(cfg, re, im, pot, n_steps, **opts):
    got_re, got_im, info = G.gpu_evolve(cfg, re, im, pot, n_steps=n_steps, **opts)
    want_re, want_im = G.oracle_evolve(cfg, re, im, pot, n_steps=n_steps)
    err, rel = G.errors(cfg, got_re, got_im, want_re, want_im)
    assert err <= G.tol(cfg), (err, info)
    assert err <= TIGHT[cfg.dtype] * max(1, n_steps / 8), (err, rel, info)
    drift = info["norm2_after"] / info["norm2_before"] - 1
    assert abs(drift) < (1e-4 if cfg.dtype == "f32" else 1e-12), drift
    return info


@pytest.mark.parametrize("nx,ny", SHAPES)
@pytest.mark.parametrize("boundary", ["closed", "periodic"])
@pytest.mark.parametrize("with_pot", [False, True])
@pytest.mark.parametrize("fuse", [1, 2, 3, 4, 5, 6])
@pytest.mark.parametrize("variant", [1, 2])
def test_fused_f32(nx, ny, boundary, with_pot, fuse, variant):
    # variant 1 = register-prefetch kernel (ts_fused.cu), 2 = TMA ring kernel (ts_stream.cu)
    if variant == 2 and nx < 128 and boundary == "periodic":
        pytest.skip("periodic in x: the TMA ring kernel needs nx >= 128 (auto falls back to variant 1)")
    if fuse > 4 and (variant == 1 or with_pot):
        pytest.skip("S = 5, 6 exist only in the TMA ring kernel, fp32, no potential")
    cfg = G.make_cfg(nx, ny, "f32", boundary, 0.3, 9)
    re, im, pot = G.random_inputs(nx, ny, "f32", nx * 1000 + ny, with_pot)
    info = check(cfg, re, im, pot, 9, path=2, fuse=fuse, seg_rows=32, variant=variant)
    assert info["fused"] == 1 and info["fuse_steps"] == fuse and info["variant"] == variant
    assert info["passes"] == math.ceil(9 / fuse)


@pytest.mark.parametrize("boundary", ["closed", "periodic"])
@pytest.mark.parametrize("with_pot", [False, True])
@pytest.mark.parametrize("dtype,fuse,seg", [("f32", 6, 8), ("f32", 4, 4), ("f32", 3, 2), ("f64", 4, 6),
                                            ("f64", 2, 2)])
def test_short_segments_whose_warmup_reaches_past_the_edge(boundary, with_pot, dtype, fuse, seg):
    # segments shorter than the 2S warm-up rows: several segments start above row 0 / end below
    # row ny-1, and in a closed lattice all of them must take the edge variant of the loop
    if with_pot and fuse > 4:
        pytest.skip("S = 5, 6 exist only without a potential")
    nx, ny = 260, 44
    cfg = G.make_cfg(nx, ny, dtype, boundary, 0.3, 13)
    re, im, pot = G.random_inputs(nx, ny, dtype, 4242 + fuse, with_pot)
    info = check(cfg, re, im, pot, 13, path=2, fuse=fuse, seg_rows=seg, variant=2)
    assert info["fused"] == 1 and info["seg_rows"] == seg


@pytest.mark.parametrize("nx,ny", [(8, 6), (124, 34), (128, 40), (252, 66), (380, 130)])
@pytest.mark.parametrize("boundary", ["closed", "periodic"])
@pytest.mark.parametrize("with_pot", [False, True])
@pytest.mark.parametrize("fuse", [1, 2, 3, 4])
@pytest.mark.parametrize("variant", [1, 2])
def test_fused_f64(nx, ny, boundary, with_pot, fuse, variant):
    if variant == 2 and nx < 128 and boundary == "periodic":
        pytest.skip("periodic in x: the TMA ring kernel needs nx >= 128")
    cfg = G.make_cfg(nx, ny, "f64", boundary, 0.3, 9)
    re, im, pot = G.random_inputs(nx, ny, "f64", nx * 1000 + ny + 1, with_pot)
    info = check(cfg, re, im, pot, 9, path=2, fuse=fuse, seg_rows=16, variant=variant)
    assert info["fused"] == 1 and info["variant"] == variant


@pytest.mark.parametrize("nx,ny", [(1, 1), (2, 1), (1, 2), (5, 3), (7, 8), (64, 64), (129, 67),
                                   (256, 30)])
@pytest.mark.parametrize("boundary", ["closed", "periodic"])
@pytest.mark.parametrize("with_pot", [False, True])
@pytest.mark.parametrize("dtype", ["f32", "f64"])
def test_generic_path(nx, ny, boundary, with_pot, dtype):
    if boundary == "periodic" and (nx % 2 or ny % 2):
        pytest.skip("periodic needs even sizes (rejected by ts_plan_create; see test_gpu_api)")
    cfg = G.make_cfg(nx, ny, dtype, boundary, 0.3, 6)
    re, im, pot = G.random_inputs(nx, ny, dtype, nx * 77 + ny, with_pot)
    info = check(cfg, re, im, pot, 6, path=1)
    assert info["fused"] == 0 and info["launches"] <= 6 * (9 if with_pot else 7)


@pytest.mark.parametrize("boundary", ["closed", "periodic"])
@pytest.mark.parametrize("fuse", [1, 3, 6])
def test_full_angle_coefficients_need_not_be_twice_the_half_angle(boundary, fuse):
    # ts.h: (a_full, b_full) belong to the middle sweep only.  The regrouped kernel merges half
    # sweeps, and must build those merged angles from the HALF coefficients, not from a_full.
    nx, ny, n = 252, 66, 7
    cfg = G.make_cfg(nx, ny, "f64", boundary, 0.3, n)
    re, im, _ = G.random_inputs(nx, ny, "f64", 321, False)
    c = (math.cos(0.15), math.sin(0.15), math.cos(0.47), math.sin(0.47))   # full != 2 * half
    got_re, got_im, info = G.gpu_evolve(cfg, re, im, None, n_steps=n, path=2, fuse=min(fuse, 4),
                                        seg_rows=16, coeffs=c)
    want_re, want_im = G.oracle_evolve(cfg, re, im, None, n_steps=n, coeffs=c)
    err, _ = G.errors(cfg, got_re, got_im, want_re, want_im)
    assert err < 1e-13, (err, info)
    cfg32 = G.make_cfg(nx, ny, "f32", boundary, 0.3, n)
    re32, im32, _ = G.random_inputs(nx, ny, "f32", 322, False)
    got_re, got_im, info = G.gpu_evolve(cfg32, re32, im32, None, n_steps=n, path=2, fuse=fuse,
                                        seg_rows=16, coeffs=c)
    want_re, want_im = G.oracle_evolve(cfg32, re32, im32, None, n_steps=n, coeffs=c)
    err, _ = G.errors(cfg32, got_re, got_im, want_re, want_im)
    assert err < 2e-5, (err, info)


@pytest.mark.parametrize("theta,expect_fused", [(0.0, 1), (-0.7, 1), (1.2, 1), (1.4, 0), (2.9, 0)])
@pytest.mark.parametrize("with_pot", [False, True])
def test_angle_range(theta, expect_fused, with_pot):
    # the fused kernels use tangents: they take angles with cos(theta) > 0.25 (theta = 0: the
    # identity, negative: backwards in time); beyond that the automatic path is the per-sweep one
    nx, ny, n = 252, 66, 5
    cfg = G.make_cfg(nx, ny, "f64", "closed", theta, n)
    re, im, pot = G.random_inputs(nx, ny, "f64", 17, with_pot)
    got_re, got_im, info = G.gpu_evolve(cfg, re, im, pot, n_steps=n)
    want_re, want_im = G.oracle_evolve(cfg, re, im, pot, n_steps=n)
    err, _ = G.errors(cfg, got_re, got_im, want_re, want_im)
    assert info["fused"] == expect_fused, info
    assert err < 1e-12, (err, info)
    if theta == 0.0 and not with_pot:
        assert np.abs(got_re - re).max() < 1e-15 and np.abs(got_im - im).max() < 1e-15


def test_auto_path_picks_generic_for_unaligned_shapes():
    cfg = G.make_cfg(130, 31, "f32", "closed", 0.2, 4)
    re, im, pot = G.random_inputs(130, 31, "f32", 5, True)
    info = check(cfg, re, im, pot, 4)
    assert info["fused"] == 0


@pytest.mark.parametrize("seg_rows", [2, 6, 64, 0])
@pytest.mark.parametrize("variant", [1, 2])
def test_segment_sizes(seg_rows, variant):
    cfg = G.make_cfg(256, 100, "f32", "periodic", 0.25, 8)
    re, im, pot = G.random_inputs(256, 100, "f32", 9, True)
    check(cfg, re, im, pot, 8, path=2, fuse=3, seg_rows=seg_rows, variant=variant)


@pytest.mark.parametrize("slots", [2, 3, 5, 12, 64])
@pytest.mark.parametrize("with_pot", [False, True])
def test_ring_depths(slots, with_pot):
    # any ring depth (clamped to what the pipeline needs and to 227 KB) gives the same result
    cfg = G.make_cfg(380, 70, "f32", "closed", 0.25, 6)
    re, im, pot = G.random_inputs(380, 70, "f32", 19, with_pot)
    check(cfg, re, im, pot, 6, path=2, fuse=2, seg_rows=32, variant=2, ring_slots=slots)


def test_negative_angle_and_reversibility_on_device():
    import torch
    from paper_1208_2407_b200.binding import Plan
    nx, ny, th, n = 256, 64, 0.2, 10
    re0, im0, pot = G.random_inputs(nx, ny, "f64", 3, True)
    plan = Plan(nx, ny, torch.float64, "periodic")
    re = torch.from_numpy(re0).cuda(); im = torch.from_numpy(im0).cuda()
    p = torch.from_numpy(pot).cuda()
    pc = p.clone(); pc[1] = -pc[1]
    ah, bh, af, bf = math.cos(th / 2), math.sin(th / 2), math.cos(th), math.sin(th)
    plan.evolve(re, im, ah, bh, af, bf, pot_phase=p, n_steps=n)
    assert (re.cpu().numpy() - re0).__abs__().max() > 1e-2
    plan.evolve(re, im, ah, -bh, af, -bf, pot_phase=pc, n_steps=n)
    torch.cuda.synchronize()
    assert np.abs(re.cpu().numpy() - re0).max() < 1e-13
    assert np.abs(im.cpu().numpy() - im0).max() < 1e-13


def test_two_site_closed_form_on_device():
    # a1 pinned on the device path too: psi = (cos n theta, i sin n theta)
    cfg = G.make_cfg(2, 1, "f64", "closed", 0.3, 7)
    re = np.array([[1.0, 0.0]]); im = np.zeros((1, 2))
    got_re, got_im, _ = G.gpu_evolve(cfg, re, im, None, n_steps=7)
    assert np.allclose(got_re.ravel(), [math.cos(2.1), 0], atol=1e-14)
    assert np.allclose(got_im.ravel(), [0, math.sin(2.1)], atol=1e-14)


@pytest.mark.parametrize("sx,sy", [(0, 0), (1, 0), (0, 1), (1, 1)])
def test_periodic_eigenstates_fused(sx, sy):
    nx, ny, theta, n = 512, 96, 0.21, 8
    cfg = G.make_cfg(nx, ny, "f64", "periodic", theta, n)
    y, x = np.mgrid[0:ny, 0:nx]
    psi0 = ((-1.0) ** (sx * x + sy * y)) / math.sqrt(nx * ny)
    got_re, got_im, info = G.gpu_evolve(cfg, psi0, np.zeros_like(psi0), None, n_steps=n, path=2)
    ph = np.exp(1j * 2 * n * theta * ((1 - 2 * sx) + (1 - 2 * sy)))
    assert np.abs((got_re + 1j * got_im) - ph * psi0).max() < 1e-15 * 50


def test_pageable_host_pointers_are_rejected_not_dereferenced():
    # include/ts.h: the planes are DEVICE memory; a pageable host pointer must come back as
    # TS_EINVAL before anything is enqueued (it would fault inside the kernel)
    import ctypes
    import torch
    from paper_1208_2407_b200 import binding
    plan = binding.Plan(64, 64, torch.float32, "closed")
    host = np.zeros((2, 64, 64), dtype=np.float32)
    dev = torch.zeros((64, 64), device="cuda:0")
    L = binding.lib()
    hp = ctypes.c_void_p(host.ctypes.data)
    rc = L.ts_evolve(plan._h, hp, ctypes.c_void_p(host[1].ctypes.data), 1.0, 0.0, 1.0, 0.0, None, 1, None)
    assert rc == binding.TS_EINVAL and "device memory" in binding.last_error()
    rc = L.ts_evolve(plan._h, ctypes.c_void_p(dev.data_ptr()), hp, 1.0, 0.0, 1.0, 0.0, None, 1, None)
    assert rc == binding.TS_EINVAL
    out = ctypes.c_double(0.0)
    assert L.ts_norm(plan._h, hp, hp, ctypes.byref(out), None) == binding.TS_EINVAL
    assert plan.info("launches") == 0
    plan.destroy()
