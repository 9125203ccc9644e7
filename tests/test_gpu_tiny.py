"""-m gpu parity of the on-chip-resident kernel (csrc/ts_tiny.cu, plan option variant = 3): the
whole lattice in the registers of one thread block, all steps in one launch -- against the oracle,
element by element, for every (rows per warp, potential, boundary, dtype) instantiation and at
the capacity limits."""
from __future__ import annotations

import numpy as np
import pytest

import gpu_util as G

pytestmark = pytest.mark.gpu

TIGHT = {"f32": 2e-5, "f64": 5e-14}

# (nx, ny): one lane; ragged lane count; C1; the fp32 / fp64 capacity limits
SHAPES = {"f32": [(4, 2), (8, 6), (64, 64), (124, 34), (128, 64), (128, 128), (36, 100)],
          "f64": [(4, 2), (8, 6), (64, 32), (124, 30), (128, 64), (20, 44)]}


@pytest.mark.parametrize("dtype", ["f32", "f64"])
@pytest.mark.parametrize("boundary", ["closed", "periodic"])
@pytest.mark.parametrize("with_pot", [False, True])
@pytest.mark.parametrize("idx", range(7))
def test_on_chip_kernel(dtype, boundary, with_pot, idx):
    if idx >= len(SHAPES[dtype]):
        pytest.skip("no such shape for this dtype")
    nx, ny = SHAPES[dtype][idx]
    rows_per_warp_2 = ny // 2 <= (32 if dtype == "f32" else 16)
    if with_pot and not rows_per_warp_2:
        pytest.skip("with a potential the kernel holds two rows per warp only")
    n = 23
    cfg = G.make_cfg(nx, ny, dtype, boundary, 0.3, n)
    re, im, pot = G.random_inputs(nx, ny, dtype, 7 * nx + ny, with_pot)
    want_re, want_im = G.oracle_evolve(cfg, re, im, pot, n_steps=n)
    # rows per warp: the default (largest that fits) and every smaller one that fits
    for rows in (0, 4, 2):
        if rows == 2 and not rows_per_warp_2:
            continue
        got_re, got_im, info = G.gpu_evolve(cfg, re, im, pot, n_steps=n, variant=3, seg_rows=rows)
        err, rel = G.errors(cfg, got_re, got_im, want_re, want_im)
        assert info["fused"] == 1 and info["variant"] == 3 and info["launches"] == 1
        assert err <= TIGHT[dtype] * 3, (rows, err, rel, info)
        drift = info["norm2_after"] / info["norm2_before"] - 1
        assert abs(drift) < (1e-4 if dtype == "f32" else 1e-12), (rows, drift)


def test_it_is_the_default_for_lattices_that_fit_and_only_for_those():
    # with a potential (without one the axis-split path is the default, tests/test_gpu_axis.py)
    cfg = G.make_cfg(64, 64, "f32", "closed", 0.01, 100)
    re, im, pot = G.random_inputs(64, 64, "f32", 3, True)
    _, _, info = G.gpu_evolve(cfg, re, im, pot, n_steps=100)
    assert info["variant"] == 3 and info["passes"] == 1
    cfg = G.make_cfg(128, 130, "f32", "closed", 0.01, 5)          # too tall: streaming kernel
    re, im, pot = G.random_inputs(128, 130, "f32", 3, True)
    _, _, info = G.gpu_evolve(cfg, re, im, pot, n_steps=5)
    assert info["variant"] == 2
    from paper_1208_2407_b200.binding import TsError, TS_EUNSUPPORTED
    with pytest.raises(TsError) as e:
        G.gpu_evolve(cfg, re, im, None, n_steps=5, variant=3)
    assert e.value.code == TS_EUNSUPPORTED


def test_long_evolution_stays_in_range():
    # the deferred cosines are multiplied in every fourth step: thousands of steps at a large angle
    # would otherwise leave the fp32 range (cos(0.45)^-7 per step).  Against the oracle: fp64 to
    # rounding, fp32 to the rounding accumulated over 2000 steps of 7 sweeps.
    for dtype, tol, drift_tol in (("f64", 1e-10, 1e-11), ("f32", 2e-3, 2e-3)):
        cfg = G.make_cfg(32, 16, dtype, "periodic", 0.9, 2000)
        re, im, _ = G.random_inputs(32, 16, dtype, 1, False)
        got_re, got_im, info = G.gpu_evolve(cfg, re, im, None, n_steps=2000, variant=3)
        want_re, want_im = G.oracle_evolve(cfg, re, im, None, n_steps=2000)
        err, rel = G.errors(cfg, got_re, got_im, want_re, want_im)
        assert info["variant"] == 3 and info["launches"] == 1
        assert err < tol, (dtype, err, rel)
        assert abs(info["norm2_after"] / info["norm2_before"] - 1) < drift_tol
    # and 20000 steps in fp32 stay finite and normalised
    cfg = G.make_cfg(32, 16, "f32", "periodic", 0.9, 20000)
    re, im, _ = G.random_inputs(32, 16, "f32", 1, False)
    got_re, got_im, info = G.gpu_evolve(cfg, re, im, None, n_steps=20000, variant=3)
    assert np.isfinite(got_re).all() and np.isfinite(got_im).all()
    assert abs(info["norm2_after"] / info["norm2_before"] - 1) < 5e-2
