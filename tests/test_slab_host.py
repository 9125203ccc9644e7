"""Host logic of the row-slab decomposition (paper_1208_2407_b200/slab.py) on CPU tensors, every
rank inside one process: with ts_evolve replaced by the oracle on the local planes, the
decomposed evolution must reproduce the undivided oracle.  (The GPU twin is test_gpu_slab.py; the
two-process exchange is test_slab_gloo.py.)"""
from __future__ import annotations

import math

import numpy as np
import pytest
import torch

import oracle
from paper_1208_2407_b200 import slab
from slab_util import oracle_evolve_fn, oracle_norm_fn, problem


def coeffs(theta):
    return (math.cos(theta / 2), math.sin(theta / 2), math.cos(theta), math.sin(theta))


def test_partition_is_even_aligned_and_covers():
    for ny, w in [(44, 3), (16384, 8), (10, 5), (64, 1)]:
        parts = slab.partition_rows(ny, w)
        assert parts[0][0] == 0 and parts[-1][1] == ny
        for (a, b), (c, d) in zip(parts, parts[1:]):
            assert b == c
        assert all(a % 2 == 0 and b % 2 == 0 and b > a for a, b in parts)
    with pytest.raises(ValueError):
        slab.partition_rows(7, 2)
    with pytest.raises(ValueError):
        slab.partition_rows(4, 3)


def test_neighbours():
    assert slab.neighbours(0, 1, True) == slab.Neighbours(None, None)
    assert slab.neighbours(0, 3, False) == slab.Neighbours(None, 1)
    assert slab.neighbours(2, 3, False) == slab.Neighbours(1, None)
    assert slab.neighbours(0, 3, True) == slab.Neighbours(2, 1)
    assert slab.neighbours(1, 2, True) == slab.Neighbours(0, 0)


def run(nx, ny, boundary, world, k, n_steps, with_pot, theta=0.3, seed=1, shrink_halo=0):
    re, im, pot = problem(nx, ny, seed, with_pot)
    g = slab.LocalGroup(nx, ny, torch.float64, boundary, world, k, evolve_fn=oracle_evolve_fn,
                        norm_fn=oracle_norm_fn)
    if shrink_halo:
        # sabotage: zero the outermost halo rows after every exchange = a halo that is too thin
        orig = g._exchange

        def thin(planes_of):
            orig(planes_of)
            for s in g.slabs:
                for p in planes_of(s):
                    if s.h_top:
                        p[:shrink_halo] = 0
                    if s.h_bot:
                        p[p.shape[0] - shrink_halo:] = 0
        g._exchange = thin
    tre, tim = torch.from_numpy(re.copy()), torch.from_numpy(im.copy())
    g.scatter(tre, tim, None if pot is None else torch.from_numpy(pot.copy()))
    n0 = g.norm()
    g.evolve(coeffs(theta), n_steps)
    out_re, out_im = torch.empty_like(tre), torch.empty_like(tim)
    g.gather(out_re, out_im)
    wre, wim = re.copy(), im.copy()
    oracle.evolve(wre, wim, *coeffs(theta), pot=None if pot is None else (pot[0], pot[1]),
                  periodic=boundary == "periodic", n_steps=n_steps)
    err = max(np.abs(out_re.numpy() - wre).max(), np.abs(out_im.numpy() - wim).max())
    return err, n0, g.norm(), oracle.norm2(re, im)


@pytest.mark.parametrize("world", [1, 2, 3, 4])
@pytest.mark.parametrize("boundary", ["closed", "periodic"])
@pytest.mark.parametrize("with_pot", [False, True])
def test_decomposed_equals_undivided_oracle(world, boundary, with_pot):
    # 11 steps with an exchange every 3: four periods, the last one shorter
    err, n0, n1, want_n0 = run(20, 48, boundary, world, 3, 11, with_pot)
    assert err < 1e-14
    assert abs(n0 - want_n0) < 1e-12 * want_n0 and abs(n1 / n0 - 1) < 1e-13


def test_halo_of_two_rows_per_step_is_tight():
    # H = 2k rows are enough (above); with the outer two rows of every halo lost the cut's error
    # reaches the own rows within k steps
    err, *_ = run(12, 40, "periodic", 2, 4, 4, False, shrink_halo=2)
    assert err > 1e-6


def test_slab_shorter_than_halo_is_rejected():
    with pytest.raises(ValueError):
        slab.LocalGroup(8, 16, torch.float64, "closed", 4, steps_per_exchange=4,
                        evolve_fn=oracle_evolve_fn, norm_fn=oracle_norm_fn)


def test_pass_cutting_and_u4_pattern():
    pat = slab.u4_pattern(0.3)
    assert len(pat) == 5 and pat[0] == pat[1] == pat[3] == pat[4] != pat[2]
    # the five angles sum to theta: cos/sin of the summed half angles
    half = sum(math.atan2(c[1], c[0]) for c in pat)
    assert abs(half - 0.15) < 1e-15
    passes = list(slab._passes(pat, 4, 6))          # 20 sub-steps in passes of at most 6
    assert [len(p) for p in passes] == [6, 6, 6, 2]
    flat = [c for p in passes for c in p]
    assert flat == pat * 4
    assert list(slab._passes([(1.0, 0.0, 1.0, 0.0)], 0, 6)) == []


def test_u4_table_of_the_library_matches_eq4():
    # ts_u4_coefficients (host arithmetic inside libts, no device needed) against the fractions of
    # Eq. 4 as the oracle states them
    import oracle
    from paper_1208_2407_b200 import binding
    theta = 0.37
    rows = binding.u4_coefficients(theta)
    assert len(rows) == 5
    for row, f in zip(rows, oracle.u4_fractions()):
        th = f * theta
        want = (math.cos(th / 2), math.sin(th / 2), math.cos(th), math.sin(th))
        assert max(abs(a - b) for a, b in zip(row, want)) < 1e-15
    assert abs(sum(oracle.u4_fractions()) - 1.0) < 1e-15
    with pytest.raises(binding.TsError):
        binding.u4_coefficients(float("nan"))
