"""CPU checks of the seeded input generators (no method arithmetic lives there)."""
from __future__ import annotations

import math

import numpy as np
import torch

from paper_1208_2407_b200 import inputs


def test_counter_based_uniform_is_index_addressable_and_in_range():
    idx = np.arange(0, 100000, dtype=np.int64)
    a = inputs.uniform_pm1(inputs.SEED, 0, idx)
    b = inputs.uniform_pm1(inputs.SEED, 0, idx[5000:5100])
    assert np.array_equal(a[5000:5100], b)
    assert a.min() >= -1.0 and a.max() < 1.0
    assert abs(a.mean()) < 0.01 and abs(a.var() - 1 / 3) < 0.01
    c = inputs.uniform_pm1(inputs.SEED, 1, idx)
    assert abs(np.corrcoef(a, c)[0, 1]) < 0.02


def test_torch_twin_is_bit_identical():
    idx = np.concatenate([np.arange(0, 4096), np.arange(2**31 - 100, 2**31 + 100),
                          np.arange(2**40, 2**40 + 777)]).astype(np.int64)
    for plane in (0, 1):
        a = inputs.uniform_pm1(inputs.SEED, plane, idx)
        b = inputs.uniform_pm1_t(inputs.SEED, plane, torch.from_numpy(idx)).numpy()
        assert np.array_equal(a, b)


def test_device_state_matches_numpy_state_on_cpu():
    cfg = inputs.scaled(inputs.CONFIGS["C4"], 96, 64, 3)
    re, im, n2 = inputs.full_state(cfg, chunk_rows=16)
    tre, tim, tn2 = inputs.device_state(cfg, torch.device("cpu"), chunk_rows=24)
    assert abs(tn2 / n2 - 1) < 1e-14
    wr, wi = inputs.state_window(cfg, np.arange(cfg.ny), np.arange(cfg.nx), tn2)
    assert np.array_equal(tre.numpy(), wr.astype(np.float32))
    assert np.array_equal(tim.numpy(), wi.astype(np.float32))
    assert abs(float(np.sum(re.astype(np.float64) ** 2 + im.astype(np.float64) ** 2)) - 1) < 1e-6


def test_gaussian_and_potential_recipes():
    cfg = inputs.CONFIGS["C1"]
    re, im, n2 = inputs.full_state(cfg)
    p = re.astype(np.float64) ** 2 + im.astype(np.float64) ** 2
    assert abs(p.sum() - 1) < 1e-6
    y, x = np.mgrid[0:64, 0:64]
    assert abs((p * x).sum() - 32) < 1e-3 and abs((p * y).sum() - 32) < 1e-3
    assert abs(math.sqrt((p * (x - 32) ** 2).sum()) - 8) < 0.05    # sigma = std of |psi|^2
    # momentum kx = 0.5: phase advances 0.5 rad per site along x
    z = re[32] + 1j * im[32]
    assert abs(np.angle(z[33] / z[32]) - 0.5) < 1e-5
    c3 = inputs.scaled(inputs.CONFIGS["C3"], 64, 64, 2)
    pot = inputs.full_pot(c3)
    assert pot.shape == (2, 64, 64) and np.allclose(pot[0] ** 2 + pot[1] ** 2, 1, atol=1e-6)
    tp = inputs.device_pot(c3, torch.device("cpu"))
    assert np.abs(tp.numpy() - pot).max() < 1e-6
    pr, pi = inputs.pot_window(inputs.CONFIGS["C3"], [2048], [2048 + 1000])
    V = 0.5 * 1e-6 * 1000 ** 2
    assert abs(pr[0, 0] - math.cos(V)) < 1e-15 and abs(pi[0, 0] + math.sin(V)) < 1e-15
