"""Pins for the fourth-order step of the oracle (Eq. 4); no GPU needed.

oracle.evolve_u4 is five calls of the pinned second-order step, so what is pinned here is what
Eq. 4 adds: the value of p, the order and angles of the five sub-steps, and the placement of the
two potential phases -- against closed forms and dense scipy.linalg.expm, not against itself.
"""
from __future__ import annotations

import math

import numpy as np
import pytest

import oracle
from dense_ref import exact_unitary, from_vec, step_unitary, to_vec


def rand_state(ny, nx, seed):
    rng = np.random.default_rng(seed)
    return rng.uniform(-1, 1, (ny, nx)), rng.uniform(-1, 1, (ny, nx))


def pots(V, dt):
    p = oracle.U4_P
    q = 1.0 - 4.0 * p
    return ((np.cos(V * p * dt), -np.sin(V * p * dt)), (np.cos(V * q * dt), -np.sin(V * q * dt)))


def test_p_is_the_root_that_cancels_the_third_order_error():
    # [13] (Suzuki): the fractions must sum to 1 and their cubes to 0; p = (4 - 4^(1/3))^-1
    p = oracle.U4_P
    assert abs(p - 0.41449077179437573) < 1e-15
    f = oracle.u4_fractions()
    assert len(f) == 5 and f[0] == f[1] == f[3] == f[4] == p
    assert abs(sum(f) - 1.0) < 1e-15
    assert abs(sum(x ** 3 for x in f)) < 1e-15
    assert f[2] < 0          # the middle sub-step runs backwards in time


@pytest.mark.parametrize("shape", [(1, 2), (2, 1)])
def test_two_site_closed_form(shape):
    # one even pair only: every sub-step is a rotation by its own angle, the angles sum to theta
    theta, n = 0.37, 6
    re = np.zeros(shape); im = np.zeros(shape)
    re.flat[0] = 1.0
    oracle.evolve_u4(re, im, theta, n_steps=n)
    assert np.allclose(re.ravel(), [math.cos(n * theta), 0.0], atol=1e-14)
    assert np.allclose(im.ravel(), [0.0, math.sin(n * theta)], atol=1e-14)


@pytest.mark.parametrize("nx,ny,periodic", [(5, 3, False), (6, 4, True), (4, 4, False)])
@pytest.mark.parametrize("with_pot", [False, True])
def test_equals_ordered_dense_product(nx, ny, periodic, with_pot):
    theta, dt = 0.4, 0.8
    rng = np.random.default_rng(5)
    V = rng.uniform(-2, 2, (ny, nx)) if with_pot else None
    re, im = rand_state(ny, nx, 3)
    v = to_vec(re, im)
    for f in oracle.u4_fractions():      # applied left to right
        v = step_unitary(nx, ny, periodic, f * theta, V, f * dt) @ v
    pp, pq = pots(V, dt) if with_pot else (None, None)
    oracle.evolve_u4(re, im, theta, pot_p=pp, pot_q=pq, periodic=periodic, n_steps=1)
    wr, wi = from_vec(v, ny, nx)
    assert np.abs(re - wr).max() < 1e-13 and np.abs(im - wi).max() < 1e-13


@pytest.mark.parametrize("periodic", [False, True])
@pytest.mark.parametrize("with_pot", [False, True])
def test_dt4_convergence_to_exact_exponential(periodic, with_pot):
    # global error of a fourth-order scheme falls 16x per halving of dt (second order: 4x)
    nx = ny = 6      # (on a periodic ring of 4 the even and odd parts commute: no error at all)
    J, T = 1.0, 1.0
    rng = np.random.default_rng(11)
    V = rng.uniform(-1, 1, (ny, nx)) if with_pot else None
    re0, im0 = rand_state(ny, nx, 8)
    want = exact_unitary(nx, ny, periodic, J, T, V) @ to_vec(re0, im0)
    errs = []
    for n in (4, 8, 16):
        dt = T / n
        re, im = re0.copy(), im0.copy()
        pp, pq = pots(V, dt) if with_pot else (None, None)
        oracle.evolve_u4(re, im, J * dt, pot_p=pp, pot_q=pq, periodic=periodic, n_steps=n)
        errs.append(np.abs(to_vec(re, im) - want).max())
    assert errs[0] < 5e-3
    for a, b in zip(errs, errs[1:]):
        assert 13.0 < a / b < 19.0, errs


def test_reversibility_and_norm():
    nx, ny = 6, 4
    rng = np.random.default_rng(2)
    V = rng.uniform(-1, 1, (ny, nx))
    re0, im0 = rand_state(ny, nx, 4)
    re, im = re0.copy(), im0.copy()
    pp, pq = pots(V, 1.0)
    n0 = oracle.norm2(re, im)
    oracle.evolve_u4(re, im, 0.3, pot_p=pp, pot_q=pq, periodic=True, n_steps=5)
    assert abs(oracle.norm2(re, im) / n0 - 1) < 1e-13
    conj = lambda P: (P[0], -P[1])
    oracle.evolve_u4(re, im, -0.3, pot_p=conj(pp), pot_q=conj(pq), periodic=True, n_steps=5)
    assert np.abs(re - re0).max() < 1e-13 and np.abs(im - im0).max() < 1e-13
