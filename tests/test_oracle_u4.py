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


# ---- time-dependent potential (the Hamiltonian may depend on time) ------------------
# oracle.evolve_tdep is the checker of ts_evolve_tdep; what it adds to the pinned single step is the
# ORDER in which the list is consumed and the potential-free (None) entry.

@pytest.mark.parametrize("nx,ny,periodic", [(6, 4, True), (5, 3, False), (4, 6, False)])
def test_tdep_equals_ordered_dense_product_and_order_matters(nx, ny, periodic):
    theta = 0.45
    c = (math.cos(theta / 2), math.sin(theta / 2), math.cos(theta), math.sin(theta))
    rng = np.random.default_rng(17)
    Vs = [rng.uniform(-2, 2, (ny, nx)) for _ in range(3)]
    order = [0, 1, None, 2, 1]                     # step k uses Vs[order[k]]; None: 7-stage step
    pots_k = [None if k is None else (np.cos(Vs[k]), -np.sin(Vs[k])) for k in order]
    re, im = rand_state(ny, nx, 23)
    v = to_vec(re, im)
    for k in order:                                # applied left to right = first step first
        v = step_unitary(nx, ny, periodic, theta, None if k is None else Vs[k], 1.0) @ v
    w_re, w_im = from_vec(v, ny, nx)
    g_re, g_im = re.copy(), im.copy()
    oracle.evolve_tdep(g_re, g_im, *c, pots_k, periodic=periodic)
    assert np.abs(g_re - w_re).max() < 1e-13 and np.abs(g_im - w_im).max() < 1e-13
    # the reversed list is a different operator: the pin above would not pass for it
    r_re, r_im = re.copy(), im.copy()
    oracle.evolve_tdep(r_re, r_im, *c, pots_k[::-1], periodic=periodic)
    assert max(np.abs(r_re - w_re).max(), np.abs(r_im - w_im).max()) > 1e-3
    # dropping the potential-free step is a different operator as well
    d_re, d_im = re.copy(), im.copy()
    oracle.evolve_tdep(d_re, d_im, *c, [p for p in pots_k if p is not None], periodic=periodic)
    assert max(np.abs(d_re - w_re).max(), np.abs(d_im - w_im).max()) > 1e-3


def test_tdep_with_one_repeated_array_is_evolve():
    nx, ny, theta, n = 6, 4, 0.3, 4
    c = (math.cos(theta / 2), math.sin(theta / 2), math.cos(theta), math.sin(theta))
    V = np.random.default_rng(2).uniform(-3, 3, (ny, nx))
    pot = (np.cos(V), -np.sin(V))
    re, im = rand_state(ny, nx, 4)
    a_re, a_im = re.copy(), im.copy()
    oracle.evolve_tdep(a_re, a_im, *c, [pot] * n, periodic=True)
    v = np.linalg.matrix_power(step_unitary(nx, ny, True, theta, V, 1.0), n) @ to_vec(re, im)
    w_re, w_im = from_vec(v, ny, nx)
    assert np.abs(a_re - w_re).max() < 1e-13 and np.abs(a_im - w_im).max() < 1e-13
    e_re, e_im = re.copy(), im.copy()
    oracle.evolve_tdep(e_re, e_im, *c, [], periodic=True)      # empty list: identity
    assert np.array_equal(e_re, re) and np.array_equal(e_im, im)
