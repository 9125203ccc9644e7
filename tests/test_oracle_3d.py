"""Pins for the THREE-dimensional CPU oracle (oracle/ts_oracle3d.c; runs without a GPU).

The 3-D step is the extension the paper announces along the lines it gives for
more than one dimension (the diagonal part and two pair parts per dimension).
Every test checks the oracle against something other than itself: dense Hermitian matrices built
here from 1-D chain adjacency matrices by Kronecker products and exponentiated by scipy, the
pinned 2-D oracle (a 3-D lattice one site thick IS a 2-D lattice), closed forms and invariants.
"""
from __future__ import annotations

import math

import numpy as np
import pytest
from scipy.linalg import expm

import oracle


def coeffs(theta):
    return (math.cos(theta / 2), math.sin(theta / 2), math.cos(theta), math.sin(theta))


def rand_state(shape, seed):
    rng = np.random.default_rng(seed)
    return rng.uniform(-1, 1, shape), rng.uniform(-1, 1, shape)


# ---- dense statements: site (x, y, z) <-> index (z*ny + y)*nx + x, i.e. kron(Az, Ay, Ax) ---------
def chain_part(n, parity, periodic):
    """Adjacency of the even (0) / odd (1) bonds of an n-site chain."""
    A = np.zeros((n, n))
    for i in range(parity, n - 1, 2):
        A[i, i + 1] += 1.0
        A[i + 1, i] += 1.0
    if periodic and parity == 1:
        A[n - 1, 0] += 1.0       # n == 2: the single bond carries weight 2 (documented, R7)
        A[0, n - 1] += 1.0
    return A


def part_adjacency(dims, axis, parity, periodic):
    nx, ny, nz = dims
    mats = [np.eye(nz), np.eye(ny), np.eye(nx)]            # kron order: z (slowest), y, x
    mats[2 - axis] = chain_part(dims[axis], parity, periodic)
    return np.kron(np.kron(mats[0], mats[1]), mats[2])


def part_unitary(dims, axis, parity, periodic, theta):
    return expm(1j * theta * part_adjacency(dims, axis, parity, periodic))


def step_unitary(dims, per, theta, V=None):
    """Ordered dense product of one step, applied to psi left to right:
    Xe Xo Ye Yo Ze [Zo(f) | Zo P Zo] Ze Yo Ye Xo Xe  (matrix product written right to left)."""
    h = theta / 2
    U = {(ax, par): part_unitary(dims, ax, par, per[ax], h) for ax in range(3) for par in (0, 1)}
    if V is None:
        mid = part_unitary(dims, 2, 1, per[2], theta)
    else:
        P = np.diag(np.exp(-1j * np.asarray(V, dtype=float).reshape(-1)))
        mid = U[2, 1] @ P @ U[2, 1]
    first = U[2, 0] @ U[1, 1] @ U[1, 0] @ U[0, 1] @ U[0, 0]       # applied first: Xe ... Ze
    last = U[0, 0] @ U[0, 1] @ U[1, 0] @ U[1, 1] @ U[2, 0]        # applied last: Ze ... Xe
    return last @ mid @ first


def exact_unitary(dims, per, J, T, V=None):
    H = -J * sum(part_adjacency(dims, ax, par, per[ax]) for ax in range(3) for par in (0, 1))
    if V is not None:
        H = H + np.diag(np.asarray(V, dtype=float).reshape(-1))
    return expm(-1j * H * T)


def vec(re, im):
    return (re + 1j * im).reshape(-1)


LATTICES = [((3, 4, 5), (False, False, False)), ((4, 4, 4), (True, True, True)),
            ((5, 2, 3), (False, True, False)), ((2, 6, 4), (True, False, True)),
            ((1, 1, 6), (False, False, True)), ((6, 1, 1), (False, False, False)),
            ((1, 5, 1), (False, False, False)), ((4, 3, 2), (True, False, True))]


# ---- every sweep equals the dense exponential of its part ------------------------------------------
@pytest.mark.parametrize("dims,per", LATTICES)
@pytest.mark.parametrize("axis", [0, 1, 2])
@pytest.mark.parametrize("parity", [0, 1])
def test_sweep_is_the_dense_exponential_of_its_part(dims, per, axis, parity):
    nx, ny, nz = dims
    re, im = rand_state((nz, ny, nx), 7 + 10 * axis + parity)
    want = part_unitary(dims, axis, parity, per[axis], 0.37) @ vec(re, im)
    oracle.sweep3(re, im, axis, parity, math.cos(0.37), math.sin(0.37), per[axis])
    assert np.abs(vec(re, im) - want).max() < 1e-13


def test_sweeps_touch_only_their_axis_and_leave_unpaired_sites():
    # closed 3 x 3 x 3: the odd sweep along z leaves the z = 0 layer alone, the even one z = 2
    re, im = rand_state((3, 3, 3), 3)
    r0, i0 = re.copy(), im.copy()
    oracle.sweep3(re, im, 2, 1, math.cos(0.4), math.sin(0.4), False)
    assert np.array_equal(re[0], r0[0]) and np.array_equal(im[0], i0[0])
    assert not np.allclose(re[1], r0[1])
    re, im = r0.copy(), i0.copy()
    oracle.sweep3(re, im, 1, 0, math.cos(0.4), math.sin(0.4), False)
    assert np.array_equal(re[:, 2, :], r0[:, 2, :]) and not np.allclose(re[:, 0, :], r0[:, 0, :])
    re, im = r0.copy(), i0.copy()
    oracle.sweep3(re, im, 0, 0, math.cos(0.4), math.sin(0.4), False)
    assert np.array_equal(re[:, :, 2], r0[:, :, 2]) and not np.allclose(re[:, :, 0], r0[:, :, 0])


# ---- the full step equals the ordered dense product -----------------------------------------------
@pytest.mark.parametrize("dims,per", LATTICES[:5] + LATTICES[7:])
@pytest.mark.parametrize("with_pot", [False, True])
def test_step_is_the_ordered_dense_product(dims, per, with_pot):
    nx, ny, nz = dims
    re, im = rand_state((nz, ny, nx), 11)
    V = None
    pot = None
    if with_pot:
        V = np.random.default_rng(5).uniform(-1.5, 1.5, (nz, ny, nx))
        pot = (np.cos(V), -np.sin(V))
    U = step_unitary(dims, per, 0.3, V)
    want = U @ U @ vec(re, im)
    oracle.evolve3(re, im, *coeffs(0.3), pot=pot, periodic=per, n_steps=2)
    assert np.abs(vec(re, im) - want).max() < 1e-13


def test_position_of_the_potential_matters_and_is_the_centre():
    # a trailing P (after the kinetic palindrome) is a different operator: the pin above would
    # fail for it.  Checked on the dense side so that the statement is about the reading (R3).
    dims, per = (3, 2, 4), (False, False, False)
    V = np.random.default_rng(9).uniform(-1, 1, (4, 2, 3))
    centre = step_unitary(dims, per, 0.3, V)
    trailing = np.diag(np.exp(-1j * V.reshape(-1))) @ step_unitary(dims, per, 0.3, None)
    assert np.abs(centre - trailing).max() > 1e-3


# ---- one site thick: the pinned 2-D oracle ----------------------------------------------------------
@pytest.mark.parametrize("periodic", [False, True])
@pytest.mark.parametrize("with_pot", [False, True])
def test_one_layer_reduces_to_the_2d_oracle(periodic, with_pot):
    # nz = 1: no z pair exists (closed in z), so Ze, Zo are identities and, without a potential,
    # the step is Xe Xo Ye Yo | Yo Ye Xo Xe with all half angles = the 2-D step (whose middle
    # Yo(full) = Yo(half)^2).  With a potential P sits between the two Yo half sweeps: the 2-D
    # 9-stage step exactly.
    ny, nx = 6, 8
    re2, im2 = rand_state((ny, nx), 21)
    pot2 = None
    if with_pot:
        V = np.random.default_rng(2).uniform(-1, 1, (ny, nx))
        pot2 = (np.cos(V), -np.sin(V))
    re3, im3 = re2.copy()[None], im2.copy()[None]
    pot3 = None if pot2 is None else (pot2[0][None], pot2[1][None])
    oracle.evolve(re2, im2, *coeffs(0.23), pot=pot2, periodic=periodic, n_steps=5)
    r3 = np.ascontiguousarray(re3); i3 = np.ascontiguousarray(im3)
    oracle.evolve3(r3, i3, *coeffs(0.23), pot=pot3, periodic=(periodic, periodic, False), n_steps=5)
    assert np.abs(r3[0] - re2).max() < 1e-13 and np.abs(i3[0] - im2).max() < 1e-13


def test_one_column_reduces_to_the_2d_oracle_with_axes_renamed():
    # nx = 1: the (y, z) lattice is a 2-D lattice with y in the role of x and z in the role of y,
    # including the full middle sweep on the innermost axis
    nz, ny = 6, 5
    re2, im2 = rand_state((nz, ny), 33)
    r3 = np.ascontiguousarray(re2.reshape(nz, ny, 1)); i3 = np.ascontiguousarray(im2.reshape(nz, ny, 1))
    oracle.evolve(re2, im2, *coeffs(0.31), periodic=False, n_steps=4)
    oracle.evolve3(r3, i3, *coeffs(0.31), periodic=False, n_steps=4)
    assert np.abs(r3[:, :, 0] - re2).max() < 1e-13 and np.abs(i3[:, :, 0] - im2).max() < 1e-13


# ---- closed forms and invariants -----------------------------------------------------------------
@pytest.mark.parametrize("axis", [0, 1, 2])
def test_two_site_closed_form_along_each_axis(axis):
    shape = [1, 1, 1]
    shape[2 - axis] = 2                      # array shape is [nz][ny][nx]
    re = np.zeros(shape); im = np.zeros(shape)
    re.flat[0] = 1.0
    oracle.evolve3(re, im, *coeffs(0.3), periodic=False, n_steps=7)
    assert np.allclose(re.ravel(), [math.cos(7 * 0.3), 0.0], atol=1e-14)
    assert np.allclose(im.ravel(), [0.0, math.sin(7 * 0.3)], atol=1e-14)


@pytest.mark.parametrize("s", [(0, 0, 0), (1, 0, 0), (0, 1, 1), (1, 1, 1)])
def test_periodic_checkerboard_eigenstates(s):
    # psi = (-1)^(sx x + sy y + sz z) / sqrt(N): every site is paired in every sweep and each pair
    # is (c, +-c), an eigenvector of the rotation with eigenvalue exp(+-i angle); per step each
    # axis contributes angle 2 theta (four half sweeps, or two half + one full)
    nx, ny, nz = 6, 4, 8
    z, y, x = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    psi = (-1.0) ** (s[0] * x + s[1] * y + s[2] * z) / math.sqrt(nx * ny * nz)
    re = psi.copy(); im = np.zeros_like(re)
    n, theta = 9, 0.17
    oracle.evolve3(re, im, *coeffs(theta), periodic=True, n_steps=n)
    ph = np.exp(1j * 2 * n * theta * sum(1 - 2 * k for k in s))
    assert np.abs((re + 1j * im) - ph * psi).max() < 1e-14


@pytest.mark.parametrize("per", [(False, False, False), (True, True, True), (True, False, True)])
@pytest.mark.parametrize("with_pot", [False, True])
def test_reversibility_and_norm(per, with_pot):
    shape = (4, 6, 8)
    re, im = rand_state(shape, 4)
    r0, i0 = re.copy(), im.copy()
    pot = conj = None
    if with_pot:
        V = np.random.default_rng(8).uniform(-2, 2, shape)
        pot, conj = (np.cos(V), -np.sin(V)), (np.cos(V), np.sin(V))
    a_h, b_h, a_f, b_f = coeffs(0.4)
    n0 = oracle.norm2_3d(re, im)
    oracle.evolve3(re, im, a_h, b_h, a_f, b_f, pot=pot, periodic=per, n_steps=6)
    assert abs(oracle.norm2_3d(re, im) / n0 - 1) < 1e-13
    assert np.abs(re - r0).max() > 1e-2
    oracle.evolve3(re, im, a_h, -b_h, a_f, -b_f, pot=conj, periodic=per, n_steps=6)
    assert np.abs(re - r0).max() < 1e-13 and np.abs(im - i0).max() < 1e-13


def test_constant_potential_is_a_global_phase():
    shape = (3, 4, 5)
    re, im = rand_state(shape, 6)
    r1, i1 = re.copy(), im.copy()
    V0, n = 0.7, 4
    pot = (np.full(shape, math.cos(V0)), np.full(shape, -math.sin(V0)))
    oracle.evolve3(re, im, *coeffs(0.2), pot=pot, periodic=False, n_steps=n)
    # without a potential the middle is one full z-odd sweep = two half sweeps
    oracle.evolve3(r1, i1, *coeffs(0.2), pot=None, periodic=False, n_steps=n)
    want = np.exp(-1j * V0 * n) * (r1 + 1j * i1)
    assert np.abs((re + 1j * im) - want).max() < 1e-13


@pytest.mark.parametrize("per", [(False, False, False), (True, True, True)])
@pytest.mark.parametrize("with_pot", [False, True])
def test_second_order_convergence_to_the_exact_propagator(per, with_pot):
    dims = (6, 2, 4)       # (the even and odd parts of a periodic 4-ring commute: no splitting error)
    nx, ny, nz = dims
    J, T = 1.0, 0.8
    V = None
    if with_pot:
        V = np.random.default_rng(12).uniform(-1, 1, (nz, ny, nx))
    re0, im0 = rand_state((nz, ny, nx), 13)
    want = exact_unitary(dims, per, J, T, V) @ vec(re0, im0)
    errs = []
    for n in (8, 16, 32):
        dt = T / n
        re, im = re0.copy(), im0.copy()
        pot = None if V is None else (np.cos(V * dt), -np.sin(V * dt))
        oracle.evolve3(re, im, *coeffs(J * dt), pot=pot, periodic=per, n_steps=n)
        errs.append(np.abs(vec(re, im) - want).max())
    assert 3.7 < errs[0] / errs[1] < 4.3 and 3.7 < errs[1] / errs[2] < 4.3, errs


def test_axes_commute_without_a_potential():
    # the property the axis-split CUDA path rests on: X, Y and Z chains may be applied one after
    # the other.  n steps = [n-step X chain][n-step Y chain][n-step Z chain], each chain being
    # E(h) O(f) E(f) O(f) ... E(h) along its axis (adjacent half sweeps merged).
    shape = (4, 6, 8)
    re, im = rand_state(shape, 17)
    r1, i1 = re.copy(), im.copy()
    n, theta = 3, 0.3
    a_h, b_h, a_f, b_f = coeffs(theta)
    oracle.evolve3(re, im, a_h, b_h, a_f, b_f, periodic=(True, False, True), n_steps=n)
    for axis, per in ((0, True), (1, False), (2, True)):
        oracle.sweep3(r1, i1, axis, 0, a_h, b_h, per)
        for k in range(n):
            oracle.sweep3(r1, i1, axis, 1, a_f, b_f, per)
            if k < n - 1:
                oracle.sweep3(r1, i1, axis, 0, a_f, b_f, per)
        oracle.sweep3(r1, i1, axis, 0, a_h, b_h, per)
    assert np.abs(re - r1).max() < 1e-13 and np.abs(im - i1).max() < 1e-13
