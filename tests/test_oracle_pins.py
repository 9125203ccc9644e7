"""Pins for the CPU oracle (runs without a GPU).

Each test checks oracle/ts_oracle.c against something OTHER than itself: closed forms, dense
scipy.linalg.expm of Hermitian matrices (tests/dense_ref.py), invariants, stored tables written
by tests/golden/make_golden.py from dense matrices.  Citations: PAPER.md = the paper's text.
"""
from __future__ import annotations

import math
from pathlib import Path

import numpy as np
import pytest

import oracle
from dense_ref import (exact_unitary, from_vec, part_unitary, step_unitary, to_vec)

GOLDEN = Path(__file__).resolve().parent / "golden"


def coeffs(theta):
    return (math.cos(theta / 2), math.sin(theta / 2), math.cos(theta), math.sin(theta))


def rand_state(ny, nx, seed):
    rng = np.random.default_rng(seed)
    return rng.uniform(-1, 1, (ny, nx)), rng.uniform(-1, 1, (ny, nx))


def load_golden(name):
    rows = [list(map(float, ln.split())) for ln in open(GOLDEN / name) if not ln.startswith("#")]
    a = np.array(rows)
    return a[:4], a[4:]


# --- a1: the pair rotation, 2-site closed form ---------------------------------
@pytest.mark.parametrize("shape", [(1, 2), (2, 1)])
@pytest.mark.parametrize("theta,n", [(0.3, 1), (0.3, 7), (-0.11, 5), (1.9, 3)])
def test_two_site_closed_form(shape, theta, n):
    # only one even pair exists: each step applies it with theta/2 twice (the full middle sweep
    # and the other axis have no pair at all) => psi = (cos n theta, i sin n theta)
    ny, nx = shape
    re = np.zeros((ny, nx)); im = np.zeros((ny, nx))
    re.flat[0] = 1.0
    oracle.evolve(re, im, *coeffs(theta), periodic=False, n_steps=n)
    assert np.allclose(re.ravel(), [math.cos(n * theta), 0.0], atol=1e-14)
    assert np.allclose(im.ravel(), [0.0, math.sin(n * theta)], atol=1e-14)


def test_sign_convention_i_times_b():
    # reading R1: block [[a, +ib],[+ib, a]]: from (1,0) the partner acquires +i*b
    re = np.array([[1.0, 0.0]]); im = np.zeros((1, 2))
    oracle.sweep(re, im, 0, 0, math.cos(0.2), math.sin(0.2), False)
    assert re[0, 0] == pytest.approx(math.cos(0.2)) and im[0, 1] == pytest.approx(+math.sin(0.2))
    assert re[0, 1] == 0.0 and im[0, 0] == 0.0


# --- a2-a5: every sweep equals the dense exponential of its part ----------------
LATTICES = [(5, 3, False), (6, 4, False), (8, 8, False), (3, 5, False), (1, 6, False),
            (6, 4, True), (8, 8, True), (2, 4, True), (4, 2, True)]


@pytest.mark.parametrize("nx,ny,periodic", LATTICES)
@pytest.mark.parametrize("axis", [0, 1])
@pytest.mark.parametrize("parity", [0, 1])
def test_sweep_equals_dense_expm(nx, ny, periodic, axis, parity):
    theta = 0.37
    re, im = rand_state(ny, nx, 100 + nx * 10 + ny)
    want = part_unitary(nx, ny, axis, parity, periodic, theta) @ to_vec(re, im)
    # n = 2 periodic: the oracle rotates the single bond twice; the dense adjacency carries
    # weight 2 on it -- the same operator
    oracle.sweep(re, im, axis, parity, math.cos(theta), math.sin(theta), periodic)
    assert np.abs(to_vec(re, im) - want).max() < 1e-13


def test_unpaired_sites_unchanged_closed():
    # odd length: last site has no even partner, first site has no odd partner (zero rows in
    # the printed H1/H2)
    re, im = rand_state(5, 7, 3)
    r0, i0 = re.copy(), im.copy()
    oracle.sweep(re, im, 0, 0, math.cos(0.4), math.sin(0.4), False)
    assert np.array_equal(re[:, 6], r0[:, 6]) and np.array_equal(im[:, 6], i0[:, 6])
    assert not np.allclose(re[:, :6], r0[:, :6])
    re, im = r0.copy(), i0.copy()
    oracle.sweep(re, im, 1, 1, math.cos(0.4), math.sin(0.4), False)
    assert np.array_equal(re[0], r0[0]) and np.array_equal(im[0], i0[0])
    re, im = r0.copy(), i0.copy()
    oracle.sweep(re, im, 0, 1, math.cos(0.4), math.sin(0.4), False)
    assert np.array_equal(re[:, 0], r0[:, 0])
    # 7 columns: odd pairs (1,2),(3,4),(5,6) -> column 6 IS paired
    assert not np.array_equal(re[:, 6], r0[:, 6])


# --- a6: potential phase -----------------------------------------------
def test_phase_is_elementwise_complex_multiply_and_unit_modulus():
    re, im = rand_state(6, 5, 7)
    rng = np.random.default_rng(8)
    V = rng.uniform(-20, 20, (6, 5))
    want = (re + 1j * im) * np.exp(-1j * V)
    n0 = oracle.norm2(re, im)
    oracle.phase(re, im, np.cos(V), -np.sin(V))
    assert np.abs((re + 1j * im) - want).max() < 1e-14
    assert abs(oracle.norm2(re, im) - n0) < 1e-13 * n0


def test_constant_potential_is_global_phase():
    # flat V => H0 only contributes a global phase
    nx, ny, theta, n, V0 = 6, 4, 0.2, 5, 0.7
    re, im = rand_state(ny, nx, 11)
    r1, i1 = re.copy(), im.copy()
    pot = (np.full((ny, nx), math.cos(V0)), np.full((ny, nx), -math.sin(V0)))
    oracle.evolve(re, im, *coeffs(theta), pot=pot, periodic=False, n_steps=n)
    oracle.evolve(r1, i1, *coeffs(theta), pot=None, periodic=False, n_steps=n)
    want = (r1 + 1j * i1) * np.exp(-1j * V0 * n)
    assert np.abs((re + 1j * im) - want).max() < 1e-13


# --- a7: the full step equals the ordered dense product (Eq. 3) ------------------
@pytest.mark.parametrize("nx,ny,periodic", [(5, 3, False), (6, 4, False), (8, 8, False),
                                            (6, 4, True), (8, 8, True), (4, 6, True)])
@pytest.mark.parametrize("with_pot", [False, True])
def test_step_equals_dense_product(nx, ny, periodic, with_pot):
    theta, n = 0.31, 3
    re, im = rand_state(ny, nx, 21)
    V = None
    pot = None
    if with_pot:
        V = np.random.default_rng(5).uniform(-3, 3, (ny, nx))
        pot = (np.cos(V), -np.sin(V))
    U = step_unitary(nx, ny, periodic, theta, V=V, dt=1.0)
    want = np.linalg.matrix_power(U, n) @ to_vec(re, im)
    oracle.evolve(re, im, *coeffs(theta), pot=pot, periodic=periodic, n_steps=n)
    assert np.abs(to_vec(re, im) - want).max() < 1e-13


def test_stage_order_matters_and_is_the_documented_one():
    # Swapping whole X and Y groups changes nothing (X parts commute with Y parts, even around
    # the phase), but swapping even and odd WITHIN an axis -- the paper's literal 1-D order has
    # the odd part outermost -- is a different second-order operator.  The oracle
    # must be the documented even-outermost one (reading R5).
    nx, ny, theta = 4, 4, 0.6
    V = np.random.default_rng(1).uniform(-2, 2, (ny, nx))
    re, im = rand_state(ny, nx, 2)
    v0 = to_vec(re, im)
    oracle.evolve(re, im, *coeffs(theta), pot=(np.cos(V), -np.sin(V)), periodic=False, n_steps=1)
    good = step_unitary(nx, ny, False, theta, V=V) @ v0
    assert np.abs(to_vec(re, im) - good).max() < 1e-13
    h = theta / 2
    Xe, Xo = part_unitary(nx, ny, 0, 0, False, h), part_unitary(nx, ny, 0, 1, False, h)
    Ye, Yo = part_unitary(nx, ny, 1, 0, False, h), part_unitary(nx, ny, 1, 1, False, h)
    P = np.diag(np.exp(-1j * V.reshape(-1)))
    xy_swapped = Ye @ Yo @ Xe @ Xo @ P @ Xo @ Xe @ Yo @ Ye @ v0
    assert np.abs(to_vec(re, im) - xy_swapped).max() < 1e-13
    odd_outermost = Xo @ Xe @ Yo @ Ye @ P @ Ye @ Yo @ Xe @ Xo @ v0
    assert np.abs(to_vec(re, im) - odd_outermost).max() > 1e-3


# --- a7: palindrome => time reversible ----------------------------------------------------------
@pytest.mark.parametrize("periodic", [False, True])
def test_reversibility(periodic):
    nx, ny, theta, n = 12, 10, 0.13, 25
    re, im = rand_state(ny, nx, 31)
    r0, i0 = re.copy(), im.copy()
    V = np.random.default_rng(6).uniform(-3, 3, (ny, nx))
    ah, bh, af, bf = coeffs(theta)
    oracle.evolve(re, im, ah, bh, af, bf, pot=(np.cos(V), -np.sin(V)), periodic=periodic, n_steps=n)
    assert np.abs(re - r0).max() > 1e-2
    oracle.evolve(re, im, ah, -bh, af, -bf, pot=(np.cos(V), +np.sin(V)), periodic=periodic, n_steps=n)
    assert np.abs(re - r0).max() < 1e-13 and np.abs(im - i0).max() < 1e-13


# --- a7: second order: error vs exp(-iHT) falls 4x per halving of dt --------
@pytest.mark.parametrize("periodic", [False, True])
@pytest.mark.parametrize("with_pot", [False, True])
def test_dt2_convergence_to_exact_exponential(periodic, with_pot):
    nx = ny = 6
    J, T = 1.0, 1.0
    re0, im0 = rand_state(ny, nx, 41)
    nrm = math.sqrt(oracle.norm2(re0, im0))
    re0 /= nrm; im0 /= nrm
    V = None
    if with_pot:
        y, x = np.mgrid[0:ny, 0:nx]
        V = 0.3 * ((x - 2.5) ** 2 + (y - 2.0) ** 2)
    exact = exact_unitary(nx, ny, periodic, J, T, V=V) @ to_vec(re0, im0)
    errs = []
    for n in (20, 40, 80, 160):
        dt = T / n
        theta = J * dt            # theta = dt*|V_tunnel|/hbar
        re, im = re0.copy(), im0.copy()
        pot = None if V is None else (np.cos(V * dt), -np.sin(V * dt))
        oracle.evolve(re, im, *coeffs(theta), pot=pot, periodic=periodic, n_steps=n)
        errs.append(np.abs(to_vec(re, im) - exact).max())
    ratios = [errs[i] / errs[i + 1] for i in range(3)]
    assert errs[0] < 5e-3 and errs[-1] < errs[0] / 50
    assert all(3.8 < r < 4.2 for r in ratios), (errs, ratios)


# --- a7: X and Y parts commute without a potential (SURVEY 8(c) reading 5) -----------------------
def test_xy_regrouping_without_potential():
    nx, ny, theta = 8, 6, 0.23
    re, im = rand_state(ny, nx, 51)
    r1, i1 = re.copy(), im.copy()
    ah, bh, af, bf = coeffs(theta)
    oracle.evolve(re, im, ah, bh, af, bf, periodic=False, n_steps=1)
    for (axis, parity, a, b) in [(0, 0, ah, bh), (0, 1, af, bf), (0, 0, ah, bh),
                                 (1, 0, ah, bh), (1, 1, af, bf), (1, 0, ah, bh)]:
        oracle.sweep(r1, i1, axis, parity, a, b, False)
    assert np.abs(re - r1).max() < 1e-14 and np.abs(im - i1).max() < 1e-14


# --- a8/a9: unitarity and the norm ---------------------------------------------------------------
def test_norm2_matches_numpy_and_is_conserved():
    nx, ny = 40, 33
    re, im = rand_state(ny, nx, 61)
    n0 = oracle.norm2(re, im)
    assert n0 == pytest.approx(float(np.sum(re * re + im * im)), rel=1e-14)
    V = np.random.default_rng(9).uniform(-5, 5, (ny, nx))
    oracle.evolve(re, im, *coeffs(0.05), pot=(np.cos(V), -np.sin(V)), periodic=False, n_steps=200)
    assert abs(oracle.norm2(re, im) / n0 - 1) < 1e-12


# --- periodic: exact eigenstates at any size -----------------------------------------------------
@pytest.mark.parametrize("sx,sy", [(0, 0), (1, 0), (0, 1), (1, 1)])
def test_periodic_checkerboard_eigenstates(sx, sy):
    nx, ny, theta, n = 16, 12, 0.21, 9
    y, x = np.mgrid[0:ny, 0:nx]
    psi0 = ((-1.0) ** (sx * x + sy * y)) / math.sqrt(nx * ny)
    re, im = psi0.copy(), np.zeros_like(psi0)
    oracle.evolve(re, im, *coeffs(theta), periodic=True, n_steps=n)
    # every site is paired in every sweep: (c,c) -> e^{i t}(c,c), (c,-c) -> e^{-i t}(c,-c);
    # per step the x parts contribute 2*theta*(1-2sx), the y parts 2*theta*(1-2sy)
    ph = np.exp(1j * 2 * n * theta * ((1 - 2 * sx) + (1 - 2 * sy)))
    assert np.abs((re + 1j * im) - ph * psi0).max() < 1e-14


# --- delta start: each hop carries a factor i ----------------------------------------------------
def test_delta_checkerboard_invariant():
    nx, ny = 20, 18
    re = np.zeros((ny, nx)); im = np.zeros((ny, nx))
    re[7, 9] = 1.0
    oracle.evolve(re, im, *coeffs(0.4), periodic=False, n_steps=6)
    y, x = np.mgrid[0:ny, 0:nx]
    odd = ((abs(x - 9) + abs(y - 7)) % 2) == 1
    assert np.all(re[odd] == 0.0) and np.all(im[~odd] == 0.0)
    assert np.abs(im[odd]).max() > 1e-3


# --- golden tables (written from dense matrices by tests/golden/make_golden.py) -------------------
def test_golden_G1_closed():
    gr, gi = load_golden("G1.txt")
    re = np.zeros((4, 4)); im = np.zeros((4, 4)); re[2, 1] = 1.0
    oracle.evolve(re, im, *coeffs(0.3), periodic=False, n_steps=3)
    assert np.abs(re - gr).max() < 1e-14 and np.abs(im - gi).max() < 1e-14
    # two entries as printed in SURVEY.md 8(c), retyped by hand
    assert gr[3, 0] == pytest.approx(-0.456940473303475, abs=1e-14)
    assert gi[0, 0] == pytest.approx(-0.220727410314480, abs=1e-14)


def test_golden_G2_periodic_potential():
    gr, gi = load_golden("G2.txt")
    y, x = np.mgrid[0:4, 0:4]
    V = 0.1 * (x + 2 * y)
    re = np.zeros((4, 4)); im = np.zeros((4, 4)); re[2, 1] = 1.0
    oracle.evolve(re, im, *coeffs(0.3), pot=(np.cos(V), -np.sin(V)), periodic=True, n_steps=3)
    assert np.abs(re - gr).max() < 1e-14 and np.abs(im - gi).max() < 1e-14
    assert gr[1, 3] == pytest.approx(-0.291735876653960, abs=1e-14)
    assert gi[0, 3] == pytest.approx(-0.323800052908717, abs=1e-14)


# --- causal-window oracle == full oracle on its interior -----------------------------------------
@pytest.mark.parametrize("periodic", [False, True])
@pytest.mark.parametrize("win", [(20, 24, 8, 6), (0, 0, 6, 6), (58, 60, 6, 4), (31, 1, 5, 7)])
def test_window_oracle_is_exact(periodic, win):
    nx, ny, theta, n = 64, 64, 0.3, 5
    x0, y0, w, h = win
    re0, im0 = rand_state(ny, nx, 71)
    V = np.random.default_rng(10).uniform(-3, 3, (ny, nx))
    pr, pi = np.cos(V), -np.sin(V)
    re, im = re0.copy(), im0.copy()
    oracle.evolve(re, im, *coeffs(theta), pot=(pr, pi), periodic=periodic, n_steps=n)
    wr, wi = oracle.window_evolve(lambda ys, xs: (re0[np.ix_(ys, xs)], im0[np.ix_(ys, xs)]),
                                  nx, ny, x0, y0, w, h, *coeffs(theta), periodic, n,
                                  fetch_pot=lambda ys, xs: (pr[np.ix_(ys, xs)], pi[np.ix_(ys, xs)]))
    assert np.array_equal(wr, re[y0:y0 + h, x0:x0 + w])
    assert np.array_equal(wi, im[y0:y0 + h, x0:x0 + w])


def test_periodic_rejects_odd_sizes():
    re, im = rand_state(4, 5, 1)
    with pytest.raises(ValueError):
        oracle.evolve(re, im, *coeffs(0.1), periodic=True, n_steps=1)


# --- per-axis boundaries (row slabs of a domain decomposition) -----------------
@pytest.mark.parametrize("px,py", [(True, False), (False, True), (True, True), (False, False)])
@pytest.mark.parametrize("with_pot", [False, True])
def test_evolve_xy_equals_dense_product_per_axis(px, py, with_pot):
    from dense_ref import step_unitary_xy
    nx, ny, theta = 6, 4, 0.37
    rng = np.random.default_rng(17)
    V = rng.uniform(-2, 2, (ny, nx)) if with_pot else None
    re, im = rand_state(ny, nx, 21)
    U = step_unitary_xy(nx, ny, px, py, theta, V)
    want = U @ (U @ to_vec(re, im))
    pot = None if V is None else (np.cos(V), -np.sin(V))
    oracle.evolve_xy(re, im, *coeffs(theta), pot=pot, periodic_x=px, periodic_y=py, n_steps=2)
    wr, wi = from_vec(want, ny, nx)
    assert np.abs(re - wr).max() < 1e-13 and np.abs(im - wi).max() < 1e-13


def test_evolve_xy_with_equal_boundaries_is_evolve():
    re, im = rand_state(10, 12, 5)
    r2, i2 = re.copy(), im.copy()
    oracle.evolve(re, im, *coeffs(0.2), periodic=True, n_steps=3)
    oracle.evolve_xy(r2, i2, *coeffs(0.2), periodic_x=True, periodic_y=True, n_steps=3)
    assert np.array_equal(re, r2) and np.array_equal(im, i2)


# --- separable potential (harmonic trap: V = Vx + Vy) --------------------------------------------
def test_evolve_sep_is_evolve_with_the_sum_potential():
    nx, ny, theta = 10, 8, 0.23
    rng = np.random.default_rng(3)
    Vx, Vy = rng.uniform(-2, 2, nx), rng.uniform(-2, 2, ny)
    re, im = rand_state(ny, nx, 6)
    r2, i2 = re.copy(), im.copy()
    V = Vy[:, None] + Vx[None, :]
    oracle.evolve(re, im, *coeffs(theta), pot=(np.cos(V), -np.sin(V)), periodic=True, n_steps=4)
    oracle.evolve_sep(r2, i2, *coeffs(theta), (np.cos(Vx), -np.sin(Vx)), (np.cos(Vy), -np.sin(Vy)),
                      periodic=True, n_steps=4)
    assert np.abs(re - r2).max() < 1e-14 and np.abs(im - i2).max() < 1e-14


# --- physics of the whole step: group velocity of a wavepacket (tight-binding dispersion) ---------
def test_wavepacket_moves_with_the_tight_binding_group_velocity():
    # H = -J * Adj has E(k) = -2J (cos kx + cos ky), so a packet of mean momentum k drifts by
    # dE/dk = 2J sin k per unit time: per step of angle theta = J dt that is 2 theta sin k sites.
    # Checks sign (R1: +i b, so positive k moves to +x), the half-angle reading (R2: a step is ONE
    # dt, not two) and the x/y assignment, independently of any matrix code.
    nx = ny = 96
    kx, ky, sigma, theta, n = 0.5, -0.3, 8.0, 0.05, 60
    x = np.arange(nx)[None, :] - 40.0
    y = np.arange(ny)[:, None] - 52.0
    env = np.exp(-(x * x + y * y) / (4 * sigma * sigma))
    re = env * np.cos(kx * x + ky * y)
    im = env * np.sin(kx * x + ky * y)
    nrm = math.sqrt((re * re + im * im).sum())
    re, im = np.ascontiguousarray(re / nrm), np.ascontiguousarray(im / nrm)

    def centre(r, i):
        p = r * r + i * i
        return (p * np.arange(nx)[None, :]).sum(), (p * np.arange(ny)[:, None]).sum()

    x0, y0 = centre(re, im)
    oracle.evolve(re, im, *coeffs(theta), periodic=False, n_steps=n)
    x1, y1 = centre(re, im)
    # finite width in k: <sin k> = sin(k0) exp(-1/(8 sigma^2)) for a Gaussian of std 1/(2 sigma)
    damp = math.exp(-1.0 / (8 * sigma * sigma))
    want_dx = 2 * theta * n * math.sin(kx) * damp
    want_dy = 2 * theta * n * math.sin(ky) * damp
    assert abs((x1 - x0) - want_dx) < 0.02 * abs(want_dx), (x1 - x0, want_dx)
    assert abs((y1 - y0) - want_dy) < 0.02 * abs(want_dy), (y1 - y0, want_dy)


def test_packet_in_a_harmonic_trap_oscillates_at_the_classical_frequency():
    # small momenta: E(k) ~ -2J + J k^2, an effective mass m = 1/(2J); in V = w^2 x^2 / 2 the
    # packet centre follows x_c + A cos(W t), W = w sqrt(2J) (Ehrenfest).  Pins the SIGN of the
    # potential phase (R9: exp(-i V dt); with +i the trap repels) and its place in the step.
    nx, ny = 192, 4
    J, w, A, dt = 0.25, 0.02, 12.0, 1.0
    W = w * math.sqrt(2 * J)
    sigma = math.sqrt(J / W) / math.sqrt(2) * math.sqrt(2)      # ground-state width of |psi|^2
    xc = 96.0
    x = np.arange(nx)[None, :] - xc
    env = np.exp(-((x - A) ** 2) / (4 * sigma * sigma)) * np.ones((ny, 1))
    re = np.ascontiguousarray(env / math.sqrt((env * env).sum()))
    im = np.zeros_like(re)
    V = 0.5 * w * w * (x * x) * np.ones((ny, 1))
    pot = (np.cos(V * dt), -np.sin(V * dt))
    quarter = int(round(math.pi / (2 * W)))

    def centre(r, i):
        p = r * r + i * i
        return (p * np.arange(nx)[None, :]).sum() / p.sum() - xc

    assert abs(centre(re, im) - A) < 1e-9
    oracle.evolve(re, im, *coeffs(J * dt), pot=pot, periodic=True, n_steps=quarter)
    assert abs(centre(re, im)) < 0.06 * A, centre(re, im)            # through the centre
    oracle.evolve(re, im, *coeffs(J * dt), pot=pot, periodic=True, n_steps=quarter)
    assert abs(centre(re, im) + A) < 0.06 * A, centre(re, im)        # at the other turning point
