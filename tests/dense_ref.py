"""Dense linear-algebra statements of the method, used ONLY to pin the oracle.

Nothing here loops over pairs and rotates them: every operator is built as a Hermitian
matrix (an adjacency matrix of one split part, or the full tight-binding
Hamiltonian) and exponentiated by scipy.linalg.expm, so a slip in the oracle's
pair enumeration, sign, index order or stage order shows up as a mismatch.

Vectorisation: site (x, y) <-> index y*nx + x (x fastest), as in the library.
"""
from __future__ import annotations

import numpy as np
from scipy.linalg import expm


def part_adjacency(nx: int, ny: int, axis: int, parity: int, periodic: bool) -> np.ndarray:
    """Adjacency matrix of one split part (H1 or H2 along one axis, for every line)."""
    n = nx * ny
    A = np.zeros((n, n))
    length = nx if axis == 0 else ny

    def idx(line, i):
        return line * nx + i if axis == 0 else i * nx + line

    lines = ny if axis == 0 else nx
    for line in range(lines):
        for i in range(parity, length - 1, 2):
            p, q = idx(line, i), idx(line, i + 1)
            A[p, q] += 1.0
            A[q, p] += 1.0
        if periodic and parity == 1:
            # wrap bond (n-1, 0); for length == 2 this doubles the single bond (documented)
            p, q = idx(line, length - 1), idx(line, 0)
            A[p, q] += 1.0
            A[q, p] += 1.0
    return A


def part_unitary(nx, ny, axis, parity, periodic, theta) -> np.ndarray:
    """exp(+i theta A_part): 2x2 blocks [[cos, i sin],[i sin, cos]] (reading R1)."""
    # length-2 periodic lines carry weight 2 on their single bond (= the bond rotated twice)
    return expm(1j * theta * part_adjacency(nx, ny, axis, parity, periodic))


def full_adjacency(nx, ny, periodic) -> np.ndarray:
    return sum(part_adjacency(nx, ny, ax, par, periodic) for ax in (0, 1) for par in (0, 1))


def step_unitary(nx, ny, periodic, theta, V=None, dt=1.0) -> np.ndarray:
    """Ordered product of the dense part exponentials = one second-order step (readings R2-R5).

    Applied to psi left to right: Xe/2 Xo/2 Ye/2 [Yo | Yo/2 P Yo/2] Ye/2 Xo/2 Xe/2, so the
    matrix product is written right to left.
    """
    h = theta / 2.0
    Xe = part_unitary(nx, ny, 0, 0, periodic, h)
    Xo = part_unitary(nx, ny, 0, 1, periodic, h)
    Ye = part_unitary(nx, ny, 1, 0, periodic, h)
    if V is None:
        mid = part_unitary(nx, ny, 1, 1, periodic, theta)
    else:
        Yo = part_unitary(nx, ny, 1, 1, periodic, h)
        P = np.diag(np.exp(-1j * np.asarray(V, dtype=float).reshape(-1) * dt))
        mid = Yo @ P @ Yo
    return Xe @ Xo @ Ye @ mid @ Ye @ Xo @ Xe


def step_unitary_xy(nx, ny, periodic_x, periodic_y, theta, V=None, dt=1.0) -> np.ndarray:
    """step_unitary with one boundary type per axis (a row slab: periodic in x, closed in y)."""
    h = theta / 2.0
    Xe = part_unitary(nx, ny, 0, 0, periodic_x, h)
    Xo = part_unitary(nx, ny, 0, 1, periodic_x, h)
    Ye = part_unitary(nx, ny, 1, 0, periodic_y, h)
    if V is None:
        mid = part_unitary(nx, ny, 1, 1, periodic_y, theta)
    else:
        Yo = part_unitary(nx, ny, 1, 1, periodic_y, h)
        P = np.diag(np.exp(-1j * np.asarray(V, dtype=float).reshape(-1) * dt))
        mid = Yo @ P @ Yo
    return Xe @ Xo @ Ye @ mid @ Ye @ Xo @ Xe


def exact_unitary(nx, ny, periodic, J, T, V=None) -> np.ndarray:
    """exp(-i H T), H = -J * Adj + diag(V): the thing the splitting approximates (Eq. 2)."""
    H = -J * full_adjacency(nx, ny, periodic)
    if V is not None:
        H = H + np.diag(np.asarray(V, dtype=float).reshape(-1))
    return expm(-1j * H * T)


def to_vec(re, im) -> np.ndarray:
    return (np.asarray(re) + 1j * np.asarray(im)).reshape(-1)


def from_vec(v, ny, nx):
    v = np.asarray(v).reshape(ny, nx)
    return np.ascontiguousarray(v.real), np.ascontiguousarray(v.imag)
