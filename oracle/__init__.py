"""CPU oracle for the second-order Trotter-Suzuki step -- TEST INFRASTRUCTURE ONLY.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  The product path
(``paper_1208_2407_b200``) never does, and this package never imports the product.

The arithmetic lives in ``ts_oracle.c`` (plain C, double precision, the paper's operator
sequence written out; citations there).  This file only builds it with gcc, loads it with
ctypes and marshals numpy arrays.  ``ts_oracle3d.c`` is the same statement for three-dimensional
lattices (``sweep3``, ``evolve3``).  ``window_evolve`` is the causal-window oracle of
SURVEY.md 8(c): the same C routine run on a cut-out whose margin exceeds the light cone
(2 sites per step when the window origin is even), so it is exact on the interior.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "ts_oracle.c"
_LIB = _HERE / "libts_oracle.so"
_lib = None
_SRC3 = _HERE / "ts_oracle3d.c"
_LIB3 = _HERE / "libts_oracle3d.so"
_lib3 = None

_D = ctypes.POINTER(ctypes.c_double)


def build(force: bool = False) -> Path:
    """Compile ts_oracle.c -> libts_oracle.so (gcc -O2 -fopenmp, no fast-math)."""
    if force or not _LIB.exists() or _LIB.stat().st_mtime < _SRC.stat().st_mtime:
        tmp = _LIB.with_suffix(f".so.tmp{os.getpid()}")
        cmd = ["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-std=c11", "-Wall", "-Wextra",
               "-o", str(tmp), str(_SRC)]
        subprocess.run(cmd, check=True)
        os.replace(tmp, _LIB)
    if force or not _LIB3.exists() or _LIB3.stat().st_mtime < _SRC3.stat().st_mtime:
        tmp = _LIB3.with_suffix(f".so.tmp{os.getpid()}")
        cmd = ["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-std=c11", "-Wall", "-Wextra",
               "-o", str(tmp), str(_SRC3)]
        subprocess.run(cmd, check=True)
        os.replace(tmp, _LIB3)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        lib = ctypes.CDLL(str(_LIB))
        i64, dbl, i32 = ctypes.c_int64, ctypes.c_double, ctypes.c_int
        lib.oracle_sweep.argtypes = [_D, _D, i64, i64, i32, i32, dbl, dbl, i32]
        lib.oracle_sweep.restype = None
        lib.oracle_phase.argtypes = [_D, _D, i64, i64, _D, _D]
        lib.oracle_phase.restype = None
        lib.oracle_step.argtypes = [_D, _D, i64, i64, dbl, dbl, dbl, dbl, _D, _D, i32]
        lib.oracle_step.restype = None
        lib.oracle_evolve.argtypes = [_D, _D, i64, i64, dbl, dbl, dbl, dbl, _D, _D, i32, i64]
        lib.oracle_evolve.restype = None
        lib.oracle_norm2.argtypes = [_D, _D, i64, i64]
        lib.oracle_norm2.restype = dbl
        lib.oracle_num_threads.argtypes = []
        lib.oracle_num_threads.restype = i32
        lib.oracle_set_num_threads.argtypes = [i32]
        lib.oracle_set_num_threads.restype = None
        _lib = lib
    return _lib


def _plane(a: np.ndarray) -> np.ndarray:
    if a.dtype != np.float64 or a.ndim != 2 or not a.flags.c_contiguous or not a.flags.writeable:
        raise ValueError("oracle planes must be writable C-contiguous float64 [ny][nx] arrays")
    return a


def _ptr(a):
    return None if a is None else a.ctypes.data_as(_D)


def num_threads() -> int:
    return int(_load().oracle_num_threads())


def set_num_threads(n: int) -> None:
    _load().oracle_set_num_threads(int(n))


def sweep(re, im, axis: int, parity: int, a: float, b: float, periodic: bool) -> None:
    """In place: one checkerboard sweep (axis 0 = x, 1 = y; parity 0 = even, 1 = odd)."""
    _plane(re), _plane(im)
    ny, nx = re.shape
    _load().oracle_sweep(_ptr(re), _ptr(im), nx, ny, axis, parity, a, b, int(bool(periodic)))


def phase(re, im, pot_re, pot_im) -> None:
    """In place: psi <- psi * (pot_re + i pot_im)."""
    _plane(re), _plane(im)
    ny, nx = re.shape
    pot_re = np.ascontiguousarray(pot_re, dtype=np.float64)
    pot_im = np.ascontiguousarray(pot_im, dtype=np.float64)
    assert pot_re.shape == re.shape and pot_im.shape == re.shape
    _load().oracle_phase(_ptr(re), _ptr(im), nx, ny, _ptr(pot_re), _ptr(pot_im))


def evolve(re, im, a_half, b_half, a_full, b_full, pot=None, periodic=False, n_steps=1) -> None:
    """In place: n_steps second-order steps.  pot = None or (pot_re, pot_im) float64 planes."""
    _plane(re), _plane(im)
    ny, nx = re.shape
    if im.shape != re.shape:
        raise ValueError("re/im shape mismatch")
    if periodic and (nx % 2 or ny % 2):
        raise ValueError("periodic needs even nx, ny (an odd ring cannot be 2-coloured)")
    pr = pi = None
    if pot is not None:
        pr = np.ascontiguousarray(pot[0], dtype=np.float64)
        pi = np.ascontiguousarray(pot[1], dtype=np.float64)
        assert pr.shape == re.shape and pi.shape == re.shape
    _load().oracle_evolve(_ptr(re), _ptr(im), nx, ny, a_half, b_half, a_full, b_full,
                          _ptr(pr), _ptr(pi), int(bool(periodic)), int(n_steps))


def evolve_xy(re, im, a_half, b_half, a_full, b_full, pot=None, periodic_x=False,
              periodic_y=False, n_steps=1) -> None:
    """In place: n_steps second-order steps with one boundary type PER AXIS.

    The stage list of SURVEY.md 8(c) / ``oracle_step`` written out with the C sweep and phase
    routines (each pinned on its own), so that the horizontal sweeps can wrap while the vertical
    ones do not: the lattice a row slab of a domain decomposition is evolved on.
    """
    _plane(re), _plane(im)
    for _ in range(int(n_steps)):
        sweep(re, im, 0, 0, a_half, b_half, periodic_x)
        sweep(re, im, 0, 1, a_half, b_half, periodic_x)
        sweep(re, im, 1, 0, a_half, b_half, periodic_y)
        if pot is None:
            sweep(re, im, 1, 1, a_full, b_full, periodic_y)
        else:
            sweep(re, im, 1, 1, a_half, b_half, periodic_y)
            phase(re, im, pot[0], pot[1])
            sweep(re, im, 1, 1, a_half, b_half, periodic_y)
        sweep(re, im, 1, 0, a_half, b_half, periodic_y)
        sweep(re, im, 0, 1, a_half, b_half, periodic_x)
        sweep(re, im, 0, 0, a_half, b_half, periodic_x)


def evolve_sep(re, im, a_half, b_half, a_full, b_full, phase_x, phase_y, periodic=False,
               n_steps=1) -> None:
    """In place: the 9-stage step with a SEPARABLE potential phase P(x, y) = px(x) * py(y),
    phase_x = (Re px, Im px) over x, phase_y likewise over y (float64).  By definition the
    diagonal step multiplies site (x, y) by that complex product, so this is ``evolve`` with the
    product written out as planes (exp(-i dt H0) with V = Vx + Vy)."""
    px = np.asarray(phase_x[0], dtype=np.float64) + 1j * np.asarray(phase_x[1], dtype=np.float64)
    py = np.asarray(phase_y[0], dtype=np.float64) + 1j * np.asarray(phase_y[1], dtype=np.float64)
    P = py[:, None] * px[None, :]
    evolve(re, im, a_half, b_half, a_full, b_full,
           pot=(np.ascontiguousarray(P.real), np.ascontiguousarray(P.imag)), periodic=periodic,
           n_steps=n_steps)


def evolve_tdep(re, im, a_half, b_half, a_full, b_full, pots, periodic=False) -> None:
    """In place: one second-order step per entry of `pots`, step k with the potential phase
    pots[k] = (pot_re, pot_im) or None (time-dependent Hamiltonian): by definition
    a chain of single steps of ``evolve``."""
    for pot in pots:
        evolve(re, im, a_half, b_half, a_full, b_full, pot=pot, periodic=periodic, n_steps=1)


# p of Eq. 4: p = (4 - 4^(1/3))^-1
U4_P = 1.0 / (4.0 - 4.0 ** (1.0 / 3.0))


def u4_fractions():
    """Time fractions of the five second-order sub-steps of Eq. 4, in order of application."""
    return (U4_P, U4_P, 1.0 - 4.0 * U4_P, U4_P, U4_P)


def evolve_u4(re, im, theta, pot_p=None, pot_q=None, periodic=False, n_steps=1) -> None:
    """In place: n_steps fourth-order steps, Eq. 4 of the paper written out:

        U4(dt) = U2(p dt) U2(p dt) U2((1-4p) dt) U2(p dt) U2(p dt),   p = (4 - 4^(1/3))^-1.

    Each U2(f dt) is ``evolve`` (the pinned second-order step) with angle f*theta, i.e.
    coefficients cos/sin(f theta/2) and cos/sin(f theta); the sequence is a palindrome, so the
    order of application equals the printed order.  With a potential the caller supplies the
    phase planes of the two distinct sub-steps: pot_p = (cos, -sin)(V p dt) and
    pot_q = (cos, -sin)(V (1-4p) dt).
    """
    if (pot_p is None) != (pot_q is None):
        raise ValueError("give both pot_p and pot_q or neither")
    import math
    for _ in range(int(n_steps)):
        for k, f in enumerate(u4_fractions()):
            th = f * theta
            pot = None if pot_p is None else (pot_q if k == 2 else pot_p)
            evolve(re, im, math.cos(th / 2), math.sin(th / 2), math.cos(th), math.sin(th),
                   pot=pot, periodic=periodic, n_steps=1)


def norm2(re, im) -> float:
    re = np.ascontiguousarray(re, dtype=np.float64)
    im = np.ascontiguousarray(im, dtype=np.float64)
    ny, nx = re.shape
    return float(_load().oracle_norm2(_ptr(re), _ptr(im), nx, ny))


def window_evolve(fetch, nx: int, ny: int, x0: int, y0: int, w: int, h: int,
                  a_half, b_half, a_full, b_full, periodic: bool, n_steps: int,
                  fetch_pot=None):
    """Causal-window oracle: exact result on the w x h window at (x0, y0) of an nx x ny lattice.

    ``fetch(ys, xs) -> (re, im)`` returns the INITIAL state (float64) at the index grids
    ``ys[:, None], xs[None, :]`` (already reduced modulo the lattice for periodic);
    ``fetch_pot`` likewise returns (pot_re, pot_im).  The window is grown by a margin of
    2*n_steps + 2 sites per side (the dependency cone is 2 sites per step when
    the cut starts on an even coordinate), snapped to even coordinates, and clipped at real
    closed edges so those coincide with the cut-out's own closed edges.  The cut-out is evolved
    as a CLOSED lattice by the same C routine; the margin is discarded.
    """
    m = 2 * n_steps + 2
    lo_x, hi_x = x0 - m, x0 + w + m
    lo_y, hi_y = y0 - m, y0 + h + m
    lo_x -= lo_x % 2
    lo_y -= lo_y % 2
    hi_x += hi_x % 2
    hi_y += hi_y % 2
    if periodic:
        if hi_x - lo_x >= nx or hi_y - lo_y >= ny:
            raise ValueError("window + margin wraps onto itself; use the full oracle")
        xs = np.arange(lo_x, hi_x) % nx
        ys = np.arange(lo_y, hi_y) % ny
    else:
        lo_x, lo_y = max(lo_x, 0), max(lo_y, 0)
        hi_x, hi_y = min(hi_x, nx), min(hi_y, ny)
        xs = np.arange(lo_x, hi_x)
        ys = np.arange(lo_y, hi_y)
    re, im = fetch(ys, xs)
    re = np.array(re, dtype=np.float64, order="C")
    im = np.array(im, dtype=np.float64, order="C")
    pot = None
    if fetch_pot is not None:
        pot = fetch_pot(ys, xs)
    evolve(re, im, a_half, b_half, a_full, b_full, pot=pot, periodic=False, n_steps=n_steps)
    ox, oy = x0 - lo_x, y0 - lo_y
    return re[oy:oy + h, ox:ox + w].copy(), im[oy:oy + h, ox:ox + w].copy()


# ---- three-dimensional lattices (ts_oracle3d.c) ------------------------------

def _load3():
    global _lib3
    if _lib3 is None:
        build()
        lib = ctypes.CDLL(str(_LIB3))
        i64, dbl, i32 = ctypes.c_int64, ctypes.c_double, ctypes.c_int
        _I = ctypes.POINTER(ctypes.c_int)
        lib.oracle3_sweep.argtypes = [_D, _D, i64, i64, i64, i32, i32, dbl, dbl, i32]
        lib.oracle3_sweep.restype = None
        lib.oracle3_phase.argtypes = [_D, _D, i64, _D, _D]
        lib.oracle3_phase.restype = None
        lib.oracle3_evolve.argtypes = [_D, _D, i64, i64, i64, dbl, dbl, dbl, dbl, _D, _D, _I, i64]
        lib.oracle3_evolve.restype = None
        _lib3 = lib
    return _lib3


def _vol(a: np.ndarray) -> np.ndarray:
    if a.dtype != np.float64 or a.ndim != 3 or not a.flags.c_contiguous or not a.flags.writeable:
        raise ValueError("3-D oracle planes must be writable C-contiguous float64 [nz][ny][nx] arrays")
    return a


def _per3(periodic):
    per = (periodic,) * 3 if isinstance(periodic, (bool, int, np.bool_)) else tuple(periodic)
    if len(per) != 3:
        raise ValueError("periodic: one flag or one per axis (x, y, z)")
    return tuple(bool(p) for p in per)


def sweep3(re, im, axis: int, parity: int, a: float, b: float, periodic: bool) -> None:
    """In place: one checkerboard sweep of a [nz][ny][nx] lattice along axis 0 = x, 1 = y, 2 = z."""
    _vol(re), _vol(im)
    nz, ny, nx = re.shape
    _load3().oracle3_sweep(_ptr(re), _ptr(im), nx, ny, nz, axis, parity, a, b, int(bool(periodic)))


def evolve3(re, im, a_half, b_half, a_full, b_full, pot=None, periodic=False, n_steps=1) -> None:
    """In place: n_steps second-order steps on a [nz][ny][nx] lattice.  periodic: one flag or
    (px, py, pz); pot = None or (pot_re, pot_im) float64 arrays of the lattice's shape."""
    _vol(re), _vol(im)
    if im.shape != re.shape:
        raise ValueError("re/im shape mismatch")
    nz, ny, nx = re.shape
    per = _per3(periodic)
    for n, p in zip((nx, ny, nz), per):
        if p and n % 2:
            raise ValueError("a periodic axis needs an even extent")
    pr = pi = None
    if pot is not None:
        pr = np.ascontiguousarray(pot[0], dtype=np.float64)
        pi = np.ascontiguousarray(pot[1], dtype=np.float64)
        assert pr.shape == re.shape and pi.shape == re.shape
    flags = (ctypes.c_int * 3)(*[int(p) for p in per])
    _load3().oracle3_evolve(_ptr(re), _ptr(im), nx, ny, nz, a_half, b_half, a_full, b_full,
                            _ptr(pr), _ptr(pi), flags, int(n_steps))


def norm2_3d(re, im) -> float:
    """sum |psi|^2 of a 3-D state: the pinned 2-D routine on the same memory viewed as [nz*ny][nx]."""
    re = np.ascontiguousarray(re, dtype=np.float64)
    im = np.ascontiguousarray(im, dtype=np.float64)
    return norm2(re.reshape(-1, re.shape[-1]), im.reshape(-1, im.shape[-1]))
