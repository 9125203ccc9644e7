"""Seeded synthetic workloads: the five configurations of BASELINE.json.

This module holds NO arithmetic of the method -- only initial states, potentials and the step
angle -- and is the one module both the CUDA tests/bench and the oracle-side tests use, so both
see bit-identical inputs.  The paper measured on "a synthetic state in a square domain" with a
flat potential; there is no dataset to stand in for.

Everything is generated in float64 on the host with numpy, normalised to sum |psi|^2 = 1 in
float64, and cast to the config's dtype by the caller.  Random states use a counter-based
generator (SplitMix64 of (seed, plane, linear index)) so that any window of a huge lattice can
be regenerated without materialising the rest.
"""
from __future__ import annotations

import math
from dataclasses import dataclass
from typing import Optional

import numpy as np

SEED = 12082407


@dataclass(frozen=True)
class Config:
    name: str
    nx: int
    ny: int
    dtype: str            # "f32" | "f64"
    boundary: str         # "closed" | "periodic"
    theta: float
    n_steps: int
    state: str            # "gaussian" | "random"
    x0: float = 0.0
    y0: float = 0.0
    sigma: float = 1.0
    kx: float = 0.0
    ky: float = 0.0
    omega: Optional[float] = None   # harmonic potential V = 0.5*omega^2*r^2, dt = 1
    cx: float = 0.0
    cy: float = 0.0

    @property
    def periodic(self) -> bool:
        return self.boundary == "periodic"

    @property
    def has_pot(self) -> bool:
        return self.omega is not None

    @property
    def sites(self) -> int:
        return self.nx * self.ny

    def coeffs(self):
        """(a_half, b_half, a_full, b_full) = cos/sin of theta/2 and theta."""
        t = self.theta
        return (math.cos(t / 2), math.sin(t / 2), math.cos(t), math.sin(t))


CONFIGS = {
    "C1": Config("C1", 64, 64, "f32", "closed", 0.01, 100, "gaussian",
                 x0=32, y0=32, sigma=8, kx=0.5, ky=0.0),
    "C2": Config("C2", 1024, 1024, "f32", "closed", 0.01, 1000, "gaussian",
                 x0=512, y0=512, sigma=64, kx=0.3, ky=0.2),
    "C3": Config("C3", 4096, 4096, "f32", "closed", 0.01, 500, "gaussian",
                 x0=1536, y0=2048, sigma=128, omega=1e-3, cx=2048, cy=2048),
    "C4": Config("C4", 16384, 16384, "f32", "periodic", 0.02, 200, "random"),
    "C5": Config("C5", 32768, 32768, "f64", "periodic", 0.01, 50, "random",
                 omega=2.5e-4, cx=16384, cy=16384),
}


def scaled(cfg: Config, nx: int, ny: int, n_steps: Optional[int] = None) -> Config:
    """The same recipe on a smaller lattice (centres and widths scaled with the size)."""
    fx, fy = nx / cfg.nx, ny / cfg.ny
    return Config(f"{cfg.name}@{nx}x{ny}", nx, ny, cfg.dtype, cfg.boundary, cfg.theta,
                  cfg.n_steps if n_steps is None else n_steps, cfg.state,
                  x0=cfg.x0 * fx, y0=cfg.y0 * fy, sigma=max(2.0, cfg.sigma * min(fx, fy)),
                  kx=cfg.kx, ky=cfg.ky, omega=cfg.omega, cx=cfg.cx * fx, cy=cfg.cy * fy)


# ---- counter-based uniform generator ------------------------------------------------------------
_M64 = np.uint64(0xFFFFFFFFFFFFFFFF)


def _splitmix64(z: np.ndarray) -> np.ndarray:
    z = (z + np.uint64(0x9E3779B97F4A7C15)) & _M64
    z = ((z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)) & _M64
    z = ((z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)) & _M64
    return z ^ (z >> np.uint64(31))


def uniform_pm1(seed: int, plane: int, index: np.ndarray) -> np.ndarray:
    """Uniform in [-1, 1) as float64, a pure function of (seed, plane, linear site index)."""
    with np.errstate(over="ignore"):
        key = _splitmix64(np.asarray([seed * 2 + plane], dtype=np.uint64))[0]
        bits = _splitmix64(np.asarray(index, dtype=np.uint64) ^ key)
    # top 53 bits -> [0, 1) -> [-1, 1)
    return (bits >> np.uint64(11)).astype(np.float64) * (2.0 / 9007199254740992.0) - 1.0


# ---- un-normalised fields on index grids ----------------------------------------------------------
def raw_state(cfg: Config, ys: np.ndarray, xs: np.ndarray):
    """Un-normalised (re, im) float64 on the grid ys[:, None] x xs[None, :] of site indices."""
    ys = np.asarray(ys, dtype=np.int64)
    xs = np.asarray(xs, dtype=np.int64)
    if cfg.state == "gaussian":
        X = xs[None, :].astype(np.float64)
        Y = ys[:, None].astype(np.float64)
        env = np.exp(-((X - cfg.x0) ** 2 + (Y - cfg.y0) ** 2) / (4.0 * cfg.sigma ** 2))
        ph = cfg.kx * X + cfg.ky * Y
        return env * np.cos(ph), env * np.sin(ph)
    idx = ys[:, None] * np.int64(cfg.nx) + xs[None, :]
    return uniform_pm1(SEED, 0, idx), uniform_pm1(SEED, 1, idx)


def raw_norm2(cfg: Config, chunk_rows: int = 1024) -> float:
    """sum |psi_raw|^2 over the whole lattice in float64 (chunked; math.fsum over chunks)."""
    xs = np.arange(cfg.nx)
    parts = []
    for y0 in range(0, cfg.ny, chunk_rows):
        re, im = raw_state(cfg, np.arange(y0, min(cfg.ny, y0 + chunk_rows)), xs)
        parts.append(float(np.sum(re * re + im * im, dtype=np.float64)))
    return math.fsum(parts)


def state_window(cfg: Config, ys, xs, norm2: float):
    """Normalised initial state (float64) on an index grid, given the global raw norm^2."""
    re, im = raw_state(cfg, ys, xs)
    s = 1.0 / math.sqrt(norm2)
    return re * s, im * s


def pot_window(cfg: Config, ys, xs):
    """(pot_re, pot_im) = (cos V, -sin V) float64, V = 0.5 omega^2 r^2, dt = 1 (readings R8/R9)."""
    assert cfg.has_pot
    X = np.asarray(xs, dtype=np.float64)[None, :]
    Y = np.asarray(ys, dtype=np.float64)[:, None]
    V = 0.5 * cfg.omega ** 2 * ((X - cfg.cx) ** 2 + (Y - cfg.cy) ** 2)
    return np.cos(V), -np.sin(V)


def np_dtype(cfg: Config):
    return np.float32 if cfg.dtype == "f32" else np.float64


def full_state(cfg: Config, chunk_rows: int = 1024):
    """(re, im, norm2_raw): full normalised planes cast to the config dtype (host numpy)."""
    n2 = raw_norm2(cfg, chunk_rows)
    dt = np_dtype(cfg)
    re = np.empty((cfg.ny, cfg.nx), dtype=dt)
    im = np.empty((cfg.ny, cfg.nx), dtype=dt)
    xs = np.arange(cfg.nx)
    for y0 in range(0, cfg.ny, chunk_rows):
        ys = np.arange(y0, min(cfg.ny, y0 + chunk_rows))
        r, i = state_window(cfg, ys, xs, n2)
        re[y0:y0 + len(ys)] = r
        im[y0:y0 + len(ys)] = i
    return re, im, n2


def full_pot(cfg: Config, chunk_rows: int = 1024):
    """pot_phase [2][ny][nx] cast to the config dtype, or None."""
    if not cfg.has_pot:
        return None
    dt = np_dtype(cfg)
    pot = np.empty((2, cfg.ny, cfg.nx), dtype=dt)
    xs = np.arange(cfg.nx)
    for y0 in range(0, cfg.ny, chunk_rows):
        ys = np.arange(y0, min(cfg.ny, y0 + chunk_rows))
        pr, pi = pot_window(cfg, ys, xs)
        pot[0, y0:y0 + len(ys)] = pr
        pot[1, y0:y0 + len(ys)] = pi
    return pot


# ---- the same generators with torch ops (any device), bit-identical to the numpy ones ------------
def _i64(v: int) -> int:
    """two's-complement int64 view of a uint64 constant"""
    v &= 0xFFFFFFFFFFFFFFFF
    return v - (1 << 64) if v >= (1 << 63) else v


def _lsr(z, k: int):
    """logical shift right of int64 tensors"""
    return (z >> k) & ((1 << (64 - k)) - 1)


def _splitmix64_t(z):
    z = z + _i64(0x9E3779B97F4A7C15)
    z = (z ^ _lsr(z, 30)) * _i64(0xBF58476D1CE4E5B9)
    z = (z ^ _lsr(z, 27)) * _i64(0x94D049BB133111EB)
    return z ^ _lsr(z, 31)


def uniform_pm1_t(seed: int, plane: int, index):
    """torch twin of uniform_pm1: index is an int64 tensor; returns float64 on its device."""
    import torch
    with np.errstate(over="ignore"):
        key = int(_splitmix64(np.asarray([seed * 2 + plane], dtype=np.uint64))[0])
    bits = _splitmix64_t(index ^ _i64(key))
    return _lsr(bits, 11).to(torch.float64) * (2.0 / 9007199254740992.0) - 1.0


def _raw_state_t(cfg: Config, y0: int, y1: int, device):
    import torch
    ys = torch.arange(y0, y1, dtype=torch.int64, device=device)
    xs = torch.arange(cfg.nx, dtype=torch.int64, device=device)
    if cfg.state == "gaussian":
        X = xs[None, :].to(torch.float64)
        Y = ys[:, None].to(torch.float64)
        env = torch.exp(-((X - cfg.x0) ** 2 + (Y - cfg.y0) ** 2) / (4.0 * cfg.sigma ** 2))
        ph = cfg.kx * X + cfg.ky * Y
        return env * torch.cos(ph), env * torch.sin(ph)
    idx = ys[:, None] * cfg.nx + xs[None, :]
    return uniform_pm1_t(SEED, 0, idx), uniform_pm1_t(SEED, 1, idx)


def device_state(cfg: Config, device, chunk_rows: int = 2048):
    """(re, im, norm2_raw) as torch tensors of the config dtype on `device`; generated in float64
    chunk by chunk, normalised by the float64 raw norm, then cast (same recipe as full_state).
    For random states the values are bit-identical to the numpy path given the same norm2."""
    import torch
    dt = torch.float32 if cfg.dtype == "f32" else torch.float64
    parts = []
    for y0 in range(0, cfg.ny, chunk_rows):
        r, i = _raw_state_t(cfg, y0, min(cfg.ny, y0 + chunk_rows), device)
        parts.append(float(torch.sum(r * r + i * i, dtype=torch.float64)))
    n2 = math.fsum(parts)
    s = 1.0 / math.sqrt(n2)
    re = torch.empty((cfg.ny, cfg.nx), dtype=dt, device=device)
    im = torch.empty((cfg.ny, cfg.nx), dtype=dt, device=device)
    for y0 in range(0, cfg.ny, chunk_rows):
        y1 = min(cfg.ny, y0 + chunk_rows)
        r, i = _raw_state_t(cfg, y0, y1, device)
        re[y0:y1] = (r * s).to(dt)
        im[y0:y1] = (i * s).to(dt)
    return re, im, n2


def device_pot(cfg: Config, device, chunk_rows: int = 2048):
    """pot_phase [2][ny][nx] of the config dtype on `device` (float64 cos/sin, then cast)."""
    import torch
    if not cfg.has_pot:
        return None
    dt = torch.float32 if cfg.dtype == "f32" else torch.float64
    pot = torch.empty((2, cfg.ny, cfg.nx), dtype=dt, device=device)
    X = torch.arange(cfg.nx, dtype=torch.float64, device=device)[None, :]
    for y0 in range(0, cfg.ny, chunk_rows):
        y1 = min(cfg.ny, y0 + chunk_rows)
        Y = torch.arange(y0, y1, dtype=torch.float64, device=device)[:, None]
        V = 0.5 * cfg.omega ** 2 * ((X - cfg.cx) ** 2 + (Y - cfg.cy) ** 2)
        pot[0, y0:y1] = torch.cos(V).to(dt)
        pot[1, y0:y1] = (-torch.sin(V)).to(dt)
    return pot


def sep_pot(cfg: Config):
    """The harmonic potential of the recipe as SEPARABLE phase factors (host numpy, config dtype):
    V = 0.5 w^2 (x-cx)^2 + 0.5 w^2 (y-cy)^2, so exp(-i V) = px(x) * py(y);
    returns (phase_x [2][nx], phase_y [2][ny]) = (cos, -sin) of the two 1-D terms, or None."""
    if not cfg.has_pot:
        return None
    dt = np_dtype(cfg)
    vx = 0.5 * cfg.omega ** 2 * (np.arange(cfg.nx, dtype=np.float64) - cfg.cx) ** 2
    vy = 0.5 * cfg.omega ** 2 * (np.arange(cfg.ny, dtype=np.float64) - cfg.cy) ** 2
    return (np.stack([np.cos(vx), -np.sin(vx)]).astype(dt),
            np.stack([np.cos(vy), -np.sin(vy)]).astype(dt))
