"""Shared by the slab tests: an oracle-backed stand-in for ts_evolve / ts_norm on CPU tensors, so
that the decomposition logic (partition, halo width, exchange order) is tested without a GPU."""
from __future__ import annotations

import numpy as np

import oracle


def oracle_evolve_fn(re, im, coeffs, pot, n_steps, periodic_x, periodic_y):
    r, i = re.numpy(), im.numpy()          # views: in place
    p = None if pot is None else (pot[0].numpy(), pot[1].numpy())
    oracle.evolve_xy(r, i, *coeffs, pot=p, periodic_x=periodic_x, periodic_y=periodic_y,
                     n_steps=n_steps)


def oracle_norm_fn(re, im):
    return oracle.norm2(re.numpy(), im.numpy())


def problem(nx, ny, seed, with_pot):
    rng = np.random.default_rng(seed)
    re = rng.uniform(-1, 1, (ny, nx))
    im = rng.uniform(-1, 1, (ny, nx))
    pot = None
    if with_pot:
        V = rng.uniform(-3, 3, (ny, nx))
        pot = np.stack([np.cos(V), -np.sin(V)])
    return re, im, pot
