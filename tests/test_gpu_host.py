"""-m gpu parity of ts_evolve_host (host-resident planes; the entry bench.py's "e2e" times): against
the oracle, and bit for bit against ts_evolve on device planes -- small lattices (one upload), and
lattices large enough that the planes go up in pieces while the row chain of the pieces already
there runs (axis-split path), with every path that must instead wait for the whole upload."""
from __future__ import annotations

import math

import numpy as np
import pytest

import gpu_util as G
import oracle

pytestmark = pytest.mark.gpu

TIGHT = {"f32": 2e-5, "f64": 5e-14}


def coeffs(theta):
    return (math.cos(theta / 2), math.sin(theta / 2), math.cos(theta), math.sin(theta))


CASES = [
    # nx, ny, dtype, boundary, with_pot, options, pinned
    (64, 40, "f32", "closed", False, {}, False),                 # one upload (small)
    (128, 66, "f64", "periodic", True, {}, True),
    (2048, 1024, "f32", "periodic", False, {}, True),             # pieces, rows resident (2 warps per line)
    (2048, 1024, "f32", "closed", False, {}, False),              # the same from pageable memory
    (1024, 1030, "f64", "closed", False, {}, True),               # pieces up, x-ranges down (fp64, pipelined columns)
    (2048, 1030, "f32", "periodic", False, {}, True),             # the same in fp32, 256-column ranges
    (4096, 600, "f32", "closed", False, {"chain": 7}, False),     # several column passes per range, pageable
    (1056, 2048, "f32", "periodic", False, {}, True),             # windowed rows: waits for the upload
    (2048, 1024, "f32", "periodic", False, {"variant": 2}, True), # tile kernel: waits for the upload
    (2048, 1024, "f32", "closed", False, {"path": 1}, True),      # per-sweep kernels: wait
    (2048, 1024, "f32", "closed", True, {}, True),                # potential: one upload
]


@pytest.mark.parametrize("nx,ny,dtype,boundary,with_pot,opts,pinned", CASES)
def test_host_entry_matches_oracle_and_device_entry(nx, ny, dtype, boundary, with_pot, opts, pinned):
    import torch
    from paper_1208_2407_b200.binding import Plan
    dev = torch.device("cuda:0")
    tdt = torch.float32 if dtype == "f32" else torch.float64
    re, im, pot = G.random_inputs(nx, ny, dtype, 5 * nx + ny, with_pot)
    n, theta = 5, 0.3
    plan = Plan(nx, ny, tdt, boundary)
    for k, v in opts.items():
        plan.set_option(k, v)
    h_re, h_im = torch.from_numpy(re.copy()), torch.from_numpy(im.copy())
    h_pot = None if pot is None else torch.from_numpy(pot.copy())
    if pinned:
        h_re, h_im = h_re.pin_memory(), h_im.pin_memory()
        h_pot = None if h_pot is None else h_pot.pin_memory()
    for _ in range(2):        # twice: the second call reuses the plan's streams, events and buffers
        h_re.copy_(torch.from_numpy(re)); h_im.copy_(torch.from_numpy(im))
        plan.evolve_host(h_re, h_im, *coeffs(theta), pot_phase=h_pot, n_steps=n)
    info = {k: plan.info(k) for k in ("fused", "variant", "launches", "passes")}
    # the device entry on the same plan
    d_re, d_im = torch.from_numpy(re).to(dev), torch.from_numpy(im).to(dev)
    d_pot = None if pot is None else torch.from_numpy(pot).to(dev)
    plan.evolve(d_re, d_im, *coeffs(theta), pot_phase=d_pot, n_steps=n)
    torch.cuda.synchronize()
    assert np.array_equal(h_re.numpy(), d_re.cpu().numpy()), info
    assert np.array_equal(h_im.numpy(), d_im.cpu().numpy()), info
    wre, wim = re.astype(np.float64), im.astype(np.float64)
    p64 = None if pot is None else (pot[0].astype(np.float64), pot[1].astype(np.float64))
    oracle.evolve(wre, wim, *coeffs(theta), pot=p64, periodic=boundary == "periodic", n_steps=n)
    err = max(np.abs(h_re.numpy() - wre).max(), np.abs(h_im.numpy() - wim).max())
    assert err <= TIGHT[dtype] * 2, (err, info)
    # zero steps: the planes come back unchanged
    h_re.copy_(torch.from_numpy(re)); h_im.copy_(torch.from_numpy(im))
    plan.evolve_host(h_re, h_im, *coeffs(theta), pot_phase=h_pot, n_steps=0)
    assert np.array_equal(h_re.numpy(), re) and np.array_equal(h_im.numpy(), im)
    plan.destroy()


def test_host_entry_rejects_bad_coefficients_after_the_upload_started():
    """An error found by ts_evolve after the pieces were enqueued: the call returns the error with
    nothing left running on the plan's streams, and the plan stays usable."""
    import torch
    from paper_1208_2407_b200.binding import Plan, TsError
    nx, ny = 2048, 1024
    re, im, _ = G.random_inputs(nx, ny, "f32", 3, False)
    plan = Plan(nx, ny, torch.float32, "periodic")
    h_re, h_im = torch.from_numpy(re.copy()).pin_memory(), torch.from_numpy(im.copy()).pin_memory()
    with pytest.raises(TsError):
        plan.evolve_host(h_re, h_im, 0.9, 0.9, 1.0, 0.0, n_steps=3)       # a^2 + b^2 != 1
    assert np.array_equal(h_re.numpy(), re) and np.array_equal(h_im.numpy(), im)
    plan.evolve_host(h_re, h_im, *coeffs(0.3), n_steps=3)
    wre, wim = re.astype(np.float64), im.astype(np.float64)
    oracle.evolve(wre, wim, *coeffs(0.3), pot=None, periodic=True, n_steps=3)
    err = max(np.abs(h_re.numpy() - wre).max(), np.abs(h_im.numpy() - wim).max())
    assert err <= TIGHT["f32"] * 2, err
    plan.destroy()
