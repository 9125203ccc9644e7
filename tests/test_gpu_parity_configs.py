"""-m gpu parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times
(default plan options, through the C ABI).

C1-C3: every element against the full-lattice oracle.  C4/C5 (periodic, 2.7e8 / 1.07e9 sites):
the causal-window oracle (exact on the window, oracle/__init__.py) on windows placed at the
centre, across the periodic wrap in x, in y and at the corner, across strip and segment seams of
the fused kernel, plus random ones; and global properties that hold at any size -- the exactly
known periodic eigenstates (closed form) and the norm.  Tolerances are north_star's: max-abs
1e-4 (fp32) / 1e-11 (fp64) after the config's step count; relative errors are printed."""
from __future__ import annotations

import math

import numpy as np
import pytest

import gpu_util as G
import oracle
from paper_1208_2407_b200 import inputs

pytestmark = pytest.mark.gpu


def _report(name, err, rel, info):
    drift = info["norm2_after"] / info["norm2_before"] - 1
    print(f"\n[{name}] max-abs err {err:.3e}  rel-to-max|psi| {rel:.3e}  norm drift {drift:+.3e}  "
          f"fused={info['fused']} S={info['fuse_steps']} passes={info['passes']}")
    return drift


@pytest.mark.parametrize("name", ["C1", "C2", "C3"])
def test_full_lattice_configs(name):
    cfg = inputs.CONFIGS[name]
    re, im, _ = inputs.full_state(cfg)
    pot = inputs.full_pot(cfg)
    got_re, got_im, info = G.gpu_evolve(cfg, re, im, pot)
    want_re, want_im = G.oracle_evolve(cfg, re, im, pot)
    err, rel = G.errors(cfg, got_re, got_im, want_re, want_im)
    drift = _report(name, err, rel, info)
    assert info["fused"] == 1
    assert err <= G.tol(cfg)
    assert rel <= 2e-4           # fp32 rounding over up to 1000 steps, relative to max |psi|
    assert abs(drift) < 1e-4
    assert abs(info["norm2_before"] - 1) < 1e-5


def _windows(cfg, S, seg):
    wi = 128 - 2 * ((2 * S + 3) // 4 * 4)
    nx, ny = cfg.nx, cfg.ny
    rng = np.random.default_rng(7)
    wins = [
        (nx // 2 - 16, ny // 2 - 16, 32, 32),          # centre
        (nx - 16, 1000, 32, 16),                        # across the x wrap
        (2000, ny - 16, 16, 32),                        # across the y wrap
        (nx - 12, ny - 12, 24, 24),                     # corner, both wraps
        (0, 0, 16, 16),                                 # origin
        (wi * 7 - 10, seg * 3 - 10, 20, 20),            # strip seam x segment seam
        (wi * (nx // wi) - 8, seg * 5 - 6, 24, 12),     # last (ragged) strip
    ]
    for _ in range(2):
        wins.append((int(rng.integers(0, nx - 40)), int(rng.integers(0, ny - 40)), 24, 24))
    return wins


def _run_periodic_config(cfg):
    import torch
    from paper_1208_2407_b200.binding import Plan
    dev = torch.device("cuda:0")
    re, im, n2 = inputs.device_state(cfg, dev)
    pot = inputs.device_pot(cfg, dev)
    plan = Plan(cfg.nx, cfg.ny, G.torch_dtype(cfg), cfg.boundary)
    c = cfg.coeffs()

    def fetch_from(t_re, t_im):
        def f(ys, xs):
            iy = torch.as_tensor(ys, device=dev); ix = torch.as_tensor(xs, device=dev)
            return (t_re[iy][:, ix].double().cpu().numpy(), t_im[iy][:, ix].double().cpu().numpy())
        return f

    # probe what the default configuration fuses, to aim windows at its seams
    plan.evolve(re.clone(), im.clone(), *c, pot_phase=pot, n_steps=1)
    S, seg = max(1, plan.info("fuse_steps")), max(2, plan.info("seg_rows"))
    S = S if cfg.n_steps >= S else cfg.n_steps

    wins = _windows(cfg, plan.info("fuse_steps") or 2, seg)
    margin = 2 * cfg.n_steps + 2
    cut = {}
    for (x0, y0, w, h) in wins:       # cut the INPUT windows out before evolving in place
        xs = np.arange(x0 - margin - 2, x0 + w + margin + 2) % cfg.nx
        ys = np.arange(y0 - margin - 2, y0 + h + margin + 2) % cfg.ny
        r, i = fetch_from(re, im)(ys, xs)
        pw = None
        if pot is not None:
            pw = fetch_from(pot[0], pot[1])(ys, xs)
        cut[(x0, y0, w, h)] = (xs, ys, r, i, pw)

    n2_before = plan.norm(re, im)
    plan.evolve(re, im, *c, pot_phase=pot, n_steps=cfg.n_steps)
    torch.cuda.synchronize()
    n2_after = plan.norm(re, im)
    info = {k: plan.info(k) for k in ("fused", "fuse_steps", "passes", "launches", "seg_rows")}
    info["norm2_before"], info["norm2_after"] = n2_before, n2_after

    worst, worst_rel = 0.0, 0.0
    for (x0, y0, w, h), (xs, ys, r, i, pw) in cut.items():
        lut_x = {int(v): k for k, v in enumerate(xs)}
        lut_y = {int(v): k for k, v in enumerate(ys)}

        def fetch(yy, xx, r=r, i=i, lut_x=lut_x, lut_y=lut_y):
            iy = [lut_y[int(v)] for v in yy]; ix = [lut_x[int(v)] for v in xx]
            return r[np.ix_(iy, ix)], i[np.ix_(iy, ix)]

        fetch_pot = None
        if pw is not None:
            def fetch_pot(yy, xx, pw=pw, lut_x=lut_x, lut_y=lut_y):
                iy = [lut_y[int(v)] for v in yy]; ix = [lut_x[int(v)] for v in xx]
                return pw[0][np.ix_(iy, ix)], pw[1][np.ix_(iy, ix)]

        want_re, want_im = oracle.window_evolve(fetch, cfg.nx, cfg.ny, x0, y0, w, h, *c, True,
                                                cfg.n_steps, fetch_pot=fetch_pot)
        oy = np.arange(y0, y0 + h) % cfg.ny
        ox = np.arange(x0, x0 + w) % cfg.nx
        got_re, got_im = fetch_from(re, im)(oy, ox)
        err, rel = G.errors(cfg, got_re, got_im, want_re, want_im)
        worst, worst_rel = max(worst, err), max(worst_rel, rel)
    plan.destroy()
    return worst, worst_rel, info, len(wins)


def test_C4_windows_and_norm():
    cfg = inputs.CONFIGS["C4"]
    err, rel, info, n = _run_periodic_config(cfg)
    drift = _report(f"C4, {n} windows", err, rel, info)
    assert info["fused"] == 1
    assert err <= G.tol(cfg)
    assert rel <= 1e-4
    assert abs(drift) < 1e-5 and abs(info["norm2_before"] - 1) < 1e-5


def test_C5_windows_and_norm():
    import torch
    if torch.cuda.get_device_properties(0).total_memory < 70e9:
        pytest.skip("C5 needs ~52 GB of device memory")
    cfg = inputs.CONFIGS["C5"]
    err, rel, info, n = _run_periodic_config(cfg)
    drift = _report(f"C5, {n} windows", err, rel, info)
    assert info["fused"] == 1
    assert err <= G.tol(cfg)
    assert rel <= 1e-10
    assert abs(drift) < 1e-12 and abs(info["norm2_before"] - 1) < 1e-12


@pytest.mark.parametrize("name,sx,sy", [("C4", 1, 0), ("C4", 1, 1), ("C5", 0, 1)])
def test_full_size_periodic_eigenstates(name, sx, sy):
    """Closed form at full size: psi = (-1)^(sx x + sy y)/sqrt(N) is an exact eigenstate of every
    sweep on a periodic lattice (no potential): U2^n psi = exp(i 2 n theta ((1-2sx)+(1-2sy))) psi."""
    import torch
    from paper_1208_2407_b200.binding import Plan
    cfg = inputs.CONFIGS[name]
    dev = torch.device("cuda:0")
    dt = G.torch_dtype(cfg)
    amp = 1.0 / math.sqrt(cfg.sites)
    sgn_x = (1 - 2 * (sx * (torch.arange(cfg.nx, device=dev) % 2))).to(dt)
    sgn_y = (1 - 2 * (sy * (torch.arange(cfg.ny, device=dev) % 2))).to(dt)
    re = (sgn_y[:, None] * sgn_x[None, :] * amp).contiguous()
    im = torch.zeros_like(re)
    ref = re.clone()
    plan = Plan(cfg.nx, cfg.ny, dt, "periodic")
    n = cfg.n_steps
    plan.evolve(re, im, *cfg.coeffs(), n_steps=n)
    torch.cuda.synchronize()
    ph = 2 * n * cfg.theta * ((1 - 2 * sx) + (1 - 2 * sy))
    err_re = float((re - math.cos(ph) * ref).abs().max())
    err_im = float((im - math.sin(ph) * ref).abs().max())
    rel = max(err_re, err_im) / amp
    print(f"\n[{name} eigenstate sx={sx} sy={sy}] rel err {rel:.3e}")
    assert plan.info("fused") == 1
    assert rel < (2e-5 if cfg.dtype == "f32" else 1e-13)
    plan.destroy()
