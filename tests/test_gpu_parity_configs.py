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


def _windows(cfg, S, seg, variant=2):
    # x seams: interior width of a strip of the 2-D streaming kernel, or of a row window of the
    # axis-split path (1024 / 512 sites less a halo of 2 per chained sub-step, in fours)
    if variant == 4:
        wi = (1024 if cfg.dtype == "f32" else 512) - 2 * ((2 * S + 3) // 4 * 4)
    else:
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


def _run_periodic_config(cfg, sep=False):
    """sep: pass the harmonic potential as separable factors (ts_evolve_sep); the oracle then gets
    the outer product of the same (cast) factors as planes, which is what the entry defines."""
    import torch
    from paper_1208_2407_b200.binding import Plan
    dev = torch.device("cuda:0")
    re, im, n2 = inputs.device_state(cfg, dev)
    plan = Plan(cfg.nx, cfg.ny, G.torch_dtype(cfg), cfg.boundary)
    c = cfg.coeffs()
    if sep:
        sx, sy = inputs.sep_pot(cfg)
        d_sx, d_sy = torch.from_numpy(sx).to(dev), torch.from_numpy(sy).to(dev)
        pot = None
        cx = sx[0].astype(np.float64) + 1j * sx[1].astype(np.float64)
        cy = sy[0].astype(np.float64) + 1j * sy[1].astype(np.float64)

        def evolve(r, i, n):
            plan.evolve_sep(r, i, *c, d_sx, d_sy, n_steps=n)
    else:
        pot = inputs.device_pot(cfg, dev)

        def evolve(r, i, n):
            plan.evolve(r, i, *c, pot_phase=pot, n_steps=n)

    def fetch_from(t_re, t_im):
        def f(ys, xs):
            iy = torch.as_tensor(ys, device=dev); ix = torch.as_tensor(xs, device=dev)
            return (t_re[iy][:, ix].double().cpu().numpy(), t_im[iy][:, ix].double().cpu().numpy())
        return f

    # probe what the default configuration fuses, to aim windows at its seams
    evolve(re.clone(), im.clone(), 1)
    S, seg = max(1, plan.info("fuse_steps")), max(2, plan.info("seg_rows"))
    S = S if cfg.n_steps >= S else cfg.n_steps

    variant = plan.info("variant")
    wins = _windows(cfg, (plan.info("chain_x") if variant == 4 else plan.info("fuse_steps")) or 2,
                    seg, variant)
    margin = 2 * cfg.n_steps + 2
    cut = {}
    for (x0, y0, w, h) in wins:       # cut the INPUT windows out before evolving in place
        xs = np.arange(x0 - margin - 2, x0 + w + margin + 2) % cfg.nx
        ys = np.arange(y0 - margin - 2, y0 + h + margin + 2) % cfg.ny
        r, i = fetch_from(re, im)(ys, xs)
        pw = None
        if pot is not None:
            pw = fetch_from(pot[0], pot[1])(ys, xs)
        elif sep:
            P = cy[ys][:, None] * cx[xs][None, :]
            pw = (np.ascontiguousarray(P.real), np.ascontiguousarray(P.imag))
        cut[(x0, y0, w, h)] = (xs, ys, r, i, pw)

    n2_before = plan.norm(re, im)
    evolve(re, im, cfg.n_steps)
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


def test_C5_separable_entry_windows_and_norm():
    import torch
    if torch.cuda.get_device_properties(0).total_memory < 40e9:
        pytest.skip("needs ~34 GB of device memory")
    cfg = inputs.CONFIGS["C5"]
    err, rel, info, n = _run_periodic_config(cfg, sep=True)
    drift = _report(f"C5 via ts_evolve_sep, {n} windows", err, rel, info)
    assert info["fused"] == 1
    assert err <= G.tol(cfg)
    assert rel <= 1e-10
    assert abs(drift) < 1e-12


def test_C4_size_fourth_order_eigenstate():
    """The same closed form for ts_evolve_u4: the five sub-step angles sum to theta, so
    U4^n psi = exp(i 2 n theta ((1-2sx)+(1-2sy))) psi at full C4 size (8 steps = 40 sub-steps
    chained through passes of 6)."""
    import torch
    from paper_1208_2407_b200.binding import Plan
    cfg = inputs.CONFIGS["C4"]
    dev = torch.device("cuda:0")
    amp = 1.0 / math.sqrt(cfg.sites)
    sgn_x = (1 - 2 * (torch.arange(cfg.nx, device=dev) % 2)).to(torch.float32)
    re = (sgn_x[None, :] * amp).expand(cfg.ny, cfg.nx).contiguous()
    im = torch.zeros_like(re)
    ref = re.clone()
    plan = Plan(cfg.nx, cfg.ny, torch.float32, "periodic")
    n, theta = 8, 0.1
    plan.evolve_u4(re, im, theta, n_steps=n)
    torch.cuda.synchronize()
    ph = 2 * n * theta * ((1 - 2 * 1) + 1)          # sx = 1, sy = 0: the two axes cancel
    ph_x = -2 * n * theta
    # (sx, sy) = (1, 0): X sweeps give exp(-i theta) per step each way, Y sweeps exp(+i theta)
    assert ph == 0.0 and ph_x != 0.0
    rel = max(float((re - ref).abs().max()), float(im.abs().max())) / amp
    print(f"\n[C4-size U4 eigenstate sx=1 sy=0] rel err {rel:.3e}  passes={plan.info('passes')}")
    assert plan.info("fused") == 1
    if plan.info("variant") == 4:       # row chain + column chain, chain_x / chain_y sub-steps per pass
        assert plan.info("passes") == (math.ceil(5 * n / plan.info("chain_x")) +
                                       math.ceil(5 * n / plan.info("chain_y")))
    else:
        assert plan.info("passes") == math.ceil(5 * n / 6)
    assert rel < 2e-5
    # and a state whose phase does not cancel: sx = sy = 0 (uniform), phase 4 n theta
    re.fill_(amp); im.zero_()
    plan.evolve_u4(re, im, theta, n_steps=n)
    torch.cuda.synchronize()
    ph = 4 * n * theta
    rel = max(float((re - math.cos(ph) * amp).abs().max()),
              float((im - math.sin(ph) * amp).abs().max())) / amp
    print(f"[C4-size U4 uniform state] rel err {rel:.3e}")
    assert rel < 2e-5
    plan.destroy()


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


# ---- every element of a full-size lattice against the full oracle ----------------------------------
def _full_lattice_check(cfg, n_steps, option_sets, sep=False):
    """Every element of the lattice against the full oracle for n_steps steps, once per set of plan
    options (the oracle runs once).  Inputs are built on the device (bit-identical to the numpy
    recipe) and downloaded for the oracle."""
    import torch
    from paper_1208_2407_b200.binding import Plan
    dev = torch.device("cuda:0")
    re0, im0, _ = inputs.device_state(cfg, dev)
    pot = inputs.device_pot(cfg, dev)
    c = cfg.coeffs()
    wre = re0.cpu().numpy().astype(np.float64)
    wim = im0.cpu().numpy().astype(np.float64)
    wpot = None
    if pot is not None:
        wpot = (pot[0].cpu().numpy().astype(np.float64), pot[1].cpu().numpy().astype(np.float64))
    oracle.evolve(wre, wim, *c, pot=wpot, periodic=cfg.periodic, n_steps=n_steps)
    del wpot
    scale = max(np.abs(wre).max(), np.abs(wim).max())
    out = []
    for opts in option_sets:
        plan = Plan(cfg.nx, cfg.ny, G.torch_dtype(cfg), cfg.boundary)
        for k, v in opts.items():
            plan.set_option(k, v)
        re, im = re0.clone(), im0.clone()
        n0 = plan.norm(re, im)
        plan.evolve(re, im, *c, pot_phase=pot, n_steps=n_steps)
        torch.cuda.synchronize()
        n1 = plan.norm(re, im)
        info = {k: plan.info(k) for k in ("fused", "fuse_steps", "passes", "seg_rows", "variant")}
        err = 0.0
        rows = 2048
        for y0 in range(0, cfg.ny, rows):       # compare in slabs: no second full-size host copy
            gr = re[y0:y0 + rows].cpu().numpy().astype(np.float64)
            gi = im[y0:y0 + rows].cpu().numpy().astype(np.float64)
            err = max(err, np.abs(gr - wre[y0:y0 + rows]).max(), np.abs(gi - wim[y0:y0 + rows]).max())
        plan.destroy()
        del re, im
        print(f"\n[{cfg.name} full lattice, {n_steps} steps, options {opts}] max-abs err {err:.3e}  "
              f"rel {err / scale:.3e}  norm drift {n1 / n0 - 1:+.3e}  {info}")
        out.append((err, err / scale, n1 / n0 - 1, info))
    return out


@pytest.mark.slow
def test_C4_full_lattice_short():
    """16384^2 fp32 periodic, 24 steps, EVERY element against the full oracle (about 20 s of oracle
    time, 9 GB of host memory): default plan options (the path bench.py times) and the 2-D
    streaming kernel at its default S = 6 (four passes)."""
    import psutil
    if psutil.virtual_memory().available < 14e9:
        pytest.skip("needs ~12 GB of host memory")
    cfg = inputs.CONFIGS["C4"]
    res = _full_lattice_check(cfg, 24, [{}, {"variant": 2}])
    for err, rel, drift, info in res:
        assert info["fused"] == 1
        assert err <= G.tol(cfg) and rel <= 2e-5 and abs(drift) < 1e-5, (err, rel, drift, info)
    assert res[1][3]["variant"] == 2 and res[1][3]["fuse_steps"] == 6 and res[1][3]["passes"] == 4


@pytest.mark.slow
def test_C5_recipe_8192_full_lattice_short():
    """The C5 recipe (fp64, periodic, harmonic trap as phase planes) on 8192^2 -- the full C5 oracle
    needs 34 GB of host memory -- with default options, 12 steps, every element."""
    cfg = inputs.scaled(inputs.CONFIGS["C5"], 8192, 8192, 12)
    (err, rel, drift, info), = _full_lattice_check(cfg, 12, [{}])
    assert info["fused"] == 1 and info["variant"] == 2
    assert err <= G.tol(cfg) and rel <= 1e-11 and abs(drift) < 1e-12, (err, rel, drift, info)


@pytest.mark.parametrize("recipe,opts", [("C4", {}), ("C4", {"variant": 2}), ("C3", {}), ("C5", {})])
def test_2048_default_options_full_lattice(recipe, opts):
    """Mid-size lattices with DEFAULT segment sizes and fusion depths (the small parity tests force
    short segments): the C4 recipe (fp32 periodic, no potential) on the default path and on the
    2-D streaming kernel, the C3 recipe (fp32 closed + trap) and the C5 recipe (fp64 periodic +
    trap), 2048^2, 24 steps, every element against the full oracle."""
    cfg = inputs.scaled(inputs.CONFIGS[recipe], 2048, 2048, 24)
    (err, rel, drift, info), = _full_lattice_check(cfg, 24, [opts])
    assert info["fused"] == 1
    if recipe == "C4" and not opts:
        assert info["variant"] == 4          # resident lines: one launch per axis, no segments
    else:
        assert info["variant"] == 2 and info["seg_rows"] != 0
    assert err <= G.tol(cfg), (err, info)
    assert rel <= (2e-5 if cfg.dtype == "f32" else 1e-11), (rel, info)
    assert abs(drift) < (1e-5 if cfg.dtype == "f32" else 1e-12)
