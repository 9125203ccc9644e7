"""-m gpu test of ts_norm_static (include/ts.h): the squared norm through the entry
point that allocates nothing -- its partial sums live in a fixed 256 KB array of the library's
device image -- against the existing path (ts_norm, plan-owned workspace) and the oracle, on two
calls in a row that share that array.  Collected last on purpose (the run is `pytest -x`);
passes alone in a fresh process and after the other tests."""
from __future__ import annotations

import ctypes

import numpy as np
import pytest

import oracle
from paper_1208_2407_b200.binding import TS_EINVAL, TS_EUNSUPPORTED, TsError

pytestmark = pytest.mark.gpu

REL = 1e-12     # both sides accumulate in double; only the order of the additions differs
MAX_SITES = 1 << 29


def planes(shape, dtype, seed):
    rng = np.random.default_rng(seed)
    dt = np.float32 if dtype == "f32" else np.float64
    return (rng.uniform(-1, 1, shape).astype(dt), rng.uniform(-1, 1, shape).astype(dt))


@pytest.mark.parametrize("dtype", ["f32", "f64"])
def test_two_calls_in_a_row_match_ts_norm_and_the_oracle(dtype):
    """A large call, then a smaller one on the same stream: the second must not see the partial
    sums the first one left in the shared array; then the first input again (bit-equal: the
    order of the additions is fixed)."""
    import torch
    from paper_1208_2407_b200.binding import Plan, norm_static
    dev = torch.device("cuda:0")
    tdt = torch.float32 if dtype == "f32" else torch.float64
    cases = [((1031, 2050), 11), ((37, 130), 12), ((1, 5), 13), ((1031, 2050), 11)]
    outs = torch.full((len(cases),), -1.0, dtype=torch.float64, device=dev)
    want_plan, want_oracle, keep = [], [], []
    for k, (shape, seed) in enumerate(cases):
        re, im = planes(shape, dtype, seed)
        dre, dim = torch.from_numpy(re).to(dev), torch.from_numpy(im).to(dev)
        keep.append((dre, dim))
        norm_static(dre, dim, outs[k:k + 1])              # no synchronisation in between
        want_oracle.append(oracle.norm2(re.astype(np.float64), im.astype(np.float64)))
    torch.cuda.synchronize()
    got = outs.cpu().numpy()
    for k, (shape, seed) in enumerate(cases):
        plan = Plan(shape[1], shape[0], tdt, "closed")
        want_plan.append(plan.norm(*keep[k]))
        plan.destroy()
    for k in range(len(cases)):
        assert abs(got[k] - want_plan[k]) <= REL * want_plan[k], (k, got[k], want_plan[k])
        assert abs(got[k] - want_oracle[k]) <= REL * want_oracle[k], (k, got[k], want_oracle[k])
    assert got[0] == got[3]


def test_allocates_nothing_and_works_at_C4_size():
    """16384^2 fp32 (2^28 sites, half the maximum): device memory in use does not change across
    the calls (the planes are allocated before the first measurement), result = ts_norm's."""
    import torch
    from paper_1208_2407_b200.binding import Plan, norm_static
    dev = torch.device("cuda:0")
    n = 16384
    g = torch.Generator(device=dev); g.manual_seed(5)
    re = torch.rand((n, n), device=dev, generator=g) - 0.5
    im = torch.rand((n, n), device=dev, generator=g) - 0.5
    out = torch.zeros(1, dtype=torch.float64, device=dev)
    norm_static(re[:4], im[:4], out)                       # set-up call (symbol address look-up)
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info(dev)
    for _ in range(2):
        norm_static(re, im, out)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info(dev)
    assert free1 == free0, (free0, free1)
    plan = Plan(n, n, torch.float32, "periodic")
    want = plan.norm(re, im)
    plan.destroy()
    assert abs(out.item() - want) <= REL * want, (out.item(), want)


def test_empty_input_and_rejections():
    import torch
    from paper_1208_2407_b200.binding import lib, last_error, norm_static
    dev = torch.device("cuda:0")
    re = torch.ones(8, device=dev); im = torch.ones(8, device=dev)
    out = torch.full((1,), 7.0, dtype=torch.float64, device=dev)
    vp = ctypes.c_void_p
    # zero sites: the sum is 0 (and the stale partials of earlier calls are not read)
    assert lib().ts_norm_static(0, vp(re.data_ptr()), vp(im.data_ptr()), 0, vp(out.data_ptr()), None) == 0
    torch.cuda.synchronize()
    assert out.item() == 0.0
    out.fill_(7.0)
    # beyond the maximum: refused before anything is enqueued, with the limit in the message
    rc = lib().ts_norm_static(0, vp(re.data_ptr()), vp(im.data_ptr()), MAX_SITES + 1,
                              vp(out.data_ptr()), None)
    assert rc == TS_EUNSUPPORTED and str(MAX_SITES) in last_error(), last_error()
    # host pointers, a NULL pointer, a bad dtype, a negative size
    host = np.ones(8, dtype=np.float32)
    hout = ctypes.c_double(0.0)
    assert lib().ts_norm_static(0, vp(host.ctypes.data), vp(im.data_ptr()), 8, vp(out.data_ptr()), None) == TS_EINVAL
    assert lib().ts_norm_static(0, vp(re.data_ptr()), vp(im.data_ptr()), 8,
                                ctypes.cast(ctypes.byref(hout), vp), None) == TS_EINVAL
    assert lib().ts_norm_static(0, None, vp(im.data_ptr()), 8, vp(out.data_ptr()), None) == TS_EINVAL
    assert lib().ts_norm_static(9, vp(re.data_ptr()), vp(im.data_ptr()), 8, vp(out.data_ptr()), None) == TS_EINVAL
    assert lib().ts_norm_static(0, vp(re.data_ptr()), vp(im.data_ptr()), -1, vp(out.data_ptr()), None) == TS_EINVAL
    torch.cuda.synchronize()
    assert out.item() == 7.0                                # none of the refused calls wrote
    with pytest.raises(ValueError):
        norm_static(re, im, torch.zeros(1, device=dev))     # out must be float64
    norm_static(re, im, out)
    torch.cuda.synchronize()
    assert out.item() == 16.0
