"""The N > 1 path over torch.distributed: two (and three) processes, gloo backend, CPU tensors.
Each rank owns a Slab, exchanges halos with DistComm (the same code that runs over NCCL on GPUs)
and evolves its local planes with the oracle standing in for ts_evolve; rank 0 gathers the slabs
and compares them with the undivided oracle."""
from __future__ import annotations

import math
import os
import socket
import sys
from pathlib import Path

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = Path(__file__).resolve().parents[1]


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, boundary, with_pot, k, n_steps, q):
    sys.path.insert(0, str(ROOT)); sys.path.insert(0, str(ROOT / "tests"))
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    torch.set_num_threads(1)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        import oracle
        from paper_1208_2407_b200 import slab
        from slab_util import oracle_evolve_fn, oracle_norm_fn, problem
        oracle.set_num_threads(1)
        nx, ny, theta = 16, 36, 0.3
        c = (math.cos(theta / 2), math.sin(theta / 2), math.cos(theta), math.sin(theta))
        re, im, pot = problem(nx, ny, 7, with_pot)          # every rank builds the same global data
        comm = slab.DistComm()
        s = slab.Slab(nx, ny, torch.float64, boundary, rank, world, k,
                      evolve_fn=oracle_evolve_fn, norm_fn=oracle_norm_fn)
        s.set_state(torch.from_numpy(re[s.r0:s.r1]), torch.from_numpy(im[s.r0:s.r1]))
        if pot is not None:
            s.set_potential(torch.from_numpy(pot[:, s.r0:s.r1]), comm)
        n0 = s.norm(comm)
        s.evolve(c, n_steps, comm)
        n1 = s.norm(comm)
        own = torch.stack([s.own_rows(s.re), s.own_rows(s.im)]).contiguous()
        parts = [None] * world
        dist.all_gather_object(parts, (s.r0, s.r1, own.numpy()))
        if rank == 0:
            out_re = np.empty((ny, nx)); out_im = np.empty((ny, nx))
            for r0, r1, a in parts:
                out_re[r0:r1], out_im[r0:r1] = a[0], a[1]
            wre, wim = re.copy(), im.copy()
            oracle.evolve(wre, wim, *c, pot=None if pot is None else (pot[0], pot[1]),
                          periodic=boundary == "periodic", n_steps=n_steps)
            err = max(np.abs(out_re - wre).max(), np.abs(out_im - wim).max())
            q.put((err, n0, n1, oracle.norm2(re, im)))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world,boundary,with_pot", [(2, "periodic", False), (2, "closed", True),
                                                     (3, "periodic", True), (3, "closed", False)])
def test_two_process_halo_exchange_matches_undivided_oracle(world, boundary, with_pot):
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, boundary, with_pot, 2, 7, q))
             for r in range(world)]
    for p in procs:
        p.start()
    for p in procs:
        p.join(120)
        assert p.exitcode == 0
    err, n0, n1, want = q.get(timeout=10)
    assert err < 1e-14
    assert abs(n0 / want - 1) < 1e-13 and abs(n1 / n0 - 1) < 1e-13
