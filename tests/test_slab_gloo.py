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


# ---- PeerRank (the fused-halo path, one process per GPU) sequenced on CPU ---------------------------
# The symmetric-memory handle is replaced by file-backed shared tensors (get_buffer = the peer's
# file mapped into this process, barrier = a gloo barrier) and ts_slab_pass by the oracle on
# [neighbour rows | own rows | neighbour rows]: what is tested is PeerRank.run itself -- which
# buffer of which neighbour a pass reads, the flip, one barrier per pass -- so that the only part
# left untested without two GPUs is the CUDA peer mapping.
class _FileMemory:
    def __init__(self, tmpdir, rank, group=None):
        self.tmpdir, self.rank, self.barriers = tmpdir, rank, 0

    def _open(self, rank, shape, dtype):
        n = int(np.prod(shape))
        return torch.from_file(f"{self.tmpdir}/buf{rank}.bin", shared=True, size=n, dtype=dtype).view(shape)

    def alloc(self, shape, dtype, device):
        return self._open(self.rank, shape, dtype)

    def rendezvous(self, buf, group):
        dist.barrier(group)                       # every rank's file exists and is zeroed
        return self

    def get_buffer(self, rank, shape, dtype, offset):
        assert offset == 0
        return self._open(rank, shape, dtype)

    def barrier(self, channel=0):
        self.barriers += 1
        dist.barrier()


def _oracle_pass(slab_, src, dst, up_src, dn_src, subs):
    import oracle
    h = 2 * len(subs)
    parts_re, parts_im = [], []
    if up_src is not None:
        parts_re.append(up_src[0][-h:].numpy()); parts_im.append(up_src[1][-h:].numpy())
    parts_re.append(src[0].numpy()); parts_im.append(src[1].numpy())
    if dn_src is not None:
        parts_re.append(dn_src[0][:h].numpy()); parts_im.append(dn_src[1][:h].numpy())
    re = np.ascontiguousarray(np.concatenate(parts_re)); im = np.ascontiguousarray(np.concatenate(parts_im))
    for c in subs:
        oracle.evolve_xy(re, im, *c, pot=None, periodic_x=slab_.boundary == "periodic",
                         periodic_y=False, n_steps=1)
    o = h if up_src is not None else 0
    dst[0].copy_(torch.from_numpy(re[o:o + slab_.own])); dst[1].copy_(torch.from_numpy(im[o:o + slab_.own]))


def _peer_worker(rank, world, port, boundary, u4, tmpdir, q):
    sys.path.insert(0, str(ROOT)); sys.path.insert(0, str(ROOT / "tests"))
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    torch.set_num_threads(1)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        import oracle
        from paper_1208_2407_b200 import slab
        from slab_util import oracle_norm_fn, problem
        oracle.set_num_threads(1)
        nx, ny, theta, n_steps = 16, 48, 0.3, 5
        re, im, _ = problem(nx, ny, 11, False)
        mem = _FileMemory(tmpdir, rank)
        pr = slab.PeerRank(nx, ny, torch.float64, boundary, memory=mem, device=torch.device("cpu"),
                           pass_fn=_oracle_pass, norm_fn=oracle_norm_fn)
        s = pr.slab
        s.set_state(torch.from_numpy(re[s.r0:s.r1]), torch.from_numpy(im[s.r0:s.r1]))
        n0 = pr.norm()
        if u4:
            pr.evolve_u4(theta, n_steps)
            n_sub = 5 * n_steps
        else:
            c = (math.cos(theta / 2), math.sin(theta / 2), math.cos(theta), math.sin(theta))
            pr.evolve(c, n_steps)
            n_sub = n_steps
        n1 = pr.norm()
        n_pass = -(-n_sub // pr.S)
        assert mem.barriers == n_pass + 1, (mem.barriers, n_pass)
        own = torch.stack(list(s.planes(s.cur))).contiguous()
        parts = [None] * world
        dist.all_gather_object(parts, (s.r0, s.r1, own.numpy()))
        if rank == 0:
            out_re = np.empty((ny, nx)); out_im = np.empty((ny, nx))
            for r0, r1, a in parts:
                out_re[r0:r1], out_im[r0:r1] = a[0], a[1]
            wre, wim = re.copy(), im.copy()
            if u4:
                oracle.evolve_u4(wre, wim, theta, periodic=boundary == "periodic", n_steps=n_steps)
            else:
                oracle.evolve(wre, wim, *c, periodic=boundary == "periodic", n_steps=n_steps)
            err = max(np.abs(out_re - wre).max(), np.abs(out_im - wim).max())
            q.put((err, n0, n1, pr.S))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world,boundary,u4", [(2, "periodic", False), (2, "closed", True),
                                               (3, "periodic", True), (3, "closed", False)])
def test_peer_rank_pass_flip_barrier_sequencing(world, boundary, u4, tmp_path):
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_peer_worker, args=(r, world, port, boundary, u4, str(tmp_path), q))
             for r in range(world)]
    for p in procs:
        p.start()
    for p in procs:
        p.join(180)
        assert p.exitcode == 0
    err, n0, n1, S = q.get(timeout=10)
    assert S == 4                                  # fp64: passes of up to four sub-steps
    assert err < 1e-13, err
    assert abs(n1 / n0 - 1) < 1e-13
