"""Row-slab domain decomposition of ONE lattice over several GPUs.

The paper's subject is the distributed solver: every process owns a tile of the lattice plus a
halo, evolves it, and exchanges halos with its neighbours.  On B200/NVSwitch
the natural cut is 1-D: rows are contiguous in memory, so a rank owns a slab of rows and a halo is
one contiguous block of rows per neighbour and plane -- no packing, no 2-D corner wave.

    local planes  [ halo_top | own rows | halo_bottom ]      (H = 2 * steps_per_exchange rows each)

Per exchange period of k steps: the ranks swap their outermost H own rows into the neighbours'
halos (torch.distributed point-to-point: NCCL over NVLink on GPUs, gloo on CPU tensors), then every
rank calls ts_evolve for k steps on its extended slab, planned as a lattice that keeps the global
boundary in x and is CLOSED in y (ts_plan_create_xy).  The closed cut is wrong physics, but the
error travels 2 rows per step (cuts are on even rows), i.e. it stays inside the halo, which the
next exchange overwrites.  At a real closed edge of the global lattice there is no halo and the
local closed edge IS the lattice edge.  k defaults to two fused passes (2 S steps), so the result
of ts_evolve lands back in the caller's planes without the odd-pass copy.

Everything numerical happens in ts_evolve / ts_norm; this file is partition arithmetic, views and
send/recv -- argument marshalling for N ranks.  `evolve_fn` / `norm_fn` exist so that the host
logic can be tested on CPU tensors with world_size 2 over gloo (tests/test_slab_gloo.py).
"""
from __future__ import annotations

from dataclasses import dataclass


def partition_rows(ny: int, world: int):
    """Even-aligned row ranges [(r0, r1)] * world covering [0, ny): cuts must fall on even rows so
    that local pair parity equals global pair parity."""
    if ny % 2:
        raise ValueError("slab decomposition needs an even number of rows")
    pairs = ny // 2
    if world < 1 or pairs < world:
        raise ValueError("more ranks than row pairs")
    cuts = [2 * ((pairs * k) // world) for k in range(world + 1)]
    return [(cuts[k], cuts[k + 1]) for k in range(world)]


@dataclass
class Neighbours:
    up: int | None      # rank owning the rows above mine (smaller y), None at a closed top edge
    down: int | None    # rank owning the rows below mine


def neighbours(rank: int, world: int, periodic_y: bool) -> Neighbours:
    if world == 1:
        return Neighbours(None, None)
    if periodic_y:
        return Neighbours((rank - 1) % world, (rank + 1) % world)
    return Neighbours(rank - 1 if rank > 0 else None, rank + 1 if rank < world - 1 else None)


def default_steps_per_exchange(dtype, with_pot: bool) -> int:
    """Two fused passes of the stream kernel's default depth (csrc/ts_fused.cu::
    fused_default_steps), so that every local ts_evolve ends in the caller's planes."""
    import torch
    if dtype == torch.float32:
        return 6 if with_pot else 12
    return 6 if with_pot else 8


class DistComm:
    """Halo exchange over torch.distributed (NCCL for CUDA tensors, gloo for CPU tensors)."""

    def __init__(self, group=None):
        import torch.distributed as dist
        self.dist = dist
        self.group = group
        self.rank = dist.get_rank(group)
        self.world = dist.get_world_size(group)

    def exchange(self, nb: Neighbours, send_up, send_down, recv_up, recv_down):
        """send_up -> nb.up's bottom halo, send_down -> nb.down's top halo; fills recv_*.
        Each argument is a list of contiguous tensors (one per plane) or None."""
        dist = self.dist
        ops = []
        # NCCL matches the messages of a pair of ranks by order, not by tag, and with two ranks
        # on a periodic lattice the up and the down neighbour are the same peer.  So every rank
        # posts the UPWARD traffic first (my top rows -> the bottom halo of the rank above; what
        # the rank below sends me lands in my bottom halo), then the DOWNWARD traffic.
        if nb.up is not None:
            for t in send_up:
                ops.append(dist.P2POp(dist.isend, t, nb.up, self.group))
        if nb.down is not None:
            for t in recv_down:
                ops.append(dist.P2POp(dist.irecv, t, nb.down, self.group))
            for t in send_down:
                ops.append(dist.P2POp(dist.isend, t, nb.down, self.group))
        if nb.up is not None:
            for t in recv_up:
                ops.append(dist.P2POp(dist.irecv, t, nb.up, self.group))
        if ops:
            for w in dist.batch_isend_irecv(ops):
                w.wait()

    def all_reduce_sum(self, value: float) -> float:
        import torch
        t = torch.tensor([value], dtype=torch.float64)
        if self.dist.get_backend(self.group) == "nccl":
            t = t.cuda()
        self.dist.all_reduce(t, group=self.group)
        return float(t.item())


class LocalComm:
    """All ranks inside one process (one GPU, or CPU tensors): the exchange is a set of copies.

    Used to run the slab path on a single device, where ranks must not wait on one another:
    `LocalGroup` steps its virtual ranks one after the other and exchanges between the steps.
    """

    def __init__(self, world: int):
        self.world = world

    @staticmethod
    def copy(dst_list, src_list):
        for d, s in zip(dst_list, src_list):
            d.copy_(s)


class Slab:
    """One rank's share of an nx x ny lattice: own rows [r0, r1) plus halo rows, and the plan that
    evolves them.  boundary = "closed" | "periodic" is the GLOBAL boundary (both axes).

    steps_per_exchange = k: halos are H = 2k rows and are refreshed every k steps.
    evolve_fn(re, im, coeffs, pot, n_steps, periodic_x, periodic_y) / norm_fn(re, im): replace
    ts_evolve / ts_norm on the
    local planes (host-logic tests on CPU tensors); by default a binding.Plan is used and the planes
    live on `device`.
    """

    def __init__(self, nx, ny, dtype, boundary, rank, world, steps_per_exchange=8, device=None,
                 evolve_fn=None, norm_fn=None):
        import torch
        if boundary not in ("closed", "periodic"):
            raise ValueError("boundary must be 'closed' or 'periodic'")
        self.nx, self.ny, self.dtype, self.boundary = int(nx), int(ny), dtype, boundary
        self.rank, self.world = int(rank), int(world)
        self.k = int(steps_per_exchange)
        if self.k < 1:
            raise ValueError("steps_per_exchange must be >= 1")
        self.r0, self.r1 = partition_rows(self.ny, self.world)[self.rank]
        self.own = self.r1 - self.r0
        self.nb = neighbours(self.rank, self.world, boundary == "periodic")
        self.H = 2 * self.k if self.world > 1 else 0
        sizes = [b - a for a, b in partition_rows(self.ny, self.world)]
        if self.world > 1 and min(sizes) < self.H:
            raise ValueError(f"slabs of {min(sizes)} rows are shorter than the halo of {self.H} "
                             "rows: lower steps_per_exchange or use fewer ranks")
        self.h_top = self.H if self.nb.up is not None else 0
        self.h_bot = self.H if self.nb.down is not None else 0
        self.ny_local = self.h_top + self.own + self.h_bot
        self.device = device if device is not None else torch.device("cpu")
        self.re = torch.zeros((self.ny_local, self.nx), dtype=dtype, device=self.device)
        self.im = torch.zeros((self.ny_local, self.nx), dtype=dtype, device=self.device)
        self.pot = None
        self._evolve_fn, self._norm_fn = evolve_fn, norm_fn
        self.plan = self.norm_plan = None
        if evolve_fn is None:
            from .binding import Plan
            # the slab keeps the global boundary in x; in y it is closed (cut or real edge)
            by = boundary if self.world == 1 else "closed"
            self.plan = Plan(self.nx, self.ny_local, dtype, boundary, by)
            self.norm_plan = Plan(self.nx, self.own, dtype, "closed")

    # ---- views ----------------------------------------------------------------------------------
    def own_rows(self, t):
        """The rows of a local plane [ny_local][nx] (or [2][ny_local][nx]) that this rank owns."""
        return t[..., self.h_top:self.h_top + self.own, :]

    def _halo_views(self, planes):
        o0, o1 = self.h_top, self.h_top + self.own
        H = self.H
        send_up = [p[o0:o0 + H] for p in planes] if self.nb.up is not None else None
        send_down = [p[o1 - H:o1] for p in planes] if self.nb.down is not None else None
        recv_up = [p[0:o0] for p in planes] if self.nb.up is not None else None
        recv_down = [p[o1:] for p in planes] if self.nb.down is not None else None
        return send_up, send_down, recv_up, recv_down

    def set_state(self, re_own, im_own):
        self.own_rows(self.re).copy_(re_own)
        self.own_rows(self.im).copy_(im_own)

    def set_potential(self, pot_own, comm):
        """pot_own: [2][own][nx] phase planes of the own rows; the halo rows are fetched once."""
        import torch
        self.pot = torch.zeros((2, self.ny_local, self.nx), dtype=self.dtype, device=self.device)
        self.own_rows(self.pot).copy_(pot_own)
        if self.world > 1 and comm is not None:
            comm.exchange(self.nb, *self._halo_views([self.pot[0], self.pot[1]]))

    # ---- the path --------------------------------------------------------------------------------
    def exchange(self, comm):
        if self.world > 1:
            comm.exchange(self.nb, *self._halo_views([self.re, self.im]))

    def evolve_local(self, coeffs, n_steps, stream=None):
        if self._evolve_fn is not None:
            per = self.boundary == "periodic"
            self._evolve_fn(self.re, self.im, coeffs, self.pot, n_steps, per,
                            per and self.world == 1)
        else:
            self.plan.evolve(self.re, self.im, *coeffs, pot_phase=self.pot, n_steps=n_steps,
                             stream=stream)

    def evolve(self, coeffs, n_steps, comm):
        """n_steps second-order steps of the GLOBAL lattice (collective over the group)."""
        left = int(n_steps)
        while left > 0:
            k = min(self.k, left)
            self.exchange(comm)
            self.evolve_local(coeffs, k)
            left -= k

    def norm_local(self) -> float:
        re, im = self.own_rows(self.re), self.own_rows(self.im)
        if self._norm_fn is not None:
            return float(self._norm_fn(re, im))
        return self.norm_plan.norm(re, im)

    def norm(self, comm) -> float:
        v = self.norm_local()
        return comm.all_reduce_sum(v) if self.world > 1 else v

    def destroy(self):
        for p in (self.plan, self.norm_plan):
            if p is not None:
                p.destroy()


class LocalGroup:
    """All ranks of a decomposition inside one process, stepped one after the other, with the
    halo exchange done by copies: the slab path on ONE device (tests, and lattices that are cut
    only to bound the scratch memory)."""

    def __init__(self, nx, ny, dtype, boundary, world, steps_per_exchange=8, device=None,
                 evolve_fn=None, norm_fn=None):
        self.slabs = [Slab(nx, ny, dtype, boundary, r, world, steps_per_exchange, device,
                           evolve_fn, norm_fn) for r in range(world)]
        self.world = world

    def _exchange(self, planes_of):
        for s in self.slabs:
            su, sd, ru, rd = s._halo_views(planes_of(s))
            if s.nb.up is not None:       # my top rows -> bottom halo of the rank above
                up = self.slabs[s.nb.up]
                LocalComm.copy(up._halo_views(planes_of(up))[3], su)
            if s.nb.down is not None:     # my bottom rows -> top halo of the rank below
                dn = self.slabs[s.nb.down]
                LocalComm.copy(dn._halo_views(planes_of(dn))[2], sd)

    def scatter(self, re, im, pot=None):
        for s in self.slabs:
            s.set_state(re[s.r0:s.r1], im[s.r0:s.r1])
            if pot is not None:
                s.set_potential(pot[:, s.r0:s.r1], None)
        if pot is not None and self.world > 1:
            self._exchange(lambda s: [s.pot[0], s.pot[1]])

    def gather(self, re, im):
        for s in self.slabs:
            re[s.r0:s.r1].copy_(s.own_rows(s.re))
            im[s.r0:s.r1].copy_(s.own_rows(s.im))

    def evolve(self, coeffs, n_steps):
        left = int(n_steps)
        k0 = self.slabs[0].k
        while left > 0:
            k = min(k0, left)
            if self.world > 1:
                self._exchange(lambda s: [s.re, s.im])
            for s in self.slabs:
                s.evolve_local(coeffs, k)
            left -= k

    def norm(self) -> float:
        return sum(s.norm_local() for s in self.slabs)

    def destroy(self):
        for s in self.slabs:
            s.destroy()


# ---- fused halo path: ts_slab_pass reads the neighbours' boundary rows in place ------------------
def max_fused_steps(dtype, with_pot: bool = False) -> int:
    """Deepest pass ts_slab_pass takes (csrc/ts_stream.cu::stream_max_steps)."""
    import torch
    return 6 if (dtype == torch.float32 and not with_pot) else 4


def u4_pattern(theta):
    """The five sub-steps of the fourth-order step, Eq. 4: the library's table
    (ts_u4_coefficients) -- the binding holds none of the method's arithmetic."""
    from .binding import u4_coefficients
    return u4_coefficients(theta)


def _passes(pattern, n_repeat, depth):
    """Cut n_repeat repetitions of a sub-step pattern into passes of at most `depth` sub-steps."""
    total = len(pattern) * int(n_repeat)
    i = 0
    while i < total:
        k = min(depth, total - i)
        yield [pattern[(i + j) % len(pattern)] for j in range(k)]
        i += k


class PeerSlab:
    """One rank's slab for the fused path: its own rows only, in two buffers that ping-pong; there
    is NO halo storage and no exchange step -- `ts_slab_pass` fetches the rows beyond the slab
    straight from the neighbours' source buffers (same GPU here, a peer GPU's mapped memory in
    `PeerRank`).  buffers: optional [2][2][rows >= own][nx] tensor to live in (symmetric memory)."""

    def __init__(self, nx, ny, dtype, boundary, rank, world, device, buffers=None, pass_fn=None,
                 norm_fn=None):
        import torch
        self.nx, self.ny, self.dtype, self.boundary = int(nx), int(ny), dtype, boundary
        self.rank, self.world = int(rank), int(world)
        self.r0, self.r1 = partition_rows(self.ny, self.world)[self.rank]
        self.own = self.r1 - self.r0
        # on a periodic lattice every rank has both neighbours -- a single rank is its own
        per = boundary == "periodic"
        self.nb = Neighbours((rank - 1) % world, (rank + 1) % world) if per else \
            neighbours(self.rank, self.world, False)
        if buffers is None:
            buffers = torch.zeros((2, 2, self.own, self.nx), dtype=dtype, device=device)
        self.buffers = buffers
        self.cur = 0
        self.sep = None
        # pass_fn / norm_fn stand in for ts_slab_pass / ts_norm in the CPU tests of the sequencing
        self.pass_fn, self.norm_fn = pass_fn, norm_fn
        self.plan = None
        if pass_fn is None:
            from .binding import Plan
            self.plan = Plan(self.nx, self.own, dtype, boundary, "closed")
        self.norm_plan = self.plan

    def planes(self, which):
        """(re, im) views of buffer `which` restricted to the own rows."""
        b = self.buffers[which]
        return b[0, :self.own], b[1, :self.own]

    def set_state(self, re_own, im_own):
        re, im = self.planes(self.cur)
        re.copy_(re_own); im.copy_(im_own)

    def set_separable_potential(self, phase_x, phase_y):
        """phase_x [2][nx], phase_y [2][ny] over the GLOBAL lattice (every rank holds both)."""
        self.sep = (phase_x, phase_y)

    def launch_pass(self, up_src, dn_src, subs, stream=None):
        """dst <- U2(subs[-1]) ... U2(subs[0]) src with the neighbours' CURRENT planes as halos;
        does not flip."""
        px, py = self.sep if self.sep is not None else (None, None)
        if self.pass_fn is not None:
            self.pass_fn(self, self.planes(self.cur), self.planes(1 - self.cur), up_src, dn_src, subs)
            return
        self.plan.slab_pass(self.planes(self.cur), self.planes(1 - self.cur), up_src, dn_src,
                            subs, px, py, self.r0, self.ny, self.boundary == "periodic",
                            stream=stream)

    def flip(self):
        self.cur = 1 - self.cur

    def norm_local(self) -> float:
        re, im = self.planes(self.cur)
        if self.norm_fn is not None:
            return self.norm_fn(re, im)
        return self.plan.norm(re, im)

    def destroy(self):
        if self.plan is not None:
            self.plan.destroy()


class SymmetricMemory:
    """Where PeerRank's buffers live: torch.distributed._symmetric_memory (CUDA, one process per
    GPU).  alloc -> a tensor every peer can map; rendezvous -> a handle with get_buffer(rank, shape,
    dtype, offset) and barrier(channel).  The CPU tests pass a stand-in with the same two calls."""

    def alloc(self, shape, dtype, device):
        import torch.distributed._symmetric_memory as symm
        return symm.empty(shape, dtype=dtype, device=device)

    def rendezvous(self, buf, group):
        import torch.distributed._symmetric_memory as symm
        return symm.rendezvous(buf, group)


class PeerGroup:
    """All ranks of the fused path in one process on one device.  One stream orders the passes:
    every slab's pass k reads only buffers written by pass k-1, so launching the slabs one after
    the other and flipping all of them afterwards is the barrier."""

    def __init__(self, nx, ny, dtype, boundary, world, device):
        self.slabs = [PeerSlab(nx, ny, dtype, boundary, r, world, device) for r in range(world)]
        self.dtype = dtype
        self.smallest = min(s.own for s in self.slabs)
        if self.smallest < 2:
            raise ValueError("slabs need at least one row pair")
        self.S = self._depth(False)

    def _depth(self, with_pot):
        # a pass consumes 2 rows per sub-step from each neighbour
        return max(1, min(max_fused_steps(self.dtype, with_pot), self.smallest // 2))

    def scatter(self, re, im, phase_x=None, phase_y=None):
        for s in self.slabs:
            s.set_state(re[s.r0:s.r1], im[s.r0:s.r1])
            if phase_x is not None:
                s.set_separable_potential(phase_x, phase_y)
        self.S = self._depth(phase_x is not None)

    def gather(self, re, im):
        for s in self.slabs:
            r, i = s.planes(s.cur)
            re[s.r0:s.r1].copy_(r); im[s.r0:s.r1].copy_(i)

    def run(self, pattern, n_repeat):
        """n_repeat repetitions of a list of sub-step coefficient tuples."""
        for subs in _passes(pattern, n_repeat, self.S):
            for s in self.slabs:
                up = self.slabs[s.nb.up].planes(self.slabs[s.nb.up].cur) if s.nb.up is not None \
                    else None
                dn = self.slabs[s.nb.down].planes(self.slabs[s.nb.down].cur) \
                    if s.nb.down is not None else None
                s.launch_pass(up, dn, subs)
            for s in self.slabs:
                s.flip()

    def evolve(self, coeffs, n_steps):
        self.run([tuple(coeffs)], n_steps)

    def evolve_u4(self, theta, n_steps):
        self.run(u4_pattern(theta), n_steps)

    def norm(self) -> float:
        return sum(s.norm_local() for s in self.slabs)

    def destroy(self):
        for s in self.slabs:
            s.destroy()


class PeerRank:
    """The fused path with one process per GPU: the two buffers of every rank live in symmetric
    memory (torch.distributed._symmetric_memory), so each rank holds mapped views of its
    neighbours' buffers and `ts_slab_pass` reads their boundary rows over NVLink inside the
    kernel's own bulk copies.  Between passes: one device-side barrier over the group
    (`handle.barrier`), which orders "everybody finished writing pass k" before "anybody reads
    pass k".  NOT RUN on hardware in this round (needs >= 2 GPUs); the single-process twin
    `PeerGroup` runs the identical kernel path with neighbours on the same device."""

    def __init__(self, nx, ny, dtype, boundary, group=None, memory=None, device=None, pass_fn=None,
                 norm_fn=None):
        import torch
        import torch.distributed as dist
        self.group = group if group is not None else dist.group.WORLD
        rank, world = dist.get_rank(self.group), dist.get_world_size(self.group)
        dev = device if device is not None else torch.device("cuda", torch.cuda.current_device())
        memory = memory if memory is not None else SymmetricMemory()
        rows = max(b - a for a, b in partition_rows(ny, world))      # same shape on every rank
        self.shape = (2, 2, rows, int(nx))
        buf = memory.alloc(self.shape, dtype, dev)
        buf.zero_()
        self.handle = memory.rendezvous(buf, self.group)
        self.slab = PeerSlab(nx, ny, dtype, boundary, rank, world, dev, buffers=buf, pass_fn=pass_fn,
                             norm_fn=norm_fn)
        parts = partition_rows(ny, world)
        self.peer_own = [b - a for a, b in parts]
        self.peer_buf = {}
        for r in {self.slab.nb.up, self.slab.nb.down} - {None}:
            self.peer_buf[r] = buf if r == rank else \
                self.handle.get_buffer(r, self.shape, dtype, 0)
        self.dtype = dtype
        self.S = max(1, min(max_fused_steps(dtype), min(self.peer_own) // 2))
        self.comm = DistComm(self.group)

    def set_separable_potential(self, phase_x, phase_y):
        self.slab.set_separable_potential(phase_x, phase_y)
        self.S = max(1, min(max_fused_steps(self.dtype, True), min(self.peer_own) // 2))

    def _peer_planes(self, r, which):
        if r is None:
            return None
        b = self.peer_buf[r][which]
        n = self.peer_own[r]
        return b[0, :n], b[1, :n]

    def run(self, pattern, n_repeat, stream=None):
        """One barrier per pass: it orders "every rank has written pass k-1" before "anybody reads
        it" (RAW) and, because a rank reaches barrier k+1 only after its own pass k, also "every
        neighbour has read my pass k-1 source" before pass k+1 overwrites it (WAR).  The barrier
        and the pass must be enqueued on the SAME stream (torch's current one by default)."""
        import torch
        s = self.slab
        if stream is not None and s.plan is not None:
            assert stream.cuda_stream == torch.cuda.current_stream().cuda_stream, \
                "PeerRank: handle.barrier runs on the current stream; launch the passes there too"
        for subs in _passes(pattern, n_repeat, self.S):
            self.handle.barrier(channel=0)          # every rank's previous pass is complete
            s.launch_pass(self._peer_planes(s.nb.up, s.cur), self._peer_planes(s.nb.down, s.cur),
                          subs, stream=stream)
            s.flip()                                # all ranks flip in step: same parity everywhere
        self.handle.barrier(channel=0)

    def evolve(self, coeffs, n_steps):
        self.run([tuple(coeffs)], n_steps)

    def evolve_u4(self, theta, n_steps):
        self.run(u4_pattern(theta), n_steps)

    def norm(self) -> float:
        return self.comm.all_reduce_sum(self.slab.norm_local())
