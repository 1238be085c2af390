"""Domain-decomposed time stepping on blocks (one block per GPU, one halo exchange of the
8 evolved fields of width 8 per Runge-Kutta stage, one all-reduce(max) of a_max per step).

Every numerical step runs in the CUDA library (echo_stage_sweeps / echo_stage_finish on a padded periodic
block, include/echo.h); this module only holds the plumbing around it: the decomposition, the halo refresh
(tensor slices, or torch.distributed send/recv between ranks) and the a_max all-reduce.

The halo refresh uses PACKED messages: per decomposed axis and side one buffer with the slabs of all fields
(echo_halo_pack / echo_halo_unpack, one kernel each), i.e. 2 sends + 2 receives per axis instead of 4 per field.
Two drivers share it:
  * LocalBlocks — all blocks in ONE process on one GPU, the packed buffers handed over as device tensors.  This is
    how the decomposed path is verified on a single GPU (bitwise against the undecomposed run) without running
    kernels that wait on one another.
  * RankBlock   — one block per process / GPU; messages by torch.distributed batch_isend_irecv (NCCL over NVLink on
    GPUs), a_max by all_reduce(MAX); the cell-field messages travel on a side stream under the UCT kernels.
exchange_packed is backend-agnostic (the CPU tests run it over gloo with the torch reference pack / unpack).
Tensors are (nz, ny, nx); axis d of the grid is tensor dim 2 - d.
"""
import math

HALO = 8          # dependency reach of one RK stage: MP5 +-3, DER +-2 (+1), INT +-3
STATE = tuple(range(0, 8))      # fields of U^n (D, Sx, Sy, Sz, U, Bx, By, Bz)
STAGE = tuple(range(8, 16))     # fields of the stage state


class Decomposition:
    """px x py x pz blocks of a periodic box of gn = (gnx, gny, gnz) cells; rank = ix + px*(iy + py*iz)."""

    def __init__(self, gn, p):
        self.gn, self.p = tuple(int(v) for v in gn), tuple(int(v) for v in p)
        for g, q in zip(self.gn, self.p):
            if q < 1 or g % q:
                raise ValueError("the blocks must tile the box evenly")
            if q > 1 and g // q < HALO:
                raise ValueError("a decomposed axis needs at least %d interior cells per block" % HALO)
        self.size = self.p[0] * self.p[1] * self.p[2]
        self.halo = tuple(HALO if q > 1 else 0 for q in self.p)
        self.interior = tuple(g // q for g, q in zip(self.gn, self.p))
        self.local = tuple(n + 2 * h for n, h in zip(self.interior, self.halo))     # padded block (nx, ny, nz)

    def coords(self, rank):
        return (rank % self.p[0], (rank // self.p[0]) % self.p[1], rank // (self.p[0] * self.p[1]))

    def rank_of(self, c):
        c = [v % q for v, q in zip(c, self.p)]
        return c[0] + self.p[0] * (c[1] + self.p[1] * c[2])

    def neighbour(self, rank, axis, step):
        c = list(self.coords(rank))
        c[axis] += step
        return self.rank_of(c)

    def global_index(self, rank, axis):
        """Global cell indices (periodically wrapped) of the padded block along `axis`."""
        c = self.coords(rank)[axis]
        start = c * self.interior[axis] - self.halo[axis]
        return [(start + i) % self.gn[axis] for i in range(self.local[axis])]

    def cut(self, rank, a):
        """The padded block of a global (gnz, gny, gnx) numpy array."""
        import numpy as np
        ix, iy, iz = (self.global_index(rank, d) for d in range(3))
        return np.ascontiguousarray(a[np.ix_(iz, iy, ix)])

    def interior_slices(self):
        return tuple(slice(h, h + n) for n, h in zip(self.interior[::-1], self.halo[::-1]))   # (z, y, x)


def slabs(t, axis, h=HALO):
    """Views (low_halo, low_interior, high_interior, high_halo) of tensor t along grid axis `axis`."""
    dim = 2 - axis
    n = t.shape[dim]
    return (t.narrow(dim, 0, h), t.narrow(dim, h, h), t.narrow(dim, n - 2 * h, h), t.narrow(dim, n - h, h))


# ---- packed halo messages: ONE buffer per axis and side with the slabs of all fields, [field][slab] ------------------
def pack_slabs(tensors, axis, side, buf, h=HALO):
    """Reference (torch) form of echo_halo_pack for tensors the library does not own (the CPU tests): gathers the
    interior slab next to `side` of every tensor (None = skipped, its part of buf is left alone) into buf."""
    per = buf.numel() // len(tensors)
    for v, t in enumerate(tensors):
        if t is not None:
            _, lo_int, hi_int, _ = slabs(t, axis, h)
            buf[v * per:(v + 1) * per].view((hi_int if side else lo_int).shape).copy_(hi_int if side else lo_int)


def unpack_slabs(tensors, axis, side, buf, h=HALO):
    """Reference form of echo_halo_unpack: scatters buf into the halo on `side` of every tensor that is not None."""
    per = buf.numel() // len(tensors)
    for v, t in enumerate(tensors):
        if t is not None:
            lo_halo, _, _, hi_halo = slabs(t, axis, h)
            dst = hi_halo if side else lo_halo
            dst.copy_(buf[v * per:(v + 1) * per].view(dst.shape))


def exchange_packed(decomp, rank, dist, bufs, pack, unpack, part=None, group=None):
    """One halo refresh with packed messages: per decomposed axis (x, then y, then z, so that edges and corners
    arrive through the later axes) pack the two interior slabs, exchange them with the two neighbours (2 sends +
    2 receives instead of 4 per field), unpack into the two halos.  bufs[axis] = (send_lo, send_hi, recv_lo,
    recv_hi), persistent 1-D tensors; pack(axis, side, buf) / unpack(axis, side, buf) move the slabs; part(axis), if
    given, is the slice of the buffers that is sent (the cell fields and the face fields of a stage travel separately);
    group: the process group (communicator) to send on."""
    for axis in range(3):
        if decomp.p[axis] == 1:
            continue
        lo, hi = decomp.neighbour(rank, axis, -1), decomp.neighbour(rank, axis, +1)
        send_lo, send_hi, recv_lo, recv_hi = bufs[axis]
        sl = part(axis) if part is not None else slice(None)
        pack(axis, 0, send_lo)
        pack(axis, 1, send_hi)
        # order matters when lo == hi (two blocks along the axis): the peer's first message is its low slab, which
        # belongs in our HIGH halo
        ops = [dist.P2POp(dist.isend, send_lo[sl], lo, group), dist.P2POp(dist.isend, send_hi[sl], hi, group),
               dist.P2POp(dist.irecv, recv_hi[sl], hi, group), dist.P2POp(dist.irecv, recv_lo[sl], lo, group)]
        for req in dist.batch_isend_irecv(ops):
            req.wait()          # NCCL: the current stream waits (no host block); gloo: the host waits
        unpack(axis, 0, recv_lo)
        unpack(axis, 1, recv_hi)


CELLS = slice(0, 5)     # the five cell fields of echo_stage_halo_fields: final when echo_stage_sweeps returns
FACES = slice(5, 8)     # the three face fields: final when echo_stage_finish returns


def _masked(fields, part):
    """The 8 field indices with those outside `part` replaced by -1 (skipped by echo_halo_pack / unpack)."""
    keep = set(range(8)[part])
    return [f if v in keep else -1 for v, f in enumerate(fields)]


class LocalBlocks:
    """All blocks of a decomposition in this process, on the current CUDA device."""

    def __init__(self, gn, p, gamma, cfl, ho=True, rec=5, rk=3):
        import torch
        from . import binding
        self.d = Decomposition(gn, p)
        blk = tuple(self.d.gn) + tuple(self.d.halo)
        self.blocks = [binding.Echo(*self.d.local, gamma, cfl, block=blk, ho=ho, rec=rec, rk=rk) for _ in range(self.d.size)]
        self.rk = rk
        b0 = self.blocks[0]
        self.bufs = [[tuple(torch.empty(b0.halo_doubles(ax), dtype=torch.float64, device=b0.device) for _ in range(2))
                      if self.d.p[ax] > 1 else None for ax in range(3)] for _ in self.blocks]

    def set_primitives(self, w, keys=("rho", "vx", "vy", "vz", "p", "bxf", "byf", "bzf")):
        """w: dict of GLOBAL (gnz, gny, gnx) numpy arrays."""
        import torch
        for r, b in enumerate(self.blocks):
            b.set_primitives(*[torch.as_tensor(self.d.cut(r, w[k]), device=b.device) for k in keys])

    def _allreduce_amax(self):
        import torch
        words = [b.ctrl_word(0) for b in self.blocks]
        m = torch.stack(words).max(dim=0).values       # bit patterns of non-negative doubles order like integers
        for wd in words:
            wd.copy_(m)

    def _refresh(self, fields):
        """The packed exchange with device buffers standing in for the messages (echo_halo_pack / echo_halo_unpack)."""
        d = self.d
        for axis in range(3):
            if d.p[axis] == 1:
                continue
            for r, b in enumerate(self.blocks):
                b.halo_pack(fields, axis, 0, self.bufs[r][axis][0])
                b.halo_pack(fields, axis, 1, self.bufs[r][axis][1])
            for r, b in enumerate(self.blocks):
                b.halo_unpack(fields, axis, 0, self.bufs[d.neighbour(r, axis, -1)][axis][1])    # their high interior
                b.halo_unpack(fields, axis, 1, self.bufs[d.neighbour(r, axis, +1)][axis][0])    # their low interior

    def step(self, nsteps, t_end=math.inf):
        for _ in range(int(nsteps)):
            for stage in range(1, self.rk + 1):
                for b in self.blocks:
                    b.stage_sweeps(stage, t_end)
                if stage == 1:
                    self._allreduce_amax()
                for b in self.blocks:
                    b.stage_finish(stage)
                self._refresh(self.blocks[0].stage_halo_fields(stage))

    def get_primitives(self):
        """Gathers the interiors into GLOBAL numpy arrays."""
        import numpy as np
        d = self.d
        names = ["rho", "vx", "vy", "vz", "p", "bx", "by", "bz", "bxf", "byf", "bzf"]
        out = {k: np.empty(d.gn[::-1]) for k in names}
        sl = d.interior_slices()
        for r, b in enumerate(self.blocks):
            q = b.get_primitives()
            c = d.coords(r)
            dst = tuple(slice(c[ax] * d.interior[ax], (c[ax] + 1) * d.interior[ax]) for ax in (2, 1, 0))
            for k in names:
                out[k][dst] = q[k][sl].cpu().numpy()
        return out

    def time(self):
        import torch
        return float(self.blocks[0].ctrl_word(1).view(torch.float64).item())


class RankBlock:
    """This process's block of a decomposition over torch.distributed (one rank per GPU).

    Per RK stage: sweeps -> [a_max all-reduce in stage 1] -> UCT + B update -> halo refresh.  The five cell fields
    the next stage needs are final once the sweeps are enqueued, so their packed messages (pack kernel, NCCL
    send/recv, unpack kernel) run on a SIDE stream while the main stream runs the UCT kernel and the B update (a third
    of a stage); only the three face fields are exchanged after them.  Nothing blocks the host: streams are ordered
    by events (wait_stream), NCCL requests by stream-side waits."""

    def __init__(self, gn, p, gamma, cfl, ho=True, rec=5, rk=3):
        import torch
        import torch.distributed as dist
        from . import binding
        self.dist = dist
        self.d = Decomposition(gn, p)
        if dist.get_world_size() != self.d.size:
            raise ValueError("world size %d != number of blocks %d" % (dist.get_world_size(), self.d.size))
        self.rank = dist.get_rank()
        self.rk = rk
        self.block = b = binding.Echo(*self.d.local, gamma, cfl, block=tuple(self.d.gn) + tuple(self.d.halo), ho=ho, rec=rec, rk=rk)
        self.bufs = [tuple(torch.empty(b.halo_doubles(ax), dtype=torch.float64, device=b.device) for _ in range(4))
                     if self.d.p[ax] > 1 else None for ax in range(3)]
        self.side = torch.cuda.Stream(device=b.device) if self.d.size > 1 else None
        # the messages of the side stream travel on their own communicator: NCCL operations of ONE communicator must not
        # run concurrently from two streams (the a_max all-reduce and the face messages use the default group)
        self.side_group = dist.new_group() if self.d.size > 1 else None

    def set_primitives(self, w, keys=("rho", "vx", "vy", "vz", "p", "bxf", "byf", "bzf")):
        import torch
        self.block.set_primitives(*[torch.as_tensor(self.d.cut(self.rank, w[k]), device=self.block.device)
                                    for k in keys])

    def _exchange(self, fields, part, stream, group=None):
        b = self.block
        f = _masked(fields, part)
        sp = stream.cuda_stream if stream is not None else None
        exchange_packed(self.d, self.rank, self.dist, self.bufs,
                        lambda ax, side, buf: b.halo_pack(f, ax, side, buf, sp),
                        lambda ax, side, buf: b.halo_unpack(f, ax, side, buf, sp),
                        part=lambda ax: slice(part.start * (b.halo_doubles(ax) // 8), part.stop * (b.halo_doubles(ax) // 8)),
                        group=group)

    def step(self, nsteps, t_end=math.inf):
        import torch
        b, dist = self.block, self.dist
        main = torch.cuda.current_stream(b.device)
        for _ in range(int(nsteps)):
            for stage in range(1, self.rk + 1):
                b.stage_sweeps(stage, t_end)
                fields = b.stage_halo_fields(stage)
                if self.side is not None:                    # cell fields: exchanged under the UCT kernels
                    self.side.wait_stream(main)
                    with torch.cuda.stream(self.side):
                        self._exchange(fields, CELLS, self.side, self.side_group)
                if stage == 1:
                    dist.all_reduce(b.ctrl_word(0), op=dist.ReduceOp.MAX)
                b.stage_finish(stage)
                if self.side is not None:
                    self._exchange(fields, FACES, None)      # face fields: after the B update, on the main stream
                    main.wait_stream(self.side)

    def get_interior(self):
        q = self.block.get_primitives()
        sl = self.d.interior_slices()
        return {k: v[sl] for k, v in q.items()}
