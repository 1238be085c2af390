"""Domain-decomposed time stepping on blocks (one block per GPU, one halo exchange of the
8 evolved fields of width 8 per Runge-Kutta stage, one all-reduce(max) of a_max per step).

Every numerical step runs in the CUDA library (echo_stage_sweeps / echo_stage_finish on a padded periodic
block, include/echo.h); this module only holds the plumbing around it: the decomposition, the halo refresh
(tensor slices, or torch.distributed send/recv between ranks) and the a_max all-reduce.

Two drivers share the slab logic:
  * LocalBlocks — all blocks in ONE process on one GPU, halos refreshed by device copies.  This is how the
    decomposed path is verified on a single GPU (bitwise against the undecomposed run) without running kernels
    that wait on one another.
  * RankBlock   — one block per process / GPU; halos by torch.distributed batch_isend_irecv (NCCL over NVLink on
    GPUs, gloo in the CPU tests), a_max by all_reduce(MAX).
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


def _step_loop(blocks, nsteps, t_end, allreduce_amax, refresh):
    for _ in range(int(nsteps)):
        for stage in (1, 2, 3):
            for b in blocks:
                b.stage_sweeps(stage, t_end)
            if stage == 1:
                allreduce_amax()
            for b in blocks:
                b.stage_finish(stage)
            refresh(STAGE if stage < 3 else STATE)


class LocalBlocks:
    """All blocks of a decomposition in this process, on the current CUDA device."""

    def __init__(self, gn, p, gamma, cfl):
        from . import binding
        self.d = Decomposition(gn, p)
        blk = tuple(self.d.gn) + tuple(self.d.halo)
        self.blocks = [binding.Echo(*self.d.local, gamma, cfl, block=blk) for _ in range(self.d.size)]

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
        d = self.d
        for axis in range(3):
            if d.p[axis] == 1:
                continue
            for f in fields:
                views = [b.field(f) for b in self.blocks]
                for r in range(d.size):
                    lo_halo, _, _, hi_halo = slabs(views[r], axis)
                    _, _, src_hi_int, _ = slabs(views[d.neighbour(r, axis, -1)], axis)
                    _, src_lo_int, _, _ = slabs(views[d.neighbour(r, axis, +1)], axis)
                    lo_halo.copy_(src_hi_int)
                    hi_halo.copy_(src_lo_int)

    def step(self, nsteps, t_end=math.inf):
        _step_loop(self.blocks, nsteps, t_end, self._allreduce_amax, self._refresh)

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


def exchange_halos(tensors, decomp, rank, dist, h=HALO):
    """Refreshes the halos of this rank's tensors from its neighbours with torch.distributed point-to-point
    operations, axis by axis (so that edges and corners arrive through the later axes).  Works on CUDA tensors
    with NCCL and on CPU tensors with gloo."""
    for axis in range(3):
        if decomp.p[axis] == 1:
            continue
        lo, hi = decomp.neighbour(rank, axis, -1), decomp.neighbour(rank, axis, +1)
        ops, pending = [], []
        for t in tensors:
            lo_halo, lo_int, hi_int, hi_halo = slabs(t, axis, h)
            send_lo, send_hi = lo_int.contiguous(), hi_int.contiguous()
            recv_hi, recv_lo = hi_halo.new_empty(hi_halo.shape), lo_halo.new_empty(lo_halo.shape)
            # order matters when lo == hi (two blocks along the axis): the peer's first message is its low slab,
            # which belongs in our HIGH halo
            ops += [dist.P2POp(dist.isend, send_lo, lo), dist.P2POp(dist.isend, send_hi, hi),
                    dist.P2POp(dist.irecv, recv_hi, hi), dist.P2POp(dist.irecv, recv_lo, lo)]
            pending.append((hi_halo, recv_hi, lo_halo, recv_lo))
        for req in dist.batch_isend_irecv(ops):
            req.wait()
        for hi_halo, recv_hi, lo_halo, recv_lo in pending:
            hi_halo.copy_(recv_hi)
            lo_halo.copy_(recv_lo)


class RankBlock:
    """This process's block of a decomposition over torch.distributed (one rank per GPU)."""

    def __init__(self, gn, p, gamma, cfl):
        import torch.distributed as dist
        from . import binding
        self.dist = dist
        self.d = Decomposition(gn, p)
        if dist.get_world_size() != self.d.size:
            raise ValueError("world size %d != number of blocks %d" % (dist.get_world_size(), self.d.size))
        self.rank = dist.get_rank()
        self.block = binding.Echo(*self.d.local, gamma, cfl, block=tuple(self.d.gn) + tuple(self.d.halo))

    def set_primitives(self, w, keys=("rho", "vx", "vy", "vz", "p", "bxf", "byf", "bzf")):
        import torch
        self.block.set_primitives(*[torch.as_tensor(self.d.cut(self.rank, w[k]), device=self.block.device)
                                    for k in keys])

    def step(self, nsteps, t_end=math.inf):
        b, dist = self.block, self.dist
        _step_loop([b], nsteps, t_end,
                   lambda: dist.all_reduce(b.ctrl_word(0), op=dist.ReduceOp.MAX),
                   lambda fields: exchange_halos([b.field(f) for f in fields], self.d, self.rank, dist))

    def get_interior(self):
        q = self.block.get_primitives()
        sl = self.d.interior_slices()
        return {k: v[sl] for k, v in q.items()}
