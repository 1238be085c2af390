"""CPU checks of the multi-rank plumbing of row (f1): the decomposition bookkeeping and the PACKED halo exchange
(blocks.exchange_packed: one message per axis and side for all fields, sent in a cell part and a face part) over
torch.distributed with the gloo backend (world sizes 2 and 4), on plain CPU tensors with the torch reference
pack / unpack (the CUDA pack kernels are compared with these in tests/test_gpu_blocks.py)."""
import json
import os
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

WORKER = r"""
import sys, json
sys.path.insert(0, %r)
import numpy as np, torch, torch.distributed as dist
from paper_2401_03008_b200 import blocks
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
p = tuple(json.loads(sys.argv[1]))
gn = (32, 16, 24)
d = blocks.Decomposition(gn, p)
assert d.size == world
rng = np.random.default_rng(5)
glob = [rng.standard_normal(gn[::-1]) for _ in range(2)]
ts = []
for a in glob:
    t = torch.from_numpy(d.cut(rank, a)).clone()
    # wipe the halos: the exchange has to restore them
    for axis in range(3):
        if d.halo[axis]:
            lo, _, _, hi = blocks.slabs(t, axis)
            lo.fill_(float("nan")); hi.fill_(float("nan"))
    ts.append(t)
# packed messages: 8 slots per buffer (5 "cell" + 3 "face"), sent in two parts as RankBlock does; slots 0-4 and
# 5-7 carry the same two tensors over and over, a skipped slot (None) must leave its part of the message alone
def per(axis):
    n = list(d.local); n[axis] = blocks.HALO
    return n[0] * n[1] * n[2]
bufs = [tuple(torch.full((8 * per(ax),), -7.0, dtype=torch.float64) for _ in range(4)) if d.p[ax] > 1 else None for ax in range(3)]
cells = [ts[0], ts[1], ts[0], ts[1], ts[0], None, None, None]
faces = [None] * 5 + [ts[1], ts[0], ts[1]]
side_group = dist.new_group()            # as RankBlock: the cell part travels on its own communicator
for tensors, part in ((cells, blocks.CELLS), (faces, blocks.FACES)):
    blocks.exchange_packed(d, rank, dist, bufs,
                           lambda ax, side, buf: blocks.pack_slabs(tensors, ax, side, buf),
                           lambda ax, side, buf: blocks.unpack_slabs(tensors, ax, side, buf),
                           part=lambda ax: slice(part.start * per(ax), part.stop * per(ax)),
                           group=side_group if part is blocks.CELLS else None)
    if part is blocks.CELLS:      # after the first part every halo is already restored (both tensors travelled)
        ok_first = all(np.array_equal(t.numpy(), d.cut(rank, a)) for t, a in zip(ts, glob))
ok = ok_first and all(np.array_equal(t.numpy(), d.cut(rank, a)) for t, a in zip(ts, glob))
assert blocks._masked(list(range(8)), blocks.FACES) == [-1] * 5 + [5, 6, 7]
# a_max style all-reduce of a bit pattern
w = torch.tensor([np.float64(0.1 * (rank + 1)).view(np.int64)], dtype=torch.int64)
dist.all_reduce(w, op=dist.ReduceOp.MAX)
ok = ok and w.view(torch.float64).item() == 0.1 * world
res = torch.tensor([1 if ok else 0])
dist.all_reduce(res, op=dist.ReduceOp.MIN)
if rank == 0:
    print(json.dumps({"ok": int(res.item()), "world": world}))
dist.destroy_process_group()
"""


def _torchrun(nproc, args, port):
    env = dict(os.environ, MASTER_ADDR="127.0.0.1")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(nproc),
           "--master-addr", "127.0.0.1", "--master-port", str(port)] + args
    return subprocess.run(cmd, capture_output=True, text=True, timeout=300, env=env, cwd=ROOT)


@pytest.mark.parametrize("p,port", [((2, 1, 1), 29741), ((1, 1, 2), 29742), ((2, 2, 1), 29743)])
def test_halo_exchange_gloo(tmp_path, p, port):
    script = tmp_path / "worker.py"
    script.write_text(WORKER % ROOT)
    r = _torchrun(p[0] * p[1] * p[2], [str(script), json.dumps(list(p))], port)
    assert r.returncode == 0, r.stderr[-3000:]
    out = json.loads([l for l in r.stdout.splitlines() if l.startswith("{")][-1])
    assert out == {"ok": 1, "world": p[0] * p[1] * p[2]}


def test_decomposition_bookkeeping():
    from paper_2401_03008_b200 import blocks
    d = blocks.Decomposition((32, 16, 24), (2, 1, 3))
    assert d.size == 6 and d.halo == (8, 0, 8) and d.interior == (16, 16, 8) and d.local == (32, 16, 24)
    assert d.coords(5) == (1, 0, 2) and d.rank_of((1, 0, 2)) == 5
    assert d.neighbour(0, 0, -1) == 1 and d.neighbour(0, 2, -1) == 4 and d.neighbour(5, 2, +1) == 1
    assert d.global_index(0, 0)[:9] == [24, 25, 26, 27, 28, 29, 30, 31, 0]
    a = np.arange(24 * 16 * 32, dtype=float).reshape(24, 16, 32)
    c = d.cut(3, a)                       # rank 3 = coords (1, 0, 1)
    assert c.shape == (24, 16, 32)
    sl = d.interior_slices()
    assert np.array_equal(c[sl], a[8:16, :, 16:32])
