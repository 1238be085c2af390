"""Row (f1): the domain-decomposed step (one padded periodic block per rank, packed halo refresh of 8 fields after
every RK stage, all-reduce(max) of a_max) against the undecomposed run of the same library.  All blocks live in
this process on one GPU (LocalBlocks): the stage halves are the ones echo_step is made of, the same arithmetic
per cell and an exact max, so the interiors must agree BIT FOR BIT; a wrong halo width, slab, corner, field list
or reduction shows up at once."""
import numpy as np
import pytest

from paper_2401_03008_b200 import inputs

pytestmark = pytest.mark.gpu
G = 4.0 / 3.0
SETK = "rho vx vy vz p bxf byf bzf".split()


def test_pack_kernels_equal_the_torch_reference():
    """echo_halo_pack / echo_halo_unpack against blocks.pack_slabs / unpack_slabs (the form the gloo test runs),
    for every axis and side, with skipped slots."""
    import torch
    from paper_2401_03008_b200 import binding as eb, blocks
    e = eb.Echo(40, 24, 32, G, 0.3, block=(64, 24, 64, 8, 0, 8))
    g = torch.Generator(device="cuda").manual_seed(3)
    fields = [24, 25, 26, -1, 28, 13, -1, 15]
    for f in range(44):
        e.field(f).copy_(torch.randn(e.shape, generator=g, device="cuda", dtype=torch.float64))
    tens = [e.field(f) if f >= 0 else None for f in fields]
    assert e.halo_doubles(1) == 0 and e.halo_doubles(0) == 8 * 8 * 24 * 32 and e.halo_doubles(2) == 8 * 8 * 40 * 24
    for axis in (0, 2):
        for side in (0, 1):
            a = torch.full((e.halo_doubles(axis),), -7.0, dtype=torch.float64, device="cuda")
            b = a.clone()
            e.halo_pack(fields, axis, side, a)
            blocks.pack_slabs(tens, axis, side, b)
            assert torch.equal(a, b), (axis, side)
            assert (a.view(8, -1)[3] == -7.0).all()                  # skipped slot untouched
            before = [e.field(f).clone() for f in range(44)]
            msg = torch.randn(e.halo_doubles(axis), generator=g, device="cuda", dtype=torch.float64)
            ref = [t.clone() for t in before]
            blocks.unpack_slabs([ref[f] if f >= 0 else None for f in fields], axis, side, msg)
            e.halo_unpack(fields, axis, side, msg)
            for f in range(44):
                assert torch.equal(e.field(f), ref[f]), (axis, side, f)
    assert e.L.echo_halo_pack(e.h, (eb.C.c_int * 8)(*[0] * 8), 1, 0, a.data_ptr(), None) == eb.ECHO_EINVAL   # y is not decomposed
    assert e.stage_halo_fields(1) == [24, 25, 26, 27, 28, 13, 14, 15]
    assert e.stage_halo_fields(2) == list(range(8, 16)) and e.stage_halo_fields(3) == list(range(8))


@pytest.mark.parametrize("p,order", [((2, 1, 1), (5, 3)), ((1, 2, 2), (5, 3)), ((2, 2, 2), (5, 3)), ((1, 1, 3), (5, 3)),
                                     ((2, 1, 2), (2, 2))])
def test_blocks_match_single_domain_bitwise(p, order):
    import torch
    from paper_2401_03008_b200 import binding as eb, blocks
    from oracle import binding as ob

    gn = (32, 32, 48)
    w = inputs.turbulence(None, shape=gn)
    bo = ob.faces_from_potential(w["ax"], w["ay"], w["az"])
    w["bxf"], w["byf"], w["bzf"] = [b + w["b0"][d] for d, b in enumerate(bo)]
    rec, rk = order                        # (2, 2): linear REC + SSP-RK2 with the second-order INT/DER
    e = eb.Echo(*gn, G, 0.3, ho=(rec == 5), rec=rec, rk=rk)
    e.set_primitives(*[torch.as_tensor(w[k], device="cuda") for k in SETK])
    lb = blocks.LocalBlocks(gn, p, G, 0.3, ho=(rec == 5), rec=rec, rk=rk)
    lb.set_primitives(w)
    t_end = 2.5 * 0.3 / 48 / 0.9          # inside the third step: exercises the clipped dt on every block
    e.step(4, t_end)
    lb.step(4, t_end)
    d = e.diagnostics()
    assert d["steps"] == 3 and lb.time() == d["t"] == t_end
    q = {k: v.cpu().numpy() for k, v in e.get_primitives().items()}
    qb = lb.get_primitives()
    for k in q:
        assert np.array_equal(q[k], qb[k]), (p, k, np.abs(q[k] - qb[k]).max())


def test_block_argument_checks():
    from paper_2401_03008_b200 import binding as eb, blocks
    L = eb.lib()
    assert not L.echo_create_block(20, 8, 8, G, 0.3, 32, 8, 8, 8, 0, 0)      # 4 interior cells < halo
    assert not L.echo_create_block(16, 8, 8, G, 0.3, 0, 8, 8, 0, 0, 0)
    with pytest.raises(ValueError):
        blocks.Decomposition((30, 32, 32), (4, 1, 1))                        # 30 % 4 != 0
    with pytest.raises(ValueError):
        blocks.Decomposition((32, 32, 32), (8, 1, 1))                        # 4 cells per block < halo


def test_rank_block_world_of_one():
    """RankBlock (the torch.distributed driver) in a world of one rank: NCCL all-reduce of the a_max word, no
    exchange; must reproduce the plain run bit for bit."""
    import os
    import torch
    import torch.distributed as dist
    from paper_2401_03008_b200 import binding as eb, blocks

    os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
    os.environ.setdefault("MASTER_PORT", "29755")
    dist.init_process_group("nccl", rank=0, world_size=1)
    try:
        gn = (24, 16, 20)
        w = inputs.cpa_wave(*gn)
        e = eb.Echo(*gn, G, 0.3)
        e.set_primitives(*[torch.as_tensor(w[k], device="cuda") for k in SETK])
        rb = blocks.RankBlock(gn, (1, 1, 1), G, 0.3)
        rb.set_primitives(w)
        e.step(3)
        rb.step(3)
        q, qb = e.get_primitives(), rb.get_interior()
        for k in q:
            assert torch.equal(q[k], qb[k]), k
    finally:
        dist.destroy_process_group()
