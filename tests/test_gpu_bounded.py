"""Row f4, first slice, on the CUDA path: non-periodic boundaries (reflecting walls, zero-gradient outflow) of a padded
block (echo_create_block with 8 ghost layers + echo_set_boundaries), advanced by echo_step itself (the ghost fill runs
inside the step, after every stage).  Element-wise against the oracle's bounded grid on the same padded inputs."""
import numpy as np
import pytest

from paper_2401_03008_b200 import inputs

pytestmark = pytest.mark.gpu
G = 4.0 / 3.0
PRIMS = "rho vx vy vz p bx by bz".split()
SETK = "rho vx vy vz p bxf byf bzf".split()
NG = 8


def _padded_turbulence(n, kinds):
    """Config-5 field on the interior n = (nx, ny, nz), extended into the ghost layers by its periodic images (the
    libraries overwrite those layers; only the low wall faces of the normal B are read)."""
    from oracle import binding as ob
    w = inputs.turbulence(None, shape=n)
    bo = ob.faces_from_potential(w["ax"], w["ay"], w["az"])
    f = [w[k] for k in ("rho", "vx", "vy", "vz", "p")] + [b + w["b0"][d] for d, b in enumerate(bo)]
    for a in range(3):
        if kinds[2 * a]:
            idx = (np.arange(-NG, n[a] + NG)) % n[a]
            f = [np.ascontiguousarray(np.take(x, idx, axis=2 - a)) for x in f]
    return f


@pytest.mark.parametrize("n,kinds", [((24, 16, 12), (1, 1, 0, 0, 0, 0)), ((20, 24, 9), (2, 2, 1, 1, 0, 0)),
                                     ((16, 12, 24), (1, 2, 0, 0, 2, 1)), ((18, 16, 20), (1, 1, 1, 1, 1, 1))])
def test_bounded_step_against_the_oracle(n, kinds):
    import torch
    from paper_2401_03008_b200 import binding as eb
    from oracle import binding as ob

    f = _padded_turbulence(n, kinds)
    ng = [NG if kinds[2 * a] else 0 for a in range(3)]
    o = ob.Oracle(*n, G, 0.3, boundaries=kinds)
    o.set_primitives(*f)
    pad = [n[a] + 2 * ng[a] for a in range(3)]
    e = eb.Echo(*pad, G, 0.3, block=tuple(n) + tuple(ng), boundaries=kinds)
    e.set_primitives(*[torch.as_tensor(a, device="cuda") for a in f])
    div0 = e.div_b(want_field=True)[1].cpu().numpy()
    # 6 steps (graph replay), then 2 more with plain launches
    e.step(6)
    assert o.step(6) == 6
    e.use_graph(False)
    e.step(2)
    o.step(2)
    dg, do = e.diagnostics(), o.diagnostics()
    assert dg["rc"] == 0 and dg["steps"] == 8 and dg["c2p_failures"] == 0 and do["c2p_failures"] == 0
    assert dg["t"] == pytest.approx(do["t"], rel=1e-13)
    qg = {k: v.cpu().numpy() for k, v in e.get_primitives().items()}
    qo = o.get_primitives()
    inner = o.interior()
    for k in PRIMS + ["bxf", "byf", "bzf"]:
        ref, got = qo[k][inner], qg[k][inner]
        err = np.abs(got - ref).max() / np.abs(ref).max()
        assert err <= 1e-10, (kinds, k, err)
        assert err <= 1e-11, ("above round-off level", kinds, k, err)
    # the ghost layers of the evolved fields agree as well (same fill rule): conserved fields and faces
    cg = {k: v.cpu().numpy() for k, v in e.get_conserved().items()}
    assert np.isfinite(cg["D"]).all()
    for k in ("bxf", "byf", "bzf"):
        assert np.abs(qg[k] - qo[k]).max() <= 1e-11 * np.abs(qo[k]).max(), k
    # the high-order div B of every interior cell keeps its initial value to round-off with walls and outflow alike
    # (UCT advances the faces by a curl; next to a wall the initial value is not zero, because the ghost faces that
    # enter the stencil are mirror images rather than the periodic images the field was made solenoidal with)
    # ... except within the stencil's reach (3 cells) of an OUTFLOW side, whose ghost faces are copies, not a curl
    div1 = e.div_b(want_field=True)[1].cpu().numpy()
    keep = tuple(slice(ng[a] + (3 if kinds[2 * a] == 2 else 0), ng[a] + n[a] - (3 if kinds[2 * a + 1] == 2 else 0))
                 for a in (2, 1, 0))
    assert np.abs(div1[keep] - div0[keep]).max() <= 1e-11 * max(n) * 5


def test_reflecting_box_conserves_mass_and_energy():
    """All six sides reflecting: no flux through a wall (the mirror image makes the normal mass and energy fluxes odd),
    so the interior sums of D and U are conserved to round-off; the momentum normal to a wall is not."""
    import torch
    from paper_2401_03008_b200 import binding as eb

    n, kinds = (20, 16, 18), (1,) * 6
    f = _padded_turbulence(n, kinds)
    pad = [m + 2 * NG for m in n]
    e = eb.Echo(*pad, G, 0.3, block=tuple(n) + (NG,) * 3, boundaries=kinds)
    e.set_primitives(*[torch.as_tensor(a, device="cuda") for a in f])
    d0 = e.diagnostics()
    e.step(10)
    d1 = e.diagnostics()
    assert d1["steps"] == 10 and d1["c2p_failures"] == 0
    for k in ("sum_D", "sum_U"):
        assert abs(d1[k] - d0[k]) <= 1e-12 * abs(d0[k]), (k, d0[k], d1[k])
    assert abs(d1["sum_Sx"] - d0["sum_Sx"]) > 1e-6


def test_boundary_argument_checks():
    import torch
    from paper_2401_03008_b200 import binding as eb
    e = eb.Echo(24, 8, 8, G, 0.3, block=(8, 8, 8, 8, 0, 0))
    k = lambda *v: (eb.C.c_int * 6)(*v)
    assert e.L.echo_set_boundaries(e.h, k(1, 1, 1, 1, 0, 0)) == eb.ECHO_EINVAL      # y has no ghost layers
    assert e.L.echo_set_boundaries(e.h, k(3, 1, 0, 0, 0, 0)) == eb.ECHO_EINVAL
    assert e.L.echo_set_boundaries(e.h, k(1, 0, 0, 0, 0, 0)) == eb.ECHO_OK          # one wall, one neighbour
    z = [torch.ones(8, 8, 24, dtype=torch.float64, device="cuda") * c for c in (1, 0, 0, 0, 1, 1, 0, 0)]
    e.set_primitives(*z)
    assert e.L.echo_step(e.h, 1, float("inf")) == eb.ECHO_EINVAL                     # the high side is the caller's
    assert e.L.echo_set_boundaries(e.h, k(1, 1, 0, 0, 0, 0)) == eb.ECHO_ESTATE
    e.stage_sweeps(1)                                                                # ... who steps it by halves
    e.stage_finish(1)
    e.fill_boundaries(e.stage_halo_fields(1))
