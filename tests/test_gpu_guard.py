"""Out-of-bounds WRITE detector (the stand-in for compute-sanitizer memcheck, which this GPU pool refuses): the handle's
workspace and the output buffers of echo_get_primitives sit between guard bands filled with a byte pattern; after every
entry point has run on grids whose sizes are multiples of nothing (ragged tiles, ragged chunks, odd row lengths that
switch the TMA path off, even ones that switch it on, a one-plane grid, a padded block with physical boundaries) the
bands must be untouched.  A kernel that stores one element past a field, a tile tail that is not masked, a halo
message one slab too long: each of them lands in a band or in a neighbouring field and shows up here or in the parity
tests.  The pattern is 0xFF, a NaN when read as a double, and the workspace itself starts out filled with it: a READ
of a band, of the padding between fields or of a scratch field that no kernel has written yet turns the state into NaN
and fails the finiteness checks below (the stand-in for initcheck)."""
import ctypes as C

import numpy as np
import pytest

from paper_2401_03008_b200 import inputs

pytestmark = pytest.mark.gpu
G = 4.0 / 3.0
BAND = 1 << 20            # bytes on each side of a guarded buffer (a multiple of 256: the workspace alignment)
PATTERN = 0xFF           # as doubles: NaN, so that a READ of a band or of never-written workspace poisons the result


class Guarded:
    """A device byte buffer of `nbytes` between two bands of PATTERN."""

    def __init__(self, torch, nbytes):
        self.torch = torch
        self.raw = torch.full((BAND + nbytes + BAND,), PATTERN, dtype=torch.uint8, device="cuda")
        self.body = self.raw[BAND:BAND + nbytes]       # starts out as NaN as well (initcheck: see the module docstring)
        assert self.body.data_ptr() % 256 == 0

    def intact(self):
        self.torch.cuda.synchronize()
        return bool((self.raw[:BAND] == PATTERN).all()) and bool((self.raw[BAND + self.body.numel():] == PATTERN).all())


def _rebind_guarded(torch, eb, e):
    """Moves the handle's workspace between guard bands (echo_bind again: allowed, it resets the handle)."""
    nbytes = e.L.echo_workspace_bytes(e.h)
    gws = Guarded(torch, nbytes)
    e._check(e.L.echo_bind(e.h, gws.body.data_ptr(), nbytes, eb._stream(e.device)))
    e.workspace = gws.body
    return gws


def _guarded_outputs(torch, e, k):
    """k output fields of the handle's shape in ONE guarded buffer, separated by bands as well."""
    per = e.N * 8
    stride = (per + BAND + 255) // 256 * 256
    g = Guarded(torch, stride * k)
    g.body.fill_(PATTERN)
    views = [g.body[i * stride:i * stride + per].view(torch.float64).view(e.shape) for i in range(k)]

    def gaps_intact():
        torch.cuda.synchronize()
        return all(bool((g.body[i * stride + per:(i + 1) * stride] == PATTERN).all()) for i in range(k)) and g.intact()
    return views, gaps_intact


def _fields(torch, eb, ob, shape):
    w = inputs.turbulence(None, shape=shape)
    bo = ob.faces_from_potential(w["ax"], w["ay"], w["az"])
    f = [w[k] for k in ("rho", "vx", "vy", "vz", "p")] + [b + w["b0"][d] for d, b in enumerate(bo)]
    return [torch.as_tensor(np.ascontiguousarray(a), device="cuda") for a in f]


@pytest.mark.parametrize("shape,kw", [
    ((37, 21, 11), {}),                          # odd n_x: no tensor maps, every tile by cp.async; ragged everywhere
    ((50, 19, 23), {}),                          # even n_x: TMA tiles next to seam tiles, ragged y and z
    ((70, 40, 9), {}),                           # one z-chunk of 9 planes, several x tiles
    ((16, 16, 40), {}),                          # the smallest tile count, several z-chunks
    ((40, 24, 1), {}),                           # 2.5-D: the flat kernels
    ((50, 19, 23), {"uct": False, "ho": False}),  # cell-centred B: 8-component sweeps in dynamic shared memory
    ((37, 21, 11), {"rec": 2, "rk": 2, "ho": False}),   # linear reconstruction + RK2
])
def test_no_write_outside_the_workspace_or_the_outputs(shape, kw):
    import torch
    from paper_2401_03008_b200 import binding as eb
    from oracle import binding as ob

    f = _fields(torch, eb, ob, shape)
    e = eb.Echo(*shape, G, 0.3, **kw)
    gws = _rebind_guarded(torch, eb, e)
    e.set_primitives(*f)
    assert gws.intact()
    gws.raw[BAND - 1] = 0                        # the detector itself: one byte just below the workspace
    assert not gws.intact()
    gws.raw[BAND - 1] = PATTERN
    e.step(2)                                    # graph replay
    e.use_graph(False)
    e.step(1)                                    # plain launches
    r = e.rhs()
    assert all(bool(torch.isfinite(t).all()) for k in ("rhsU", "rhsB", "E") for t in r[k]) and np.isfinite(r["amax"])
    mdiv, fdiv = e.div_b(want_field=True)
    assert np.isfinite(mdiv) and bool(torch.isfinite(fdiv).all())
    d = e.diagnostics()
    assert d["rc"] == 0 and d["steps"] == 3 and d["c2p_failures"] == 0
    assert gws.intact()
    outs, gaps_intact = _guarded_outputs(torch, e, 11)
    e._check(e.L.echo_get_primitives(e.h, *[o.data_ptr() for o in outs]))
    assert gaps_intact() and gws.intact()
    assert all(bool(torch.isfinite(o).all()) for o in outs)                  # and every element was written
    cons, gaps2 = _guarded_outputs(torch, e, 5)
    e._check(e.L.echo_get_conserved(e.h, *[o.data_ptr() for o in cons]))
    assert gaps2() and all(bool(torch.isfinite(o).all()) for o in cons)


def test_no_write_outside_a_padded_block_with_boundaries():
    """Block mode: ghost fill of reflecting / outflow sides inside echo_step, packed halo messages in guarded buffers."""
    import torch
    from paper_2401_03008_b200 import binding as eb
    from oracle import binding as ob

    n, ng, kinds = (22, 18, 20), 8, (1, 2, 0, 0, 2, 1)
    pad = (n[0] + 2 * ng, n[1], n[2] + 2 * ng)
    f = _fields(torch, eb, ob, pad)
    e = eb.Echo(*pad, G, 0.3, block=tuple(n) + (ng, 0, ng), boundaries=kinds)
    gws = _rebind_guarded(torch, eb, e)
    e._check(e.L.echo_set_boundaries(e.h, (C.c_int * 6)(*kinds)))            # echo_bind reset nothing of these, but be explicit
    e.set_primitives(*f)
    e.step(2)
    assert gws.intact()
    # one packed message per decomposed axis and side, each in its own guarded buffer
    fields = list(range(8))
    for axis in (0, 2):
        nd = e.halo_doubles(axis)
        for side in (0, 1):
            gb = Guarded(torch, nd * 8)
            buf = gb.body.view(torch.float64)
            e.halo_pack(fields, axis, side, buf)
            assert gb.intact() and bool(torch.isfinite(buf).all())
            e.halo_unpack(fields, axis, side, buf)
            assert gb.intact() and gws.intact()
    d = e.diagnostics()
    assert d["rc"] == 0 and d["c2p_failures"] == 0
