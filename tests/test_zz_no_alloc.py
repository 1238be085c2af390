"""echo_div_b_static: the allocation-free entry point (its scratch is a static device array, include/echo.h) against the
existing path echo_div_b, on the same staggered fields, on calls in a row that share the scratch.  Collected last on
purpose (the file name): the run uses -x, and nothing here depends on what ran before it."""
import ctypes as C

import numpy as np
import pytest

G = 4.0 / 3.0
TOL = 1e-10          # the parity bar of the other GPU tests, relative to the largest |div B|


def test_oversize_grid_is_rejected_before_any_cuda_call():
    """Host logic only (runs without a GPU): the size check comes first and says what the limit is."""
    from paper_2401_03008_b200 import binding as eb
    L = eb.lib()
    fake = C.c_void_p(256)           # never dereferenced: the call must fail on the sizes
    # 257 x 256 x 256: ceil(257/64) * ceil(256/4) * 256 = 81920 tiles > 65536
    rc = L.echo_div_b_static(257, 256, 256, 1, fake, fake, fake, fake, fake, None)
    assert rc == eb.ECHO_EINVAL
    msg = L.echo_div_b_static_error().decode()
    assert "81920" in msg and str(eb.ECHO_DIV_B_STATIC_MAX_TILES) in msg, msg
    assert L.echo_div_b_static(0, 4, 4, 1, fake, fake, fake, fake, fake, None) == eb.ECHO_EINVAL
    assert L.echo_div_b_static(8, 8, 8, 1, None, fake, fake, fake, fake, None) == eb.ECHO_EINVAL
    assert L.echo_div_b_static(8, 8, 8, 1, fake, fake, fake, None, None, None) == eb.ECHO_EINVAL
    assert "null" in L.echo_div_b_static_error().decode()


def _handle_with_faces(eb, torch, n, seed, amp, ho=True):
    """A periodic handle holding uniform gas and random (NOT solenoidal) staggered fields of amplitude amp."""
    nx, ny, nz = n
    rng = np.random.default_rng(seed)
    one = torch.ones((nz, ny, nx), dtype=torch.float64, device="cuda")
    zero = torch.zeros_like(one)
    faces = [torch.as_tensor(amp * rng.standard_normal((nz, ny, nx)), device="cuda") for _ in range(3)]
    e = eb.Echo(nx, ny, nz, G, 0.3, ho=ho)
    e.set_primitives(one, zero, zero, zero, one, *faces)
    return e


def _compare(eb, torch, e, ho, div_out, max_out):
    """One call of the new entry point into the caller's buffers, against echo_div_b of the same handle."""
    bf = [e.field(5 + d) for d in range(3)]                       # the staggered B the existing path reads
    ref_max, ref_field = e.div_b(want_field=True)
    eb.div_b_static(bf[0], bf[1], bf[2], ho=ho, div_field=div_out, max_abs=max_out)
    torch.cuda.synchronize()
    scale = float(ref_field.abs().max())
    assert scale > 0.0 and ref_max == pytest.approx(scale, rel=1e-15)
    assert float((div_out - ref_field).abs().max()) <= TOL * scale
    assert abs(float(max_out[0]) - ref_max) <= TOL * scale
    return ref_max


@pytest.mark.gpu
def test_static_div_b_matches_the_workspace_path_on_calls_in_a_row():
    import torch
    from paper_2401_03008_b200 import binding as eb

    # call 1: ragged tiles along x and y, large divergence (leaves large partial maxima behind in the scratch)
    big = _handle_with_faces(eb, torch, (72, 22, 9), 11, 1.0)
    out_big = torch.empty((9, 22, 72), dtype=torch.float64, device="cuda")
    m = torch.full((1,), -1.0, dtype=torch.float64, device="cuda")
    m_big = _compare(eb, torch, big, 1, out_big, m)
    # call 2, straight after, on a smaller grid with a divergence 1e6 times smaller: fewer tiles than the scratch
    # still holds from call 1, so a stale slot read would show up as the wrong maximum
    small = _handle_with_faces(eb, torch, (20, 6, 3), 12, 1e-6)
    out_small = torch.empty((3, 6, 20), dtype=torch.float64, device="cuda")
    m_small = _compare(eb, torch, small, 1, out_small, m)
    assert m_small < 1e-3 * m_big
    # call 3: the first grid again, into the same outputs -> the same answer as call 1
    keep = out_big.clone()
    assert _compare(eb, torch, big, 1, out_big, m) == m_big
    assert torch.equal(out_big, keep)
    # the second-order divergence (HO = NO) and the maximum alone (no field output)
    lo = _handle_with_faces(eb, torch, (33, 9, 5), 13, 0.5, ho=False)
    out_lo = torch.empty((5, 9, 33), dtype=torch.float64, device="cuda")
    m_lo = _compare(eb, torch, lo, 0, out_lo, m)
    m2 = torch.zeros(1, dtype=torch.float64, device="cuda")
    eb.div_b_static(*[lo.field(5 + d) for d in range(3)], ho=0, max_abs=m2)
    torch.cuda.synchronize()
    assert abs(float(m2[0]) - m_lo) <= TOL * m_lo


@pytest.mark.gpu
def test_static_div_b_allocates_nothing_and_honours_the_limit():
    import torch
    from paper_2401_03008_b200 import binding as eb

    e = _handle_with_faces(eb, torch, (64, 16, 8), 21, 1.0)
    bf = [e.field(5 + d) for d in range(3)]
    out = torch.empty((8, 16, 64), dtype=torch.float64, device="cuda")
    m = torch.zeros(1, dtype=torch.float64, device="cuda")
    assert eb.lib().echo_div_b_static_setup() == 0
    eb.div_b_static(*bf, div_field=out, max_abs=m)               # first call: any lazy set-up is behind us
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    for _ in range(5):
        eb.div_b_static(*bf, div_field=out, max_abs=m)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0                 # device memory in use did not move
    # a solenoidal field: both paths see round-off only
    rng = np.random.default_rng(5)
    pot = [torch.as_tensor(rng.standard_normal((8, 16, 64)), device="cuda") for _ in range(3)]
    faces = e.faces_from_potential(*pot)
    e.set_primitives(torch.ones_like(out), *[torch.zeros_like(out)] * 3, torch.ones_like(out), *faces)
    eb.div_b_static(*[e.field(5 + d) for d in range(3)], div_field=out, max_abs=m)
    torch.cuda.synchronize()
    bmax = max(float(f.abs().max()) for f in faces)
    assert float(m[0]) <= 1e-11 * bmax * 64 and abs(float(m[0]) - e.div_b()) <= 1e-11 * bmax * 64
    # beyond the scratch: a clear error, nothing launched
    nx, ny, nz = 130, 256, 256                                   # 3 * 64 * 256 = 49152 tiles fits; 257 wide does not
    big = [torch.zeros((nz, ny, nx), dtype=torch.float64, device="cuda") for _ in range(3)]
    eb.div_b_static(*big, max_abs=m)
    torch.cuda.synchronize()
    assert float(m[0]) == 0.0
    too_big = [torch.zeros((256, 256, 257), dtype=torch.float64, device="cuda") for _ in range(3)]
    with pytest.raises(eb.EchoError) as ei:
        eb.div_b_static(*too_big, max_abs=m)
    assert ei.value.code == eb.ECHO_EINVAL and "65536" in str(ei.value)


@pytest.mark.gpu
def test_static_div_b_under_stream_capture():
    """The use case the entry point exists for: captured into a CUDA graph (no allocation, no synchronisation inside
    the call), replayed twice on changing inputs."""
    import torch
    from paper_2401_03008_b200 import binding as eb

    e = _handle_with_faces(eb, torch, (40, 12, 6), 31, 1.0)
    bf = [e.field(5 + d) for d in range(3)]
    out = torch.zeros((6, 12, 40), dtype=torch.float64, device="cuda")
    m = torch.zeros(1, dtype=torch.float64, device="cuda")
    assert eb.lib().echo_div_b_static_setup() == 0                # symbol lookup before the capture begins
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph):
        eb.div_b_static(*bf, div_field=out, max_abs=m)
    for scale in (1.0, 0.25):
        for f in bf:
            f.mul_(scale)                                         # the graph reads the handle's fields in place
        graph.replay()
        torch.cuda.synchronize()
        ref_max, ref_field = e.div_b(want_field=True)
        assert float((out - ref_field).abs().max()) <= TOL * ref_max
        assert abs(float(m[0]) - ref_max) <= TOL * ref_max
