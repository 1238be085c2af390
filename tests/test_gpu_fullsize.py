"""Parity at BASELINE.json's full size (configs[2]: 256^3 CPA wave) in the launch configuration bench.py
times.  The oracle cannot sweep 256^3 in seconds, so it recomputes SAMPLED outputs one by one: a 64^3
periodic sub-box cut out of the same initial data around each sample is advanced one full RK3 step by the
oracle with the SAME time step (the scheme has no length scale: rhs ~ 1/h, so dt_sub = dt * 256/64 on the
64^3 unit box reproduces the update exactly up to rounding); after one step the wrong periodic images have
travelled at most 3 stages x 8 cells = 24 cells, so the inner 8^3 cells of the sub-box must agree with the
256^3 run to round-off.  Plus properties that hold at any size: div B, conservation, wave symmetry."""
import numpy as np
import pytest

from paper_2401_03008_b200 import inputs

pytestmark = pytest.mark.gpu
G = 4.0 / 3.0
SETK = "rho vx vy vz p bxf byf bzf".split()
PRIMS = "rho vx vy vz p bx by bz".split()


def subbox_check(ob, w, q, n, dt, centres, m=64, inner=8, tight=1e-12):
    """The oracle advances an m^3 periodic sub-box cut out of the initial data `w` (n^3) around each centre
    (x, y, z) by one step of the same dt; the inner `inner`^3 cells must agree with the full-size CUDA result q."""
    lo = (m - inner) // 2
    sl = slice(lo, lo + inner)
    for centre in centres:
        ix = [(np.arange(m) + c - m // 2) % n for c in centre]
        sub = {k: np.ascontiguousarray(w[k][np.ix_(ix[2], ix[1], ix[0])]) for k in SETK}
        o = ob.Oracle(m, m, m, G, 1e3)                                   # cfl so large that dt = t_end
        o.set_primitives(*[sub[k] for k in SETK])
        assert o.step(1, dt * n / m) == 1
        assert o.diagnostics()["dt_last"] == dt * n / m
        qo = o.get_primitives()
        for k in PRIMS + ["bxf", "byf", "bzf"]:
            ref = qo[k][sl, sl, sl]
            got = q[k][np.ix_(ix[2][sl], ix[1][sl], ix[0][sl])]
            err = np.abs(got - ref).max() / np.abs(qo[k]).max()                 # S16 norm
            assert err <= 1e-10, (centre, k, err)
            assert err <= tight, ("above round-off level", centre, k, err)


def seam_planes(e):
    """First plane of every z-chunk but the first of the plane-marching kernels (echo_get_tiling): where their
    register / shared-memory windows restart."""
    t = e.tiling()
    out = set()
    for key in ("cz_prim", "cz_uct", "cz_bupd"):
        cz = t[key]
        if 0 < cz < e.n[2]:
            out.update(range(cz, e.n[2], cz))
    return sorted(out), t


def test_256_sampled_parity_and_invariants():
    import torch
    from paper_2401_03008_b200 import binding as eb
    from oracle import binding as ob

    n = 256
    w = inputs.cpa_wave(n, n, n)
    e = eb.Echo(n, n, n, G, 0.3)
    e.set_primitives(*[torch.as_tensor(w[k], device="cuda") for k in SETK])
    d0 = e.diagnostics()
    e.step(1)
    d1 = e.diagnostics()
    assert d1["rc"] == 0 and d1["steps"] == 1
    dt = d1["dt_last"]
    assert dt == pytest.approx(0.3 / n / d1["amax"], rel=1e-14)          # S9, on the device
    q = {k: v.cpu().numpy() for k, v in e.get_primitives().items()}

    # ---- sampled outputs recomputed by the oracle: the periodic seams, an interior point, and a box whose inner
    # cells straddle a z-chunk seam of the plane-marching kernels (computed from the launch configuration in force)
    seams, til = seam_planes(e)
    assert seams, til                                                   # 256 planes are cut into several chunks
    zs = seams[len(seams) // 2]
    subbox_check(ob, w, q, n, dt, [(0, 0, 0), (100, 37, 201), (255, 128, 5), (77, 130, zs), (8, 251, seams[-1])])

    # ---- properties at full size
    assert d1["max_div_b"] * (1.0 / n) <= 1e-12 * 2.0                    # P5 (|B| <= 2)
    for k in ("sum_D", "sum_Sx", "sum_Sy", "sum_Sz", "sum_U", "sum_Bx", "sum_By", "sum_Bz"):
        assert abs(d1[k] - d0[k]) <= 1e-12 * max(abs(d0[k]), 1.0), k    # P4
    # the diagonal wave depends on x + y + z only: (i+1, j-1, k) carries the same value to round-off
    for k in PRIMS:
        a = q[k]
        assert np.abs(np.roll(a, (1, -1), axis=(1, 2)) - a).max() <= 1e-12, k
    # and one step stays within truncation error of the exact solution (P1)
    ex = inputs.cpa_wave(n, n, n, t=d1["t"])
    for k in PRIMS:
        assert np.abs(q[k] - ex[k]).max() <= 1e-8, k


def test_384_turbulence_sampled_parity():
    """BASELINE.json configs[4] at its full size (384^3 Alfvenic turbulence, the launch configuration bench.py
    --workload turb3d times): one step, sampled sub-boxes recomputed by the oracle (the trick is field-agnostic:
    the periodic images of the cut only reach 24 cells in one step), div B and conservation at full size."""
    import torch
    from paper_2401_03008_b200 import binding as eb
    from oracle import binding as ob

    n = 384
    w = inputs.turbulence(n)
    e = eb.Echo(n, n, n, G, 0.3)
    faces = e.faces_from_potential(*[torch.as_tensor(w[k], device="cuda") for k in ("ax", "ay", "az")], w["b0"])
    for k, f in zip(("bxf", "byf", "bzf"), faces):
        w[k] = f.cpu().numpy()
    del faces
    for k in ("ax", "ay", "az"):
        del w[k]
    e.set_primitives(*[torch.as_tensor(w[k], device="cuda") for k in SETK])
    d0 = e.diagnostics()
    e.step(1)
    d1 = e.diagnostics()
    assert d1["rc"] == 0 and d1["steps"] == 1 and d1["c2p_failures"] == 0
    dt = d1["dt_last"]
    assert dt == pytest.approx(0.3 / n / d1["amax"], rel=1e-14)
    q = {k: v.cpu().numpy() for k, v in e.get_primitives().items()}
    seams, til = seam_planes(e)
    assert seams, til
    subbox_check(ob, w, q, n, dt, [(0, 0, 0), (383, 200, 17), (150, 301, seams[0]), (9, 64, seams[-1])], tight=1e-11)
    assert d1["max_div_b"] <= 1e-12 * w["B0"] * n * 50                   # P5 on a multi-mode field
    for k in ("sum_D", "sum_Sx", "sum_Sy", "sum_Sz", "sum_U", "sum_Bx", "sum_By", "sum_Bz"):
        assert abs(d1[k] - d0[k]) <= 1e-12 * max(abs(d0[k]), 1.0), k    # P4


def test_512_x_aligned_sampled_parity():
    """BASELINE.json configs[3], the x-aligned wave at 512^3 (47 GB workspace, the launch configuration bench.py
    --n 512 --direction x times): one step, sampled sub-boxes recomputed by the oracle, the y/z independence of
    the x-aligned wave bit for bit, div B and conservation."""
    import torch
    from paper_2401_03008_b200 import binding as eb
    from oracle import binding as ob

    n = 512
    w = inputs.cpa_wave(n, n, n, direction="x")
    e = eb.Echo(n, n, n, G, 0.3)
    e.set_primitives(*[torch.as_tensor(w[k], device="cuda") for k in SETK])
    d0 = e.diagnostics()
    e.step(1)
    d1 = e.diagnostics()
    assert d1["rc"] == 0 and d1["steps"] == 1
    dt = d1["dt_last"]
    assert dt == pytest.approx(0.3 / n / d1["amax"], rel=1e-14)
    q = {k: v.cpu().numpy() for k, v in e.get_primitives().items()}
    seams, til = seam_planes(e)
    subbox_check(ob, w, q, n, dt, [(0, 0, 0), (511, 300, seams[0] if seams else 100)])
    for k in PRIMS:                                                      # P7(i): no dependence on y, z, bitwise
        a = q[k]
        assert np.array_equal(a, np.broadcast_to(a[:1, :1, :], a.shape)), k
    assert d1["max_div_b"] * (1.0 / n) <= 1e-12 * 2.0
    for k in ("sum_D", "sum_Sx", "sum_Sy", "sum_Sz", "sum_U", "sum_Bx", "sum_By", "sum_Bz"):
        assert abs(d1[k] - d0[k]) <= 1e-12 * max(abs(d0[k]), 1.0), k


def test_640_diag_sampled_parity():
    """The largest grid of the suite: 640^3 (2.6e8 cells, 92 GB workspace, about 135 GB of device memory at the peak of
    this test), where every sweep axis is longer than the 512-cell chunk limit (two chunks per column) and the
    plane-marching kernels run 3-4 z-chunks.  One step of the diagonal wave, sampled sub-boxes recomputed by the
    oracle (one of them across a z-chunk seam), div B and conservation.  Skipped on a device with less free memory."""
    import torch
    from paper_2401_03008_b200 import binding as eb
    from oracle import binding as ob

    torch.cuda.empty_cache()
    if torch.cuda.mem_get_info()[0] < 150e9:
        pytest.skip("needs 150 GB of free device memory")
    n = 640
    w = inputs.cpa_wave(n, n, n)
    e = eb.Echo(n, n, n, G, 0.3)
    e.set_primitives(*[torch.as_tensor(w[k], device="cuda") for k in SETK])
    d0 = e.diagnostics()
    e.step(1)
    d1 = e.diagnostics()
    assert d1["rc"] == 0 and d1["steps"] == 1
    dt = d1["dt_last"]
    assert dt == pytest.approx(0.3 / n / d1["amax"], rel=1e-14)
    q = {k: v.cpu().numpy() for k, v in e.get_primitives().items()}
    seams, til = seam_planes(e)
    assert til["cx_flux"] < n and til["cy_flux"] < n and til["cz_flux"] < n        # multi-chunk sweeps on all three axes
    subbox_check(ob, w, q, n, dt, [(0, 0, 0), (n - 1, 300, seams[0] if seams else 100), (til["cx_flux"], n - 1, til["cz_flux"])])
    assert d1["max_div_b"] * (1.0 / n) <= 1e-12 * 2.0
    for k in ("sum_D", "sum_Sx", "sum_Sy", "sum_Sz", "sum_U", "sum_Bx", "sum_By", "sum_Bz"):
        assert abs(d1[k] - d0[k]) <= 1e-12 * max(abs(d0[k]), 1.0), k
    del e, q, w
    torch.cuda.empty_cache()
