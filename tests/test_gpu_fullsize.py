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


def test_256_sampled_parity_and_invariants():
    import torch
    from paper_2401_03008_b200 import binding as eb
    from oracle import binding as ob

    n, m, inner = 256, 64, 8
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

    # ---- sampled outputs recomputed by the oracle
    lo = (m - inner) // 2
    for centre in [(0, 0, 0), (100, 37, 201), (255, 128, 5)]:            # (x, y, z) incl. the periodic seams
        ix = [(np.arange(m) + c - m // 2) % n for c in centre]
        sub = {k: np.ascontiguousarray(w[k][np.ix_(ix[2], ix[1], ix[0])]) for k in SETK}
        o = ob.Oracle(m, m, m, G, 1e3)                                   # cfl so large that dt = t_end
        o.set_primitives(*[sub[k] for k in SETK])
        assert o.step(1, dt * n / m) == 1
        assert o.diagnostics()["dt_last"] == dt * n / m
        qo = o.get_primitives()
        sl = slice(lo, lo + inner)
        for k in PRIMS + ["bxf", "byf", "bzf"]:
            ref = qo[k][sl, sl, sl]
            got = q[k][np.ix_(ix[2][sl], ix[1][sl], ix[0][sl])]
            err = np.abs(got - ref).max() / np.abs(qo[k]).max()
            assert err <= 1e-10, (centre, k, err)
            assert err <= 1e-12, ("above round-off level", centre, k, err)

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
