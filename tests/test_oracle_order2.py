"""Pins of the oracle's second-order variant of P:L304 ("second order time-stepping and linear reconstruction rather
than MP5"): REC = limited linear (monotonized-central slope, reading O3b) and SSP-RK2.  What fixes them:
hand-computed values and the defining properties of the limiter, the two-stage update rebuilt in numpy from L(U)
(itself pinned in test_oracle_scheme.py), and the orders in dt and in h the variant must show on the exact wave."""
import math

import numpy as np
import pytest

from oracle import binding as ob
from oracle.binding import Oracle
from paper_2401_03008_b200 import inputs

G = 4.0 / 3.0


def test_tvd2_hand_values_and_limiter_properties():
    # v_i + MC(a, b)/2, MC = minmod(2a, 2b, (a+b)/2), a = v_i - v_{i-1}, b = v_{i+1} - v_i; worked by hand:
    assert ob.tvd2([0, 1, 2, 3, 4]) == 2.5                 # a = b = 1: slope 1 (exact on linear data)
    assert ob.tvd2([0, 0, 1, 4, 0]) == 2.0                 # a = 1, b = 3: min(2, 6, 2) = 2
    assert ob.tvd2([9, 3, 1, 0.5, 7]) == 0.5               # a = -2, b = -0.5: max(-4, -1, -1.25) = -1
    assert ob.tvd2([0, 1, 2, 2, 0]) == 2.0                 # b = 0: no slope
    assert ob.tvd2([0, 1, 3, 2, 0]) == 3.0                 # extremum: slopes of opposite sign
    assert ob.tvd2([0, 1, 2, 12, 0]) == 3.0                # a = 1, b = 10: 2a = 2 bounds the central slope 5.5
    rng = np.random.default_rng(3)
    for _ in range(2000):
        v = rng.standard_normal(5)
        r = ob.tvd2(v)
        lo, hi = min(v[2], v[3]), max(v[2], v[3])
        assert lo - 1e-15 <= r <= hi + 1e-15               # between the two neighbours of the face (monotone)
        assert ob.tvd2([5.0, v[1], v[2], v[3], -7.0]) == r            # a three-point stencil
        assert ob.tvd2(-v) == -r                                      # odd
        assert ob.tvd2(3.0 * v + 1.0) == pytest.approx(3.0 * r + 1.0, abs=1e-14)
    for k in range(50):                                    # exact for linear data of any slope
        s, c = rng.standard_normal(2)
        v = c + s * np.arange(-2, 3)
        assert ob.tvd2(v) == pytest.approx(c + 0.5 * s, abs=1e-15)
        assert ob.tvd2(v[::-1]) == pytest.approx(c - 0.5 * s, abs=1e-15)   # mirrored stencil: right-biased value


def _conserved(o):
    u = o.get_conserved()
    q = o.get_primitives()
    return [np.array(u[k]) for k in ("D", "Sx", "Sy", "Sz", "U")] + [np.array(q[k]) for k in ("bxf", "byf", "bzf")]


@pytest.mark.parametrize("uct", [True, False])
def test_rk2_step_is_heun_of_the_pinned_operator(uct):
    """One oracle step with rk = 2 against U^{n+1} = 1/2 U^n + 1/2 (U1 + dt L(U1)), U1 = U^n + dt L(U^n), rebuilt in
    numpy from rhs() calls; U1 enters a second oracle through con2prim (exact to 1e-12, test_oracle_units.py)."""
    n = (12, 10, 8)
    w = inputs.turbulence(None, shape=n)
    if uct:
        b = [x + w["b0"][d] for d, x in enumerate(ob.faces_from_potential(w["ax"], w["ay"], w["az"], ho=False))]
    else:
        b = [w["b0"][d] + 0.1 * np.cos(2 * np.pi * (d + 1) * np.arange(n[0]) / n[0]) * np.ones(w["rho"].shape) for d in range(3)]
    args = [w[k] for k in ("rho", "vx", "vy", "vz", "p")] + b
    kw = dict(uct=uct, ho=False, rec=2)
    o = Oracle(*n, G, 0.3, rk=2, **kw)
    o.set_primitives(*args)
    a = Oracle(*n, G, 0.3, rk=3, **kw)               # same operator; only used for rhs() and the state
    a.set_primitives(*args)
    u0, r0 = _conserved(a), a.rhs()
    hmin = min(1.0 / m for m in n)
    dt = 0.3 * hmin / r0["amax"]
    L0 = list(r0["rhsU"]) + list(r0["rhsB"])
    u1 = [x + dt * y for x, y in zip(u0, L0)]
    if uct:
        bc1 = Oracle(*n, G, 0.3, **kw)
        bc1.set_primitives(*args[:5], *u1[5:])       # only to centre the staggered B of U1 (INT, second order)
        q = bc1.get_primitives()
        Bc = [q["bx"], q["by"], q["bz"]]
    else:
        Bc = u1[5:]
    p1 = ob.con2prim(G, *[x.ravel() for x in u1[:5]], *[x.ravel() for x in Bc])
    b1 = Oracle(*n, G, 0.3, **kw)
    b1.set_primitives(*[p1[k].reshape(w["rho"].shape) for k in ("rho", "vx", "vy", "vz", "p")], *u1[5:])
    r1 = b1.rhs()
    L1 = list(r1["rhsU"]) + list(r1["rhsB"])
    expect = [0.5 * x0 + 0.5 * (x1 + dt * y) for x0, x1, y in zip(u0, u1, L1)]
    assert o.step(1) == 1
    got = _conserved(o)
    assert o.diagnostics()["t"] == pytest.approx(dt, rel=1e-14)
    for k, (g_, e_) in enumerate(zip(got, expect)):
        assert np.abs(g_ - e_).max() <= 2e-11 * max(1.0, np.abs(e_).max()), k


def _wave_error(n, cfl, **kw):
    w = inputs.cpa_wave(n, 1, 1, direction="x")
    o = Oracle(n, 1, 1, G, cfl, **kw)
    bk = ("bxf", "byf", "bzf") if kw.get("uct", True) else ("bx", "by", "bz")
    o.set_primitives(w["rho"], w["vx"], w["vy"], w["vz"], w["p"], *[w[k] for k in bk])
    d0 = o.diagnostics()
    o.step(10 ** 9, w["T"])
    d1 = o.diagnostics()
    assert d1["t"] == w["T"]
    for k in ("sum_D", "sum_Sx", "sum_Sy", "sum_Sz", "sum_U", "sum_By", "sum_Bz"):
        assert abs(d1[k] - d0[k]) <= 1e-12 * max(abs(d0[k]), 1.0), k      # eq.(9): conservation form
    q = o.get_primitives()
    return {k: float(np.abs(q[k] - w[k]).mean()) for k in ("vy", "vz", "by", "bz")}


def test_rk2_is_second_order_in_dt():
    """MP5 + HO at n = 64 leaves a spatial error far below the temporal one, so halving the Courant number must
    divide the one-period error of the RK2 run by 4; the RK3 run with the same operator sits well below it."""
    e2a, e2b = _wave_error(64, 0.6, rk=2), _wave_error(64, 0.3, rk=2)
    e3b = _wave_error(64, 0.3, rk=3)
    for k in e2a:
        assert 1.85 < math.log2(e2a[k] / e2b[k]) < 2.15, (k, e2a[k], e2b[k])
        assert e3b[k] < 0.2 * e2b[k]                              # the third-order scheme is well below it


@pytest.mark.parametrize("uct", [True, False])
def test_linear_rk2_variant_is_second_order_on_the_exact_wave(uct):
    """The whole second-order variant (linear REC, second-order INT/DER, RK2) on one period of the x-aligned CPA wave
    (P:L229-233): L1 error falls by about 4 per doubling (the limiter clips the extrema, so a little less)."""
    kw = dict(uct=uct, ho=False, rec=2, rk=2)
    a, b = _wave_error(64, 0.3, **kw), _wave_error(128, 0.3, **kw)
    mp5 = _wave_error(64, 0.3, uct=uct, ho=False)                 # MP5 with the same second-order INT/DER
    for k in a:
        assert 1.6 < math.log2(a[k] / b[k]) < 2.3, (k, a[k], b[k])
        assert a[k] > mp5[k]                                      # linear REC is the more diffusive one
