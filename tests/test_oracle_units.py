"""Pins for the point/stencil routines of the CPU oracle (no GPU).

Each test checks the oracle against something other than itself: a closed form, polynomial
exactness that fixes the stencil coefficients, a textbook special case, an identity between
two different routines, or a library routine (numpy polyfit / numpy.linalg).
"""
import math

import numpy as np
import pytest

from oracle import binding as ob
from paper_2401_03008_b200 import inputs

G = 4.0 / 3.0


# ----------------------------------------------------------------------------- O1 INT
@pytest.mark.parametrize("m", range(6))
def test_int6_exact_for_degree_le_5(m):
    h, xc = 0.37, 0.81
    faces = xc + h * (np.arange(6) - 2.5)            # i-5/2 .. i+5/2
    got = ob.int6(faces ** m)
    assert got == pytest.approx(xc ** m, rel=0, abs=2e-14)


def test_int6_is_sixth_order_not_more():
    # 6-point Lagrange remainder at the midpoint: f^(6)(xi)/6! * prod(x - x_j) = -(225/64) h^6 / 720 * 720 ...
    # for f = x^6 the error is exactly -prod_j (xc - x_j) = -(0.5*1.5*2.5)^2 h^6 (sign: interp - exact)
    h, xc = 0.1, 0.3
    faces = xc + h * (np.arange(6) - 2.5)
    err = ob.int6(faces ** 6) - xc ** 6
    assert err == pytest.approx((0.5 * 1.5 * 2.5) ** 2 * h ** 6, rel=1e-6)


# ----------------------------------------------------------------------------- O6 DER
@pytest.mark.parametrize("m", range(7))
def test_der5_difference_reproduces_derivative_up_to_degree_6(m):
    h, xc = 0.23, 0.4
    # faces i-5/2 .. i+5/2 ; F^_{i+1/2} uses faces[1:6], F^_{i-1/2} uses faces[0:5]
    faces = xc + h * (np.arange(6) - 2.5)
    F = faces ** m
    d = (ob.der5(F[1:6]) - ob.der5(F[0:5])) / h
    exact = m * xc ** (m - 1) if m > 0 else 0.0
    assert d == pytest.approx(exact, rel=0, abs=5e-14)


def test_der5_fails_at_degree_7_and_weights_sum_to_one():
    h, xc = 0.23, 0.4
    faces = xc + h * (np.arange(6) - 2.5)
    F = faces ** 7
    d = (ob.der5(F[1:6]) - ob.der5(F[0:5])) / h
    assert abs(d - 7 * xc ** 6) > 1e-6          # 6th order, not 8th
    assert ob.der5(np.ones(5)) == pytest.approx(1.0, abs=1e-15)   # constants pass unchanged
    # symmetric stencil
    v = np.array([0.3, -1.2, 0.7, 2.0, 0.1])
    assert ob.der5(v) == pytest.approx(ob.der5(v[::-1]), abs=1e-15)


# ----------------------------------------------------------------------------- O3 MP5
def test_mp5_smooth_equals_quartic_interpolation():
    # on smooth data MP5 returns the 5-point Lagrange interpolant at i+1/2: compare with numpy polyfit
    rng = np.random.default_rng(1)
    for _ in range(50):
        c = rng.normal(size=5)
        x = np.arange(-2, 3) * 0.01 + 0.2
        v = np.polyval(c, x)
        want = np.polyval(np.polyfit(x, v, 4), x[2] + 0.005)
        assert ob.mp5(v) == pytest.approx(want, rel=0, abs=1e-12 * max(1, abs(want)))


def test_mp5_exact_for_quartics_is_point_value_not_cell_average():
    # point-value weights (3,-20,90,60,-5)/128: exact for x^4 point values (S1/O3);
    # the cell-average weights (2,-13,47,27,-3)/60 would give a different number
    x = 1.0 + 0.05 * np.arange(-2, 3, dtype=float)      # resolved, monotone: the limiter stays off
    for m in range(5):
        assert ob.mp5(x ** m) == pytest.approx(1.025 ** m, abs=1e-14)
    v = x ** 2
    avg = np.dot([2, -13, 47, 27, -3], v) / 60.0
    assert abs(ob.mp5(v) - avg) > 1e-4                  # differs by h^2/12 f'' = 0.05^2/6


def test_mp5_limiter_invariants():
    rng = np.random.default_rng(2)
    # step: no new extrema at the face next to a discontinuity
    for v in ([0, 0, 0, 1, 1], [0, 0, 1, 1, 1], [1, 1, 1, 0, 0], [1, 1, 0, 0, 0], [0, 0, 1, 0, 0]):
        r = ob.mp5(np.array(v, float))
        assert min(v[2], v[3]) - 1e-14 <= r <= max(v[2], v[3]) + 1e-14
    # monotone data: the face value stays between its two neighbours (monotonicity preserving)
    for _ in range(2000):
        v = np.cumsum(rng.uniform(0, 1, 5) ** 4) * rng.choice([-1.0, 1.0])
        r = ob.mp5(v)
        # the absolute switch eps = 1e-10 (S2) lets the unlimited value through while
        # (vor-v0)(vor-vmp) <= eps, i.e. overshoots are bounded by sqrt(eps)
        assert min(v[2], v[3]) - 1e-5 <= r <= max(v[2], v[3]) + 1e-5
    for _ in range(2000):                                  # well above the switch: strict bounds
        v = np.cumsum(rng.uniform(0.02, 1, 5)) * rng.choice([-1.0, 1.0])
        r = ob.mp5(v)
        assert min(v[2], v[3]) - 1e-12 <= r <= max(v[2], v[3]) + 1e-12 or \
            abs((r - v[2]) * (r - (v[2] + (v[3] - v[2])))) <= 1e-10
    # odd symmetry and (for large data, where the absolute eps does not matter) positive scaling
    for _ in range(500):
        v = rng.normal(size=5) * 10.0
        assert ob.mp5(-v) == pytest.approx(-ob.mp5(v), abs=1e-13)
    # constant shift
    for _ in range(200):
        v = rng.normal(size=5)
        assert ob.mp5(v + 3.0) == pytest.approx(ob.mp5(v) + 3.0, abs=1e-9)


def test_mp5_median_bound_is_the_linear_extrapolation_from_the_right():
    """The constant 1/2 of v^MD (O3).  v^MD = v^AV - d^M4/2 is Suresh & Huynh's median of v_i, v_{i+1} and the value
    extrapolated linearly to the face from the right, v^FR = v_{i+1} + (v_{i+1} - v_{i+2})/2: with d^M4 = d_{i+1} the
    two are the same number, (v_i + v_{i+1})/2 - (v_i - 2 v_{i+1} + v_{i+2})/2 = v^FR.  On the stencils below the
    unlimited value lies beyond that bound, d^M4_{i+1/2} = d_{i+1} and the other bound (v^UL, v^LC) is wider, so MP5
    must return v^FR exactly; with 1 or 1/4 in place of 1/2 it returns something else by more than 0.02."""
    cases = [[-1.8, 1.56, 0.87, 0.79, 0.93], [1.59, -1.65, -1.59, -0.69, 0.63],
             [-1.94, 1.22, 0.44, 0.45, 0.73], [1.98, -1.43, -0.23, -0.04, -0.21]]
    for v in cases:
        v = np.array(v)
        fr = v[3] + 0.5 * (v[3] - v[4])
        vor = np.dot([3, -20, 90, 60, -5], v) / 128.0
        dj, dj1 = v[1] - 2 * v[2] + v[3], v[2] - 2 * v[3] + v[4]
        # the premises, from the data alone: d_{i+1} is the minmod of (4 d_i - d_{i+1}, 4 d_{i+1} - d_i, d_i, d_{i+1})
        four = np.array([4 * dj - dj1, 4 * dj1 - dj, dj, dj1])
        assert (np.sign(four) == np.sign(dj1)).all() and np.abs(four).min() == abs(dj1)
        assert abs(vor - fr) > 0.05                       # the unlimited value is somewhere else
        for sgn in (1.0, -1.0):                           # and the odd image
            assert ob.mp5(sgn * v) == pytest.approx(sgn * fr, abs=2e-15)
        vav = 0.5 * (v[2] + v[3])
        assert min(abs(vav - 1.0 * dj1 - fr), abs(vav - 0.25 * dj1 - fr)) > 0.02


def test_mp5_clips_overshoot_of_the_linear_scheme():
    # data with a kink where the unlimited quartic overshoots: the limited value must differ from it
    v = np.array([0.0, 0.0, 0.0, 1.0, 2.0])
    vor = np.dot([3, -20, 90, 60, -5], v) / 128.0
    r = ob.mp5(v)
    assert 0.0 <= r <= 1.0
    assert vor == pytest.approx(50.0 / 128.0)
    v = np.array([1.0, 1.0, 1.0, 0.0, 5.0])     # vor = (3-20+90-25)/128 = 0.375, inside -> kept or limited within
    r = ob.mp5(v)
    assert 0.0 <= r <= 1.0


# ----------------------------------------------------------------------------- O4 speeds
def _state(rho, v, p, B):
    return np.array([rho, v[0], v[1], v[2], p, B[0], B[1], B[2]], float)


def test_fast_speeds_static_unmagnetised_is_sound_speed():
    rho, p = 1.3, 0.7
    cs = math.sqrt(G * p / (rho + G / (G - 1) * p))
    for d in range(3):
        lam = ob.fast_speeds(G, _state(rho, (0, 0, 0), p, (0, 0, 0)), d)
        assert lam[0] == pytest.approx(cs, rel=1e-15)
        assert lam[1] == pytest.approx(-cs, rel=1e-15)


def test_fast_speeds_aligned_flow_is_relativistic_velocity_addition():
    rho, p = 0.8, 2.0
    cs = math.sqrt(G * p / (rho + G / (G - 1) * p))
    for d in range(3):
        for vd in (-0.9, -0.3, 0.2, 0.85):
            v = [0.0, 0.0, 0.0]
            v[d] = vd
            lam = ob.fast_speeds(G, _state(rho, v, p, (0, 0, 0)), d)
            assert lam[0] == pytest.approx((vd + cs) / (1 + vd * cs), rel=1e-13)
            assert lam[1] == pytest.approx((vd - cs) / (1 - vd * cs), rel=1e-13)


def test_fast_speeds_static_perpendicular_field_is_exact_magnetosonic():
    # v = 0, B perpendicular to d: exact fast speed a^2 = cs^2 + ca^2 - cs^2 ca^2, ca^2 = B^2/(rho h + B^2)
    rho, p, B = 1.0, 0.5, 1.7
    rhoh = rho + G / (G - 1) * p
    cs2, ca2 = G * p / rhoh, B * B / (rhoh + B * B)
    a = math.sqrt(cs2 + ca2 - cs2 * ca2)
    lam = ob.fast_speeds(G, _state(rho, (0, 0, 0), p, (0, B, 0)), 0)
    assert lam[0] == pytest.approx(a, rel=1e-14) and lam[1] == pytest.approx(-a, rel=1e-14)
    # parallel field: the approximation is an upper bound of the exact fast speed max(cs, ca)
    lam = ob.fast_speeds(G, _state(rho, (0, 0, 0), p, (B, 0, 0)), 0)
    assert lam[0] >= max(math.sqrt(cs2), math.sqrt(ca2)) - 1e-15
    assert lam[0] < 1.0


def test_fast_speeds_are_subluminal_and_ordered_on_random_states():
    s = inputs.random_states(2000, seed=5)
    for i in range(2000):
        q = _state(s["rho"][i], (s["vx"][i], s["vy"][i], s["vz"][i]), s["p"][i], (s["bx"][i], s["by"][i], s["bz"][i]))
        for d in range(3):
            lp, lm = ob.fast_speeds(G, q, d)
            assert -1.0 < lm <= q[1 + d] <= lp < 1.0


def test_cpa_state_amax_matches_the_value_implied_by_the_paper_tables(golden_dir):
    # P2: steps per period = T_diag * N * amax / cfl must fall inside what Tables 1-2 print
    from conftest import read_golden_table
    rows = read_golden_table(golden_dir + "/paper_tables_1_2.txt")
    w = inputs.cpa_wave(1, 1, 1)
    amax = 0.0
    for ph in np.linspace(0, 2 * math.pi, 721):
        X, Y, Z, _ = inputs._cpa_frame("diag")
        dB = math.cos(ph) * Y + math.sin(ph) * Z
        q = _state(1.0, -w["vA"] * dB, 1.0, X + dB)
        for d in range(3):
            lp, lm = ob.fast_speeds(G, q, d)
            amax = max(amax, lp, -lm)
    assert amax == pytest.approx(0.81327, abs=2e-5)
    ratios = []
    for N, nodes, wt_no, sp_no, wt_yes, sp_yes in rows:
        steps = w["T"] * N * amax / 0.3
        for wt, sp in ((wt_no, sp_no), (wt_yes, sp_yes)):
            # printed speed has 2 decimals and W-time includes start-up: allow the rounding + 1 %
            lo, hi = wt * (sp - 0.005) * 0.99, wt * (sp + 0.005) * 1.01
            assert lo <= steps <= hi, (N, nodes, steps, lo, hi)
            ratios.append(wt * sp / steps)
    # on average the rule dt = 0.3 h / amax reproduces the printed step counts to 0.5 %;
    # a sum-over-directions rule (3x smaller dt) or cfl = 0.4 / 0.25 would not
    assert np.mean(ratios) == pytest.approx(1.0, abs=5e-3)


# ----------------------------------------------------------------------------- prim2cons / flux
def _covariant(q):
    """Textbook covariant RMHD: T^{mu nu} = (rho h + b^2) u^mu u^nu + (p + b^2/2) eta^{mu nu} - b^mu b^nu."""
    rho, v, p, B = q[0], q[1:4], q[4], q[5:8]
    W = 1 / math.sqrt(1 - v @ v)
    u = np.concatenate([[W], W * v])
    b0 = W * (v @ B)
    b = np.concatenate([[b0], B / W + b0 * v])
    b2 = -b[0] ** 2 + b[1:] @ b[1:]
    eta = np.diag([-1.0, 1, 1, 1])
    rhoh = rho + G / (G - 1) * p
    T = (rhoh + b2) * np.outer(u, u) + (p + b2 / 2) * eta - np.outer(b, b)
    return rho * u, T


def test_prim2cons_and_flux_match_covariant_stress_energy_tensor():
    s = inputs.random_states(300, seed=3, wmax=5.0)
    for i in range(300):
        q = _state(s["rho"][i], (s["vx"][i], s["vy"][i], s["vz"][i]), s["p"][i], (s["bx"][i], s["by"][i], s["bz"][i]))
        J, T = _covariant(q)
        c = ob.prim2cons(G, *[np.array([x]) for x in q])
        scale = abs(T[0, 0])
        assert c["D"][0] == pytest.approx(J[0], rel=1e-13)
        assert c["U"][0] == pytest.approx(T[0, 0], rel=1e-12)
        for a, k in enumerate(("Sx", "Sy", "Sz")):
            assert c[k][0] == pytest.approx(T[0, 1 + a], abs=1e-12 * scale)
        for d in range(3):
            F = ob.phys_flux(G, q, d)
            assert F[0] == pytest.approx(J[1 + d], abs=1e-13 * abs(J[0]))
            for a in range(3):
                assert F[1 + a] == pytest.approx(T[1 + a, 1 + d], abs=1e-12 * scale)
            assert F[4] == pytest.approx(T[0, 1 + d], abs=1e-12 * scale)     # energy flux = momentum density


def test_prim2cons_static_textbook_values():
    c = ob.prim2cons(G, *[np.array([x]) for x in (2.0, 0, 0, 0, 0.5, 0.3, -0.4, 1.2)])
    B2 = 0.09 + 0.16 + 1.44
    assert c["D"][0] == 2.0
    assert c["Sx"][0] == 0 and c["Sy"][0] == 0 and c["Sz"][0] == 0
    assert c["U"][0] == pytest.approx(2.0 + 3 * 0.5 + B2 / 2, rel=1e-15)      # rho + p/(g-1) + B^2/2
    F = ob.phys_flux(G, _state(2.0, (0, 0, 0), 0.5, (0.3, -0.4, 1.2)), 0)
    assert F[0] == 0 and F[4] == 0
    assert F[1] == pytest.approx(0.5 + B2 / 2 - 0.09, rel=1e-15)             # Maxwell stress
    assert F[2] == pytest.approx(0.3 * 0.4, rel=1e-15)
    assert F[3] == pytest.approx(-0.3 * 1.2, rel=1e-15)


# ----------------------------------------------------------------------------- O5 HLL
def test_hll_consistency_and_upwinding():
    s = inputs.random_states(100, seed=9, wmax=3.0, sigma_max=1.0)
    for i in range(100):
        q = _state(s["rho"][i], (s["vx"][i], s["vy"][i], s["vz"][i]), s["p"][i], (s["bx"][i], s["by"][i], s["bz"][i]))
        for d in range(3):
            F, ex = ob.hll(G, q, q, d)
            np.testing.assert_allclose(F, ob.phys_flux(G, q, d), rtol=1e-12, atol=1e-12 * abs(F).max())
            lp, lm = ob.fast_speeds(G, q, d)
            assert ex[0] == max(0.0, lp) and ex[1] == max(0.0, -lm)
            assert ex[2] == pytest.approx(q[1 + (d + 1) % 3], abs=1e-14)
            assert ex[3] == pytest.approx(q[1 + (d + 2) % 3], abs=1e-14)
    # supersonic to the right: a- = 0 and the flux is the left flux
    qL = _state(1.0, (0.95, 0.0, 0.0), 0.01, (0.0, 0.0, 0.0))
    qR = _state(0.5, (0.96, 0.0, 0.0), 0.02, (0.0, 0.0, 0.0))
    F, ex = ob.hll(G, qL, qR, 0)
    assert ex[1] == 0.0
    np.testing.assert_allclose(F, ob.phys_flux(G, qL, 0), rtol=1e-14)


def test_hll_contact_at_rest_diffuses_mass_downhill_and_vbar_weights():
    qL = _state(2.0, (0.0, 0.1, -0.2), 1.0, (0, 0, 0))
    qR = _state(1.0, (0.0, 0.3, 0.4), 1.0, (0, 0, 0))
    F, ex = ob.hll(G, qL, qR, 0)
    assert F[0] > 0            # -a+a-(D_R - D_L)/(a+ + a-) with D_L > D_R
    ap, am = ex[0], ex[1]
    assert ex[2] == pytest.approx((ap * 0.1 + am * 0.3) / (ap + am), rel=1e-14)      # v_y (t1 of x)
    assert ex[3] == pytest.approx((ap * -0.2 + am * 0.4) / (ap + am), rel=1e-14)     # v_z (t2 of x)
    # cyclic slots: for d = 1 the transverse components are (z, x)
    qL = _state(1.0, (0.1, 0.0, -0.2), 1.0, (0, 0, 0))
    qR = _state(1.0, (0.3, 0.0, 0.4), 1.0, (0, 0, 0))
    F, ex = ob.hll(G, qL, qR, 1)
    assert ex[2] == pytest.approx(0.1, abs=1e-15)       # v_z: (a+ * -0.2 + a- * 0.4)/(a+ + a-) with a+ = a-
    assert ex[3] == pytest.approx(0.2, abs=1e-15)       # v_x


# ----------------------------------------------------------------------------- O2 con2prim
def test_con2prim_hydro_static_closed_form():
    r = ob.con2prim(G, [1.5], [0], [0], [0], [1.5 + 0.9 / (G - 1)], [0], [0], [0])
    assert r["rc"] == 0
    assert r["rho"][0] == pytest.approx(1.5, rel=1e-14)
    assert r["p"][0] == pytest.approx(0.9, rel=1e-13)
    assert r["vx"][0] == 0 and r["vy"][0] == 0 and r["vz"][0] == 0


def test_con2prim_round_trip_P6():
    """BJ north_star: prim->cons->prim <= 1e-12 relative up to W = 10, sigma = 10.

    Acceptance as derived in SURVEY 8(c) "conditioning caveat": rho, v, W <= 1e-12 on every sample;
    p <= 1e-12 at the 99.9th percentile and |dp| <= 5e-15 U everywhere (p is a difference of O(U) terms).
    """
    n = 200000
    s = inputs.random_states(n, seed=12345)
    c = ob.prim2cons(G, s["rho"], s["vx"], s["vy"], s["vz"], s["p"], s["bx"], s["by"], s["bz"])
    r = ob.con2prim(G, c["D"], c["Sx"], c["Sy"], c["Sz"], c["U"], s["bx"], s["by"], s["bz"])
    assert r["rc"] == 0 and (r["iters"] > 0).all()
    assert r["iters"].max() <= 12
    vmod = np.sqrt(s["vx"] ** 2 + s["vy"] ** 2 + s["vz"] ** 2)
    dv = np.sqrt((r["vx"] - s["vx"]) ** 2 + (r["vy"] - s["vy"]) ** 2 + (r["vz"] - s["vz"]) ** 2)
    W2 = 1 / np.sqrt(1 - (r["vx"] ** 2 + r["vy"] ** 2 + r["vz"] ** 2))
    assert (np.abs(r["rho"] / s["rho"] - 1)).max() <= 1e-12
    assert (dv / np.maximum(vmod, 1e-300)).max() <= 1e-12 or dv.max() <= 1e-13
    assert (np.abs(W2 / s["W"] - 1)).max() <= 1e-12
    ep = np.abs(r["p"] / s["p"] - 1)
    assert np.quantile(ep, 0.999) <= 1e-12
    assert (np.abs(r["p"] - s["p"]) / c["U"]).max() <= 5e-15
    # moderate regime of all evolution configs: every variable tight
    m = (s["W"] <= 3) & (s["sigma"] <= 1)
    assert ep[m].max() <= 1e-12


def test_con2prim_safeguard_branch_reaches_the_same_root():
    """The safeguard of O2 (an iterate with y <= 0 or x(y) outside [0, 1) is replaced by the midpoint with the last
    valid one).  No state of BJ's P6 range (W <= 10) enters it, but physical states do: for cold ultra-relativistic
    flows (W = 20..40, p/rho = 1e-6..1e-2) the first Newton step from the upper bound y0 overshoots below the root
    into x(y) >= 1 for most samples (the instrumented count `nsafe` says which).  What the branch must deliver is
    fixed by the mathematics, not by the rule: the root is unique, so the primitives must still be the ones the
    conserved state was built from, to the conditioning of the problem (relative error ~ eps W^2)."""
    n = 20000
    s = inputs.random_states(n, seed=777, wmin=20.0, wmax=40.0, log_p_over_rho=(-6.0, -2.0))
    assert s["W"].min() >= 20.0 - 1e-9 and s["W"].max() <= 40.0 + 1e-9
    c = ob.prim2cons(G, s["rho"], s["vx"], s["vy"], s["vz"], s["p"], s["bx"], s["by"], s["bz"])
    r = ob.con2prim_trace(G, c["D"], c["Sx"], c["Sy"], c["Sz"], c["U"], s["bx"], s["by"], s["bz"])
    hit = r["nsafe"] > 0
    assert hit.mean() > 0.5, hit.mean()                    # the branch is what this sample exercises
    assert r["rc"] == 0 and (r["iters"] > 0).all() and r["iters"].max() <= 20
    assert (r["iters"][hit] >= 3).all()                    # at least: failed step, midpoint, converging step
    W2 = 1 / np.sqrt(1 - (r["vx"] ** 2 + r["vy"] ** 2 + r["vz"] ** 2))
    eps_w2 = 2.2e-16 * s["W"] ** 2
    assert (np.abs(r["rho"] / s["rho"] - 1) <= 60 * eps_w2).all()
    assert (np.abs(W2 / s["W"] - 1) <= 60 * eps_w2).all()
    dv = np.sqrt((r["vx"] - s["vx"]) ** 2 + (r["vy"] - s["vy"]) ** 2 + (r["vz"] - s["vz"]) ** 2)
    assert dv.max() <= 1e-13
    assert (np.abs(r["p"] - s["p"]) <= 5e-15 * c["U"]).all()
    # same accuracy whether or not the safeguard was used: it only changes the path to the root
    e = np.abs(r["rho"] / s["rho"] - 1) / eps_w2
    assert np.median(e[hit]) < 10 * max(np.median(e[~hit]), 0.05)
    # and the plain entry point returns the same numbers (the instrumentation changes nothing)
    r0 = ob.con2prim(G, c["D"], c["Sx"], c["Sy"], c["Sz"], c["U"], s["bx"], s["by"], s["bz"])
    assert np.array_equal(r0["iters"], r["iters"]) and np.array_equal(r0["rho"], r["rho"]) and np.array_equal(r0["p"], r["p"])
    # in BJ's own range the branch is never entered (so parity there never depended on it)
    s6 = inputs.random_states(100000, seed=12345)
    c6 = ob.prim2cons(G, s6["rho"], s6["vx"], s6["vy"], s6["vz"], s6["p"], s6["bx"], s6["by"], s6["bz"])
    r6 = ob.con2prim_trace(G, c6["D"], c6["Sx"], c6["Sy"], c6["Sz"], c6["U"], s6["bx"], s6["by"], s6["bz"])
    assert r6["rc"] == 0 and r6["nsafe"].max() == 0


def test_con2prim_flags_unphysical_input():
    r = ob.con2prim(G, [1.0], [0], [0], [0], [-1.0], [0], [0], [0])
    assert r["rc"] != 0 and r["iters"][0] < 0 and np.isnan(r["rho"][0])


def test_alfven_speed_closed_form_and_limits(golden_dir):
    from conftest import read_golden_table
    rhoh, vA, W, Td, Tx = read_golden_table(golden_dir + "/cpa_paper_values.txt")[0]
    assert (3 - math.sqrt(5)) / 2 == pytest.approx(vA, rel=1e-15)
    assert inputs.alfven_speed() == pytest.approx(vA, rel=1e-14)
    assert inputs.cpa_period("diag") == pytest.approx(Td, rel=1e-14)
    assert inputs.cpa_period("x") == pytest.approx(Tx, rel=1e-14)
    # P9: eta -> 0 gives vA^2 = B0^2/(rho h + B0^2)
    assert inputs.alfven_speed(eta=1e-8) ** 2 == pytest.approx(1.0 / 6.0, rel=1e-12)
