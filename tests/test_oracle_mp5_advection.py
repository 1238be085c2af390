"""Pins of the oracle's MP5 limiter (O3: "holib_rec ... MP5") on NON-SMOOTH data, from what the
limiter is for rather than from its formula: used as the upwind interface value of the linear advection equation
u_t + u_x = 0 (forward differences of the interface values, SSP-RK3, Courant number 1/(1 + alpha) = 0.2, the bound of
Suresh & Huynh's monotonicity proof), it must

  (a) keep a square pulse and a triangle inside their initial range and create no oscillations (total variation
      stays below that of the data), up to the sqrt(eps) = 1e-5 the absolute switch eps = 1e-10 (S2) lets through;
  (b) leave a resolved smooth profile WITH extrema exactly as the unlimited fifth-order scheme leaves it
      (accuracy-preserving at extrema: the whole point of MP5 over a TVD limiter), bit for bit;
  (c) on steep convex monotone data let the face value rise to v_j + alpha (v_j - v_{j-1}) and no further
      (the defining MP bound, alpha = 4).

Checked beforehand against deliberately broken limiters (a scratch re-implementation that is not part of the
repository): (a) fails when the two curvature measures d^{M4}_{j+1/2}, d^{M4}_{j-1/2} are interchanged or when the
two brackets are united instead of intersected; (b) fails when v^MD or v^LC is dropped, has the wrong sign, or
when the factor 4/3 is 1/3 or the 4 inside d^{M4} is 1; (c) fails for alpha != 4.  NOT distinguished by any of them
(and by nothing the paper prints): the published design constants 1/2 in v^MD, 4/3 in v^LC and 4 in d^{M4} against
nearby values (1, 3/4, 2): that part of the limiter stays "parity unpinned" (oracle header)."""
import numpy as np

from oracle import binding as ob

NU = 0.2          # 1 / (1 + alpha), alpha = 4


def _unlimited(v):
    return (3.0 * v[0] - 20.0 * v[1] + 90.0 * v[2] + 60.0 * v[3] - 5.0 * v[4]) / 128.0


def _advect(rec, u0, steps):
    n = len(u0)
    idx = (np.arange(n)[:, None] + np.arange(-2, 3)[None, :]) % n

    def L(u):
        f = np.array([rec(s) for s in u[idx]])
        return -(f - np.roll(f, 1))

    u = u0.copy()
    for _ in range(steps):
        u1 = u + NU * L(u)
        u2 = 0.75 * u + 0.25 * (u1 + NU * L(u1))
        u = u / 3.0 + 2.0 / 3.0 * (u2 + NU * L(u2))
    return u


def _tv(u):
    return float(np.abs(u - np.roll(u, 1)).sum())


def test_mp5_advection_of_a_pulse_and_a_triangle_stays_monotone():
    n = 80
    x = (np.arange(n) + 0.5) / n
    u0 = np.where((x > 0.25) & (x < 0.5), 1.0, 0.0) + np.where((x > 0.6) & (x < 0.9), 1.0 - np.abs(x - 0.75) / 0.15, 0.0)
    u = _advect(ob.mp5, u0, 200)                              # half a box length
    assert u.min() >= -1e-5 and u.max() <= 1.0 + 1e-5
    assert _tv(u) <= _tv(u0) + 1e-4
    assert abs(u.sum() - u0.sum()) <= 1e-12 * n              # flux form: conservative
    # the unlimited scheme on the same data oscillates visibly: the bounds above are the limiter's doing
    w = _advect(_unlimited, u0, 200)
    assert w.min() < -0.02 and w.max() > 1.02 and _tv(w) > _tv(u0) + 0.1
    # and the pulse is still a pulse (not smeared away by an over-restrictive limiter)
    assert u.max() > 0.99 and _tv(u) > 3.7


def test_mp5_is_transparent_on_resolved_smooth_extrema():
    n = 80
    x = (np.arange(n) + 0.5) / n
    u0 = np.sin(2.0 * np.pi * x) + 0.5 * np.sin(4.0 * np.pi * x + 1.0)
    a = _advect(ob.mp5, u0, 100)
    b = _advect(_unlimited, u0, 100)
    assert np.abs(a - b).max() <= 1e-13
    # the S&H test does fire on these data (around the extrema), so the limiter proper was exercised
    idx = (np.arange(n)[:, None] + np.arange(-2, 3)[None, :]) % n
    fired = 0
    for s in u0[idx]:
        vor = _unlimited(s)
        da, db = s[3] - s[2], 4.0 * (s[2] - s[1])
        mm = 0.0 if da * db <= 0.0 else (da if abs(da) < abs(db) else db)
        fired += (vor - s[2]) * (vor - s[2] - mm) > 1e-10
    assert fired >= 4


def test_mp5_bound_on_steep_convex_data_is_v_plus_alpha_times_the_backward_difference():
    # v_j - v_{j-1} = 1, then a jump: the unlimited value 8.53 exceeds v_j + 4 = 5; the curvature brackets do not bind
    assert ob.mp5(np.array([-1.0, 0.0, 1.0, 20.0, 39.0])) == 5.0
    assert ob.mp5(np.array([1.0, 0.0, -1.0, -20.0, -39.0])) == -5.0
    assert ob.mp5(np.array([-2.0, 0.0, 2.0, 40.0, 78.0]) + 3.0) == 13.0
    # inside the bound nothing is changed: unlimited value 4.625 < 5
    assert ob.mp5(np.array([-1.0, 0.0, 1.0, 10.0, 19.0])) == 4.625
