"""Pins for the non-periodic boundaries of the oracle ("next" row f4, first slice).

Reflecting wall: a periodic box of 2n cells along an axis with data that is mirror-symmetric about the planes at 0
and at n stays mirror-symmetric (the reflection covariance of the scheme, P7iv), so its half 0 <= c < n is the
solution of the wall-bounded problem on n cells.  The bounded oracle run (ghost layers refilled by the mirror rule
before every L(U)) must reproduce that half to round-off: this fixes the ghost index map, the face staggering of the
normal B (wall faces are evolved, not filled) and the parity of every field (a wrong sign or an off-by-one changes
the result at O(1)).  Outflow: while a compact pulse has not reached the boundary the zero-gradient ghost layers hold
the same uniform background as the periodic images, so the two runs agree to the last bit."""
import numpy as np
import pytest

from oracle import binding as ob
from oracle.binding import Oracle
from paper_2401_03008_b200 import inputs

G = 4.0 / 3.0
PRIMS = "rho vx vy vz p bx by bz".split()
SETK = "rho vx vy vz p bxf byf bzf".split()
NG = 8


def _symmetric_box(shape, axis):
    """Multi-mode config-5 field on `shape` (nx, ny, nz), made mirror-symmetric about the plane x_axis = 0 (and,
    by periodicity, about the middle of the box): q_sym = (q + R q)/2 with R the reflection of P7iv."""
    from test_oracle_scheme import _mirror, _turb
    tb, bf = _turb(shape)
    f = [tb["rho"], tb["vx"], tb["vy"], tb["vz"], tb["p"]] + bf
    sv = [(-1.0 if c == axis else 1.0) for c in range(3)]
    sb = [-sv[c] for c in range(3)]                       # axial vector, one reflected axis
    m = [_mirror(f[0], (axis,))] + [sv[c] * _mirror(f[1 + c], (axis,)) for c in range(3)] + [_mirror(f[4], (axis,))] + \
        [sb[c] * _mirror(f[5 + c], (axis,), stag=c) for c in range(3)]
    return [0.5 * (a + b) for a, b in zip(f, m)]


def _pad(a, axis, lo, n):
    """Cells lo-8 .. lo+n+8 (periodic) of a along grid axis `axis`."""
    ax = 2 - axis
    idx = (np.arange(-NG, n + NG) + lo) % a.shape[ax]
    return np.ascontiguousarray(np.take(a, idx, axis=ax))


@pytest.mark.parametrize("axis", [0, 1, 2])
def test_reflecting_walls_equal_the_mirror_symmetric_periodic_run(axis):
    full = [24, 12, 10]
    full[axis] = 32                                       # 2n = 32 cells along the reflected axis
    n = 16
    f = _symmetric_box(tuple(full), axis)
    o = Oracle(*full, G, 0.3)
    o.set_primitives(*f)
    half = list(full)
    half[axis] = n
    kinds = [0] * 6
    kinds[2 * axis] = kinds[2 * axis + 1] = 1
    b = Oracle(*half, G, 0.3, boundaries=kinds, gn=full)      # the same spacing as the periodic box
    fp = [_pad(a, axis, 0, n) for a in f]
    # ghost entries are the library's business: poison them, except the low wall face of the normal B
    sl = [slice(None)] * 3
    for k, a in enumerate(fp):
        keep = a.copy()
        sl_lo, sl_hi = list(sl), list(sl)
        sl_lo[2 - axis] = slice(0, NG)
        sl_hi[2 - axis] = slice(NG + n, None)
        a[tuple(sl_lo)] = 1e30
        a[tuple(sl_hi)] = 1e30
        if k == 5 + axis:
            w = list(sl)
            w[2 - axis] = NG - 1
            a[tuple(w)] = keep[tuple(w)]
    b.set_primitives(*fp)
    assert o.step(4) == 4 and b.step(4) == 4
    do, db = o.diagnostics(), b.diagnostics()
    assert db["t"] == pytest.approx(do["t"], rel=1e-13) and db["c2p_failures"] == 0
    q, qb = o.get_primitives(), b.get_primitives()
    for k in PRIMS + ["bxf", "byf", "bzf"]:
        ref = _pad(q[k], axis, 0, n)[b.interior()]
        got = qb[k][b.interior()]
        assert np.abs(got - ref).max() <= 1e-12 * max(1.0, np.abs(ref).max()), (axis, k, np.abs(got - ref).max())
    # the low wall face of the normal B is evolved, not filled
    kf = ["bxf", "byf", "bzf"][axis]
    w = [slice(None)] * 3
    w[2 - axis] = NG - 1
    wi = list(b.interior())
    wi[2 - axis] = NG - 1
    assert np.abs(qb[kf][tuple(wi)] - _pad(q[kf], axis, 0, n)[tuple(wi)]).max() <= 1e-12
    # teeth: the run moved, and the wall matters (the plain periodic half-box differs at O(1))
    assert np.abs(qb["vx"][b.interior()] - fp[1][b.interior()]).max() > 1e-3


def test_outflow_is_transparent_to_a_uniform_background():
    n = (96, 4, 4)
    z, y, x = np.meshgrid(*[(np.arange(m) + 0.5) / m for m in n[::-1]], indexing="ij")
    bump = np.exp(-((x - 0.5) / 0.02) ** 2)
    bump[np.abs(x - 0.5) > 0.05] = 0.0                    # compact support, 43 cells from either x-boundary
    one = np.ones_like(x)
    f = [one + 0.3 * bump, 0.2 * one, 0.0 * one, 0.0 * one, one + 0.3 * bump, 0.5 * one, 0.3 * one, 0.2 * one]
    o = Oracle(*n, G, 0.3)
    o.set_primitives(*f)
    b = Oracle(*n, G, 0.3, boundaries=(2, 2, 0, 0, 0, 0))
    b.set_primitives(*[_pad(a, 0, 0, n[0]) for a in f])
    # one step: the numerical domain of dependence (8 cells per sub-step) has not reached the boundary, where the
    # zero-gradient ghost layers hold the same uniform background as the periodic images: identical to the last bit
    o.step(1)
    b.step(1)
    q, qb = o.get_primitives(), b.get_primitives()
    assert o.diagnostics()["t"] == b.diagnostics()["t"]
    for k in PRIMS + ["bxf", "byf", "bzf"]:
        assert np.array_equal(qb[k][b.interior()], q[k]), k
    assert np.abs(q["rho"] - f[0]).max() > 1e-3           # (the pulse moved)
    # the ghost layers hold the boundary value (zero gradient)
    assert np.array_equal(qb["rho"][:, :, 0], qb["rho"][:, :, NG]) and np.array_equal(qb["rho"][:, :, -1], qb["rho"][:, :, -NG - 1])
    # later the two differ only by what has physically reached the boundary: nothing yet after 8 more steps
    o.step(8)
    b.step(8)
    q, qb = o.get_primitives(), b.get_primitives()
    for k in PRIMS:
        assert np.abs(qb[k][b.interior()] - q[k]).max() <= 1e-9, k


def test_bounded_argument_checks():
    L = ob.lib()
    import ctypes as C
    k = lambda *v: (C.c_int * 6)(*v)
    assert not L.oracle_create_bounded(16, 8, 8, G, 0.3, k(1, 0, 0, 0, 0, 0), None)    # one side periodic, the other not
    assert not L.oracle_create_bounded(4, 8, 8, G, 0.3, k(1, 1, 0, 0, 0, 0), None)     # fewer interior cells than ghosts
    assert not L.oracle_create_bounded(16, 8, 8, G, 0.3, k(3, 3, 0, 0, 0, 0), None)
