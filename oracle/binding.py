"""ctypes access to the CPU oracle (oracle/echo_oracle.cpp).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may
import this module.  It holds no arithmetic of the method: it compiles the C++ file with
g++ (if the shared object is missing or stale) and marshals numpy arrays.
"""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "echo_oracle.cpp")
_LIB = os.path.join(_HERE, "libecho_oracle.so")

_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int)


def build(force=False):
    """Compile the oracle with plain g++ -O2 (no intrinsics, no fast-math)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".tmp%d" % os.getpid()
        subprocess.check_call(["g++", "-O2", "-std=c++17", "-shared", "-fPIC", "-ffp-contract=off",
                               "-o", tmp, _SRC])
        os.replace(tmp, _LIB)
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        L.oracle_create.restype = C.c_void_p
        L.oracle_create.argtypes = [C.c_int, C.c_int, C.c_int, C.c_double, C.c_double]
        L.oracle_create_bounded.restype = C.c_void_p
        L.oracle_create_bounded.argtypes = [C.c_int, C.c_int, C.c_int, C.c_double, C.c_double, _ip, _ip]
        L.oracle_destroy.argtypes = [C.c_void_p]
        L.oracle_destroy.restype = None
        L.oracle_set_scheme.argtypes = [C.c_void_p, C.c_int, C.c_int]
        L.oracle_set_order.argtypes = [C.c_void_p, C.c_int, C.c_int]
        L.oracle_tvd2.restype = C.c_double
        L.oracle_tvd2.argtypes = [_dp]
        L.oracle_faces_from_potential_ho.argtypes = [C.c_int] * 4 + [_dp] * 6
        L.oracle_set_primitives.argtypes = [C.c_void_p] + [_dp] * 8
        L.oracle_step.argtypes = [C.c_void_p, C.c_int, C.c_double]
        L.oracle_get_primitives.argtypes = [C.c_void_p] + [_dp] * 11
        L.oracle_get_conserved.argtypes = [C.c_void_p] + [_dp] * 5
        L.oracle_rhs.argtypes = [C.c_void_p] + [C.POINTER(_dp)] * 4 + [_dp]
        L.oracle_con2prim.argtypes = [C.c_double, C.c_long] + [_dp] * 13 + [_ip]
        L.oracle_con2prim_trace.argtypes = [C.c_double, C.c_long] + [_dp] * 13 + [_ip, _ip]
        L.oracle_prim2cons.argtypes = [C.c_double, C.c_long] + [_dp] * 13
        L.oracle_div_b.argtypes = [C.c_void_p, _dp, _dp]
        L.oracle_diagnostics.argtypes = [C.c_void_p, _dp]
        L.oracle_faces_from_potential.argtypes = [C.c_int] * 3 + [_dp] * 6
        L.oracle_int6.restype = C.c_double
        L.oracle_int6.argtypes = [_dp]
        L.oracle_der5.restype = C.c_double
        L.oracle_der5.argtypes = [_dp]
        L.oracle_mp5.restype = C.c_double
        L.oracle_mp5.argtypes = [_dp]
        L.oracle_fast_speeds.restype = None
        L.oracle_fast_speeds.argtypes = [C.c_double, _dp, C.c_int, _dp]
        L.oracle_phys_flux.restype = None
        L.oracle_phys_flux.argtypes = [C.c_double, _dp, C.c_int, _dp]
        L.oracle_hll.restype = None
        L.oracle_hll.argtypes = [C.c_double, _dp, _dp, C.c_int, _dp, _dp]
        _lib = L
    return _lib


def _c(a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a


def _p(a):
    return a.ctypes.data_as(_dp)


DIAG_NAMES = ["t", "dt_last", "steps", "amax", "sum_D", "sum_Sx", "sum_Sy", "sum_Sz", "sum_U",
              "sum_Bx", "sum_By", "sum_Bz", "max_div_b", "max_W", "min_rho", "min_p",
              "c2p_max_iters", "c2p_mean_iters", "c2p_failures"]


class Oracle:
    """One periodic unit box.  Arrays are numpy float64 of shape (nz, ny, nx) (x fastest)."""

    def __init__(self, nx, ny, nz, gamma, cfl, uct=True, ho=True, rec=5, rk=3, boundaries=None, gn=None):
        """uct / ho: the paper's scheme switches.  With uct=False the three B arrays given to
        set_primitives (and returned as bxf, byf, bzf) are CELL-CENTRED.  rec / rk: 5 / 3 = MP5 + SSP-RK3 (default),
        2 / 2 = limited linear reconstruction + SSP-RK2.
        boundaries = (x_lo, x_hi, y_lo, y_hi, z_lo, z_hi) with 0 periodic, 1 reflecting, 2 outflow (row f4): nx, ny, nz
        are then the INTERIOR cells and every array has 8 ghost layers on each side of a bounded axis; gn = (gnx, gny,
        gnz): the spacing is h_d = 1/gn_d (default gn = n: the interior is the unit box)."""
        self.L = lib()
        self.n = (nx, ny, nz)
        if boundaries is None:
            self.ng = (0, 0, 0)
            self.h = self.L.oracle_create(nx, ny, nz, gamma, cfl)
        else:
            kinds = (C.c_int * 6)(*[int(k) for k in boundaries])
            self.ng = tuple(8 if boundaries[2 * a] else 0 for a in range(3))
            gnp = (C.c_int * 3)(*[int(v) for v in gn]) if gn is not None else None
            self.h = self.L.oracle_create_bounded(nx, ny, nz, gamma, cfl, kinds, gnp)
        self.shape = (nz + 2 * self.ng[2], ny + 2 * self.ng[1], nx + 2 * self.ng[0])
        if not self.h:
            raise ValueError("oracle_create: bad arguments")
        if not (uct and ho):
            rc = self.L.oracle_set_scheme(self.h, int(bool(uct)), int(bool(ho)))
            assert rc == 0, rc
        if (rec, rk) != (5, 3):
            rc = self.L.oracle_set_order(self.h, int(rec), int(rk))
            assert rc == 0, rc

    def __del__(self):
        if getattr(self, "h", None):
            self.L.oracle_destroy(self.h)
            self.h = None

    def _new(self, k):
        return [np.empty(self.shape, dtype=np.float64) for _ in range(k)]

    def interior(self):
        """Slices (z, y, x) of the interior cells of a bounded grid's arrays."""
        return tuple(slice(g, s - g) for g, s in zip(self.ng[::-1], self.shape))

    def set_primitives(self, rho, vx, vy, vz, p, bxf, byf, bzf):
        arrs = [_c(a) for a in (rho, vx, vy, vz, p, bxf, byf, bzf)]
        for a in arrs:
            assert a.shape == self.shape, (a.shape, self.shape)
        rc = self.L.oracle_set_primitives(self.h, *[_p(a) for a in arrs])
        if rc:
            raise RuntimeError("oracle_set_primitives rc=%d" % rc)

    def step(self, nsteps, t_end=float("inf")):
        rc = self.L.oracle_step(self.h, int(nsteps), float(t_end))
        if rc < 0:
            raise RuntimeError("oracle_step rc=%d" % rc)
        return rc

    def get_primitives(self):
        """-> dict rho,vx,vy,vz,p,bx,by,bz (centres) and bxf,byf,bzf (faces)."""
        out = self._new(11)
        rc = self.L.oracle_get_primitives(self.h, *[_p(a) for a in out])
        names = ["rho", "vx", "vy", "vz", "p", "bx", "by", "bz", "bxf", "byf", "bzf"]
        d = dict(zip(names, out))
        d["rc"] = rc
        return d

    def get_conserved(self):
        out = self._new(5)
        self.L.oracle_get_conserved(self.h, *[_p(a) for a in out])
        return dict(zip(["D", "Sx", "Sy", "Sz", "U"], out))

    def rhs(self):
        """L(U) of the current state: dict with rhsU[5], rhsB[3], E[3], F[3][5], amax."""
        rU, rB, E, F = self._new(5), self._new(3), self._new(3), self._new(15)

        def pp(lst):
            return (_dp * len(lst))(*[_p(a) for a in lst])

        amax = C.c_double(0.0)
        rc = self.L.oracle_rhs(self.h, pp(rU), pp(rB), pp(E), pp(F), C.byref(amax))
        if rc:
            raise RuntimeError("oracle_rhs rc=%d" % rc)
        return {"rhsU": rU, "rhsB": rB, "E": E, "F": [F[0:5], F[5:10], F[10:15]], "amax": amax.value}

    def div_b(self, want_field=False):
        m = C.c_double(0.0)
        f = np.empty(self.shape) if want_field else None
        self.L.oracle_div_b(self.h, _p(f) if want_field else None, C.byref(m))
        return (m.value, f) if want_field else m.value

    def diagnostics(self):
        out = np.zeros(24)
        rc = self.L.oracle_diagnostics(self.h, _p(out))
        if rc:
            raise RuntimeError("oracle_diagnostics rc=%d" % rc)
        d = dict(zip(DIAG_NAMES, out[:len(DIAG_NAMES)]))
        d["raw"] = out
        return d


def con2prim(gamma, D, Sx, Sy, Sz, U, Bx, By, Bz):
    ins = [_c(a).ravel() for a in (D, Sx, Sy, Sz, U, Bx, By, Bz)]
    n = ins[0].size
    outs = [np.empty(n) for _ in range(5)]
    iters = np.empty(n, dtype=np.int32)
    rc = lib().oracle_con2prim(gamma, n, *[_p(a) for a in ins], *[_p(a) for a in outs],
                               iters.ctypes.data_as(_ip))
    return dict(rho=outs[0], vx=outs[1], vy=outs[2], vz=outs[3], p=outs[4], iters=iters, rc=rc)


def con2prim_trace(gamma, D, Sx, Sy, Sz, U, Bx, By, Bz):
    """con2prim + per-state count of safeguard activations (nsafe)."""
    ins = [_c(a).ravel() for a in (D, Sx, Sy, Sz, U, Bx, By, Bz)]
    n = ins[0].size
    outs = [np.empty(n) for _ in range(5)]
    iters = np.empty(n, dtype=np.int32)
    nsafe = np.empty(n, dtype=np.int32)
    rc = lib().oracle_con2prim_trace(gamma, n, *[_p(a) for a in ins], *[_p(a) for a in outs],
                                     iters.ctypes.data_as(_ip), nsafe.ctypes.data_as(_ip))
    return dict(rho=outs[0], vx=outs[1], vy=outs[2], vz=outs[3], p=outs[4], iters=iters, nsafe=nsafe, rc=rc)


def prim2cons(gamma, rho, vx, vy, vz, p, Bx, By, Bz):
    ins = [_c(a).ravel() for a in (rho, vx, vy, vz, p, Bx, By, Bz)]
    n = ins[0].size
    outs = [np.empty(n) for _ in range(5)]
    lib().oracle_prim2cons(gamma, n, *[_p(a) for a in ins], *[_p(a) for a in outs])
    return dict(D=outs[0], Sx=outs[1], Sy=outs[2], Sz=outs[3], U=outs[4])


def faces_from_potential(ax, ay, az, ho=True):
    a = [_c(x) for x in (ax, ay, az)]
    nz, ny, nx = a[0].shape
    out = [np.empty_like(a[0]) for _ in range(3)]
    if ho:
        rc = lib().oracle_faces_from_potential(nx, ny, nz, *[_p(x) for x in a], *[_p(x) for x in out])
    else:
        rc = lib().oracle_faces_from_potential_ho(nx, ny, nz, 0, *[_p(x) for x in a], *[_p(x) for x in out])
    if rc:
        raise RuntimeError("oracle_faces_from_potential rc=%d" % rc)
    return out


def int6(b):
    b = _c(b); assert b.size == 6
    return lib().oracle_int6(_p(b))


def der5(f):
    f = _c(f); assert f.size == 5
    return lib().oracle_der5(_p(f))


def mp5(v):
    v = _c(v); assert v.size == 5
    return lib().oracle_mp5(_p(v))


def tvd2(v):
    v = _c(v); assert v.size == 5
    return lib().oracle_tvd2(_p(v))


def fast_speeds(gamma, q, d):
    q = _c(q); assert q.size == 8
    out = np.empty(2)
    lib().oracle_fast_speeds(gamma, _p(q), d, _p(out))
    return out


def phys_flux(gamma, q, d):
    q = _c(q); assert q.size == 8
    out = np.empty(5)
    lib().oracle_phys_flux(gamma, _p(q), d, _p(out))
    return out


def hll(gamma, qL, qR, d):
    qL, qR = _c(qL), _c(qR)
    F, ex = np.empty(5), np.empty(4)
    lib().oracle_hll(gamma, _p(qL), _p(qR), d, _p(F), _p(ex))
    return F, ex
