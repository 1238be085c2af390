"""Thin ctypes binding of libecho_b200.so (include/echo.h): argument marshalling only.

PyTorch supplies device memory (FP64 tensors, the workspace byte tensor) and the CUDA stream;
every step of the path runs in the library's kernels.  There is NO CPU fallback: if the shared
library cannot be loaded, or no CUDA device is present when a compute call is made, this module
raises.
"""
import ctypes as C
import math
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libecho_b200.so")

ECHO_OK, ECHO_EINVAL, ECHO_ENOMEM, ECHO_ECUDA, ECHO_ESTATE, ECHO_EC2P = 0, -1, -2, -3, -4, -5
ECHO_NDIAG = 24
_vp, _dbl, _int, _long, _sz = C.c_void_p, C.c_double, C.c_int, C.c_long, C.c_size_t

# name -> (restype, argtypes): every symbol include/echo.h declares
SIGNATURES = {
    "echo_create": (_vp, [_int, _int, _int, _dbl, _dbl]),
    "echo_destroy": (None, [_vp]),
    "echo_set_scheme": (_int, [_vp, _int, _int]),
    "echo_set_order": (_int, [_vp, _int, _int]),
    "echo_workspace_bytes": (_sz, [_vp]),
    "echo_bind": (_int, [_vp, _vp, _sz, _vp]),
    "echo_last_error": (C.c_char_p, [_vp]),
    "echo_set_primitives": (_int, [_vp] + [_vp] * 8),
    "echo_set_primitives_host": (_int, [_vp] + [_vp] * 8),
    "echo_faces_from_potential": (_int, [_vp] + [_vp] * 3 + [_dbl] * 3 + [_vp] * 3),
    "echo_step": (_int, [_vp, _int, _dbl]),
    "echo_run_until": (_int, [_vp, _dbl, C.c_long, C.POINTER(C.c_long)]),
    "echo_get_primitives": (_int, [_vp] + [_vp] * 11),
    "echo_get_primitives_host": (_int, [_vp] + [_vp] * 11),
    "echo_get_primitives_host_async": (_int, [_vp] + [_vp] * 11),
    "echo_synchronize": (_int, [_vp]),
    "echo_get_conserved": (_int, [_vp] + [_vp] * 5),
    "echo_rhs": (_int, [_vp, C.POINTER(_vp), C.POINTER(_vp), C.POINTER(_vp), C.POINTER(_dbl)]),
    "echo_con2prim": (_int, [_dbl, _long] + [_vp] * 13 + [_vp, _vp]),
    "echo_prim2cons": (_int, [_dbl, _long] + [_vp] * 13 + [_vp]),
    "echo_div_b": (_int, [_vp, _vp, C.POINTER(_dbl)]),
    "echo_div_b_static": (_int, [_int, _int, _int, _int, _vp, _vp, _vp, _vp, _vp, _vp]),
    "echo_div_b_static_setup": (_int, []),
    "echo_div_b_static_error": (C.c_char_p, []),
    "echo_diagnostics": (_int, [_vp, C.POINTER(_dbl)]),
    "echo_create_block": (_vp, [_int, _int, _int, _dbl, _dbl, _int, _int, _int, _int, _int, _int]),
    "echo_set_boundaries": (_int, [_vp, C.POINTER(_int)]),
    "echo_fill_boundaries": (_int, [_vp, C.POINTER(_int)]),
    "echo_field_offset": (_sz, [_vp, _int]),
    "echo_ctrl_offset": (_sz, [_int]),
    "echo_stage_sweeps": (_int, [_vp, _int, _dbl]),
    "echo_stage_finish": (_int, [_vp, _int]),
    "echo_stage_halo_fields": (_int, [_vp, _int, C.POINTER(_int)]),
    "echo_halo_doubles": (_sz, [_vp, _int]),
    "echo_halo_pack": (_int, [_vp, C.POINTER(_int), _int, _int, _vp, _vp]),
    "echo_halo_unpack": (_int, [_vp, C.POINTER(_int), _int, _int, _vp, _vp]),
    "echo_get_tiling": (_int, [_vp, C.POINTER(_int)]),
    "echo_use_graph": (_int, [_vp, _int]),
    "echo_timing": (_int, [_vp, _int]),
    "echo_get_timing": (_int, [_vp, C.POINTER(_dbl), C.POINTER(_long)]),
    "echo_fp64_peak": (_int, [_int, C.POINTER(_dbl), _vp]),
}
ECHO_DIV_B_STATIC_MAX_TILES = 65536
ECHO_NKCLASS = 8
KCLASS_NAMES = ["k_prim", "k_flux_x", "k_flux_y", "k_flux_z", "k_uct", "k_update", "control", "other"]

DIAG_NAMES = ["t", "dt_last", "steps", "amax", "sum_D", "sum_Sx", "sum_Sy", "sum_Sz", "sum_U",
              "sum_Bx", "sum_By", "sum_Bz", "max_div_b", "max_W", "min_rho", "min_p",
              "c2p_max_iters", "c2p_mean_iters", "c2p_failures"]

_lib = None


def lib():
    """Loads the CUDA library; raises (never falls back) if it is missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError("libecho_b200.so is not built: run `python -m paper_2401_03008_b200.build` "
                               "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        for name, (res, args) in SIGNATURES.items():
            fn = getattr(L, name)
            fn.restype = res
            fn.argtypes = args
        _lib = L
    return _lib


def _torch():
    import torch
    if not torch.cuda.is_available():
        raise RuntimeError("paper_2401_03008_b200 needs a CUDA device (sm_100a); there is no CPU fallback")
    return torch


def _dev(t, n=None):
    """Device pointer of a contiguous FP64 CUDA tensor."""
    assert t.is_cuda and t.is_contiguous() and t.dtype.is_floating_point and t.element_size() == 8, "need FP64 CUDA tensor"
    if n is not None:
        assert t.numel() == n, (t.numel(), n)
    return t.data_ptr()


def _stream(device=None):
    return _torch().cuda.current_stream(device).cuda_stream


class EchoError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("echo error %d: %s" % (code, msg))
        self.code = code


class Echo:
    """One periodic unit box on the current CUDA device.  Tensors are torch.float64, shape (nz, ny, nx)."""

    def __init__(self, nx, ny, nz, gamma, cfl, device=None, block=None, ho=True, uct=True, rec=5, rk=3, boundaries=None):
        """block = (gnx, gny, gnz, halo_x, halo_y, halo_z): a domain-decomposition block (echo_create_block).
        boundaries = (x_lo, x_hi, y_lo, y_hi, z_lo, z_hi), 0 none / 1 reflecting / 2 outflow (echo_set_boundaries): needs a
        block with halo 8 on the bounded axes; nx, ny, nz are then the PADDED sizes.
        ho / uct: the paper's scheme switches (echo_set_scheme); with uct=False the three "face" arrays of
        set_primitives / get_primitives are the cell-centred B."""
        torch = _torch()
        self.L = lib()
        self.n = (nx, ny, nz)
        self.shape = (nz, ny, nx)
        self.N = nx * ny * nz
        self.device = torch.device("cuda", torch.cuda.current_device()) if device is None else torch.device(device)
        if block is None:
            self.h = self.L.echo_create(nx, ny, nz, gamma, cfl)
        else:
            self.h = self.L.echo_create_block(nx, ny, nz, gamma, cfl, *[int(b) for b in block])
        if not self.h:
            raise ValueError("echo_create: bad arguments")
        if not (ho and uct):
            self._check(self.L.echo_set_scheme(self.h, int(bool(uct)), int(bool(ho))))
        if (rec, rk) != (5, 3):     # echo_set_order: 2 / 2 = limited linear REC + SSP-RK2
            self._check(self.L.echo_set_order(self.h, int(rec), int(rk)))
        if boundaries is not None:
            self._check(self.L.echo_set_boundaries(self.h, (_int * 6)(*[int(k) for k in boundaries])))
        nbytes = self.L.echo_workspace_bytes(self.h)
        self.workspace = torch.empty(nbytes, dtype=torch.uint8, device=self.device)   # owned by the caller side
        # the stream of the workspace's device: the library runs every kernel of this handle there (echo_bind)
        self._check(self.L.echo_bind(self.h, self.workspace.data_ptr(), nbytes, _stream(self.device)))

    def __del__(self):
        if getattr(self, "h", None):
            self.L.echo_destroy(self.h)
            self.h = None

    def _check(self, rc, allow=()):
        if rc != ECHO_OK and rc not in allow:
            raise EchoError(rc, self.L.echo_last_error(self.h).decode())
        return rc

    def _new(self, k):
        torch = _torch()
        return [torch.empty(self.shape, dtype=torch.float64, device=self.device) for _ in range(k)]

    # ---- echo_set_primitives / echo_set_primitives_host
    def set_primitives(self, rho, vx, vy, vz, p, bxf, byf, bzf):
        self._check(self.L.echo_set_primitives(self.h, *[_dev(a, self.N) for a in (rho, vx, vy, vz, p, bxf, byf, bzf)]))

    def set_primitives_host(self, *arrs):
        """arrs: 8 host FP64 buffers (numpy arrays or CPU torch tensors, ideally pinned)."""
        self._check(self.L.echo_set_primitives_host(self.h, *[_host_ptr(a, self.N) for a in arrs]))

    def faces_from_potential(self, ax, ay, az, b0=(0.0, 0.0, 0.0)):
        out = self._new(3)
        self._check(self.L.echo_faces_from_potential(self.h, _dev(ax, self.N), _dev(ay, self.N), _dev(az, self.N),
                                                     float(b0[0]), float(b0[1]), float(b0[2]),
                                                     *[_dev(o) for o in out]))
        return out

    # ---- echo_step
    def step(self, nsteps, t_end=math.inf):
        self._check(self.L.echo_step(self.h, int(nsteps), float(t_end)))

    # ---- echo_get_primitives / _host
    def get_primitives(self, faces=True):
        out = self._new(11 if faces else 8)
        ptrs = [_dev(o) for o in out] + [None] * (11 - len(out))
        self._check(self.L.echo_get_primitives(self.h, *ptrs))
        names = ["rho", "vx", "vy", "vz", "p", "bx", "by", "bz", "bxf", "byf", "bzf"]
        return dict(zip(names, out))

    def get_primitives_host(self, outs, sync=True):
        """outs: 8 or 11 host FP64 buffers; synchronises unless sync=False (then call synchronize())."""
        ptrs = [_host_ptr(a, self.N) for a in outs] + [None] * (11 - len(outs))
        fn = self.L.echo_get_primitives_host if sync else self.L.echo_get_primitives_host_async
        self._check(fn(self.h, *ptrs))

    def synchronize(self):
        self._check(self.L.echo_synchronize(self.h))

    def get_conserved(self):
        out = self._new(5)
        self._check(self.L.echo_get_conserved(self.h, *[_dev(o) for o in out]))
        return dict(zip(["D", "Sx", "Sy", "Sz", "U"], out))

    def rhs(self):
        rU, rB, E = self._new(5), self._new(3), self._new(3)

        def tab(lst):
            return (_vp * len(lst))(*[_dev(t) for t in lst])

        amax = _dbl(0.0)
        self._check(self.L.echo_rhs(self.h, tab(rU), tab(rB), tab(E), C.byref(amax)))
        return {"rhsU": rU, "rhsB": rB, "E": E, "amax": amax.value}

    def div_b(self, want_field=False):
        m = _dbl(0.0)
        f = self._new(1)[0] if want_field else None
        self._check(self.L.echo_div_b(self.h, _dev(f) if want_field else None, C.byref(m)))
        return (m.value, f) if want_field else m.value

    def diagnostics(self):
        out = (_dbl * ECHO_NDIAG)()
        rc = self._check(self.L.echo_diagnostics(self.h, out), allow=(ECHO_EC2P,))
        d = dict(zip(DIAG_NAMES, list(out)[:len(DIAG_NAMES)]))
        d["rc"] = rc
        return d


    # ---- domain-decomposition blocks
    def field(self, idx):
        """Field idx (0..43) of the workspace as a (nz, ny, nx) float64 tensor VIEW (no copy)."""
        off = self.L.echo_field_offset(self.h, int(idx))
        return self.workspace[off:off + 8 * self.N].view(_torch().float64).view(self.shape)

    def ctrl_word(self, what):
        """8-byte control word as an int64 tensor view: 0 = a_max bits, 1 = t, 2 = dt, 3 = con2prim failures."""
        off = self.L.echo_ctrl_offset(int(what))
        return self.workspace[off:off + 8].view(_torch().int64)

    def run_until(self, t_end, max_steps=2 ** 31 - 1):
        """echo_run_until: steps taken (synchronises); raises on a con2prim failure."""
        n = C.c_long(0)
        self._check(self.L.echo_run_until(self.h, float(t_end), int(max_steps), C.byref(n)))
        return n.value

    def stage_sweeps(self, stage, t_end=math.inf):
        self._check(self.L.echo_stage_sweeps(self.h, int(stage), float(t_end)))

    def stage_finish(self, stage):
        self._check(self.L.echo_stage_finish(self.h, int(stage)))

    def tiling(self):
        """echo_get_tiling: the launch configuration in force (chunk lengths of the sweeps and marching kernels)."""
        out = (_int * 8)()
        self._check(self.L.echo_get_tiling(self.h, out))
        names = ["cx_flux", "cy_flux", "cz_flux", "cz_prim", "cz_uct", "cz_bupd", "tile_x", "tile_y"]
        return dict(zip(names, list(out)))

    def fill_boundaries(self, fields):
        self._check(self.L.echo_fill_boundaries(self.h, (_int * 8)(*[int(f) for f in fields])))

    def stage_halo_fields(self, stage):
        """The 8 workspace fields whose halos the next half needs after stage `stage` (5 cell fields, 3 face fields)."""
        out = (_int * 8)()
        self._check(self.L.echo_stage_halo_fields(self.h, int(stage), out))
        return list(out)

    def halo_doubles(self, axis):
        return int(self.L.echo_halo_doubles(self.h, int(axis)))

    def halo_pack(self, fields, axis, side, buf, stream=None):
        """Gathers the interior slabs next to `side` of the 8 `fields` into the FP64 CUDA tensor buf (one kernel)."""
        arr = (_int * 8)(*[int(f) for f in fields])
        self._check(self.L.echo_halo_pack(self.h, arr, int(axis), int(side), _dev(buf, self.halo_doubles(axis)), stream))

    def halo_unpack(self, fields, axis, side, buf, stream=None):
        arr = (_int * 8)(*[int(f) for f in fields])
        self._check(self.L.echo_halo_unpack(self.h, arr, int(axis), int(side), _dev(buf, self.halo_doubles(axis)), stream))

    def use_graph(self, enable=True):
        """echo_use_graph: replay one captured step (default) or launch its kernels one by one."""
        self._check(self.L.echo_use_graph(self.h, 1 if enable else 0))

    # ---- measurement aids
    def timing(self, enable=True):
        self._check(self.L.echo_timing(self.h, 1 if enable else 0))

    def get_timing(self):
        """-> {class name: (total ms, launches)}; synchronises."""
        ms = (_dbl * ECHO_NKCLASS)()
        cnt = (_long * ECHO_NKCLASS)()
        self._check(self.L.echo_get_timing(self.h, ms, cnt))
        return {k: (ms[i], cnt[i]) for i, k in enumerate(KCLASS_NAMES)}


def fp64_peak(reps=20):
    """Measured FP64 DFMA peak of the current device in TFLOP/s: (burst, sustained)."""
    _torch()
    out = (_dbl * 2)()
    rc = lib().echo_fp64_peak(int(reps), out, _stream())
    if rc:
        raise EchoError(rc, "echo_fp64_peak")
    return out[0], out[1]


def div_b_static(bx_face, by_face, bz_face, ho=1, div_field=None, max_abs=None):
    """echo_div_b_static: div B of (nz, ny, nx) FP64 CUDA face arrays on the periodic unit box into the CALLER's
    outputs -- div_field (same shape) and/or max_abs (one double on the device), written asynchronously on the current
    stream.  Allocates nothing; grids beyond ECHO_DIV_B_STATIC_MAX_TILES tiles of 64 x 4 x 1 cells raise EchoError."""
    torch = _torch()
    nz, ny, nx = bx_face.shape
    n = nx * ny * nz
    L = lib()
    with torch.cuda.device(bx_face.device):      # the scratch address is the current device's
        rc = L.echo_div_b_static(nx, ny, nz, int(ho), _dev(bx_face, n), _dev(by_face, n), _dev(bz_face, n),
                                 _dev(div_field, n) if div_field is not None else None,
                                 _dev(max_abs, 1) if max_abs is not None else None, _stream(bx_face.device))
    if rc:
        raise EchoError(rc, L.echo_div_b_static_error().decode())


def _host_ptr(a, n):
    """Pointer of a host FP64 buffer: numpy array or CPU torch tensor."""
    if hasattr(a, "data_ptr"):
        assert not a.is_cuda and a.is_contiguous() and a.element_size() == 8 and a.numel() == n
        return a.data_ptr()
    assert a.dtype.itemsize == 8 and a.flags["C_CONTIGUOUS"] and a.size == n
    return a.ctypes.data


def con2prim(gamma, D, Sx, Sy, Sz, U, Bx, By, Bz):
    """echo_con2prim on 1-D FP64 CUDA tensors -> dict of tensors (+ int32 iters)."""
    torch = _torch()
    ins = [D, Sx, Sy, Sz, U, Bx, By, Bz]
    n = ins[0].numel()
    outs = [torch.empty(n, dtype=torch.float64, device=D.device) for _ in range(5)]
    iters = torch.empty(n, dtype=torch.int32, device=D.device)
    rc = lib().echo_con2prim(float(gamma), n, *[_dev(a, n) for a in ins], *[_dev(o) for o in outs],
                             iters.data_ptr(), _stream())
    if rc:
        raise EchoError(rc, "echo_con2prim")
    return dict(rho=outs[0], vx=outs[1], vy=outs[2], vz=outs[3], p=outs[4], iters=iters)


def prim2cons(gamma, rho, vx, vy, vz, p, Bx, By, Bz):
    torch = _torch()
    ins = [rho, vx, vy, vz, p, Bx, By, Bz]
    n = ins[0].numel()
    outs = [torch.empty(n, dtype=torch.float64, device=rho.device) for _ in range(5)]
    rc = lib().echo_prim2cons(float(gamma), n, *[_dev(a, n) for a in ins], *[_dev(o) for o in outs], _stream())
    if rc:
        raise EchoError(rc, "echo_prim2cons")
    return dict(D=outs[0], Sx=outs[1], Sy=outs[2], Sz=outs[3], U=outs[4])
