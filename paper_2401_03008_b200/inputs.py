"""Seeded synthetic workloads (numpy, host).  Serves BOTH the oracle tests and the CUDA path.

This module holds problem set-up only — closed-form initial data and random samples —
and none of the method's arithmetic (no INT/REC/DER stencils, no con2prim, no fluxes).
Staggered B is either an analytic point value at the face centre or is left as an
edge-centred vector potential for the solver under test to curl (echo_faces_from_potential /
oracle_faces_from_potential), see DESIGN.md "Input recipe".

Arrays are float64 with shape (nz, ny, nx): x fastest.
Citations: P:L<n> = /root/reference/PAPER.md line n.
"""
import math

import numpy as np

TWO_PI = 2.0 * math.pi


# --------------------------------------------------------------------------------------
# grid helpers: unit periodic box, cell (i,j,k) centred at ((i+1/2)hx, ...)
def _coords(n, offset, start=0, gn=None):
    """(start + i + offset)/gn for i < n: the same expression whether a whole box (start = 0, gn = n) or a block
    of a larger box is sampled, so a block carries bit-identical values to the corresponding part of the box."""
    gn = n if gn is None else gn
    i = (np.arange(n, dtype=np.int64) + int(start)) % int(gn)
    return (i.astype(np.float64) + offset) / gn


def _mesh(nx, ny, nz, ox, oy, oz, box=None):
    """Coordinates of points displaced by (ox,oy,oz) cells from the cell corner, shape (nz,ny,nx).
    box = ((gnx, gny, gnz), (sx, sy, sz)): the nx*ny*nz cells starting at (sx, sy, sz) of a periodic gn box."""
    (gx, gy, gz), (sx, sy, sz) = box if box is not None else ((nx, ny, nz), (0, 0, 0))
    z, y, x = np.meshgrid(_coords(nz, oz, sz, gz), _coords(ny, oy, sy, gy), _coords(nx, ox, sx, gx), indexing="ij")
    return x, y, z


CENTRE = (0.5, 0.5, 0.5)
FACE = [(1.0, 0.5, 0.5), (0.5, 1.0, 0.5), (0.5, 0.5, 1.0)]     # d-face on the + side of the cell
EDGE = [(0.5, 1.0, 1.0), (1.0, 0.5, 1.0), (1.0, 1.0, 0.5)]     # k-edge: +1/2 in the two other directions


# --------------------------------------------------------------------------------------
# Circularly polarised Alfven wave, eq.(11)-(12)
def alfven_speed(rho=1.0, p=1.0, B0=1.0, eta=1.0, gamma=4.0 / 3.0):
    """Exact propagation speed of the large-amplitude CPA wave, eq.(12)."""
    rhoh = rho + gamma / (gamma - 1.0) * p
    w = rhoh + B0 * B0 * (1.0 + eta * eta)
    s = math.sqrt(1.0 - (2.0 * eta * B0 * B0 / w) ** 2)
    return math.sqrt(B0 * B0 / w / (0.5 * (1.0 + s)))


def _cpa_frame(direction):
    if direction == "diag":      # S12: X along the main diagonal
        X = np.array([1.0, 1.0, 1.0]) / math.sqrt(3.0)
        Y = np.array([1.0, -1.0, 0.0]) / math.sqrt(2.0)
        Z = np.array([1.0, 1.0, -2.0]) / math.sqrt(6.0)
        kvec = TWO_PI * np.array([1.0, 1.0, 1.0])
    elif direction == "x":       # S13: config 4, wave along the x axis
        X = np.array([1.0, 0.0, 0.0])
        Y = np.array([0.0, 1.0, 0.0])
        Z = np.array([0.0, 0.0, 1.0])
        kvec = TWO_PI * np.array([1.0, 0.0, 0.0])
    else:
        raise ValueError(direction)
    return X, Y, Z, kvec


def cpa_period(direction="diag", **kw):
    vA = alfven_speed(**kw)
    _, _, _, kvec = _cpa_frame(direction)
    return TWO_PI / (np.linalg.norm(kvec) * vA)


def cpa_wave(nx, ny, nz, t=0.0, direction="diag", rho=1.0, p=1.0, B0=1.0, eta=1.0, gamma=4.0 / 3.0, box=None):
    """Exact CPA-wave fields at time t (phase k.x - |k| vA t).

    Returns a dict: rho, vx, vy, vz, p, bx, by, bz at cell centres; bxf, byf, bzf analytic
    point values at the staggered faces; vA, T (period), kvec.
    box = ((gnx, gny, gnz), (sx, sy, sz)) samples a block of a larger periodic box (domain decomposition).
    """
    X, Y, Z, kvec = _cpa_frame(direction)
    vA = alfven_speed(rho, p, B0, eta, gamma)
    kmod = float(np.linalg.norm(kvec))

    def fields(off):
        x, y, z = _mesh(nx, ny, nz, *off, box=box)
        phi = kvec[0] * x + kvec[1] * y + kvec[2] * z - kmod * vA * t
        c, s = np.cos(phi), np.sin(phi)
        dB = [eta * B0 * (c * Y[a] + s * Z[a]) for a in range(3)]
        B = [B0 * X[a] + dB[a] for a in range(3)]
        v = [-vA * dB[a] / B0 for a in range(3)]
        return B, v

    Bc, vc = fields(CENTRE)
    out = {"rho": np.full((nz, ny, nx), rho), "p": np.full((nz, ny, nx), p),
           "vx": vc[0], "vy": vc[1], "vz": vc[2], "bx": Bc[0], "by": Bc[1], "bz": Bc[2]}
    for d, name in enumerate(("bxf", "byf", "bzf")):
        Bf, _ = fields(FACE[d])
        out[name] = np.ascontiguousarray(Bf[d])
    out.update(vA=vA, T=TWO_PI / (kmod * vA), kvec=kvec, gamma=gamma)
    return out


# --------------------------------------------------------------------------------------
# splitmix64: the documented 64-bit generator for the turbulence phases (S18 / SURVEY 8(d))
class SplitMix64:
    def __init__(self, seed):
        self.s = seed & 0xFFFFFFFFFFFFFFFF

    def next_u64(self):
        self.s = (self.s + 0x9E3779B97F4A7C15) & 0xFFFFFFFFFFFFFFFF
        z = self.s
        z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & 0xFFFFFFFFFFFFFFFF
        z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & 0xFFFFFFFFFFFFFFFF
        return z ^ (z >> 31)

    def uniform(self):
        return (self.next_u64() >> 11) * (1.0 / 9007199254740992.0)   # 53 bits in [0,1)


def turbulence_modes():
    """The 14 integer vectors m with 1<=|m|^2<=4, (mx,my)!=(0,0), first non-zero component > 0."""
    modes = []
    for mx in range(-2, 3):
        for my in range(-2, 3):
            for mz in range(-2, 3):
                m2 = mx * mx + my * my + mz * mz
                if not (1 <= m2 <= 4) or (mx == 0 and my == 0):
                    continue
                first = next(c for c in (mx, my, mz) if c != 0)
                if first > 0:
                    modes.append((mx, my, mz))
    modes.sort()
    assert len(modes) == 14
    return modes


def turbulence(n, seed=2401, rho0=1.0, p0=0.1, sigma=1.0, amp=0.5, gamma=4.0 / 3.0, vmax_guard=0.95,
               shape=None):
    """3-D analogue of the paper's Alfvenic turbulence set-up (eq.(13)-(17)); BJ config 5.

    rho=rho0, p=p0, B0 along z with sigma = B0^2/(rho h); transverse Alfvenic modes
    delta B = curl(a z^), delta v = curl(psi z^), a = sum_m cos(k.x+phi_m)/|k| over the 14 modes,
    independent phases for B (drawn first) and v, each field scaled to an rms of amp*B0 (amp*vA)
    using the exact (orthogonal-mode) rms.  If max|v| >= vmax_guard the seed is incremented.

    Returns centre primitives, the edge-centred potential az (ax=ay=0) for the solver under test
    to curl, and the uniform part b0 = (0,0,B0) to add to the faces.
    """
    nx, ny, nz = (n, n, n) if shape is None else shape
    rhoh = rho0 + gamma / (gamma - 1.0) * p0
    B0 = math.sqrt(sigma * rhoh)
    vA = B0 / math.sqrt(rhoh + B0 * B0)
    modes = turbulence_modes()
    ms2 = sum(0.5 * (mx * mx + my * my) / float(mx * mx + my * my + mz * mz) for mx, my, mz in modes)
    xe, ye, ze = _mesh(nx, ny, nz, *EDGE[2])       # z-edges carry a
    xc, yc, zc = _mesh(nx, ny, nz, *CENTRE)
    while True:
        rng = SplitMix64(seed)
        phB = [TWO_PI * rng.uniform() for _ in modes]
        phV = [TWO_PI * rng.uniform() for _ in modes]
        cB = amp * B0 / math.sqrt(ms2)
        cV = amp * vA / math.sqrt(ms2)
        az = np.zeros((nz, ny, nx))
        vx = np.zeros((nz, ny, nx))
        vy = np.zeros((nz, ny, nx))
        for (mx, my, mz), pb, pv in zip(modes, phB, phV):
            kx, ky, kz = TWO_PI * mx, TWO_PI * my, TWO_PI * mz
            kk = math.sqrt(kx * kx + ky * ky + kz * kz)
            az += cB * np.cos(kx * xe + ky * ye + kz * ze + pb) / kk
            s = np.sin(kx * xc + ky * yc + kz * zc + pv)
            vx += cV * (-ky * s) / kk          # d(psi)/dy
            vy += cV * (kx * s) / kk           # -d(psi)/dx
        vmax = float(np.sqrt(vx * vx + vy * vy).max())
        if vmax < vmax_guard:
            break
        seed += 1
    full = lambda v: np.full((nz, ny, nx), v)
    return {"rho": full(rho0), "p": full(p0), "vx": vx, "vy": vy, "vz": full(0.0),
            "ax": full(0.0), "ay": full(0.0), "az": az, "b0": (0.0, 0.0, B0),
            "B0": B0, "vA": vA, "seed": seed, "vmax": vmax, "gamma": gamma}


# --------------------------------------------------------------------------------------
# 2.5-D decaying RMHD turbulence of the paper, eq.(13)-(17)  (row f3)
def turbulence_2d(nx, ny=None, seed=2401, eta_mean=0.25, gamma=4.0 / 3.0):
    """The paper's own turbulence set-up on an nx x ny x 1 grid (fluctuations in the x-y plane, B0 along z).

    rho0 = 1, sigma0 = B0^2/rho0 = 100, beta0 = 2 p0/B0^2 = 1  =>  B0 = 10, p0 = 50 (eq.(13));
    vA = B0/sqrt(rho0 + 4 p0 + B0^2) (eq.(14)); modes m = (mx, my), mx = 0..4, my = -4..4 (eq.(15)-(16)),
    kept when 1 <= |m| <= 4 ("spectral radius of 4") and, for mx = 0, my > 0 (the conjugate would be the
    same mode); delta v = eta vA sum (m x e_z)/|m| cos(2 pi m.x + phi_v), delta B likewise with B0 and phi_B,
    independent random phases (splitmix64(seed), B phases first); the staggered delta B comes from the potential
    a_z = sum sin(2 pi m.x + phi_B)/(2 pi |m|) at the z-edges, curled by the solver under test (S11).  eta is
    fixed a posteriori so that the MEAN magnitudes satisfy <|dv|>/vA = <|dB|>/B0 = eta_mean (eq.(17), read
    literally; |dB| is evaluated from the analytic field at the cell centres).  The paper's box has L = 2 pi; the
    equations have no length scale, so the unit box is used and one paper time unit is 1/(2 pi) here.
    """
    ny = nx if ny is None else ny
    rho0, B0 = 1.0, 10.0
    p0 = 0.5 * B0 * B0
    vA = B0 / math.sqrt(rho0 + gamma / (gamma - 1.0) * p0 + B0 * B0)
    modes = [(mx, my) for mx in range(0, 5) for my in range(-4, 5)
             if 1 <= mx * mx + my * my <= 16 and (mx > 0 or my > 0)]
    rng = SplitMix64(seed)
    phB = [TWO_PI * rng.uniform() for _ in modes]
    phV = [TWO_PI * rng.uniform() for _ in modes]
    xc, yc, _ = _mesh(nx, ny, 1, *CENTRE)
    xe, ye, _ = _mesh(nx, ny, 1, *EDGE[2])
    sh = (1, ny, nx)
    vx, vy, bxc, byc, az = (np.zeros(sh) for _ in range(5))
    for (mx, my), pb, pv in zip(modes, phB, phV):
        km = math.sqrt(mx * mx + my * my)
        cv = np.cos(TWO_PI * (mx * xc + my * yc) + pv)
        cb = np.cos(TWO_PI * (mx * xc + my * yc) + pb)
        vx += (my / km) * cv
        vy += (-mx / km) * cv
        bxc += (my / km) * cb
        byc += (-mx / km) * cb
        az += np.sin(TWO_PI * (mx * xe + my * ye) + pb) / (TWO_PI * km)
    sv = eta_mean / float(np.sqrt(vx * vx + vy * vy).mean())
    sb = eta_mean / float(np.sqrt(bxc * bxc + byc * byc).mean())
    full = lambda v: np.full(sh, v)
    return {"rho": full(rho0), "p": full(p0), "vx": sv * vA * vx, "vy": sv * vA * vy, "vz": full(0.0),
            "ax": full(0.0), "ay": full(0.0), "az": sb * B0 * az, "b0": (0.0, 0.0, B0),
            "B0": B0, "vA": vA, "gamma": gamma, "modes": modes,
            "vmax": float(sv * vA * np.sqrt(vx * vx + vy * vy).max())}


# --------------------------------------------------------------------------------------
def random_states(n, seed=12345, gamma=4.0 / 3.0, wmax=10.0, sigma_max=10.0, wmin=1.0, log_p_over_rho=(-2.0, 2.0)):
    """P6 sample: random primitive states up to Lorentz factor wmax and magnetisation sigma_max.

    rho ~ logU[1e-2,1e2], p/rho ~ logU[1e-2,1e2], u = W v uniform in [0, sqrt(wmax^2-1)] with an
    isotropic direction, sigma = b^2/(rho h) ~ logU[1e-3, sigma_max] with isotropic B direction.
    wmin > 1 and a colder log10(p/rho) range give the ultra-relativistic cold states (W of 20-40, p/rho of
    1e-6..1e-2) on which the Newton iteration of con2prim leaves its domain and needs its safeguard (O2).
    """
    rng = np.random.default_rng(seed)

    def iso(k):
        mu = rng.uniform(-1.0, 1.0, k)
        ph = rng.uniform(0.0, TWO_PI, k)
        st = np.sqrt(1.0 - mu * mu)
        return np.stack([st * np.cos(ph), st * np.sin(ph), mu])

    rho = 10.0 ** rng.uniform(-2.0, 2.0, n)
    p = rho * 10.0 ** rng.uniform(log_p_over_rho[0], log_p_over_rho[1], n)
    u = rng.uniform(math.sqrt(wmin * wmin - 1.0), math.sqrt(wmax * wmax - 1.0), n)
    W = np.sqrt(1.0 + u * u)
    v = iso(n) * (u / W)
    sigma = 10.0 ** rng.uniform(-3.0, math.log10(sigma_max), n)
    nb = iso(n)
    rhoh = rho + gamma / (gamma - 1.0) * p
    vn = (v * nb).sum(axis=0)
    beta = np.sqrt(sigma * rhoh / (1.0 / (W * W) + vn * vn))
    B = nb * beta
    return {"rho": rho, "vx": v[0].copy(), "vy": v[1].copy(), "vz": v[2].copy(), "p": p,
            "bx": B[0].copy(), "by": B[1].copy(), "bz": B[2].copy(), "W": W, "sigma": sigma}


def sample_cells(shape, count=4096, seed=7):
    """Deterministic flat indices for sampled parity checks at sizes the oracle cannot sweep."""
    total = int(np.prod(shape))
    rng = np.random.default_rng(seed)
    return np.sort(rng.choice(total, size=min(count, total), replace=False))
