// echo_oracle.cpp — ORACLE. TEST INFRASTRUCTURE ONLY, NOT THE PRODUCT.
//
// A plain, slow, single-threaded FP64 CPU implementation of one explicit time step of
// 3-D special-relativistic ideal MHD on a uniform periodic Cartesian unit box, as the
// ECHO scheme is described in /root/reference/PAPER.md ("P:L<n>" below) and read in
// SURVEY.md §8(c) / DESIGN.md ("O1".."O9", "S1".."S19").
//
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg
// may call this file.  It shares no code, header, table or helper with the CUDA path
// under paper_2401_03008_b200/csrc/ and neither includes the other.
//
// Style: every operation is a full-domain loop over whole arrays in the paper's order
// (the five points of a Runge-Kutta sub-step); no blocking, fusion or
// reordering beyond what the definitions state.  Arrays are SoA, x fastest,
// index = i + nx*(j + ny*k), all indices wrap periodically (no ghost cells).
//
// Staggering conventions:
//   cell (i,j,k) centre at ((i+1/2)hx, (j+1/2)hy, (k+1/2)hz), h_d = 1/n_d  (unit box)
//   face array  Bf[d][c]  : point value of B_d at the d-face on the + side of cell c
//   edge array  E[k][c]   : point value of E_k at the k-edge displaced +1/2 in the two
//                           directions (k+1)%3 and (k+2)%3 from the centre of cell c
//
// Scheme switches of the paper (oracle_set_scheme; defaults UCT=YES, HO=YES are the scheme of every test that
// does not say otherwise): HO=NO makes INT and DER second order ("INT and DER ... only if higher than
// second order accuracy is imposed (with the specific flag HO=YES)"); UCT=NO evolves a cell-centred B like the
// other conserved variables, with no divergence control ("the magnetic field is not staggered but it is
// treated as the other cell-centered variables").
//
// Non-periodic boundaries ("next" row f4, first slice; the paper's production runs are periodic, its code has
// ghost cells filled before every stencil loop): oracle_create_bounded pads the grid with NG = 8
// ghost cells on each side of every bounded axis (the dependency reach of one sub-step) and refills them before every
// evaluation of L(U) - reflecting wall (mirror image with the parity of each field under the reflection) or
// zero-gradient outflow (copy of the nearest interior value).  DESIGN.md section 12.
//
// Pins (tests/test_oracle_*.py): see the list in DESIGN.md §"Oracle pins".
// parity unpinned: inside the MP5 limiter branch, the published design constants 4/3 (v^LC) and 4 (inside d^M4)
// against nearby values.  The paper prints nothing that fixes them; what IS pinned about the branch
// (tests/test_oracle_units.py, tests/test_oracle_mp5_advection.py): its bounds and symmetries, monotone advection
// of a pulse at Courant number 1/(1+alpha), transparency on resolved smooth extrema, the bound v_j + alpha dv, and
// the 1/2 of v^MD (with d^M4 = d_{i+1} the bound is the linear extrapolation to the face from the right).

#include <cmath>
#include <cstddef>
#include <cstdint>
#include <cstring>
#include <limits>
#include <vector>

namespace {

typedef std::vector<double> Field;

// ----------------------------------------------------------------------------------
// O1 — INT: 6th-order centred interpolation of staggered point values to the midpoint.
// P:L128 ("staggered magnetic fields are first interpolated at cell centers (INT
// procedure) along the longitudinal direction"); order from HO=YES.
// b[0..5] = b_{i-5/2}, b_{i-3/2}, b_{i-1/2}, b_{i+1/2}, b_{i+3/2}, b_{i+5/2}.
// Coefficients = 6-point Lagrange interpolation at the midpoint: (3,-25,150,150,-25,3)/256.
double int6(const double b[6]) {
    return (150.0 / 256.0) * (b[2] + b[3]) - (25.0 / 256.0) * (b[1] + b[4]) +
           (3.0 / 256.0) * (b[0] + b[5]);
}

// ----------------------------------------------------------------------------------
// O6 — DER: high-order correction turning face point values F into the "hatted" numerical
// flux whose two-point difference is a 6th-order derivative of the point values (eq.(9),
// P:L120; "DER procedure").  f[0..4] = F_{i-3/2}, F_{i-1/2}, F_{i+1/2}, F_{i+3/2},
// F_{i+5/2}; returns F^_{i+1/2}.  (d0,d2,d4) = (1067/960, -29/480, 3/640)
// == 1 - D^2/24 + 3 D^4/640 in terms of the second difference D^2.
double der5(const double f[5]) {
    const double d0 = 1067.0 / 960.0, d2 = -29.0 / 480.0, d4 = 3.0 / 640.0;
    return d0 * f[2] + d2 * (f[1] + f[3]) + d4 * (f[0] + f[4]);
}
// HO switch: second-order INT = two-point average, second-order DER = identity
double int_ho(const double b[6], int ho) { return ho ? int6(b) : 0.5 * (b[2] + b[3]); }
double der_ho(const double f[5], int ho) { return ho ? der5(f) : f[2]; }

// ----------------------------------------------------------------------------------
// O3 — REC: MP5 (Suresh & Huynh 1997) on POINT values ("five elements ... MP5 ...
// centered at cell i ... reconstructed value at the right intercell i+1/2").
// v[0..4] = v_{i-2}, v_{i-1}, v_i, v_{i+1}, v_{i+2}; returns the left-biased value at i+1/2.
double minmod2(double a, double b) {
    if (a > 0.0 && b > 0.0) return a < b ? a : b;
    if (a < 0.0 && b < 0.0) return a > b ? a : b;
    return 0.0;
}
double minmod4(double a, double b, double c, double d) {
    if (a > 0.0 && b > 0.0 && c > 0.0 && d > 0.0) return std::fmin(std::fmin(a, b), std::fmin(c, d));
    if (a < 0.0 && b < 0.0 && c < 0.0 && d < 0.0) return std::fmax(std::fmax(a, b), std::fmax(c, d));
    return 0.0;
}
double min3(double a, double b, double c) { return std::fmin(a, std::fmin(b, c)); }
double max3(double a, double b, double c) { return std::fmax(a, std::fmax(b, c)); }

double mp5(const double v[5]) {
    const double alpha = 4.0, eps = 1e-10;  // S2
    const double vm2 = v[0], vm1 = v[1], v0 = v[2], vp1 = v[3], vp2 = v[4];
    // 5-point Lagrange interpolation of point values at +1/2
    const double vor = (3.0 * vm2 - 20.0 * vm1 + 90.0 * v0 + 60.0 * vp1 - 5.0 * vp2) / 128.0;
    const double vmp = v0 + minmod2(vp1 - v0, alpha * (v0 - vm1));
    if ((vor - v0) * (vor - vmp) <= eps) return vor;
    const double dm1 = vm2 - 2.0 * vm1 + v0;
    const double d0 = vm1 - 2.0 * v0 + vp1;
    const double dp1 = v0 - 2.0 * vp1 + vp2;
    const double dm4p = minmod4(4.0 * d0 - dp1, 4.0 * dp1 - d0, d0, dp1);   // d^{M4}_{i+1/2}
    const double dm4m = minmod4(4.0 * dm1 - d0, 4.0 * d0 - dm1, dm1, d0);   // d^{M4}_{i-1/2}
    const double vul = v0 + alpha * (v0 - vm1);
    const double vav = 0.5 * (v0 + vp1);
    const double vmd = vav - 0.5 * dm4p;
    const double vlc = v0 + 0.5 * (v0 - vm1) + (4.0 / 3.0) * dm4m;
    const double vmin = std::fmax(min3(v0, vp1, vmd), min3(v0, vul, vlc));
    const double vmax = std::fmin(max3(v0, vp1, vmd), max3(v0, vul, vlc));
    return vor + minmod2(vmin - vor, vmax - vor);
}

// "Linear reconstruction rather than MP5": v_{i+1/2}^L = v_i + sigma_i / 2 with the limited slope
// sigma_i = MC(v_i - v_{i-1}, v_{i+1} - v_i), the monotonized-central limiter
//   MC(a, b) = minmod(2a, 2b, (a + b)/2)
// (reading O3b: the paper names no limiter; MC is the choice).  Same argument convention as mp5
// (v[0] and v[4] are not used), so the mirrored stencil gives the right-biased value.
double minmod3(double a, double b, double c) {
    if (a > 0.0 && b > 0.0 && c > 0.0) return std::fmin(a, std::fmin(b, c));
    if (a < 0.0 && b < 0.0 && c < 0.0) return std::fmax(a, std::fmax(b, c));
    return 0.0;
}
double tvd2(const double v[5]) {
    const double a = v[2] - v[1], b = v[3] - v[2];
    return v[2] + 0.5 * minmod3(2.0 * a, 2.0 * b, 0.5 * (a + b));
}
// REC of the scheme in force: rec = 5 -> MP5, rec = 2 -> limited linear
double rec_value(int which, const double v[5]) { return which == 2 ? tvd2(v) : mp5(v); }

// ----------------------------------------------------------------------------------
// Point physics.  A primitive state is q[8] = (rho, vx, vy, vz, p, Bx, By, Bz).
// Definitions: D = rho W, S = rho h W^2 v + E x B, U = rho h W^2 - p + (E^2+B^2)/2,
// W_ij = rho h W^2 v_i v_j - E_i E_j - B_i B_j + p_tot delta_ij, p_tot = p + (E^2+B^2)/2;
// ideal MHD E = -v x B; ideal gas h = 1 + g/(g-1) p/rho (eq.(6)).

void cross(const double a[3], const double b[3], double c[3]) {
    c[0] = a[1] * b[2] - a[2] * b[1];
    c[1] = a[2] * b[0] - a[0] * b[2];
    c[2] = a[0] * b[1] - a[1] * b[0];
}
double dot(const double a[3], const double b[3]) { return a[0] * b[0] + a[1] * b[1] + a[2] * b[2]; }

// physics_prim2cons: u[5] = (D, Sx, Sy, Sz, U)
void prim2cons(double gam, const double q[8], double u[5]) {
    const double rho = q[0], p = q[4];
    const double *v = q + 1, *B = q + 5;
    const double v2 = dot(v, v);
    const double W2 = 1.0 / (1.0 - v2);
    const double W = std::sqrt(W2);
    const double rhoh = rho + gam / (gam - 1.0) * p;
    const double y = rhoh * W2;
    double E[3], vxB[3], ExB[3];
    cross(v, B, vxB);
    for (int a = 0; a < 3; ++a) E[a] = -vxB[a];
    cross(E, B, ExB);
    const double E2 = dot(E, E), B2 = dot(B, B);
    u[0] = rho * W;
    for (int a = 0; a < 3; ++a) u[1 + a] = y * v[a] + ExB[a];
    u[4] = y - p + 0.5 * (E2 + B2);
}

// Physical flux along direction d (eq.(8)): F[5] for (D, Sx, Sy, Sz, U).
void phys_flux(double gam, const double q[8], int d, double F[5]) {
    const double rho = q[0], p = q[4];
    const double *v = q + 1, *B = q + 5;
    const double v2 = dot(v, v);
    const double W2 = 1.0 / (1.0 - v2);
    const double W = std::sqrt(W2);
    const double rhoh = rho + gam / (gam - 1.0) * p;
    const double y = rhoh * W2;
    double E[3], vxB[3], ExB[3];
    cross(v, B, vxB);
    for (int a = 0; a < 3; ++a) E[a] = -vxB[a];
    cross(E, B, ExB);
    const double ptot = p + 0.5 * (dot(E, E) + dot(B, B));
    F[0] = rho * W * v[d];
    for (int a = 0; a < 3; ++a)
        F[1 + a] = y * v[a] * v[d] - E[a] * E[d] - B[a] * B[d] + (a == d ? ptot : 0.0);
    F[4] = y * v[d] + ExB[d];
}

// UCT=NO: induction fluxes of the cell-centred B (eq.(8): dB/dt + curl E = 0, E = -v x B):
// F_d(B_i) = v_d B_i - v_i B_d  (zero for i = d).
void phys_flux_b(const double q[8], int d, double F[3]) {
    const double *v = q + 1, *B = q + 5;
    for (int a = 0; a < 3; ++a) F[a] = v[d] * B[a] - v[a] * B[d];
}

// O4 — fast characteristic speeds along d ("fast characteristic speeds"; S5):
// lam[0] = lambda_+, lam[1] = lambda_-.
void fast_speeds(double gam, const double q[8], int d, double lam[2]) {
    const double rho = q[0], p = q[4];
    const double *v = q + 1, *B = q + 5;
    const double v2 = dot(v, v), B2 = dot(B, B), vB = dot(v, B);
    const double rhoh = rho + gam / (gam - 1.0) * p;
    const double b2 = B2 * (1.0 - v2) + vB * vB;
    const double cs2 = gam * p / rhoh;
    const double ca2 = b2 / (rhoh + b2);
    const double a2 = cs2 + ca2 - cs2 * ca2;
    const double vd = v[d];
    const double den = 1.0 - v2 * a2;
    const double disc = a2 * (1.0 - v2) * ((1.0 - v2 * a2) - (1.0 - a2) * vd * vd);
    const double root = std::sqrt(disc);
    lam[0] = ((1.0 - a2) * vd + root) / den;
    lam[1] = ((1.0 - a2) * vd - root) / den;
}

// O5 — two-state HLL flux at a d-face (S4).  qL, qR carry the SAME normal B_d.
// F[5]; ex[4] = (a+, a-, vbar_{t1}, vbar_{t2}) with t1=(d+1)%3, t2=(d+2)%3 — the "fast
// characteristic speeds and contributions for UCT" that P:L129 says are stored.
void hll(double gam, const double qL[8], const double qR[8], int d, double F[5], double ex[4], double *FB = nullptr) {
    double lamL[2], lamR[2], FL[5], FR[5], UL[5], UR[5];
    fast_speeds(gam, qL, d, lamL);
    fast_speeds(gam, qR, d, lamR);
    const double ap = std::fmax(0.0, std::fmax(lamL[0], lamR[0]));
    const double am = std::fmax(0.0, std::fmax(-lamL[1], -lamR[1]));
    phys_flux(gam, qL, d, FL);
    phys_flux(gam, qR, d, FR);
    prim2cons(gam, qL, UL);
    prim2cons(gam, qR, UR);
    for (int c = 0; c < 5; ++c) F[c] = (ap * FL[c] + am * FR[c] - ap * am * (UR[c] - UL[c])) / (ap + am);
    if (FB) {   // UCT=NO: the same two-state formula for the three cell-centred B components
        double BL[3], BR[3];
        phys_flux_b(qL, d, BL);
        phys_flux_b(qR, d, BR);
        for (int a = 0; a < 3; ++a) FB[a] = (ap * BL[a] + am * BR[a] - ap * am * (qR[5 + a] - qL[5 + a])) / (ap + am);
    }
    const int t1 = (d + 1) % 3, t2 = (d + 2) % 3;
    ex[0] = ap;
    ex[1] = am;
    ex[2] = (ap * qL[1 + t1] + am * qR[1 + t1]) / (ap + am);
    ex[3] = (ap * qL[1 + t2] + am * qR[1 + t2]) / (ap + am);
}

// O2 — conservative -> primitive inversion, Newton on y = rho h W^2 ("iterative
// Newton scheme"; S7).  Returns the number of Newton updates applied (>=1) or -(count)
// on failure (cap, non-physical start).  q receives (rho, v, p); B is passed through.
struct C2PAux { double x, p, f, df; };

// x(y) = v^2 from the momentum relation; returns false if not evaluable / unphysical
bool c2p_eval(double gam, double D, double S2, double B2, double T, double U, double y, C2PAux &a) {
    if (!(y > 0.0) || !std::isfinite(y)) return false;
    const double g1 = (gam - 1.0) / gam;
    const double yb = y + B2;
    const double x = (S2 * y * y + T * (2.0 * y + B2)) / (y * y * yb * yb);
    if (!(x < 1.0) || !(x >= 0.0)) return false;
    const double omx = 1.0 - x;
    const double sq = std::sqrt(omx);
    const double p = g1 * (y * omx - D * sq);
    const double xp = -2.0 * (S2 * y * y * y + T * (3.0 * y * y + 3.0 * y * B2 + B2 * B2)) /
                      (y * y * y * yb * yb * yb);
    a.x = x;
    a.p = p;
    a.f = y - p + 0.5 * (1.0 + x) * B2 - T / (2.0 * y * y) - U;
    a.df = 1.0 - g1 * omx - g1 * (-y + D / (2.0 * sq)) * xp + 0.5 * B2 * xp + T / (y * y * y);
    return true;
}

// nsafe (optional, instrumentation for the pins only): receives the number of times the safeguard replaced an iterate.
int con2prim(double gam, const double u[5], const double B[3], double q[5], int *nsafe = nullptr) {
    const double tol = 1e-12;
    const int maxit = 30;
    const double D = u[0], *S = u + 1, U = u[4];
    const double S2 = dot(S, S), B2 = dot(B, B), SB = dot(S, B), T = SB * SB;
    double y = gam * (U - 0.5 * B2);  // upper bound of the root (O2)
    double ylast = y;
    C2PAux a;
    int it = 0;
    bool conv = false;
    const double nan = std::numeric_limits<double>::quiet_NaN();
    while (it < maxit) {
        if (!c2p_eval(gam, D, S2, B2, T, U, y, a)) {
            if (it == 0) break;  // the start itself is unphysical: fail
            ++it;                // safeguard: halve the step back towards the last valid iterate
            if (nsafe) ++*nsafe;
            y = 0.5 * (y + ylast);
            if (!std::isfinite(y)) break;
            continue;
        }
        ylast = y;
        const double dy = -a.f / a.df;
        y = y + dy;
        ++it;
        if (std::fabs(dy) <= tol * std::fabs(y)) { conv = true; break; }
    }
    if (!conv || !c2p_eval(gam, D, S2, B2, T, U, y, a)) {
        q[0] = q[1] = q[2] = q[3] = q[4] = nan;
        return -(it > 0 ? it : 1);
    }
    q[0] = D * std::sqrt(1.0 - a.x);
    q[4] = a.p;
    for (int c = 0; c < 3; ++c) q[1 + c] = (S[c] + (SB / y) * B[c]) / (y + B2);
    return it;
}

// ----------------------------------------------------------------------------------
struct Grid {
    int n[3];
    double h[3];
    long N;
    long idx(int i, int j, int k) const { return (long)i + (long)n[0] * ((long)j + (long)n[1] * (long)k); }
    static int wrap(int a, int n) { int r = a % n; return r < 0 ? r + n : r; }
    // index of the cell reached from (c[0],c[1],c[2]) by s steps along direction d
    long shift(const int c[3], int d, int s) const {
        int cc[3] = {c[0], c[1], c[2]};
        cc[d] = wrap(cc[d] + s, n[d]);
        return idx(cc[0], cc[1], cc[2]);
    }
    long shift2(const int c[3], int d1, int s1, int d2, int s2) const {
        int cc[3] = {c[0], c[1], c[2]};
        cc[d1] = wrap(cc[d1] + s1, n[d1]);
        cc[d2] = wrap(cc[d2] + s2, n[d2]);
        return idx(cc[0], cc[1], cc[2]);
    }
};

#define FOR_CELLS(g, c)                                   \
    for (int c##k_ = 0; c##k_ < (g).n[2]; ++c##k_)       \
        for (int c##j_ = 0; c##j_ < (g).n[1]; ++c##j_)   \
            for (int c##i_ = 0; c##i_ < (g).n[0]; ++c##i_)
#define CELL(c) const int c[3] = {c##i_, c##j_, c##k_}

struct State {
    Field U[5];   // D, Sx, Sy, Sz, U at cell centres
    Field Bf[3];  // UCT=YES: staggered B_d at d-faces;  UCT=NO: the cell-centred B_d (evolved like U)
    void resize(long N) {
        for (auto &f : U) f.assign(N, 0.0);
        for (auto &f : Bf) f.assign(N, 0.0);
    }
};

struct Stats { long calls = 0, fails = 0, sumit = 0; int maxit = 0; };

struct Ctx {
    Grid g;
    double gam, cfl;
    int uct = 1, ho = 1;   // scheme switches
    int rec = 5, rk = 3;   // REC: 5 = MP5, 2 = limited linear; time stepping: SSP-RK3 or RK2
    State s;
    bool has_state = false;
    double t = 0.0, dt_last = 0.0, amax = 0.0;
    long steps = 0;
    Stats c2p;  // statistics of the most recent full-domain con2prim pass
    long c2p_fail_total = 0;
    // non-periodic boundaries: ghost width per axis (0 = periodic) and kind per (axis, side): 1 reflecting, 2 outflow
    int ng[3] = {0, 0, 0};
    int bc[3][2] = {{0, 0}, {0, 0}, {0, 0}};
    bool interior(const int c[3]) const {
        for (int d = 0; d < 3; ++d)
            if (c[d] < ng[d] || c[d] >= g.n[d] - ng[d]) return false;
        return true;
    }
    // d-faces of the interior: entry c is the face on the + side of cell c, so along d the low wall face (entry
    // ng - 1) belongs to it as well
    bool interior_face(const int c[3], int d) const {
        for (int a = 0; a < 3; ++a) {
            const int lo = (a == d && ng[a]) ? ng[a] - 1 : ng[a];
            if (c[a] < lo || c[a] >= g.n[a] - ng[a]) return false;
        }
        return true;
    }
};

// Ghost fill of the evolved fields of a bounded grid (state or, equally, its rhs: the rules are linear).  Along a
// bounded axis a with interior cells lo <= c_a < hi, ghost layer m = 0 .. NG-1:
//   cell-centred along a (D, S, U and the two transverse B components):
//        low:  ghost lo-1-m  <-  interior lo+m        high: ghost hi+m  <-  interior hi-1-m        (reflecting)
//        low:  ghost lo-1-m  <-  interior lo          high: ghost hi+m  <-  interior hi-1          (outflow)
//   B_a itself is staggered along a (entry c = face on the + side of cell c): the wall faces lo-1 and hi-1 are evolved,
//        low:  face lo-1-m   <-  face lo-1+m (m >= 1)  high: face hi-1+m <-  face hi-1-m (m >= 1)   (reflecting)
//        low:  face lo-1-m   <-  face lo-1   (m >= 1)  high: face hi-1+m <-  face hi-1   (m >= 1)   (outflow)
// Reflecting parity (the mirror symmetry of the equations, pinned for the periodic scheme by P7iv): scalars D, U even;
// the momentum component normal to the wall odd, the tangential ones even (polar vector); B_a even, the tangential B
// components odd (axial vector).  Axes are filled in the order x, y, z over the full padded extent of the other axes,
// so edges and corners get the composition of the two (three) rules.
void fill_ghosts(const Ctx &cx, Field U[5], Field Bf[3]) {
    const Grid &g = cx.g;
    for (int a = 0; a < 3; ++a) {
        const int NG = cx.ng[a];
        if (!NG) continue;
        const int lo = NG, hi = g.n[a] - NG;
        for (int side = 0; side < 2; ++side) {
            const int kind = cx.bc[a][side];
            FOR_CELLS(g, c) {
                CELL(c);
                const int ca = c[a];
                const bool ghost = side == 0 ? ca < lo : ca >= hi;
                if (!ghost) continue;
                const int m = side == 0 ? lo - 1 - ca : ca - hi;          // ghost layer 0 .. NG-1
                int src[3] = {c[0], c[1], c[2]};
                const long dst = g.idx(c[0], c[1], c[2]);
                // cell-centred fields
                src[a] = kind == 1 ? (side == 0 ? lo + m : hi - 1 - m) : (side == 0 ? lo : hi - 1);
                const long sc = g.idx(src[0], src[1], src[2]);
                for (int v = 0; v < 5; ++v) {
                    const double sgn = (kind == 1 && v == 1 + a) ? -1.0 : 1.0;   // normal momentum is odd
                    U[v][dst] = sgn * U[v][sc];
                }
                for (int b = 0; b < 3; ++b)
                    if (b != a) Bf[b][dst] = (kind == 1 ? -1.0 : 1.0) * Bf[b][sc];   // tangential B is odd
                // the normal B: faces; the wall face (low side: entry lo-1) is not a ghost
                const int mf = side == 0 ? lo - 1 - ca : ca - (hi - 1);   // distance of this face from the wall face
                if (mf >= 1) {
                    src[a] = kind == 1 ? (side == 0 ? lo - 1 + mf : hi - 1 - mf) : (side == 0 ? lo - 1 : hi - 1);
                    Bf[a][dst] = Bf[a][g.idx(src[0], src[1], src[2])];
                }
            }
        }
    }
}

// Step 1 of a sub-step: INT of the staggered B to centres, then con2prim everywhere.
void centre_b(const Grid &g, const Field Bf[3], Field Bc[3], int ho = 1) {
    for (int d = 0; d < 3; ++d) {
        Bc[d].assign(g.N, 0.0);
        FOR_CELLS(g, c) {
            CELL(c);
            double b[6];
            for (int m = 0; m < 6; ++m) b[m] = Bf[d][g.shift(c, d, m - 3)];  // faces i-5/2 .. i+5/2
            Bc[d][g.idx(c[0], c[1], c[2])] = int_ho(b, ho);
        }
    }
}

void primitives(const Ctx &cx, const State &s, Field P[5], Field Bc[3], Stats &st) {
    const Grid &g = cx.g;
    if (cx.uct) centre_b(g, s.Bf, Bc, cx.ho);
    else for (int d = 0; d < 3; ++d) Bc[d] = s.Bf[d];   // UCT=NO: the evolved field is already cell-centred
    for (int v = 0; v < 5; ++v) P[v].assign(g.N, 0.0);
    st = Stats();
    FOR_CELLS(g, cc) {
        CELL(cc);
        const long c = g.idx(cc[0], cc[1], cc[2]);
        const double u[5] = {s.U[0][c], s.U[1][c], s.U[2][c], s.U[3][c], s.U[4][c]};
        const double B[3] = {Bc[0][c], Bc[1][c], Bc[2][c]};
        double q[5];
        const int it = con2prim(cx.gam, u, B, q);
        for (int v = 0; v < 5; ++v) P[v][c] = q[v];
        if (!cx.interior(cc)) continue;   // ghost cells of a bounded grid: inverted, but not part of the statistics
        ++st.calls;
        if (it < 0) ++st.fails;
        const int ai = it < 0 ? -it : it;
        st.sumit += ai;
        if (ai > st.maxit) st.maxit = ai;
    }
}

struct Rhs {
    Field U[5];
    Field B[3];
    Field E[3];      // edge EMFs (kept for tests)
    Field F[3][5];   // face fluxes per direction (kept for tests)
    Field FB[3][3];  // UCT=NO: face fluxes of the three cell-centred B components, per direction
    double amax;
};

// The spatial operator L(U) of eq.(9)-(10): points 1-4 of P:L128-135.
void compute_rhs(Ctx &cx, const State &s, Rhs &r) {
    const Grid &g = cx.g;
    const double gam = cx.gam;
    Field P[5], Bc[3];
    primitives(cx, s, P, Bc, cx.c2p);
    cx.c2p_fail_total += cx.c2p.fails;

    // ---- point 2: per direction REC -> L/R -> HLL flux; store speeds + UCT pieces
    Field ap[3], am[3], vbar[3][2];
    double amax = 0.0;
    for (int d = 0; d < 3; ++d) {
        const int t1 = (d + 1) % 3, t2 = (d + 2) % 3;
        for (int c = 0; c < 5; ++c) r.F[d][c].assign(g.N, 0.0);
        for (int a = 0; a < 3; ++a) r.FB[d][a].assign(cx.uct ? 0 : g.N, 0.0);
        ap[d].assign(g.N, 0.0);
        am[d].assign(g.N, 0.0);
        vbar[d][0].assign(g.N, 0.0);
        vbar[d][1].assign(g.N, 0.0);
        FOR_CELLS(g, c) {
            CELL(c);
            const long i0 = g.idx(c[0], c[1], c[2]);
            long nb[6];  // cells i-2 .. i+3 along d
            for (int m = 0; m < 6; ++m) nb[m] = g.shift(c, d, m - 2);
            double qL[8], qR[8];
            // reconstructed: rho, vx, vy, vz, p and the two transverse centre-B components (S3)
            const Field *rec[7] = {&P[0], &P[1], &P[2], &P[3], &P[4], &Bc[t1], &Bc[t2]};
            const int slot[7] = {0, 1, 2, 3, 4, 5 + t1, 5 + t2};
            for (int v = 0; v < 7; ++v) {
                const Field &f = *rec[v];
                const double sl[5] = {f[nb[0]], f[nb[1]], f[nb[2]], f[nb[3]], f[nb[4]]};
                const double sr[5] = {f[nb[5]], f[nb[4]], f[nb[3]], f[nb[2]], f[nb[1]]};  // mirrored
                qL[slot[v]] = rec_value(cx.rec, sl);
                qR[slot[v]] = rec_value(cx.rec, sr);
            }
            double F[5], ex[4], FB[3];
            if (cx.uct) {
                qL[5 + d] = qR[5 + d] = s.Bf[d][i0];  // the normal B is the staggered value itself
                hll(gam, qL, qR, d, F, ex);
            } else {                                  // UCT=NO: the normal B is reconstructed like the rest
                const Field &f = Bc[d];
                const double sl[5] = {f[nb[0]], f[nb[1]], f[nb[2]], f[nb[3]], f[nb[4]]};
                const double sr[5] = {f[nb[5]], f[nb[4]], f[nb[3]], f[nb[2]], f[nb[1]]};
                qL[5 + d] = rec_value(cx.rec, sl);
                qR[5 + d] = rec_value(cx.rec, sr);
                hll(gam, qL, qR, d, F, ex, FB);
                for (int a = 0; a < 3; ++a) r.FB[d][a][i0] = FB[a];
            }
            for (int cc = 0; cc < 5; ++cc) r.F[d][cc][i0] = F[cc];
            ap[d][i0] = ex[0];
            am[d][i0] = ex[1];
            vbar[d][0][i0] = ex[2];
            vbar[d][1][i0] = ex[3];
            if (cx.interior_face(c, d)) amax = std::fmax(amax, std::fmax(ex[0], ex[1]));  // point 5
        }
    }
    r.amax = amax;

    // ---- point 3: DER + divergence, per direction; sources vanish (Minkowski)
    for (int c = 0; c < 5; ++c) r.U[c].assign(g.N, 0.0);
    for (int a = 0; a < 3; ++a) r.B[a].assign(g.N, 0.0);
    for (int d = 0; d < 3; ++d) {
        for (int cc = 0; cc < (cx.uct ? 5 : 8); ++cc) {
            const Field &F = cc < 5 ? r.F[d][cc] : r.FB[d][cc - 5];
            Field &out = cc < 5 ? r.U[cc] : r.B[cc - 5];
            Field Fh(g.N);
            FOR_CELLS(g, c) {
                CELL(c);
                double f[5];
                for (int m = 0; m < 5; ++m) f[m] = F[g.shift(c, d, m - 2)];
                Fh[g.idx(c[0], c[1], c[2])] = der_ho(f, cx.ho);
            }
            FOR_CELLS(g, c) {
                CELL(c);
                const long i0 = g.idx(c[0], c[1], c[2]);
                out[i0] -= (Fh[i0] - Fh[g.shift(c, d, -1)]) / g.h[d];
            }
        }
    }
    if (!cx.uct) {   // UCT=NO: no edge EMFs, the rhs of the cell-centred B is the flux divergence above
        for (int k = 0; k < 3; ++k) r.E[k].assign(g.N, 0.0);
        return;
    }

    // ---- point 4: UCT edge EMFs with REC + upwind formula (O7)
    for (int k = 0; k < 3; ++k) {
        const int i = (k + 1) % 3, j = (k + 2) % 3;
        r.E[k].assign(g.N, 0.0);
        // v_i saved at j-faces: direction j has transverse slots t1=(j+1)%3=k, t2=(j+2)%3=i
        const Field &vi_at_j = vbar[j][1];
        // v_j saved at i-faces: direction i has t1=(i+1)%3=j
        const Field &vj_at_i = vbar[i][0];
        FOR_CELLS(g, c) {
            CELL(c);
            const long i0 = g.idx(c[0], c[1], c[2]);
            // first bracket: j-face quantities reconstructed along i
            double sl[5], sr[5];
            long nbi[6], nbj[6];
            for (int m = 0; m < 6; ++m) { nbi[m] = g.shift(c, i, m - 2); nbj[m] = g.shift(c, j, m - 2); }
            for (int m = 0; m < 5; ++m) { sl[m] = vi_at_j[nbi[m]]; sr[m] = vi_at_j[nbi[5 - m]]; }
            const double viL = rec_value(cx.rec, sl), viR = rec_value(cx.rec, sr);
            for (int m = 0; m < 5; ++m) { sl[m] = s.Bf[j][nbi[m]]; sr[m] = s.Bf[j][nbi[5 - m]]; }
            const double BjL = rec_value(cx.rec, sl), BjR = rec_value(cx.rec, sr);
            // second bracket: i-face quantities reconstructed along j
            for (int m = 0; m < 5; ++m) { sl[m] = vj_at_i[nbj[m]]; sr[m] = vj_at_i[nbj[5 - m]]; }
            const double vjL = rec_value(cx.rec, sl), vjR = rec_value(cx.rec, sr);
            for (int m = 0; m < 5; ++m) { sl[m] = s.Bf[i][nbj[m]]; sr[m] = s.Bf[i][nbj[5 - m]]; }
            const double BiL = rec_value(cx.rec, sl), BiR = rec_value(cx.rec, sr);
            // edge speeds: max over the two faces adjacent to the edge
            const long cj = g.shift(c, j, 1), ci = g.shift(c, i, 1);
            const double aip = std::fmax(ap[i][i0], ap[i][cj]), aim = std::fmax(am[i][i0], am[i][cj]);
            const double ajp = std::fmax(ap[j][i0], ap[j][ci]), ajm = std::fmax(am[j][i0], am[j][ci]);
            r.E[k][i0] = -(aip * viL * BjL + aim * viR * BjR - aip * aim * (BjR - BjL)) / (aip + aim) +
                         (ajp * vjL * BiL + ajm * vjR * BiR - ajp * ajm * (BiR - BiL)) / (ajp + ajm);
        }
    }

    // ---- point 4, second half (eq.(10)): curl of the hatted EMFs (O8)
    for (int i = 0; i < 3; ++i) {
        const int j = (i + 1) % 3, k = (i + 2) % 3;
        Field Ekh(g.N), Ejh(g.N);  // DER of E_k along j, DER of E_j along k
        FOR_CELLS(g, c) {
            CELL(c);
            double f[5];
            for (int m = 0; m < 5; ++m) f[m] = r.E[k][g.shift(c, j, m - 2)];
            Ekh[g.idx(c[0], c[1], c[2])] = der_ho(f, cx.ho);
            for (int m = 0; m < 5; ++m) f[m] = r.E[j][g.shift(c, k, m - 2)];
            Ejh[g.idx(c[0], c[1], c[2])] = der_ho(f, cx.ho);
        }
        r.B[i].assign(g.N, 0.0);
        FOR_CELLS(g, c) {
            CELL(c);
            const long i0 = g.idx(c[0], c[1], c[2]);
            r.B[i][i0] = -((Ekh[i0] - Ekh[g.shift(c, j, -1)]) / g.h[j] - (Ejh[i0] - Ejh[g.shift(c, k, -1)]) / g.h[k]);
        }
    }
}

// O9 — SSP-RK3 (S8), dt from the stage-1 speeds of the same step (S9).
void rk3_step(Ctx &cx, double t_end) {
    const Grid &g = cx.g;
    State &s = cx.s;
    fill_ghosts(cx, s.U, s.Bf);          // (bounded grids only; no-op on a periodic box)
    State s0 = s;
    Rhs r;
    compute_rhs(cx, s, r);
    cx.amax = r.amax;
    double hmin = std::fmin(g.h[0], std::fmin(g.h[1], g.h[2]));
    double dt = cx.cfl * hmin / r.amax;
    if (cx.t + dt > t_end) dt = t_end - cx.t;
    for (long c = 0; c < g.N; ++c) {
        for (int v = 0; v < 5; ++v) s.U[v][c] = s0.U[v][c] + dt * r.U[v][c];
        for (int v = 0; v < 3; ++v) s.Bf[v][c] = s0.Bf[v][c] + dt * r.B[v][c];
    }
    fill_ghosts(cx, s.U, s.Bf);
    compute_rhs(cx, s, r);
    for (long c = 0; c < g.N; ++c) {
        for (int v = 0; v < 5; ++v) s.U[v][c] = 0.75 * s0.U[v][c] + 0.25 * (s.U[v][c] + dt * r.U[v][c]);
        for (int v = 0; v < 3; ++v) s.Bf[v][c] = 0.75 * s0.Bf[v][c] + 0.25 * (s.Bf[v][c] + dt * r.B[v][c]);
    }
    fill_ghosts(cx, s.U, s.Bf);
    compute_rhs(cx, s, r);
    for (long c = 0; c < g.N; ++c) {
        for (int v = 0; v < 5; ++v)
            s.U[v][c] = (1.0 / 3.0) * s0.U[v][c] + (2.0 / 3.0) * (s.U[v][c] + dt * r.U[v][c]);
        for (int v = 0; v < 3; ++v)
            s.Bf[v][c] = (1.0 / 3.0) * s0.Bf[v][c] + (2.0 / 3.0) * (s.Bf[v][c] + dt * r.B[v][c]);
    }
    fill_ghosts(cx, s.U, s.Bf);
    cx.t += dt;
    cx.dt_last = dt;
    ++cx.steps;
}

// "Second order time-stepping": the two-stage SSP Runge-Kutta scheme (Heun),
//   U1 = U^n + dt L(U^n),  U^{n+1} = 1/2 U^n + 1/2 (U1 + dt L(U1)),   dt as in rk3_step (S9).
void rk2_step(Ctx &cx, double t_end) {
    const Grid &g = cx.g;
    State &s = cx.s;
    State s0 = s;
    Rhs r;
    compute_rhs(cx, s, r);
    cx.amax = r.amax;
    double hmin = std::fmin(g.h[0], std::fmin(g.h[1], g.h[2]));
    double dt = cx.cfl * hmin / r.amax;
    if (cx.t + dt > t_end) dt = t_end - cx.t;
    for (long c = 0; c < g.N; ++c) {
        for (int v = 0; v < 5; ++v) s.U[v][c] = s0.U[v][c] + dt * r.U[v][c];
        for (int v = 0; v < 3; ++v) s.Bf[v][c] = s0.Bf[v][c] + dt * r.B[v][c];
    }
    compute_rhs(cx, s, r);
    for (long c = 0; c < g.N; ++c) {
        for (int v = 0; v < 5; ++v) s.U[v][c] = 0.5 * s0.U[v][c] + 0.5 * (s.U[v][c] + dt * r.U[v][c]);
        for (int v = 0; v < 3; ++v) s.Bf[v][c] = 0.5 * s0.Bf[v][c] + 0.5 * (s.Bf[v][c] + dt * r.B[v][c]);
    }
    cx.t += dt;
    cx.dt_last = dt;
    ++cx.steps;
}

// S10 — the discrete divergence that UCT + DER preserves: sum_d D_d[DER_d B_d].
void div_b(const Grid &g, const Field Bf[3], Field &div, int ho = 1) {
    div.assign(g.N, 0.0);
    for (int d = 0; d < 3; ++d) {
        Field Bh(g.N);
        FOR_CELLS(g, c) {
            CELL(c);
            double f[5];
            for (int m = 0; m < 5; ++m) f[m] = Bf[d][g.shift(c, d, m - 2)];
            Bh[g.idx(c[0], c[1], c[2])] = der_ho(f, ho);
        }
        FOR_CELLS(g, c) {
            CELL(c);
            const long i0 = g.idx(c[0], c[1], c[2]);
            div[i0] += (Bh[i0] - Bh[g.shift(c, d, -1)]) / g.h[d];
        }
    }
}

// S11 — staggered B from an edge-centred vector potential: the same discrete curl as O8
// (B = +curl A), so that div_b of the result vanishes to round-off for any A.
void curl_of_potential(const Grid &g, const double *const A[3], double *const B[3], int ho = 1) {
    for (int i = 0; i < 3; ++i) {
        const int j = (i + 1) % 3, k = (i + 2) % 3;
        Field Akh(g.N), Ajh(g.N);
        FOR_CELLS(g, c) {
            CELL(c);
            double f[5];
            for (int m = 0; m < 5; ++m) f[m] = A[k][g.shift(c, j, m - 2)];
            Akh[g.idx(c[0], c[1], c[2])] = der_ho(f, ho);
            for (int m = 0; m < 5; ++m) f[m] = A[j][g.shift(c, k, m - 2)];
            Ajh[g.idx(c[0], c[1], c[2])] = der_ho(f, ho);
        }
        FOR_CELLS(g, c) {
            CELL(c);
            const long i0 = g.idx(c[0], c[1], c[2]);
            B[i][i0] = (Akh[i0] - Akh[g.shift(c, j, -1)]) / g.h[j] - (Ajh[i0] - Ajh[g.shift(c, k, -1)]) / g.h[k];
        }
    }
}

Grid make_grid(int nx, int ny, int nz) {
    Grid g;
    g.n[0] = nx; g.n[1] = ny; g.n[2] = nz;
    for (int d = 0; d < 3; ++d) g.h[d] = 1.0 / g.n[d];
    g.N = (long)nx * ny * nz;
    return g;
}

}  // namespace

// ====================================================================================
// C ABI for ctypes (host pointers everywhere).  Return 0 on success, <0 on error.
extern "C" {

void *oracle_create(int nx, int ny, int nz, double gamma, double cfl) {
    if (nx < 1 || ny < 1 || nz < 1 || !(gamma > 1.0) || !(cfl > 0.0)) return nullptr;
    Ctx *cx = new Ctx();
    cx->g = make_grid(nx, ny, nz);
    cx->gam = gamma;
    cx->cfl = cfl;
    cx->s.resize(cx->g.N);
    return cx;
}

void oracle_destroy(void *h) { delete static_cast<Ctx *>(h); }

// Bounded grid (row f4): nx, ny, nz INTERIOR cells with the spacing h_d = 1/gn_d of a unit box of gn cells (gn = NULL:
// gn_d = n_d, the interior IS the unit box); kinds[2 a + side] = 0 periodic axis
// (both sides), 1 reflecting wall, 2 zero-gradient outflow.  Every array passed in or out then has n_d + 16 entries
// along a bounded axis (8 ghost layers on each side); ghost entries given to oracle_set_primitives are ignored
// except the normal B at the low wall face (entry 7 of that axis).  UCT=HO=YES, MP5, RK3 only.
void *oracle_create_bounded(int nx, int ny, int nz, double gamma, double cfl, const int *kinds, const int *gn) {
    if (nx < 1 || ny < 1 || nz < 1 || !(gamma > 1.0) || !(cfl > 0.0) || !kinds) return nullptr;
    const int n[3] = {nx, ny, nz};
    int ng[3];
    for (int a = 0; a < 3; ++a) {
        const int k0 = kinds[2 * a], k1 = kinds[2 * a + 1];
        if ((k0 == 0) != (k1 == 0) || k0 < 0 || k0 > 2 || k1 < 0 || k1 > 2) return nullptr;
        ng[a] = k0 ? 8 : 0;
        if (ng[a] && n[a] < 8) return nullptr;
    }
    Ctx *cx = new Ctx();
    cx->g = make_grid(nx + 2 * ng[0], ny + 2 * ng[1], nz + 2 * ng[2]);
    for (int a = 0; a < 3; ++a) {
        if (gn && gn[a] < 1) { delete cx; return nullptr; }
        cx->g.h[a] = 1.0 / (gn ? gn[a] : n[a]);
        cx->ng[a] = ng[a];
        cx->bc[a][0] = kinds[2 * a];
        cx->bc[a][1] = kinds[2 * a + 1];
    }
    cx->gam = gamma;
    cx->cfl = cfl;
    cx->s.resize(cx->g.N);
    return cx;
}

// Scheme switches of the paper; call before oracle_set_primitives.  With uct = 0 the three
// "face" arrays of set/get_primitives are the CELL-CENTRED B.
int oracle_set_scheme(void *h, int uct, int ho) {
    Ctx *cx = static_cast<Ctx *>(h);
    if (!cx || cx->has_state) return -4;
    cx->uct = uct ? 1 : 0;
    cx->ho = ho ? 1 : 0;
    return 0;
}

// Order switches of P:L304 ("second order time-stepping and linear reconstruction rather than MP5"); call before
// oracle_set_primitives.  rec: 5 = MP5 (default), 2 = limited linear (MC); rk: 3 = SSP-RK3 (default), 2 = SSP-RK2.
int oracle_set_order(void *h, int rec, int rk) {
    Ctx *cx = static_cast<Ctx *>(h);
    if (!cx || cx->has_state) return -4;
    if ((rec != 5 && rec != 2) || (rk != 3 && rk != 2)) return -1;
    cx->rec = rec;
    cx->rk = rk;
    return 0;
}
double oracle_tvd2(const double v[5]) { return tvd2(v); }

// faces from an edge potential with the second-order (HO=NO) or sixth-order curl
int oracle_faces_from_potential_ho(int nx, int ny, int nz, int ho, const double *ax, const double *ay, const double *az,
                                   double *bx, double *by, double *bz) {
    if (nx < 1 || ny < 1 || nz < 1) return -1;
    Grid g;
    g.n[0] = nx; g.n[1] = ny; g.n[2] = nz;
    for (int d = 0; d < 3; ++d) g.h[d] = 1.0 / g.n[d];
    g.N = (long)nx * ny * nz;
    const double *const A[3] = {ax, ay, az};
    double *const B[3] = {bx, by, bz};
    curl_of_potential(g, A, B, ho);
    return 0;
}

// Cell-centred rho, v, p and face-staggered B point values -> conserved state; t = 0.
int oracle_set_primitives(void *h, const double *rho, const double *vx, const double *vy, const double *vz,
                          const double *p, const double *bxf, const double *byf, const double *bzf) {
    Ctx *cx = static_cast<Ctx *>(h);
    if (!cx) return -1;
    const Grid &g = cx->g;
    const double *bf[3] = {bxf, byf, bzf};
    for (int d = 0; d < 3; ++d) cx->s.Bf[d].assign(bf[d], bf[d] + g.N);
    {   // bounded grids: the ghost layers of B come from the interior before INT reads them
        Field dummy[5];
        for (auto &f : dummy) f.assign(g.N, 0.0);
        fill_ghosts(*cx, dummy, cx->s.Bf);
    }
    Field Bc[3];
    if (cx->uct) centre_b(g, cx->s.Bf, Bc, cx->ho);
    else for (int d = 0; d < 3; ++d) Bc[d] = cx->s.Bf[d];   // UCT=NO: the arrays given are cell-centred
    for (long c = 0; c < g.N; ++c) {
        const double q[8] = {rho[c], vx[c], vy[c], vz[c], p[c], Bc[0][c], Bc[1][c], Bc[2][c]};
        double u[5];
        prim2cons(cx->gam, q, u);
        for (int v = 0; v < 5; ++v) cx->s.U[v][c] = u[v];
    }
    fill_ghosts(*cx, cx->s.U, cx->s.Bf);
    cx->t = 0.0; cx->dt_last = 0.0; cx->amax = 0.0; cx->steps = 0;
    cx->c2p = Stats(); cx->c2p_fail_total = 0;
    cx->has_state = true;
    return 0;
}

// Advance nsteps full RK3 steps, or fewer if t reaches t_end (last dt clipped).  Returns steps taken.
int oracle_step(void *h, int nsteps, double t_end) {
    Ctx *cx = static_cast<Ctx *>(h);
    if (!cx || !cx->has_state) return -4;
    int done = 0;
    for (int s = 0; s < nsteps; ++s) {
        if (!(cx->t < t_end)) break;
        if (cx->rk == 2) rk2_step(*cx, t_end);
        else rk3_step(*cx, t_end);
        ++done;
    }
    return done;
}

int oracle_get_primitives(void *h, double *rho, double *vx, double *vy, double *vz, double *p, double *bxc,
                          double *byc, double *bzc, double *bxf, double *byf, double *bzf) {
    Ctx *cx = static_cast<Ctx *>(h);
    if (!cx || !cx->has_state) return -4;
    const Grid &g = cx->g;
    Field P[5], Bc[3];
    Stats st;
    primitives(*cx, cx->s, P, Bc, st);
    double *out[8] = {rho, vx, vy, vz, p, bxc, byc, bzc};
    for (int v = 0; v < 5; ++v) std::memcpy(out[v], P[v].data(), sizeof(double) * g.N);
    for (int d = 0; d < 3; ++d) std::memcpy(out[5 + d], Bc[d].data(), sizeof(double) * g.N);
    double *bf[3] = {bxf, byf, bzf};
    for (int d = 0; d < 3; ++d)
        if (bf[d]) std::memcpy(bf[d], cx->s.Bf[d].data(), sizeof(double) * g.N);
    return st.fails ? -5 : 0;
}

int oracle_get_conserved(void *h, double *D, double *Sx, double *Sy, double *Sz, double *U) {
    Ctx *cx = static_cast<Ctx *>(h);
    if (!cx || !cx->has_state) return -4;
    double *out[5] = {D, Sx, Sy, Sz, U};
    for (int v = 0; v < 5; ++v) std::memcpy(out[v], cx->s.U[v].data(), sizeof(double) * cx->g.N);
    return 0;
}

// L(U) of the current state and its intermediates: out arrays may be NULL.
// rhsU: 5 arrays, rhsB: 3 face arrays, E: 3 edge arrays, F: 15 arrays (d-major), amax: scalar.
int oracle_rhs(void *h, double *const *rhsU, double *const *rhsB, double *const *E, double *const *F, double *amax) {
    Ctx *cx = static_cast<Ctx *>(h);
    if (!cx || !cx->has_state) return -4;
    Rhs r;
    compute_rhs(*cx, cx->s, r);
    const size_t nb = sizeof(double) * cx->g.N;
    if (rhsU) for (int v = 0; v < 5; ++v) std::memcpy(rhsU[v], r.U[v].data(), nb);
    if (rhsB) for (int v = 0; v < 3; ++v) std::memcpy(rhsB[v], r.B[v].data(), nb);
    if (E) for (int v = 0; v < 3; ++v) std::memcpy(E[v], r.E[v].data(), nb);
    if (F) for (int d = 0; d < 3; ++d) for (int v = 0; v < 5; ++v) std::memcpy(F[d * 5 + v], r.F[d][v].data(), nb);
    if (amax) *amax = r.amax;
    return 0;
}

int oracle_con2prim(double gamma, long n, const double *D, const double *Sx, const double *Sy, const double *Sz,
                    const double *U, const double *Bx, const double *By, const double *Bz, double *rho, double *vx,
                    double *vy, double *vz, double *p, int *iters) {
    int bad = 0;
    for (long c = 0; c < n; ++c) {
        const double u[5] = {D[c], Sx[c], Sy[c], Sz[c], U[c]};
        const double B[3] = {Bx[c], By[c], Bz[c]};
        double q[5];
        const int it = con2prim(gamma, u, B, q);
        rho[c] = q[0]; vx[c] = q[1]; vy[c] = q[2]; vz[c] = q[3]; p[c] = q[4];
        if (iters) iters[c] = it;
        if (it < 0) bad = 1;
    }
    return bad ? -5 : 0;
}

// the same, also reporting how often the safeguard of O2 replaced an iterate (nsafe[i]); same arithmetic
int oracle_con2prim_trace(double gamma, long n, const double *D, const double *Sx, const double *Sy, const double *Sz,
                          const double *U, const double *Bx, const double *By, const double *Bz, double *rho, double *vx,
                          double *vy, double *vz, double *p, int *iters, int *nsafe) {
    int bad = 0;
    for (long c = 0; c < n; ++c) {
        const double u[5] = {D[c], Sx[c], Sy[c], Sz[c], U[c]};
        const double B[3] = {Bx[c], By[c], Bz[c]};
        double q[5];
        nsafe[c] = 0;
        const int it = con2prim(gamma, u, B, q, &nsafe[c]);
        rho[c] = q[0]; vx[c] = q[1]; vy[c] = q[2]; vz[c] = q[3]; p[c] = q[4];
        iters[c] = it;
        if (it < 0) bad = 1;
    }
    return bad ? -5 : 0;
}

int oracle_prim2cons(double gamma, long n, const double *rho, const double *vx, const double *vy, const double *vz,
                     const double *p, const double *Bx, const double *By, const double *Bz, double *D, double *Sx,
                     double *Sy, double *Sz, double *U) {
    for (long c = 0; c < n; ++c) {
        const double q[8] = {rho[c], vx[c], vy[c], vz[c], p[c], Bx[c], By[c], Bz[c]};
        double u[5];
        prim2cons(gamma, q, u);
        D[c] = u[0]; Sx[c] = u[1]; Sy[c] = u[2]; Sz[c] = u[3]; U[c] = u[4];
    }
    return 0;
}

int oracle_div_b(void *h, double *div_field, double *max_abs) {
    Ctx *cx = static_cast<Ctx *>(h);
    if (!cx || !cx->has_state) return -4;
    Field div;
    div_b(cx->g, cx->s.Bf, div, cx->ho);
    double m = 0.0;
    for (long c = 0; c < cx->g.N; ++c) m = std::fmax(m, std::fabs(div[c]));
    if (div_field) std::memcpy(div_field, div.data(), sizeof(double) * cx->g.N);
    if (max_abs) *max_abs = m;
    return 0;
}

// out[24] = {t, dt_last, steps, amax, sum D, sum Sx, sum Sy, sum Sz, sum U (x cell volume),
//            sum Bx, sum By, sum Bz over faces (x volume), max|div_HO B|, max W, min rho, min p,
//            c2p max iterations, c2p mean iterations, c2p failures (since set_primitives), 0...}
int oracle_diagnostics(void *h, double out[24]) {
    Ctx *cx = static_cast<Ctx *>(h);
    if (!cx || !cx->has_state) return -4;
    const Grid &g = cx->g;
    for (int m = 0; m < 24; ++m) out[m] = 0.0;
    out[0] = cx->t; out[1] = cx->dt_last; out[2] = (double)cx->steps; out[3] = cx->amax;
    const double vol = g.h[0] * g.h[1] * g.h[2];
    for (int v = 0; v < 5; ++v) {
        long double sum = 0.0L;  // extended accumulation: drift at 1e-15 must be measurable (P4)
        for (long c = 0; c < g.N; ++c) sum += cx->s.U[v][c];
        out[4 + v] = (double)(sum * vol);
    }
    for (int d = 0; d < 3; ++d) {
        long double sum = 0.0L;
        for (long c = 0; c < g.N; ++c) sum += cx->s.Bf[d][c];
        out[9 + d] = (double)(sum * vol);
    }
    Field div;
    div_b(g, cx->s.Bf, div, cx->ho);   // (UCT=NO: the same stencil applied to the cell-centred field; not preserved)
    double m = 0.0;
    for (long c = 0; c < g.N; ++c) m = std::fmax(m, std::fabs(div[c]));
    out[12] = m;
    Field P[5], Bc[3];
    Stats st;
    primitives(*cx, cx->s, P, Bc, st);
    double wmax = 0.0, rmin = std::numeric_limits<double>::infinity(), pmin = rmin;
    for (long c = 0; c < g.N; ++c) {
        const double v2 = P[1][c] * P[1][c] + P[2][c] * P[2][c] + P[3][c] * P[3][c];
        wmax = std::fmax(wmax, 1.0 / std::sqrt(1.0 - v2));
        rmin = std::fmin(rmin, P[0][c]);
        pmin = std::fmin(pmin, P[4][c]);
    }
    out[13] = wmax; out[14] = rmin; out[15] = pmin;
    out[16] = (double)st.maxit;
    out[17] = st.calls ? (double)st.sumit / (double)st.calls : 0.0;
    out[18] = (double)(cx->c2p_fail_total + st.fails);
    return 0;
}

int oracle_faces_from_potential(int nx, int ny, int nz, const double *ax, const double *ay, const double *az,
                                double *bx, double *by, double *bz) {
    if (nx < 1 || ny < 1 || nz < 1) return -1;
    const Grid g = make_grid(nx, ny, nz);
    const double *const A[3] = {ax, ay, az};
    double *const B[3] = {bx, by, bz};
    curl_of_potential(g, A, B);
    return 0;
}

// ---- unit-level entry points for the pins -----------------------------------------
double oracle_int6(const double b[6]) { return int6(b); }
double oracle_der5(const double f[5]) { return der5(f); }
double oracle_mp5(const double v[5]) { return mp5(v); }
void oracle_fast_speeds(double gamma, const double q[8], int d, double lam[2]) { fast_speeds(gamma, q, d, lam); }
void oracle_phys_flux(double gamma, const double q[8], int d, double F[5]) { phys_flux(gamma, q, d, F); }
void oracle_hll(double gamma, const double qL[8], const double qR[8], int d, double F[5], double ex[4]) {
    hll(gamma, qL, qR, d, F, ex);
}

}  // extern "C"
