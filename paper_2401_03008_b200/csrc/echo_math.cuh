// echo_math.cuh — per-point device functions of the ECHO RMHD step (FP64, sm_100a).
// Stencil operators INT / DER / REC (coefficients: DESIGN.md O1, O3, O6), point
// physics (definitions, eq.(6), eq.(8)), fast speeds (O4), HLL (O5) and
// the Newton conservative->primitive inversion (O2).  Written from the paper / DESIGN.md;
// shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <math.h>

namespace echo {

// ---------------------------------------------------------------- stencils
// O1 — INT: 6-point Lagrange interpolation of staggered point values to the midpoint.
__device__ __forceinline__ double int6(double b0, double b1, double b2, double b3, double b4, double b5) {
    return (150.0 / 256.0) * (b2 + b3) - (25.0 / 256.0) * (b1 + b4) + (3.0 / 256.0) * (b0 + b5);
}

// O6 — DER then two-point difference, folded into one antisymmetric 6-point stencil:
// F^_{i+1/2} - F^_{i-1/2} with F^ = d0 F + d2 (F_-1 + F_+1) + d4 (F_-2 + F_+2),
// (d0,d2,d4) = (1067/960, -29/480, 3/640)  =>  (75/64, -25/384, 3/640) on the three differences.
// f0..f5 = F at faces i-5/2, i-3/2, i-1/2, i+1/2, i+3/2, i+5/2.
__device__ __forceinline__ double der_diff(double f0, double f1, double f2, double f3, double f4, double f5) {
    return (75.0 / 64.0) * (f3 - f2) + ((-25.0 / 384.0) * (f4 - f1) + (3.0 / 640.0) * (f5 - f0));
}

// HO switch: with ho = 0 INT is the two-point average and DER the identity (second order)
__device__ __forceinline__ double int_ho(int ho, double b0, double b1, double b2, double b3, double b4, double b5) {
    return ho ? int6(b0, b1, b2, b3, b4, b5) : 0.5 * (b2 + b3);
}
__device__ __forceinline__ double der_diff_ho(int ho, double f0, double f1, double f2, double f3, double f4, double f5) {
    return ho ? der_diff(f0, f1, f2, f3, f4, f5) : f3 - f2;
}

// ---------------------------------------------------------------- fast FP64 helpers
// min / max without the IEEE NaN bookkeeping of fmin/fmax (one DSETP + selects)
__device__ __forceinline__ double dmin(double a, double b) { return a < b ? a : b; }
__device__ __forceinline__ double dmax(double a, double b) { return a > b ? a : b; }

// Reciprocal, reciprocal square root and square root for NORMAL positive arguments: the MUFU
// seed (about 20 good bits) refined by one third-order step (error ~ e^3, then rounding), ~1 ulp.
// No denormal / special-case slow path: the arguments here are O(1) physical quantities; a zero
// or negative argument yields inf/NaN exactly like the exact operation would, and propagates.
__device__ __forceinline__ double rcp_fast(double x) {
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    const double e = fma(-x, y, 1.0);
    return fma(y * e, 1.0 + e, y);
}
__device__ __forceinline__ double rsqrt_fast(double x) {
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    const double e = fma(-(x * y), y, 1.0);
    return fma(y * e, fma(0.375, e, 0.5), y);
}
__device__ __forceinline__ double sqrt_fast(double x) {   // x >= 0; exact 0 -> 0; ~1-2 ulp (x * rsqrt(x))
    const double t = x * rsqrt_fast(x);
    return x > 0.0 ? t : 0.0;
}

__device__ __forceinline__ double minmod2(double a, double b) {
    // same sign: the one of smaller magnitude; else 0.  The sign test is done on the high words
    // (integer pipe); a zero argument selects itself as the smaller magnitude, so it needs no test.
    const double m = (fabs(a) < fabs(b)) ? a : b;
    return ((__double2hiint(a) ^ __double2hiint(b)) >= 0) ? m : 0.0;
}
__device__ __forceinline__ double minmod4(double a, double b, double c, double d) {
    // all four of one sign: the one of smallest magnitude; else 0.  Sign agreement on the high
    // words (integer pipe); the magnitude minimum with |.| operand modifiers (3 DSETP).  A zero
    // argument makes the magnitude minimum 0, so its sign bit does not matter.
    const int ha = __double2hiint(a);
    const int diff = (ha ^ __double2hiint(b)) | (ha ^ __double2hiint(c)) | (ha ^ __double2hiint(d));
    double m = (fabs(a) < fabs(b)) ? a : b;
    m = (fabs(m) < fabs(c)) ? m : c;
    m = (fabs(m) < fabs(d)) ? m : d;
    return diff >= 0 ? m : 0.0;
}

// O3 — REC: MP5 (Suresh & Huynh 1997) on POINT values, left-biased value at i+1/2 from v_{i-2..i+2};
// alpha = 4, eps = 1e-10 (S2).  The unlimited 5-point value vor = (3, -20, 90, 60, -5)/128 . v and the S&H test
// (vor - v_i)(vor - v^MP) > eps come first (mp5_pair, mp5_pair_fast below, two sides at a time); mp5_limit is the
// limiter proper, evaluated only where the test fires: on smooth data that is the few cells around each extremum.
__device__ __forceinline__ double mp5_limit(double vm2, double vm1, double v0, double vp1, double vp2, double vor) {
    const double dm1 = fma(-2.0, vm1, vm2) + v0;
    const double d0 = fma(-2.0, v0, vm1) + vp1;
    const double dp1 = fma(-2.0, vp1, v0) + vp2;
    const double dm4p = minmod4(fma(4.0, d0, -dp1), fma(4.0, dp1, -d0), d0, dp1);
    const double dm4m = minmod4(fma(4.0, dm1, -d0), fma(4.0, d0, -dm1), dm1, d0);
    const double dv = v0 - vm1;
    const double vul = fma(4.0, dv, v0);
    const double vmd = fma(0.5, v0 + vp1, -0.5 * dm4p);
    const double vlc = fma(0.5, dv, v0) + (4.0 / 3.0) * dm4m;
    // min/max of (v0, vp1, vmd) and of (v0, vul, vlc), sharing the comparisons
    const bool c1 = v0 < vp1;
    const double lo1 = c1 ? v0 : vp1, hi1 = c1 ? vp1 : v0;
    const double mn1 = dmin(lo1, vmd), mx1 = dmax(hi1, vmd);
    const bool c2 = v0 < vul;
    const double lo2 = c2 ? v0 : vul, hi2 = c2 ? vul : v0;
    const double mn2 = dmin(lo2, vlc), mx2 = dmax(hi2, vlc);
    const double vmin = dmax(mn1, mn2);
    const double vmax = dmin(mx1, mx2);
    return vor + minmod2(vmin - vor, vmax - vor);
}
__device__ __noinline__ double mp5_limit_call(double vm2, double vm1, double v0, double vp1, double vp2, double vor) {
    return mp5_limit(vm2, vm1, v0, vp1, vp2, vor);
}
// Both one-sided values at the face between s2 and s3 from the six cells s0..s5 around it:
// L = MP5(s0..s4) centred on s2, R = MP5(s5..s1) centred on s3 (mirrored).  The S&H test is evaluated
// as t (t - mm) > eps with t = vOR - v_i and mm = minmod(v_{i+1} - v_i, 4 (v_i - v_{i-1})): the two sides
// share s3 - s2, and the factor 4 is an exact exponent bump on the integer pipe (a zero becomes
// 2^-1021, which minmod treats like the zero it stands for).
__device__ __forceinline__ double times4(double d) {
    return __hiloint2double(__double2hiint(d) + 0x00200000, __double2loint(d));
}
// INL: limiter inlined behind a branch (flux sweeps) or called out of line.
#ifndef ECHO_SH_SUPERSET
#define ECHO_SH_SUPERSET 1       // sweeps: x 0.785 -> 0.776, y 0.757 -> 0.741, z 0.808 -> 0.804 ms at 256^3
#endif
template <bool INL = true>
__device__ __forceinline__ void mp5_pair(double s0, double s1, double s2, double s3, double s4, double s5, double &L,
                                         double &R) {
    const double vorL = (3.0 / 128.0) * s0 + ((-20.0 / 128.0) * s1 + ((90.0 / 128.0) * s2 +
                        ((60.0 / 128.0) * s3 + (-5.0 / 128.0) * s4)));
    const double vorR = (3.0 / 128.0) * s5 + ((-20.0 / 128.0) * s4 + ((90.0 / 128.0) * s3 +
                        ((60.0 / 128.0) * s2 + (-5.0 / 128.0) * s1)));
    const double d23 = s3 - s2;
    const double tL = vorL - s2, tR = vorR - s3;
    L = vorL;
    R = vorR;
#if ECHO_SH_SUPERSET
    // t (t - minmod(a, b)) > eps implies t (t - a) > eps or t (t - b) > eps (same signs: minmod is one of the two;
    // opposite signs: minmod = 0 and one of -t a, -t b is >= 0), so the FP64-only disjunction is a superset of the
    // S&H test that needs no selects; the exact test is repeated inside the rare branch.
    const double dL = s2 - s1, dR = s3 - s4;
    if (tL * (tL - d23) > 1e-10 || tL * fma(-4.0, dL, tL) > 1e-10) {
        asm volatile("" ::: "memory");
        if (tL * (tL - minmod2(d23, times4(dL))) > 1e-10) {
            if (INL) L = mp5_limit(s0, s1, s2, s3, s4, vorL);
            else L = mp5_limit_call(s0, s1, s2, s3, s4, vorL);
        }
    }
    if (tR * (tR + d23) > 1e-10 || tR * fma(-4.0, dR, tR) > 1e-10) {
        asm volatile("" ::: "memory");
        if (tR * (tR - minmod2(-d23, times4(dR))) > 1e-10) {
            if (INL) R = mp5_limit(s5, s4, s3, s2, s1, vorR);
            else R = mp5_limit_call(s5, s4, s3, s2, s1, vorR);
        }
    }
#else
    const double mmL = minmod2(d23, times4(s2 - s1));
    const double mmR = minmod2(-d23, times4(s3 - s4));
    if (tL * (tL - mmL) > 1e-10) {
        if (INL) { asm volatile("" ::: "memory"); L = mp5_limit(s0, s1, s2, s3, s4, vorL); }
        else L = mp5_limit_call(s0, s1, s2, s3, s4, vorL);
    }
    if (tR * (tR - mmR) > 1e-10) {
        if (INL) { asm volatile("" ::: "memory"); R = mp5_limit(s5, s4, s3, s2, s1, vorR); }
        else R = mp5_limit_call(s5, s4, s3, s2, s1, vorR);
    }
#endif
}

// O3b — the second-order REC of P:L304: v_i + MC(a, b)/2 with the monotonized-central slope
// MC(a, b) = minmod(2a, 2b, (a + b)/2); both one-sided values at the face between s2 and s3.
__device__ __forceinline__ double mc_slope(double a, double b) {
    const double s = 0.5 * (a + b);
    double m = (fabs(a) < fabs(b)) ? a : b;      // same sign: 2 min(|a|, |b|) against |a + b|/2
    m = 2.0 * m;
    m = (fabs(s) < fabs(m)) ? s : m;
    return ((__double2hiint(a) ^ __double2hiint(b)) >= 0) ? m : 0.0;
}
__device__ __forceinline__ void tvd2_pair(double s1, double s2, double s3, double s4, double &L, double &R) {
    const double b = s3 - s2;
    L = s2 + 0.5 * mc_slope(s2 - s1, b);
    R = s3 - 0.5 * mc_slope(b, s4 - s3);
}
// REC of the scheme in force
template <int REC>
__device__ __forceinline__ void rec_pair(double s0, double s1, double s2, double s3, double s4, double s5, double &L,
                                         double &R) {
    if (REC == 2) tvd2_pair(s1, s2, s3, s4, L, R);
    else mp5_pair<true>(s0, s1, s2, s3, s4, s5, L, R);
}

// Branch-free first half of mp5_pair: the two unlimited values and the two S&H test bits (bit 0: L needs the
// limiter, bit 1: R); mp5_pair_fix applies the limiter afterwards.  Used where several stencils should be
// interleaved by the compiler before any branch (the UCT kernels).
__device__ __forceinline__ unsigned mp5_pair_fast(double s0, double s1, double s2, double s3, double s4, double s5,
                                                  double &L, double &R) {
    L = (3.0 / 128.0) * s0 + ((-20.0 / 128.0) * s1 + ((90.0 / 128.0) * s2 + ((60.0 / 128.0) * s3 + (-5.0 / 128.0) * s4)));
    R = (3.0 / 128.0) * s5 + ((-20.0 / 128.0) * s4 + ((90.0 / 128.0) * s3 + ((60.0 / 128.0) * s2 + (-5.0 / 128.0) * s1)));
    const double d23 = s3 - s2;
    const double tL = L - s2, tR = R - s3;
    // the exact S&H test: its select-free superset (mp5_pair) makes the UCT kernel slower (1.16 -> 1.19-1.22 ms)
    const double mmL = minmod2(d23, times4(s2 - s1));
    const double mmR = minmod2(-d23, times4(s3 - s4));
    return (tL * (tL - mmL) > 1e-10 ? 1u : 0u) | (tR * (tR - mmR) > 1e-10 ? 2u : 0u);
}
__device__ __forceinline__ void mp5_pair_fix(unsigned bits, double s0, double s1, double s2, double s3, double s4,
                                             double s5, double &L, double &R) {
    if (bits & 1u) L = mp5_limit_call(s0, s1, s2, s3, s4, L);
    if (bits & 2u) R = mp5_limit_call(s5, s4, s3, s2, s1, R);
}

// ---------------------------------------------------------------- point physics
// q[8] = (rho, vx, vy, vz, p, Bx, By, Bz); u[5] = (D, Sx, Sy, Sz, U).  gg = gamma/(gamma-1).
// Identities used (E = -v x B): E x B = B^2 v - (v.B) B, E^2 = v^2 B^2 - (v.B)^2.
__device__ __forceinline__ void prim2cons(double gg, const double q[8], double u[5]) {
    const double v2 = q[1] * q[1] + q[2] * q[2] + q[3] * q[3];
    const double B2 = q[5] * q[5] + q[6] * q[6] + q[7] * q[7];
    const double vB = q[1] * q[5] + q[2] * q[6] + q[3] * q[7];
    const double W = rsqrt_fast(1.0 - v2);
    const double y = (q[0] + gg * q[4]) * (W * W);
    const double yb = y + B2;
    u[0] = q[0] * W;
    u[1] = yb * q[1] - vB * q[5];
    u[2] = yb * q[2] - vB * q[6];
    u[3] = yb * q[3] - vB * q[7];
    u[4] = y - q[4] + 0.5 * ((v2 * B2 - vB * vB) + B2);
}

// One side of a D-face: conserved state u, physical flux f (eq.(8)), fast speeds lp, lm (O4).
// With E = -v x B:  E^2 = B^2 - b2,  b2 = B^2 (1 - v^2) + (v.B)^2,  S = (y + B^2) v - (v.B) B, and
//   F_D(S_a) = S_a v_D - B_D beta_a + delta_aD (p + b2/2),  beta_a = (1 - v^2) B_a + (v.B) v_a,
// which is eq.(8)'s  y v_a v_D - E_a E_D - B_a B_D + p_tot delta_aD  after expanding (v x B)_a (v x B)_D.
template <int D>
__device__ __forceinline__ void side_state(double gam, double gg, const double q[8], double u[5], double f[5],
                                           double &lp, double &lm) {
    const double rho = q[0], p = q[4];
    const double v[3] = {q[1], q[2], q[3]};
    const double B[3] = {q[5], q[6], q[7]};
    const double v2 = v[0] * v[0] + v[1] * v[1] + v[2] * v[2];
    const double B2 = B[0] * B[0] + B[1] * B[1] + B[2] * B[2];
    const double vB = v[0] * B[0] + v[1] * B[1] + v[2] * B[2];
    const double omv2 = 1.0 - v2;
    const double W = rsqrt_fast(omv2);
    const double rhoh = rho + gg * p;
    const double y = rhoh * (W * W);
    const double yb = y + B2;
    const double b2 = fma(B2, omv2, vB * vB);
    u[0] = rho * W;
    u[4] = fma(-0.5, b2, (y - p) + B2);
    f[0] = u[0] * v[D];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        u[1 + a] = yb * v[a] - vB * B[a];
        const double beta = fma(omv2, B[a], vB * v[a]);
        f[1 + a] = fma(u[1 + a], v[D], -(B[D] * beta));
    }
    f[1 + D] += fma(0.5, b2, p);
    f[4] = u[1 + D];
    // O4.  a^2 = cs^2 + ca^2 - cs^2 ca^2 with cs^2 = gamma p/(rho h), ca^2 = b^2/w, w = rho h + b^2 collapses to
    // a^2 = A/w, A = gamma p + b^2.  Multiplying numerator and denominator of lambda+- by w:
    //   lambda+- = [ (w - A) v_D +- sqrt( A (1-v^2) [ (w - v^2 A) - (w - A) v_D^2 ] ) ] / (w - v^2 A)
    // — one square root and one reciprocal per side, no division.
    const double w = rhoh + b2;
    const double A = fma(gam, p, b2);
    const double N = fma(-v2, A, w);
    const double M = w - A;
    const double vd = v[D];
    const double sq = sqrt_fast(A * omv2 * fma(-M, vd * vd, N));
    const double rN = rcp_fast(N);
    lp = fma(M, vd, sq) * rN;
    lm = fma(M, vd, -sq) * rN;
}

// O5 — two-state HLL flux at a D-face; also the stored UCT pieces:
// ap, am and the upwind-averaged transverse velocities vb1 = vbar_{(D+1)%3}, vb2 = vbar_{(D+2)%3}.
template <int D>
__device__ __forceinline__ void hll_face(double gam, double gg, const double qL[8], const double qR[8], double F[5],
                                         double &ap, double &am, double &vb1, double &vb2) {
    double uL[5], fL[5], uR[5], fR[5], lpL, lmL, lpR, lmR;
    side_state<D>(gam, gg, qL, uL, fL, lpL, lmL);
    side_state<D>(gam, gg, qR, uR, fR, lpR, lmR);
    ap = dmax(0.0, dmax(lpL, lpR));
    am = dmax(0.0, dmax(-lmL, -lmR));
    const double inv = rcp_fast(ap + am);
    const double wl = ap * inv, wr = am * inv, wd = ap * am * inv;
#pragma unroll
    for (int c = 0; c < 5; ++c) F[c] = wl * fL[c] + wr * fR[c] - wd * (uR[c] - uL[c]);
    constexpr int t1 = (D + 1) % 3, t2 = (D + 2) % 3;
    vb1 = wl * qL[1 + t1] + wr * qR[1 + t1];
    vb2 = wl * qL[1 + t2] + wr * qR[1 + t2];
}

// UCT=NO: the cell-centred B is a conserved variable like the others.  Same two-state formula as O5 for
// 8 components; the induction fluxes are F_D(B_a) = v_D B_a - v_a B_D (eq.(8), with E = -v x B).  Both
// sides carry their own reconstructed normal B.
template <int D>
__device__ __forceinline__ void hll_face_cc(double gam, double gg, const double qL[8], const double qR[8], double F[8],
                                            double &ap, double &am) {
    double uL[5], fL[5], uR[5], fR[5], lpL, lmL, lpR, lmR;
    side_state<D>(gam, gg, qL, uL, fL, lpL, lmL);
    side_state<D>(gam, gg, qR, uR, fR, lpR, lmR);
    ap = dmax(0.0, dmax(lpL, lpR));
    am = dmax(0.0, dmax(-lmL, -lmR));
    const double inv = rcp_fast(ap + am);
    const double wl = ap * inv, wr = am * inv, wd = ap * am * inv;
#pragma unroll
    for (int c = 0; c < 5; ++c) F[c] = wl * fL[c] + wr * fR[c] - wd * (uR[c] - uL[c]);
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const double bL = qL[1 + D] * qL[5 + a] - qL[1 + a] * qL[5 + D];
        const double bR = qR[1 + D] * qR[5 + a] - qR[1 + a] * qR[5 + D];
        F[5 + a] = wl * bL + wr * bR - wd * (qR[5 + a] - qL[5 + a]);
    }
}

// ---------------------------------------------------------------- O2: con2prim
// Newton on y = rho h W^2 from the upper bound y0 = gamma (U - B^2/2); safeguard and stopping
// rule as in DESIGN.md O2.  Returns the number of Newton updates (>=1) or -(count) on failure.
struct C2PEval { double x, sq, p, f, df, xp; };

__device__ __forceinline__ bool c2p_eval(double g1, double D, double S2, double B2, double T, double U, double y,
                                         C2PEval &a) {
    if (!(y > 0.0) || !isfinite(y)) return false;
    const double yb = y + B2;
    const double y2 = y * y, yb2 = yb * yb;
    const double r = rcp_fast(y2 * y * yb2 * yb);   // 1/(y^3 (y+B^2)^3)
    const double x = (S2 * y2 + T * (2.0 * y + B2)) * (y * yb) * r;
    if (!(x < 1.0) || !(x >= 0.0)) return false;
    const double omx = 1.0 - x;
    const double rsq = rsqrt_fast(omx);
    const double sq = omx * rsq;
    const double xp = -2.0 * (S2 * y2 * y + T * (3.0 * y2 + 3.0 * y * B2 + B2 * B2)) * r;
    const double Ty3 = T * (yb2 * yb) * r;        // T / y^3
    a.x = x;
    a.xp = xp;
    a.sq = sq;
    a.p = g1 * (y * omx - D * sq);
    a.f = y - a.p + 0.5 * (1.0 + x) * B2 - 0.5 * Ty3 * y - U;
    a.df = 1.0 - g1 * omx - g1 * (-y + 0.5 * D * rsq) * xp + 0.5 * B2 * xp + Ty3;
    return true;
}

__device__ __forceinline__ int con2prim(double gam, const double u[5], const double B[3], double q[5]) {
    const double tol = 1e-12;
    const int maxit = 30;
    const double g1 = (gam - 1.0) / gam;
    const double D = u[0], U = u[4];
    const double S2 = u[1] * u[1] + u[2] * u[2] + u[3] * u[3];
    const double B2 = B[0] * B[0] + B[1] * B[1] + B[2] * B[2];
    const double SB = u[1] * B[0] + u[2] * B[1] + u[3] * B[2];
    const double T = SB * SB;
    double y = gam * (U - 0.5 * B2);
    double ylast = y;
    C2PEval a;
    int it = 0;
    bool conv = false;
    while (it < maxit) {
        if (!c2p_eval(g1, D, S2, B2, T, U, y, a)) {
            if (it == 0) break;
            ++it;
            y = 0.5 * (y + ylast);
            if (!isfinite(y)) break;
            continue;
        }
        ylast = y;
        const double dy = -a.f * rcp_fast(a.df);
        y = y + dy;
        ++it;
        if (fabs(dy) <= tol * fabs(y)) { conv = true; break; }
    }
    // x, sqrt(1-x) and p at the converged y from the last evaluation (made at ylast) and the last update
    // dy = y - ylast, |dy| <= 1e-12 |y|:  x(y) = x(ylast) + x'(ylast) dy + O(dy^2) -- the second-order term is 1e-24
    // relative, so this equals a fresh evaluation at y to rounding and saves a fifth of the arithmetic of a 4-iteration
    // inversion (k_prim_march 0.525 -> 0.519 ms at 256^3: the kernel is not bound by this chain).
    bool ok = conv;
    if (ok) {
        const double x = fma(a.xp, y - ylast, a.x);
        ok = (x < 1.0) && (x >= 0.0) && (y > 0.0);
        const double omx = 1.0 - x;
        a.sq = omx * rsqrt_fast(omx);
        a.p = g1 * (y * omx - D * a.sq);
    }
    if (!ok) {
        const double nan = __longlong_as_double(0x7ff8000000000000LL);
        q[0] = q[1] = q[2] = q[3] = q[4] = nan;
        return -(it > 0 ? it : 1);
    }
    q[0] = D * a.sq;
    q[4] = a.p;
    const double ryb = rcp_fast(y + B2);
    const double sby = SB * rcp_fast(y);
    q[1] = (u[1] + sby * B[0]) * ryb;
    q[2] = (u[2] + sby * B[1]) * ryb;
    q[3] = (u[3] + sby * B[2]) * ryb;
    return it;
}

}  // namespace echo
