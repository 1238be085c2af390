// echo_uct.cuh — point 4 of a sub-step: the UCT edge EMFs (O7), plane-marching, and the other kernels that
// march 16 x 8 tiles of (x, y) along z: curl + update of the staggered B (k_bupd), INT + con2prim (k_prim_march).
//
// k_uct3: a block owns a TX x TY = 16 x 8 tile of (x, y) and marches along z over a chunk of planes, one plane per
// round, one cell (three edges) per thread.  What a plane needs:
//   XR  4 fields reconstructed along x  (vbar_x@y-face, B_y, vbar_x@z-face, B_z): 22 x 8 (x0-2 .. x0+19)
//   YR  4 fields reconstructed along y  (vbar_y@x-face, B_x, vbar_y@z-face, B_z): 16 x 13 (y0-2 .. y0+10)
//   ZW  4 fields reconstructed along z  (vbar_z@x-face, B_x, vbar_z@y-face, B_y): a 6-plane sliding window per
//       thread, held in REGISTERS (one new value per field and plane)
//   AX, AY, AZ  the saved a+/a- of the three directions at the cell and its +1 neighbours along the two other axes
//       (the edge speed is the max over the two faces adjacent to the edge)
// The 14 tiles of a plane form one "package" in shared memory, moved by TMA (tiles inside the grid) or cp.async (tiles
// on the periodic seams) and completed on an mbarrier; three packages are resident (plane k, the x/y speeds of k+1,
// and k+2 landing), so every input is read from L2/HBM about once (plus tile halos) and its latency hides behind two
// planes of arithmetic.
#pragma once
#include "echo_async.cuh"
#include "echo_math.cuh"
#include "echo_types.cuh"

namespace echo {

constexpr int UCT_TX = 16, UCT_TY = 8, UCT_NT = UCT_TX * UCT_TY;
constexpr int UCT_XRW = UCT_TX + 5, UCT_XR = UCT_XRW * UCT_TY;          // 21 x 8
constexpr int UCT_YRH = UCT_TY + 5, UCT_YR = UCT_TX * UCT_YRH;          // 16 x 13
constexpr int UCT_AX = UCT_TX * (UCT_TY + 1);                           // 16 x 9   (c, c+e_y)
constexpr int UCT_AYW = UCT_TX + 1, UCT_AY = UCT_AYW * UCT_TY;          // 17 x 8   (c, c+e_x)
constexpr int UCT_AZ = UCT_AYW * (UCT_TY + 1);                          // 17 x 9   (c, c+e_x, c+e_y)

// HLL-upwinded product of O7: [a+ vL BL + a- vR BR - a+ a- (BR - BL)] / (a+ + a-)
__device__ __forceinline__ double uct_hll(double ap, double am, double vL, double vR, double BL, double BR) {
    return (ap * vL * BL + am * vR * BR - ap * am * (BR - BL)) * rcp_fast(ap + am);
}

// One upwinded product of O7: MP5 L/R (O3) of (vbar, B) to the edge from the six stencil values p[0], p[S], ...,
// p[5 S] (vbar) and q[0], ..., q[5 S] (B), then the two-state formula with the edge speeds ap, am.  Shared by the
// plane-marching kernel (k_uct3) and the flat one (k_uct2_flat), so that the two stay bit-identical.  LIN: the limited linear REC of O3b instead of MP5 (echo_set_order).
template <bool LIN>
__device__ __forceinline__ double uct_bracket(const double *p, const double *q, int S, double ap, double am) {
    double vL, vR, BL, BR;
    if (LIN) {
        tvd2_pair(p[S], p[2 * S], p[3 * S], p[4 * S], vL, vR);
        tvd2_pair(q[S], q[2 * S], q[3 * S], q[4 * S], BL, BR);
        return uct_hll(ap, am, vL, vR, BL, BR);
    }
    const unsigned nv = mp5_pair_fast(p[0], p[S], p[2 * S], p[3 * S], p[4 * S], p[5 * S], vL, vR);
    const unsigned nb = mp5_pair_fast(q[0], q[S], q[2 * S], q[3 * S], q[4 * S], q[5 * S], BL, BR);
    if (nv | nb) {
        mp5_pair_fix(nv, p[0], p[S], p[2 * S], p[3 * S], p[4 * S], p[5 * S], vL, vR);
        mp5_pair_fix(nb, q[0], q[S], q[2 * S], q[3 * S], q[4 * S], q[5 * S], BL, BR);
    }
    return uct_hll(ap, am, vL, vR, BL, BR);
}

// ------------------------------------------------------------------ k_uct3: tiles moved by TMA
// In the round-1 kernel (k_uct2) every thread issued 10-14 eight-byte cp.async per plane, each with its own wrapped
// source index (a sixth of the kernel's instructions and 40 % of its shared-memory wavefronts,
// profiles/r1_ncu_full.md).  Here the 14 tiles of a
// plane (XR, YR: 4 fields each; AZ, AX, AY: 2 each; 19 488 bytes) are 14 TMA box copies (cp.async.bulk.tensor, SASS
// UTMALDG) issued by ONE thread, completing on one mbarrier by transaction bytes (SASS SYNCS); the other 127
// threads issue nothing.  A TMA box cannot wrap periodically (out-of-range elements are zero-filled), so only the
// tiles whose boxes lie inside the grid take this path - at 256^3 that is 82 % of the blocks, at 512^3 91 %; the
// blocks along the periodic seams of x and y (and every block of a grid without tensor maps: odd n_x, small grids)
// fill the same shared-memory layout with per-thread 8-byte cp.async copies, which arrive on the same
// mbarrier (cp.async.mbarrier.arrive.noinc).  z never needs a split: a copy moves one plane, whose index is wrapped
// by the issuing thread.  The packages of three consecutive planes live in a ring (plane k and the x/y speeds of
// k+1 are in use while k+2 lands): 57 KB of dynamic shared memory, 3 blocks per SM.
#ifndef ECHO_UCT_TY
#define ECHO_UCT_TY 8
#endif
constexpr int U3_TY = ECHO_UCT_TY;                                       // tile height of k_uct3 in force
constexpr int U3_XRP = 22, U3_AP = 18;                                   // row pitches (doubles) of the x-halo tiles
constexpr int u3_pad16(int n) { return (n + 15) / 16 * 16; }             // tiles start 128-byte aligned (TMA destination)
// geometry of a plane package for tiles of UCT_TX x TY cells (TY = 8: 4 warps per block; TY = 4: 2 warps)
template <int TY>
struct U3 {
    static constexpr int NT = UCT_TX * TY;                               // threads per block = cells per tile
    static constexpr int YRH = TY + 5;
    static constexpr int NXR = U3_XRP * TY, NYR = UCT_TX * YRH;          // elements per field tile
    static constexpr int NAZ = U3_AP * (TY + 1), NAX = UCT_TX * (TY + 1), NAY = U3_AP * TY;
    static constexpr int SXR = u3_pad16(NXR), SYR = u3_pad16(NYR), SAZ = u3_pad16(NAZ), SAX = u3_pad16(NAX), SAY = u3_pad16(NAY);
    static constexpr int XR = 0, YR = XR + 4 * SXR, AZ = YR + 4 * SYR, AX = AZ + 2 * SAZ, AY = AX + 2 * SAX;   // offsets
    static constexpr int PKG = AY + 2 * SAY;                             // doubles per package (TY = 8: 2464)
    static constexpr unsigned BYTES = 8u * (4 * NXR + 4 * NYR + 2 * NAZ + 2 * NAX + 2 * NAY);   // bytes that land (19 488)
    static constexpr int NSLOT = 3;
    static constexpr size_t SMEM = sizeof(double) * NSLOT * PKG + 128 + 64;
    static constexpr int NCOPY = (NYR + NT - 1) / NT;                    // cp.async path: elements per thread and region
};

template <bool LIN = false, int TY = U3_TY>
__global__ void __launch_bounds__(UCT_TX * TY) k_uct3(Grid g, Stage st, int CZ, const __grid_constant__ UctMaps maps) {
    using G3 = U3<TY>;
    constexpr int NT = G3::NT;
    extern __shared__ __align__(128) unsigned char u3_raw[];
    double *const pkg = reinterpret_cast<double *>(u3_raw + ((128u - (smem_u32(u3_raw) & 127u)) & 127u));   // [slot][G3::PKG]
    uint64_t *const full = reinterpret_cast<uint64_t *>(pkg + G3::NSLOT * G3::PKG);  // one barrier per slot

    const int tid = threadIdx.x;
    const int tx = tid % UCT_TX, ty = tid / UCT_TX;
    const int nx = g.n[0], ny = g.n[1], nz = g.n[2];
    const int x0 = blockIdx.x * UCT_TX, y0 = blockIdx.y * TY, z0 = blockIdx.z * CZ;
    const int CZv = min(CZ, nz - z0);
    const int sy = g.s[1], sz = g.s[2];
    // all 14 boxes inside the grid?  (block-uniform)
    const bool tma = maps.ok && x0 >= 2 && x0 + UCT_TX + 4 <= nx && y0 >= 2 && y0 + TY + 3 <= ny;

    // cp.async path (seam tiles): in-plane source offsets of the (at most two) elements this thread copies per region
    int oXR[G3::NCOPY], oYR[G3::NCOPY], oAX[G3::NCOPY], oAY[G3::NCOPY], oAZ[G3::NCOPY];
    if (!tma) {
#pragma unroll
        for (int it = 0; it < G3::NCOPY; ++it) {
            const int e = tid + NT * it;
            oXR[it] = (e < G3::NXR) ? wrapi(x0 - 2 + e % U3_XRP, nx) + sy * wrapi(y0 + e / U3_XRP, ny) : -1;
            oYR[it] = (e < G3::NYR) ? wrapi(x0 + e % UCT_TX, nx) + sy * wrapi(y0 - 2 + e / UCT_TX, ny) : -1;
            oAX[it] = (e < G3::NAX) ? wrapi(x0 + e % UCT_TX, nx) + sy * wrapi(y0 + e / UCT_TX, ny) : -1;
            oAY[it] = (e < G3::NAY) ? wrapi(x0 + e % U3_AP, nx) + sy * wrapi(y0 + e / U3_AP, ny) : -1;
            oAZ[it] = (e < G3::NAZ) ? wrapi(x0 + e % U3_AP, nx) + sy * wrapi(y0 + e / U3_AP, ny) : -1;
        }
    }
    // XR = {vbar_x@y, B_y, vbar_x@z, B_z}; YR = {vbar_y@x, B_x, vbar_y@z, B_z}; ZW = {vbar_z@x, B_x, vbar_z@y, B_y}
    const double *fXR[4] = {st.vb[1][1], st.Bf[1], st.vb[2][0], st.Bf[2]};
    const double *fYR[4] = {st.vb[0][0], st.Bf[0], st.vb[2][1], st.Bf[2]};
    const double *fZW[4] = {st.vb[0][1], st.Bf[0], st.vb[1][0], st.Bf[1]};

    auto issue_package = [&](int k, int slot) {            // all tiles of plane k into ring slot `slot`
        const int kz = wrapi(k, nz);
        double *base = pkg + slot * G3::PKG;
        if (tma) {
            if (tid == 0) {
                mbar_arrive_expect_tx(&full[slot], G3::BYTES);
#pragma unroll
                for (int f = 0; f < 4; ++f) tma_load_3d(base + G3::XR + f * G3::SXR, &maps.xr[f], x0 - 2, y0, kz, &full[slot]);
#pragma unroll
                for (int f = 0; f < 4; ++f) tma_load_3d(base + G3::YR + f * G3::SYR, &maps.yr[f], x0, y0 - 2, kz, &full[slot]);
#pragma unroll
                for (int f = 0; f < 2; ++f) {
                    tma_load_3d(base + G3::AZ + f * G3::SAZ, &maps.az[f], x0, y0, kz, &full[slot]);
                    tma_load_3d(base + G3::AX + f * G3::SAX, &maps.ax[f], x0, y0, kz, &full[slot]);
                    tma_load_3d(base + G3::AY + f * G3::SAY, &maps.ay[f], x0, y0, kz, &full[slot]);
                }
            }
        } else {
            const int pz = sz * kz;
#pragma unroll
            for (int it = 0; it < G3::NCOPY; ++it) {
                const int e = tid + NT * it;
                if (oXR[it] >= 0) {
#pragma unroll
                    for (int f = 0; f < 4; ++f) cp_async8(base + G3::XR + f * G3::SXR + e, fXR[f] + (pz + oXR[it]));
                }
                if (oYR[it] >= 0) {
#pragma unroll
                    for (int f = 0; f < 4; ++f) cp_async8(base + G3::YR + f * G3::SYR + e, fYR[f] + (pz + oYR[it]));
                }
                if (oAZ[it] >= 0) {
                    cp_async8(base + G3::AZ + e, st.ap[2] + (pz + oAZ[it]));
                    cp_async8(base + G3::AZ + G3::SAZ + e, st.am[2] + (pz + oAZ[it]));
                }
                if (oAX[it] >= 0) {
                    cp_async8(base + G3::AX + e, st.ap[0] + (pz + oAX[it]));
                    cp_async8(base + G3::AX + G3::SAX + e, st.am[0] + (pz + oAX[it]));
                }
                if (oAY[it] >= 0) {
                    cp_async8(base + G3::AY + e, st.ap[1] + (pz + oAY[it]));
                    cp_async8(base + G3::AY + G3::SAY + e, st.am[1] + (pz + oAY[it]));
                }
            }
            cp_async_arrive_on(&full[slot]);               // this thread's share of the package has landed
        }
    };

    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < G3::NSLOT; ++s) mbar_init(&full[s], tma ? 1u : (unsigned)NT);
        mbar_init_fence();
    }
    __syncthreads();

    const bool cellok = (x0 + tx < nx) && (y0 + ty < ny);
    const int ccol = min(x0 + tx, nx - 1) + sy * min(y0 + ty, ny - 1);

    // prologue: packages of planes z0 and z0+1; z-window planes z0-2 .. z0+3 directly
    issue_package(z0, 0);
    issue_package(z0 + 1, 1);
    double zw[4][6];
#pragma unroll
    for (int m = 0; m < 6; ++m) {
        const int pz = sz * wrapi(z0 - 2 + m, nz);
#pragma unroll
        for (int f = 0; f < 4; ++f) zw[f][m] = __ldg(fZW[f] + (pz + ccol));
    }

    int s0 = 0;                                            // ring slot of plane k
    for (int r = 0; r < CZv; ++r) {
        const int k = z0 + r;
        const int s1 = (s0 + 1 == G3::NSLOT) ? 0 : s0 + 1, s2 = (s1 + 1 == G3::NSLOT) ? 0 : s1 + 1;
        // plane z0 + r is the (r / 3)-th package of its slot: the parity of that phase
        mbar_wait(&full[s0], (unsigned)((r / G3::NSLOT) & 1));
        mbar_wait(&full[s1], (unsigned)(((r + 1) / G3::NSLOT) & 1));
        __syncthreads();                                   // every warp is through plane k-1: its slot (s2) is free
        if (r + 2 <= CZv) issue_package(k + 2, s2);        // (plane z0+CZv only lends its x/y speeds to the last plane)
        double znew[4];
        {
            const int pz = sz * wrapi(k + 4, nz);
#pragma unroll
            for (int f = 0; f < 4; ++f) znew[f] = __ldg(fZW[f] + (pz + ccol));
        }

        if (cellok) {
            const double *P0 = pkg + s0 * G3::PKG, *P1 = pkg + s1 * G3::PKG;
            const int ixr = ty * U3_XRP + tx, iyr = ty * UCT_TX + tx, iax = ty * UCT_TX + tx, iay = ty * U3_AP + tx;
            const double *AX0 = P0 + G3::AX, *AY0 = P0 + G3::AY, *AZ0 = P0 + G3::AZ, *AX1 = P1 + G3::AX, *AY1 = P1 + G3::AY;
            const double axp = AX0[iax], axm = AX0[G3::SAX + iax];
            const double ayp = AY0[iay], aym = AY0[G3::SAY + iay];
            const double azp = AZ0[iay], azm = AZ0[G3::SAZ + iay];
            auto along_x = [&](int f, double ap, double am) {
                const double *p = P0 + G3::XR + f * G3::SXR + ixr;
                return uct_bracket<LIN>(p, p + G3::SXR, 1, ap, am);
            };
            auto along_y = [&](int f, double ap, double am) {
                const double *p = P0 + G3::YR + f * G3::SYR + iyr;
                return uct_bracket<LIN>(p, p + G3::SYR, UCT_TX, ap, am);
            };
            auto along_z = [&](int f, double ap, double am) { return uct_bracket<LIN>(zw[f], zw[f + 1], 1, ap, am); };
            // E_z: i = x, j = y
            const double ez = -along_x(0, dmax(axp, AX0[iax + UCT_TX]), dmax(axm, AX0[G3::SAX + iax + UCT_TX])) +
                              along_y(0, dmax(ayp, AY0[iay + 1]), dmax(aym, AY0[G3::SAY + iay + 1]));
            // E_y: i = z, j = x
            const double ey = -along_z(0, dmax(azp, AZ0[iay + 1]), dmax(azm, AZ0[G3::SAZ + iay + 1])) +
                              along_x(2, dmax(axp, AX1[iax]), dmax(axm, AX1[G3::SAX + iax]));
            // E_x: i = y, j = z
            const double ex = -along_y(2, dmax(ayp, AY1[iay]), dmax(aym, AY1[G3::SAY + iay])) +
                              along_z(2, dmax(azp, AZ0[iay + U3_AP]), dmax(azm, AZ0[G3::SAZ + iay + U3_AP]));
            const int o = sz * k + ccol;
            st.E[0][o] = ex;
            st.E[1][o] = ey;
            st.E[2][o] = ez;
        }
#pragma unroll
        for (int f = 0; f < 4; ++f) {
#pragma unroll
            for (int m = 0; m < 5; ++m) zw[f][m] = zw[f][m + 1];
            zw[f][5] = znew[f];
        }
        s0 = s1;
    }
}

}  // namespace echo

// ------------------------------------------------------------------ points 4b + 5 for the staggered B
// k_bupd: curl of the DER-corrected edge EMFs (O8, eq.(10)) and the Runge-Kutta combination of the
// three face fields (O9), plane-marching like k_uct3: the x- and y-stencils of a plane come from
// cp.async-fed tiles (one plane ahead), the z-stencils from a 6-plane register window, the old B values
// of the next plane are loaded one round early.  Pure streaming: 12 doubles per cell.
//   dB_x/dt = -[D_y E_z - D_z E_y],  dB_y/dt = -[D_z E_x - D_x E_z],  dB_z/dt = -[D_x E_y - D_y E_x]
// with D_d the 6-point DER+difference stencil over cells c-3 .. c+2 along d.
namespace echo {

constexpr int BU_XE = UCT_XRW * UCT_TY;     // 21 x 8, x offsets -3 .. TX+1
constexpr int BU_YE = UCT_TX * UCT_YRH;     // 16 x 13, y offsets -3 .. TY+1

// curl (O8) + RK combination (O9) of the three face fields of ONE cell from its stencils: pz_x / py_x = E_z / E_y along
// x, pz_y / px_y = E_z / E_x along y (stride S), wy / wx = E_y / E_x along z; bc / bb = current and base B of the cell.
// Shared by k_bupd and k_bupd_flat so that the two stay bit-identical.
__device__ __forceinline__ void bupd_cell(const Grid &g, const double *pz_x, const double *py_x, const double *pz_y,
                                          const double *px_y, int S, const double wy[6], const double wx[6],
                                          const double bc[3], const double bb[3], const Update &up, double dt, int o) {
    const double dxEz = der_diff_ho(g.ho, pz_x[0], pz_x[1], pz_x[2], pz_x[3], pz_x[4], pz_x[5]);
    const double dxEy = der_diff_ho(g.ho, py_x[0], py_x[1], py_x[2], py_x[3], py_x[4], py_x[5]);
    const double dyEz = der_diff_ho(g.ho, pz_y[0], pz_y[S], pz_y[2 * S], pz_y[3 * S], pz_y[4 * S], pz_y[5 * S]);
    const double dyEx = der_diff_ho(g.ho, px_y[0], px_y[S], px_y[2 * S], px_y[3 * S], px_y[4 * S], px_y[5 * S]);
    const double dzEy = der_diff_ho(g.ho, wy[0], wy[1], wy[2], wy[3], wy[4], wy[5]);
    const double dzEx = der_diff_ho(g.ho, wx[0], wx[1], wx[2], wx[3], wx[4], wx[5]);
    double rb[3];
    rb[0] = -(g.rh[1] * dyEz - g.rh[2] * dzEy);
    rb[1] = -(g.rh[2] * dzEx - g.rh[0] * dxEz);
    rb[2] = -(g.rh[0] * dxEy - g.rh[1] * dyEx);
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        const double adv = bc[d] + dt * rb[d];
        up.out[5 + d][o] = (up.c0 == 0.0) ? adv : up.c0 * bb[d] + up.c1 * adv;
    }
}

__global__ void __launch_bounds__(UCT_NT) k_bupd(Grid g, const double *E0, const double *E1, const double *E2, Update up,
                                                 const Ctrl *ctrl, int CZ) {
    __shared__ double sXE[2][2][BU_XE];    // fields: E_z, E_y (differenced along x)
    __shared__ double sYE[2][2][BU_YE];    // fields: E_z, E_x (differenced along y)
    const int tid = threadIdx.x;
    const int tx = tid % UCT_TX, ty = tid / UCT_TX;
    const int nx = g.n[0], ny = g.n[1], nz = g.n[2];
    const int x0 = blockIdx.x * UCT_TX, y0 = blockIdx.y * UCT_TY, z0 = blockIdx.z * CZ;
    const int CZv = min(CZ, nz - z0);
    const int sy = g.s[1], sz = g.s[2];
    const double dt = ctrl->dt;
    const int active = ctrl->active;

    int oXE[2], oYE[2];
#pragma unroll
    for (int it = 0; it < 2; ++it) {
        const int e = tid + UCT_NT * it;
        oXE[it] = (e < BU_XE) ? wrapi(x0 - 3 + e % UCT_XRW, nx) + sy * wrapi(y0 + e / UCT_XRW, ny) : -1;
        oYE[it] = (e < BU_YE) ? wrapi(x0 + e % UCT_TX, nx) + sy * wrapi(y0 - 3 + e / UCT_TX, ny) : -1;
    }
    auto issue_plane = [&](int k, int slot) {
        const int pz = sz * wrapi(k, nz);
#pragma unroll
        for (int it = 0; it < 2; ++it) {
            const int e = tid + UCT_NT * it;
            if (oXE[it] >= 0) {
                cp_async8(&sXE[slot][0][e], E2 + (pz + oXE[it]));
                cp_async8(&sXE[slot][1][e], E1 + (pz + oXE[it]));
            }
            if (oYE[it] >= 0) {
                cp_async8(&sYE[slot][0][e], E2 + (pz + oYE[it]));
                cp_async8(&sYE[slot][1][e], E0 + (pz + oYE[it]));
            }
        }
        cp_async_commit();
    };
    const bool cellok = (x0 + tx < nx) && (y0 + ty < ny);
    const int ccol = min(x0 + tx, nx - 1) + sy * min(y0 + ty, ny - 1);

    issue_plane(z0, 0);
    double wy[6], wx[6];                   // z-windows of E_y and E_x: planes k-3 .. k+2
#pragma unroll
    for (int m = 0; m < 6; ++m) {
        const int pz = sz * wrapi(z0 - 3 + m, nz);
        wy[m] = __ldg(E1 + (pz + ccol));
        wx[m] = __ldg(E0 + (pz + ccol));
    }
    double bc[3], bb[3];                   // cur and base B of the plane about to be updated
    {
        const int o = sz * z0 + ccol;
#pragma unroll
        for (int d = 0; d < 3; ++d) { bc[d] = up.cur[5 + d][o]; bb[d] = __ldg(up.base[5 + d] + o); }
    }

    for (int r = 0; r < CZv; ++r) {
        const int k = z0 + r;
        cp_async_wait_all();
        __syncthreads();
        const bool more = (r + 1 < CZv);
        double nwy = 0.0, nwx = 0.0, nbc[3] = {0.0, 0.0, 0.0}, nbb[3] = {0.0, 0.0, 0.0};
        if (more) {
            issue_plane(k + 1, (r + 1) & 1);
            const int pz = sz * wrapi(k + 3, nz);
            nwy = __ldg(E1 + (pz + ccol));
            nwx = __ldg(E0 + (pz + ccol));
            const int o = sz * (k + 1) + ccol;
#pragma unroll
            for (int d = 0; d < 3; ++d) { nbc[d] = up.cur[5 + d][o]; nbb[d] = __ldg(up.base[5 + d] + o); }
        }
        if (cellok && active) {
            const int ps = r & 1;
            const double *pz_x = &sXE[ps][0][ty * UCT_XRW + tx], *py_x = pz_x + BU_XE;     // E_z, E_y along x
            const double *pz_y = &sYE[ps][0][ty * UCT_TX + tx], *px_y = pz_y + BU_YE;      // E_z, E_x along y
            bupd_cell(g, pz_x, py_x, pz_y, px_y, UCT_TX, wy, wx, bc, bb, up, dt, sz * k + ccol);
        }
#pragma unroll
        for (int m = 0; m < 5; ++m) { wy[m] = wy[m + 1]; wx[m] = wx[m + 1]; }
        wy[5] = nwy; wx[5] = nwx;
#pragma unroll
        for (int d = 0; d < 3; ++d) { bc[d] = nbc[d]; bb[d] = nbb[d]; }
    }
}

}  // namespace echo

// ------------------------------------------------------------------ 2.5-D grids (n_z = 1): march along y
// With one plane there is nothing to march along in z and a block of the kernels above would load one tile, wait
// for it, compute and exit.  k_uct2_flat / k_bupd_flat run the same arithmetic with the roles of "plane" taken by
// consecutive (x, y) tiles along y: the tiles of y-tile t+1 arrive by cp.async while tile t is computed.  Through the
// periodic wrap the six z-stencil values of a cell are all the cell's own value and plane k+1 is plane k, so the
// z-brackets see six equal values (the generic arithmetic applied to them: bitwise what k_uct3 / k_bupd give on a
// one-plane grid, and what a thicker grid with z-independent data gives - the dimensional-reduction tests).
namespace echo {

template <bool LIN = false>
__global__ void __launch_bounds__(UCT_NT) k_uct2_flat(Grid g, Stage st, int CY) {
    __shared__ double sXR[2][4][UCT_XR];
    __shared__ double sYR[2][4][UCT_YR];
    __shared__ double sAZ[2][2][UCT_AZ];
    __shared__ double sAX[2][2][UCT_AX];
    __shared__ double sAY[2][2][UCT_AY];

    const int tid = threadIdx.x;
    const int tx = tid % UCT_TX, ty = tid / UCT_TX;
    const int nx = g.n[0], ny = g.n[1];
    const int ntile = (ny + UCT_TY - 1) / UCT_TY;
    const int x0 = blockIdx.x * UCT_TX, t0 = blockIdx.y * CY;
    const int CYv = min(CY, ntile - t0);
    const int sy = g.s[1];

    // per-thread copy map: wrapped x offset and row of the (at most two) elements per region
    int xXR[2], xYR[2], xAX[2], xAY[2];
#pragma unroll
    for (int it = 0; it < 2; ++it) {
        const int e = tid + UCT_NT * it;
        xXR[it] = (e < UCT_XR) ? wrapi(x0 - 2 + e % UCT_XRW, nx) : -1;
        xYR[it] = (e < UCT_YR) ? wrapi(x0 + e % UCT_TX, nx) : -1;
        xAX[it] = (e < UCT_AX) ? wrapi(x0 + e % UCT_TX, nx) : -1;
        xAY[it] = (e < UCT_AZ) ? wrapi(x0 + e % UCT_AYW, nx) : -1;      // AY (8 rows) and AZ (9 rows) share it
    }
    const double *fXR[4] = {st.vb[1][1], st.Bf[1], st.vb[2][0], st.Bf[2]};
    const double *fYR[4] = {st.vb[0][0], st.Bf[0], st.vb[2][1], st.Bf[2]};
    const double *fZW[4] = {st.vb[0][1], st.Bf[0], st.vb[1][0], st.Bf[1]};

    auto issue_tile = [&](int y0, int slot) {
#pragma unroll
        for (int it = 0; it < 2; ++it) {
            const int e = tid + UCT_NT * it;
            if (xXR[it] >= 0) {
                const int o = xXR[it] + sy * wrapi(y0 + e / UCT_XRW, ny);
#pragma unroll
                for (int f = 0; f < 4; ++f) cp_async8(&sXR[slot][f][e], fXR[f] + o);
            }
            if (xYR[it] >= 0) {
                const int o = xYR[it] + sy * wrapi(y0 - 2 + e / UCT_TX, ny);
#pragma unroll
                for (int f = 0; f < 4; ++f) cp_async8(&sYR[slot][f][e], fYR[f] + o);
            }
            if (xAX[it] >= 0) {
                const int o = xAX[it] + sy * wrapi(y0 + e / UCT_TX, ny);
                cp_async8(&sAX[slot][0][e], st.ap[0] + o);
                cp_async8(&sAX[slot][1][e], st.am[0] + o);
            }
            if (xAY[it] >= 0) {
                const int o = xAY[it] + sy * wrapi(y0 + e / UCT_AYW, ny);
                if (e < UCT_AY) {
                    cp_async8(&sAY[slot][0][e], st.ap[1] + o);
                    cp_async8(&sAY[slot][1][e], st.am[1] + o);
                }
                cp_async8(&sAZ[slot][0][e], st.ap[2] + o);
                cp_async8(&sAZ[slot][1][e], st.am[2] + o);
            }
        }
        cp_async_commit();
    };
    const bool xok = (x0 + tx) < nx;
    const int cx = min(x0 + tx, nx - 1);
    auto cell = [&](int t) { return cx + sy * min(t * UCT_TY + ty, ny - 1); };

    issue_tile(t0 * UCT_TY, 0);
    double zc[4];
#pragma unroll
    for (int f = 0; f < 4; ++f) zc[f] = __ldg(fZW[f] + cell(t0));

    for (int r = 0; r < CYv; ++r) {
        const int t = t0 + r;
        cp_async_wait_all();
        __syncthreads();
        double zn[4] = {0.0, 0.0, 0.0, 0.0};
        if (r + 1 < CYv) {
            issue_tile((t + 1) * UCT_TY, (r + 1) & 1);
#pragma unroll
            for (int f = 0; f < 4; ++f) zn[f] = __ldg(fZW[f] + cell(t + 1));
        }
        if (xok && (t * UCT_TY + ty) < ny) {
            const int ps = r & 1;
            const int iax = ty * UCT_TX + tx, iay = ty * UCT_AYW + tx;
            const double axp = sAX[ps][0][iax], axm = sAX[ps][1][iax];
            const double ayp = sAY[ps][0][iay], aym = sAY[ps][1][iay];
            const double azp = sAZ[ps][0][iay], azm = sAZ[ps][1][iay];
            auto bracket = [&](const double *p, const double *q, int S, double ap, double am) {
                return uct_bracket<LIN>(p, q, S, ap, am);
            };
            auto along_x = [&](int f, double ap, double am) {
                const double *p = &sXR[ps][f][ty * UCT_XRW + tx];
                return bracket(p, p + UCT_XR, 1, ap, am);
            };
            auto along_y = [&](int f, double ap, double am) {
                const double *p = &sYR[ps][f][ty * UCT_TX + tx];
                return bracket(p, p + UCT_YR, UCT_TX, ap, am);
            };
            auto along_z = [&](int f, double ap, double am) {      // six equal values: the cell's own
                const double a = zc[f], b = zc[f + 1];
                const double pa[6] = {a, a, a, a, a, a}, qb[6] = {b, b, b, b, b, b};
                return bracket(pa, qb, 1, ap, am);
            };
            // E_z: i = x, j = y
            const double ez = -along_x(0, dmax(axp, sAX[ps][0][iax + UCT_TX]), dmax(axm, sAX[ps][1][iax + UCT_TX])) +
                              along_y(0, dmax(ayp, sAY[ps][0][iay + 1]), dmax(aym, sAY[ps][1][iay + 1]));
            // E_y: i = z, j = x   (plane k+1 is plane k)
            const double ey = -along_z(0, dmax(azp, sAZ[ps][0][iay + 1]), dmax(azm, sAZ[ps][1][iay + 1])) +
                              along_x(2, dmax(axp, axp), dmax(axm, axm));
            // E_x: i = y, j = z
            const double ex = -along_y(2, dmax(ayp, ayp), dmax(aym, aym)) +
                              along_z(2, dmax(azp, sAZ[ps][0][iay + UCT_AYW]), dmax(azm, sAZ[ps][1][iay + UCT_AYW]));
            const int o = cell(t);
            st.E[0][o] = ex;
            st.E[1][o] = ey;
            st.E[2][o] = ez;
        }
#pragma unroll
        for (int f = 0; f < 4; ++f) zc[f] = zn[f];
    }
}

__global__ void __launch_bounds__(UCT_NT) k_bupd_flat(Grid g, const double *E0, const double *E1, const double *E2, Update up,
                                                      const Ctrl *ctrl, int CY) {
    __shared__ double sXE[2][2][BU_XE];    // E_z, E_y (differenced along x)
    __shared__ double sYE[2][2][BU_YE];    // E_z, E_x (differenced along y)
    const int tid = threadIdx.x;
    const int tx = tid % UCT_TX, ty = tid / UCT_TX;
    const int nx = g.n[0], ny = g.n[1];
    const int ntile = (ny + UCT_TY - 1) / UCT_TY;
    const int x0 = blockIdx.x * UCT_TX, t0 = blockIdx.y * CY;
    const int CYv = min(CY, ntile - t0);
    const int sy = g.s[1];
    const double dt = ctrl->dt;
    const int active = ctrl->active;

    int xXE[2], xYE[2];
#pragma unroll
    for (int it = 0; it < 2; ++it) {
        const int e = tid + UCT_NT * it;
        xXE[it] = (e < BU_XE) ? wrapi(x0 - 3 + e % UCT_XRW, nx) : -1;
        xYE[it] = (e < BU_YE) ? wrapi(x0 + e % UCT_TX, nx) : -1;
    }
    auto issue_tile = [&](int y0, int slot) {
#pragma unroll
        for (int it = 0; it < 2; ++it) {
            const int e = tid + UCT_NT * it;
            if (xXE[it] >= 0) {
                const int o = xXE[it] + sy * wrapi(y0 + e / UCT_XRW, ny);
                cp_async8(&sXE[slot][0][e], E2 + o);
                cp_async8(&sXE[slot][1][e], E1 + o);
            }
            if (xYE[it] >= 0) {
                const int o = xYE[it] + sy * wrapi(y0 - 3 + e / UCT_TX, ny);
                cp_async8(&sYE[slot][0][e], E2 + o);
                cp_async8(&sYE[slot][1][e], E0 + o);
            }
        }
        cp_async_commit();
    };
    const bool xok = (x0 + tx) < nx;
    const int cx = min(x0 + tx, nx - 1);
    auto cell = [&](int t) { return cx + sy * min(t * UCT_TY + ty, ny - 1); };

    issue_tile(t0 * UCT_TY, 0);
    double ec[2], bc[3], bb[3];            // E_y, E_x of the cell (its whole z-stencil), cur and base B
    {
        const int o = cell(t0);
        ec[0] = __ldg(E1 + o);
        ec[1] = __ldg(E0 + o);
#pragma unroll
        for (int d = 0; d < 3; ++d) { bc[d] = up.cur[5 + d][o]; bb[d] = __ldg(up.base[5 + d] + o); }
    }
    for (int r = 0; r < CYv; ++r) {
        const int t = t0 + r;
        cp_async_wait_all();
        __syncthreads();
        double nec[2] = {0.0, 0.0}, nbc[3] = {0.0, 0.0, 0.0}, nbb[3] = {0.0, 0.0, 0.0};
        if (r + 1 < CYv) {
            issue_tile((t + 1) * UCT_TY, (r + 1) & 1);
            const int o = cell(t + 1);
            nec[0] = __ldg(E1 + o);
            nec[1] = __ldg(E0 + o);
#pragma unroll
            for (int d = 0; d < 3; ++d) { nbc[d] = up.cur[5 + d][o]; nbb[d] = __ldg(up.base[5 + d] + o); }
        }
        if (xok && (t * UCT_TY + ty) < ny && active) {
            const int ps = r & 1;
            const double *pz_x = &sXE[ps][0][ty * UCT_XRW + tx], *py_x = pz_x + BU_XE;
            const double *pz_y = &sYE[ps][0][ty * UCT_TX + tx], *px_y = pz_y + BU_YE;
            const double wy[6] = {ec[0], ec[0], ec[0], ec[0], ec[0], ec[0]};      // the z-stencils of a one-plane grid:
            const double wx[6] = {ec[1], ec[1], ec[1], ec[1], ec[1], ec[1]};      // six times the cell's own value
            bupd_cell(g, pz_x, py_x, pz_y, px_y, UCT_TX, wy, wx, bc, bb, up, dt, cell(t));
        }
        ec[0] = nec[0]; ec[1] = nec[1];
#pragma unroll
        for (int d = 0; d < 3; ++d) { bc[d] = nbc[d]; bb[d] = nbb[d]; }
    }
}

}  // namespace echo

// ------------------------------------------------------------------ point 1 inside echo_step (UCT = YES)
// k_prim_march: INT of the staggered B + con2prim (O1, O2) with the data movement of k_bupd: a 16 x 8 tile
// of (x, y) marches along z; B_x with its x-halo and B_y with its y-halo of plane k+1 arrive by cp.async while plane
// k is inverted, B_z lives in a 6-plane register window, the conserved fields (and, UPD, the stage-1 rhs) of plane
// k+1 are loaded into registers one round early.  The Newton iterations of one plane thus overlap the memory
// latency of the next, which the thread-per-cell k_prim (kept for the STATS passes and UCT = NO) cannot do.
// Same formulas on the same operands as k_prim; the compiler schedules and contracts them differently in the two
// kernels, so the results agree to round-off (a few ulp), not bit for bit.
namespace echo {

template <bool UPD>
__global__ void __launch_bounds__(UCT_NT) k_prim_march(Grid g, Stage st, double gam, Ctrl *ctrl, PrimUpd pu, int CZ,
                                                       const int *gate) {
    __shared__ double sBX[2][BU_XE];       // B_x, x offsets -3 .. TX+1
    __shared__ double sBY[2][BU_YE];       // B_y, y offsets -3 .. TY+1
    const int tid = threadIdx.x;
    const int tx = tid % UCT_TX, ty = tid / UCT_TX;
    const int nx = g.n[0], ny = g.n[1], nz = g.n[2];
    const int x0 = blockIdx.x * UCT_TX, y0 = blockIdx.y * UCT_TY, z0 = blockIdx.z * CZ;
    const int CZv = min(CZ, nz - z0);
    const int sy = g.s[1], sz = g.s[2];
    const double dt = UPD ? ctrl->dt : 0.0;

    int oXE[2], oYE[2];
#pragma unroll
    for (int it = 0; it < 2; ++it) {
        const int e = tid + UCT_NT * it;
        oXE[it] = (e < BU_XE) ? wrapi(x0 - 3 + e % UCT_XRW, nx) + sy * wrapi(y0 + e / UCT_XRW, ny) : -1;
        oYE[it] = (e < BU_YE) ? wrapi(x0 + e % UCT_TX, nx) + sy * wrapi(y0 - 3 + e / UCT_TX, ny) : -1;
    }
    auto issue_plane = [&](int k, int slot) {
        const int pz = sz * wrapi(k, nz);
#pragma unroll
        for (int it = 0; it < 2; ++it) {
            const int e = tid + UCT_NT * it;
            if (oXE[it] >= 0) cp_async8(&sBX[slot][e], st.Bf[0] + (pz + oXE[it]));
            if (oYE[it] >= 0) cp_async8(&sBY[slot][e], st.Bf[1] + (pz + oYE[it]));
        }
        cp_async_commit();
    };
    const bool cellok = (x0 + tx < nx) && (y0 + ty < ny);
    const int ccol = min(x0 + tx, nx - 1) + sy * min(y0 + ty, ny - 1);
    const bool inxy = (x0 + tx) >= g.lo[0] && (x0 + tx) < g.hi[0] && (y0 + ty) >= g.lo[1] && (y0 + ty) < g.hi[1];

    issue_plane(z0, 0);
    double wz[6];                          // B_z of planes k-3 .. k+2
#pragma unroll
    for (int m = 0; m < 6; ++m) wz[m] = __ldg(st.Bf[2] + (sz * wrapi(z0 - 3 + m, nz) + ccol));
    double un[5], rn[5];
#pragma unroll
    for (int v = 0; v < 5; ++v) {
        un[v] = __ldg(st.U[v] + (sz * z0 + ccol));
        rn[v] = UPD ? __ldg(st.R[v] + (sz * z0 + ccol)) : 0.0;
    }

    for (int r = 0; r < CZv; ++r) {
        const int k = z0 + r;
        cp_async_wait_all();
        __syncthreads();
        const bool more = (r + 1 < CZv);
        double nwz = 0.0, nu[5] = {0.0, 0.0, 0.0, 0.0, 0.0}, nr[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
        if (more) {
            issue_plane(k + 1, (r + 1) & 1);
            nwz = __ldg(st.Bf[2] + (sz * wrapi(k + 3, nz) + ccol));
            const int o = sz * (k + 1) + ccol;
#pragma unroll
            for (int v = 0; v < 5; ++v) {
                nu[v] = __ldg(st.U[v] + o);
                if (UPD) nr[v] = __ldg(st.R[v] + o);
            }
        }
        if (cellok) {
            const int ps = r & 1;
            const double *px = &sBX[ps][ty * UCT_XRW + tx], *py = &sBY[ps][ty * UCT_TX + tx];
            constexpr int S = UCT_TX;
            double B[3];
            B[0] = int_ho(g.ho, px[0], px[1], px[2], px[3], px[4], px[5]);
            B[1] = int_ho(g.ho, py[0], py[S], py[2 * S], py[3 * S], py[4 * S], py[5 * S]);
            B[2] = int_ho(g.ho, wz[0], wz[1], wz[2], wz[3], wz[4], wz[5]);
            const int o = sz * k + ccol;
            double u[5];
#pragma unroll
            for (int v = 0; v < 5; ++v) {
                u[v] = un[v];
                if (UPD) {
                    u[v] = u[v] + dt * rn[v];
                    pu.uout[v][o] = u[v];
                }
            }
            double q[5];
            const int it = con2prim(gam, u, B, q);
#pragma unroll
            for (int v = 0; v < 5; ++v) st.P[v][o] = q[v];
#pragma unroll
            for (int d = 0; d < 3; ++d) st.Bc[d][o] = B[d];
            if (it < 0 && inxy && k >= g.lo[2] && k < g.hi[2] && *gate) atomicAdd(&ctrl->c2p_fail_total, 1ull);
        }
#pragma unroll
        for (int m = 0; m < 5; ++m) wz[m] = wz[m + 1];
        wz[5] = nwz;
#pragma unroll
        for (int v = 0; v < 5; ++v) { un[v] = nu[v]; rn[v] = nr[v]; }
    }
}

}  // namespace echo
