// echo_types.cuh — plain structs shared by the kernels and the C-ABI layer (device + host).
#pragma once
#include <cuda_runtime.h>

namespace echo {

// Grid geometry: unit periodic box, h_d = 1/n_d, x fastest.
struct Grid {
    int n[3];
    int s[3];         // linear strides in elements: 1, nx, nx*ny (N < 2^31: 32-bit cell indices)
    long long N;
    double h[3], rh[3];   // spacing and its reciprocal (n_d exactly)
    // interior of a domain-decomposition block (echo_create_block): cells lo_d <= c_d < hi_d; the rest is halo
    // that the caller refreshes after every stage.  Global reductions (a_max, con2prim failures) only look at
    // the interior.  A plain periodic box has lo = 0, hi = n.
    int lo[3], hi[3];
    // scheme switches of the paper (echo_set_scheme): ho = 0 makes INT and DER second order;
    // uct = 0 evolves a cell-centred B like the other conserved variables
    int ho, uct;
    int rec;                  // REC: 5 = MP5, 2 = limited linear (MC), echo_set_order
};

// Device control block (first bytes of the workspace).  Everything echo_step needs between
// kernels lives here so that no host synchronisation is needed inside a step.
struct Ctrl {
    double t, dt, dt_last, t_end;
    double amax;                       // last stage-1 maximum characteristic speed (a8)
    unsigned long long amax_bits;      // running max of non-negative doubles, as their bit pattern
    long long steps;
    int active;                        // 0 once t >= t_end: every kernel of the step returns at once
    int one;                           // constant 1 (the "always active" flag)
    // con2prim statistics: of the most recent full pass, and failures since set_primitives
    unsigned long long c2p_sumit, c2p_calls, c2p_fail, c2p_fail_total;
    int c2p_maxit;
    int pad_;
};

constexpr int NFIELD = 44;         // U[5] Bf[3] | U0[5] Bf0[3] | P[5] Bc[3] | R[5] | ap[3] am[3] vb[6] | E[3]
constexpr int NPART = 1024;        // chunks of the deterministic reductions
constexpr int NPARTF = 16;         // partial rows (8 sums + spare)
constexpr size_t CTRL_BYTES = 4096;
constexpr size_t PART_BYTES = sizeof(double) * NPART * NPARTF;

// Pointers of one stage, passed by value to the kernels.
struct Stage {
    const double *U[5];    // conserved state the operator L is applied to
    const double *Bf[3];   // staggered B of that state
    double *P[5];          // primitives rho, vx, vy, vz, p
    double *Bc[3];         // centred B (INT of the faces)
    double *R[5];          // rhs of the 5 conserved cell fields
    double *ap[3], *am[3]; // a+ and a- saved at the d-faces
    double *vb[3][2];      // vbar_{(d+1)%3}, vbar_{(d+2)%3} saved at the d-faces
    double *E[3];          // edge EMFs
};

// Tensor maps (TMA descriptors, 128 bytes each, built on the host by cuTensorMapEncodeTiled) of the fields the
// plane-marching UCT kernel stages, one per (field, tile shape); passed by value as a __grid_constant__ parameter.
struct alignas(64) TmaDesc { unsigned long long w[16]; };     // same size and alignment as CUtensorMap
struct UctMaps {
    TmaDesc xr[4];      // vbar_x@y, B_y, vbar_x@z, B_z : boxes 22 x 8   (x0-2 .. x0+19)
    TmaDesc yr[4];      // vbar_y@x, B_x, vbar_y@z, B_z : boxes 16 x 13  (y0-2 .. y0+10)
    TmaDesc az[2];      // a+_z, a-_z : 18 x 9
    TmaDesc ax[2];      // a+_x, a-_x : 16 x 9
    TmaDesc ay[2];      // a+_y, a-_y : 18 x 8
    int ok;             // 0: no maps (rows not 16-byte aligned or grid too small): every tile takes the cp.async path
};

// RK combination  out = c0 * base + c1 * (cur + dt * rhs)   (O9)
struct Update {
    const double *base[8];   // U^n, Bf^n
    const double *cur[8];    // state the stage started from
    double *out[8];
    double c0, c1;
};

}  // namespace echo
