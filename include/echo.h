/* echo.h — C ABI of libecho_b200: one explicit time step of 3-D special-relativistic ideal MHD
 * (the ECHO scheme of arXiv:2401.03008) on a uniform periodic Cartesian unit box, FP64, as
 * hand-written CUDA kernels for sm_100a.
 *
 * Citations: "P:L<n>" = line n of the paper text; "O1".."O9", "S1".."S19" = the
 * readings of the paper recorded in DESIGN.md (same labels as SURVEY.md §8(c)).
 *
 * Conventions (all calls)
 *   - extern "C", opaque handle, plain pointers and sizes; no exceptions cross the ABI.
 *   - Unless a parameter says "host", every array pointer is a DEVICE pointer to a caller-owned
 *     FP64 buffer of N = nx*ny*nz elements, x fastest: index = i + nx*(j + ny*k).  The
 *     library never frees caller memory and keeps no pointer beyond the call, except the
 *     workspace and the stream given to echo_bind.
 *   - Staggering: cell (i,j,k) is centred at ((i+1/2)/nx, (j+1/2)/ny, (k+1/2)/nz); a face array
 *     Bd[i,j,k] is the point value of B_d at the d-face on the + side of the cell; an edge
 *     array Ek[i,j,k] sits at the k-edge displaced +1/2 in the two other directions.  All indices
 *     wrap periodically; there are no ghost cells.
 *   - Calls enqueue work on the bound CUDA stream and do NOT synchronise unless stated.
 *   - Return value: ECHO_OK (0) or a negative ECHO_E* code; echo_last_error(ctx) gives a message.
 *   - There is no CPU fallback: without a CUDA device every compute call returns ECHO_ECUDA.
 */
#ifndef ECHO_B200_H
#define ECHO_B200_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

#define ECHO_OK 0
#define ECHO_EINVAL (-1) /* bad argument or size */
#define ECHO_ENOMEM (-2) /* workspace missing or too small */
#define ECHO_ECUDA (-3)  /* CUDA runtime error (message in echo_last_error) */
#define ECHO_ESTATE (-4) /* called before echo_bind / echo_set_primitives */
#define ECHO_EC2P (-5)   /* at least one cell failed the conservative->primitive inversion */

#define ECHO_NDIAG 24

typedef struct echo_ctx echo_ctx;

/* Host only.  Periodic unit box of nx*ny*nz cells (each >= 1; a size-1 axis is legal and makes
 * the problem 2-D / 1-D through the periodic wrap), ideal-gas index gamma > 1 (eq.(6)),
 * Courant number cfl > 0 (dt = cfl * min_d h_d / a_max, S9).  Returns NULL on bad arguments, on
 * nx*ny*nz >= 2^31 - 64 (32-bit cell indices) and on nz > 65535, ny > 262140 or (nz > 1 and ny > 65535)
 * (grid-dimension limits of the launches). */
echo_ctx *echo_create(int nx, int ny, int nz, double gamma, double cfl);

/* Host only.  The paper's scheme switches, to be called before echo_set_primitives.
 * ho = 0: INT and DER second order (two-point average, identity) instead of sixth; everything else unchanged; the
 * divergence UCT then preserves is the plain two-point one.  uct = 0: the cell-centred B is evolved by flux
 * differences like the other conserved variables, with no divergence control; the three "face" arrays of
 * echo_set_primitives[_host] / echo_get_primitives[_host] then hold (and return) the CELL-CENTRED B, echo_rhs returns
 * the rhs of that B in rhsB and zeros in E, echo_div_b applies its face formula to those arrays (not a conserved
 * quantity of this scheme).  uct = 0 on a block handle (echo_create_block): ECHO_EINVAL, and echo_stage_sweeps /
 * echo_stage_finish return ECHO_EINVAL on a uct = 0 handle.  ECHO_ESTATE once a state exists.
 * Defaults: uct = 1, ho = 1. */
int echo_set_scheme(echo_ctx *ctx, int uct, int ho);

/* Host only.  The second-order variant the paper quotes a throughput for ("second order time-stepping and
 * linear reconstruction rather than MP5"), to be called before echo_set_primitives and after echo_set_scheme.
 * rec = 5: MP5 (default); rec = 2: v_i + MC(v_i - v_{i-1}, v_{i+1} - v_i)/2 with the monotonized-central slope
 * MC(a, b) = minmod(2a, 2b, (a+b)/2) (reading O3b), used by the sweeps and by UCT; built with the
 * second-order INT/DER only: ECHO_EINVAL unless echo_set_scheme(ctx, uct, 0) was called first.
 * rk = 3: SSP-RK3 (default); rk = 2: U1 = U^n + dt L(U^n), U^{n+1} = (U^n + U1 + dt L(U1))/2, dt as for RK3.
 * ECHO_EINVAL on other values, ECHO_ESTATE once a state exists. */
int echo_set_order(echo_ctx *ctx, int rec, int rk);

/* Host only.  Frees the handle (never the workspace). */
void echo_destroy(echo_ctx *ctx);

/* Host only.  Bytes of device workspace the handle needs (44 fields of N doubles + control block,
 * DESIGN.md "Data layout in HBM"). */
size_t echo_workspace_bytes(const echo_ctx *ctx);

/* Binds a caller-owned device workspace (256-byte aligned, >= echo_workspace_bytes) and a CUDA
 * stream (cudaStream_t passed as void*; NULL = default stream).  The workspace must outlive the
 * handle.  Zero-fills the control block.  ECHO_ENOMEM if too small or misaligned, ECHO_EINVAL if it is
 * not device memory.  The handle remembers the device the workspace lives on: every later call runs its
 * kernels there (the stream must belong to that device) and restores the caller's current device. */
int echo_bind(echo_ctx *ctx, void *dev_workspace, size_t bytes, void *cuda_stream);

/* Message of the last error on this handle (host string owned by the handle; "" if none). */
const char *echo_last_error(const echo_ctx *ctx);

/* Initial data: cell-centred rho, v, p and FACE-staggered B point values.  Computes the centred B
 * by INT (O1) and the conserved variables by prim2cons (definitions);
 * sets t = 0, steps = 0.  The caller is responsible for divergence-free faces (S11). */
int echo_set_primitives(echo_ctx *ctx, const double *rho, const double *vx, const double *vy,
                        const double *vz, const double *p, const double *bx_face,
                        const double *by_face, const double *bz_face);

/* Same, from HOST buffers (pageable or pinned): eight cudaMemcpyAsync host->device into workspace
 * scratch, then echo_set_primitives.  Used by the end-to-end measurement. */
int echo_set_primitives_host(echo_ctx *ctx, const double *rho, const double *vx, const double *vy,
                             const double *vz, const double *p, const double *bx_face,
                             const double *by_face, const double *bz_face);

/* Staggered B from an edge-centred vector potential (S11): B = curl A with the same DER-corrected
 * discrete curl as the induction equation (O8, eq.(10)), so that echo_div_b of the result
 * vanishes to round-off; then adds the uniform field (b0x,b0y,b0z).  ax/ay/az are edge arrays,
 * bx/by/bz face arrays (outputs), all device. */
int echo_faces_from_potential(echo_ctx *ctx, const double *ax, const double *ay, const double *az,
                              double b0x, double b0y, double b0z, double *bx_face, double *by_face,
                              double *bz_face);

/* Advances nsteps full SSP-RK3 steps (O9; five points of a sub-step), or fewer if t
 * reaches t_end: the last dt is clipped to t_end - t on the device and later steps are no-ops
 * (pass +inf to disable).  The time step is formed on the device from the stage-1 characteristic
 * speeds of the same step (S9).  No host synchronisation.  ECHO_EINVAL on a block
 * handle with halos (echo_create_block) that the caller has to refresh: those are stepped stage by stage
 * by their owner (a block whose padded sides are all physical boundaries, echo_set_boundaries, is fine). */
int echo_step(echo_ctx *ctx, int nsteps, double t_end);

/* Host loop around echo_step: advances until t >= t_end (last dt clipped), max_steps steps were taken, or a
 * con2prim failure was counted.  echo_step cannot know on the host when t_end is reached, and steps enqueued past
 * it still run their kernels; this call enqueues chunks sized from the current a_max (at most 2048 steps, about 2 %
 * more than needed) and reads the 4 KB control block back after each chunk, so it SYNCHRONISES the stream a few
 * times.  steps_taken_host (host pointer, may be NULL) receives the number of steps actually taken.  Returns
 * ECHO_EC2P if the run stopped on a con2prim failure, ECHO_EINVAL for NaN / negative arguments and for block
 * handles. */
int echo_run_until(echo_ctx *ctx, double t_end, long max_steps, long *steps_taken_host);

/* Runs INT + con2prim on the current state and writes the 8 cell-centred fields; the three face
 * pointers may be NULL.  Does not synchronise.  (con2prim failures are reported by
 * echo_diagnostics, not here, because that would need a synchronisation.) */
int echo_get_primitives(echo_ctx *ctx, double *rho, double *vx, double *vy, double *vz, double *p,
                        double *bx_c, double *by_c, double *bz_c, double *bx_face, double *by_face,
                        double *bz_face);

/* Same into HOST buffers; synchronises the stream before returning. */
int echo_get_primitives_host(echo_ctx *ctx, double *rho, double *vx, double *vy, double *vz,
                             double *p, double *bx_c, double *by_c, double *bz_c, double *bx_face,
                             double *by_face, double *bz_face);

/* Same, without the final synchronisation: the host buffers (which must be PINNED for the copies to be
 * asynchronous) are valid after echo_synchronize(ctx).  Lets a caller overlap the transfers of one handle with
 * the kernels of another handle bound to a different stream. */
int echo_get_primitives_host_async(echo_ctx *ctx, double *rho, double *vx, double *vy, double *vz,
                                   double *p, double *bx_c, double *by_c, double *bz_c, double *bx_face,
                                   double *by_face, double *bz_face);

/* Blocks the host until everything enqueued on the handle's stream has finished. */
int echo_synchronize(echo_ctx *ctx);

/* Copies the 5 conserved cell fields D, Sx, Sy, Sz, U of the current state (device). */
int echo_get_conserved(echo_ctx *ctx, double *D, double *Sx, double *Sy, double *Sz, double *U);

/* Spatial operator L(U) of eq.(9)-(10) for the current state, without changing it:
 * rhsU[5] cell arrays, rhsB[3] face arrays, E[3] edge arrays (O7); any of the three pointer
 * tables (HOST arrays of DEVICE pointers) may be NULL.  amax_host (host, may be NULL) receives
 * the maximum characteristic speed (a8); synchronises if amax_host != NULL. */
int echo_rhs(echo_ctx *ctx, double *const *rhsU, double *const *rhsB, double *const *E,
             double *amax_host);

/* Stateless batched conservative->primitive inversion (O2, "iterative Newton scheme") of n
 * independent states on the given stream (void* cudaStream_t).  iters[i] (device int array, may
 * be NULL) = Newton updates applied, negative on failure (outputs NaN).  Does not synchronise. */
int echo_con2prim(double gamma, long n, const double *D, const double *Sx, const double *Sy,
                  const double *Sz, const double *U, const double *Bx, const double *By,
                  const double *Bz, double *rho, double *vx, double *vy, double *vz, double *p,
                  int *iters, void *cuda_stream);

/* Stateless batched primitive->conservative map. */
int echo_prim2cons(double gamma, long n, const double *rho, const double *vx, const double *vy,
                   const double *vz, const double *p, const double *Bx, const double *By,
                   const double *Bz, double *D, double *Sx, double *Sy, double *Sz, double *U,
                   void *cuda_stream);

/* High-order divergence sum_d (DER_d(B_d)_{+1/2} - DER_d(B_d)_{-1/2})/h_d at cell centres (S10),
 * the one UCT preserves.  div_field (device, N doubles) may be NULL; max_abs_host (host)
 * may be NULL.  Synchronises. */
int echo_div_b(echo_ctx *ctx, double *div_field, double *max_abs_host);

/* The same divergence (S10) for callers that may not allocate: no handle, no workspace, no cudaMalloc,
 * cudaFree or allocating library routine, no synchronisation -- two kernel launches on cuda_stream, legal under
 * stream capture once echo_div_b_static_setup has run on the device.  Periodic unit box of nx*ny*nz cells (h_d =
 * 1/n_d, x fastest), ho as in echo_set_scheme; bx/by/bz_face: device, N doubles each, entry c = face on the + side
 * of cell c (the layout of echo_set_primitives).  Outputs (device, written asynchronously on cuda_stream):
 * div_field (N doubles) may be NULL; max_abs_dev (ONE double, the maximum of |div B|) may be NULL; not both.
 * Scratch: one partial maximum per tile of 64 x 4 x 1 cells in a static device array of
 * ECHO_DIV_B_STATIC_MAX_TILES doubles (512 KiB, held by every GPU that loads the library until exit), so
 *     ceil(nx/64) * ceil(ny/4) * nz <= ECHO_DIV_B_STATIC_MAX_TILES      (256^3 fits exactly);
 * a larger grid returns ECHO_EINVAL before anything is launched, with the sizes in echo_div_b_static_error().
 * The array is shared by every call on a device and keeps the last call's contents; each call overwrites every
 * slot it reads, so nothing needs clearing, but two calls that can overlap on the GPU (different streams, no
 * ordering between them) race on it: serialise them.  Results equal echo_div_b's (same arithmetic per cell).
 * Errors: ECHO_EINVAL (sizes, null pointers), ECHO_ECUDA (symbol lookup or launch failed). */
#define ECHO_DIV_B_STATIC_MAX_TILES 65536
int echo_div_b_static(int nx, int ny, int nz, int ho, const double *bx_face, const double *by_face,
                      const double *bz_face, double *div_field, double *max_abs_dev, void *cuda_stream);

/* Host only.  Looks up the device address of the static scratch for the CURRENT device (once per device; later
 * calls return at once).  echo_div_b_static calls it itself; call it before stream capture begins. */
int echo_div_b_static_setup(void);

/* Host only.  Message of the last failed echo_div_b_static[_setup] call of this thread ("" if none). */
const char *echo_div_b_static_error(void);

/* out (HOST, ECHO_NDIAG doubles) = {t, dt_last, steps, amax, sum D, sum Sx, sum Sy, sum Sz, sum U
 * (each x cell volume), sum Bx, sum By, sum Bz over faces (x volume), max|div_HO B|, max W,
 * min rho, min p, con2prim max iterations, con2prim mean iterations (both of the pass run by this
 * call), con2prim failures since echo_set_primitives, 0...}.  Sums are taken in a fixed order
 * (fixed chunks on the device, extended precision across chunks on the host) so that drift at
 * 1e-15 is measurable.  Synchronises.  Returns ECHO_EC2P if the failure count is non-zero. */
int echo_diagnostics(echo_ctx *ctx, double *out);

/* ---- domain-decomposition blocks ("next" row f1: multi-GPU) ----------------------------
 * A block is a periodic box of nx*ny*nz cells INCLUDING halo_d cells on each side of every decomposed axis
 * (halo_d = 0: the block spans the whole periodic axis), with the spacing h_d = 1/gn_d of the GLOBAL unit box of
 * gnx*gny*gnz cells.  The kernels are the periodic ones of echo_step; the periodic wrap of the padded block only
 * corrupts the halo, 8 cells per RK stage (the dependency reach of one stage, P:L138 + HO stencils), so with
 * halo_d = 8 the interior stays exact provided the caller refreshes the halos of the 8 evolved fields from the
 * neighbouring blocks after every stage.  a_max and the con2prim failure count only look at the interior.
 * One step of a block, driven by the caller (paper_2401_03008_b200/blocks.py):
 *     for stage in 1, 2, 3:
 *         echo_stage_sweeps(ctx, stage, t_end)      INT + con2prim + the three sweeps (+ a_max in stage 1)
 *         [stage 1: all-reduce(max) of the 8-byte a_max word at echo_ctrl_offset(0) across the blocks]
 *         echo_stage_finish(ctx, stage)             (stage 1: dt) UCT, update of the staggered B
 *         [refresh the halos of the 8 fields echo_stage_halo_fields names from the neighbours: packed messages,
 *          echo_halo_pack / echo_halo_unpack; the 5 cell fields may already travel while echo_stage_finish runs]
 * echo_set_primitives / echo_get_primitives work on the padded block as on a plain box. */
echo_ctx *echo_create_block(int nx, int ny, int nz, double gamma, double cfl, int gnx, int gny, int gnz,
                            int halo_x, int halo_y, int halo_z);

/* ---- physical boundaries ("next" row f4, first slice: non-periodic boundaries in flat space) -----------------------
 * Host only, before echo_set_primitives, on a handle made by echo_create_block with halo_d = 8 on the bounded axes
 * (the paper's code keeps ghost cells that are filled before every stencil loop; here they are
 * filled once per RK stage, which the 8 layers allow).  kinds (HOST, 6 ints) = {x_lo, x_hi, y_lo, y_hi, z_lo, z_hi}:
 *   0  none: the axis is periodic (halo 0) or that halo is refreshed by the caller from a neighbouring block;
 *   1  reflecting wall: ghost layers = mirror image of the interior with the parity of each field under the reflection
 *      (scalars even, the momentum normal to the wall odd; B is axial: normal component even, tangential ones odd);
 *   2  outflow: zero gradient (ghost layers = the nearest interior value).
 * The wall lies on the face between the last ghost layer and the first interior cell: entry lo-1 (resp. hi-1) of the
 * face array of the normal B is the wall face; it is evolved by the scheme and must be given in echo_set_primitives
 * (all other ghost entries passed in are ignored and overwritten).  a_max, the con2prim failure count, the sums and the
 * maximum of div B of echo_diagnostics look at the interior only.  A handle whose every padded side has a kind != 0 is
 * advanced by echo_step / echo_run_until like a plain box (the ghost fill runs inside the step, after every stage).
 * ECHO_EINVAL: bad kind, fewer than 8 ghost layers on that side, uct = 0.  ECHO_ESTATE once a state exists. */
int echo_set_boundaries(echo_ctx *ctx, const int *kinds);

/* The ghost fill itself, for callers that drive a block stage by stage (a block at the edge of a decomposed bounded
 * domain: physical boundary on one side, neighbour on the other): fills the ghost layers of the 8 given workspace
 * fields (HOST array; slots 0-4 are treated as D, S_x, S_y, S_z, U - or their rhs -, slots 5-7 as B_x, B_y, B_z; -1 =
 * skip) on every side that has a boundary kind, axes in the order x, y, z.  No synchronisation. */
int echo_fill_boundaries(echo_ctx *ctx, const int *fields);

/* Host only.  Byte offset, inside the workspace given to echo_bind, of field `field` (0..43; 0-7 the state U^n =
 * D, Sx, Sy, Sz, U, Bx, By, Bz; 8-15 the stage state); each field is nx*ny*nz doubles. */
size_t echo_field_offset(const echo_ctx *ctx, int field);

/* Host only.  Byte offset inside the workspace of a control word: 0 = a_max as the bit pattern of a non-negative
 * double (8 bytes, ordered like an unsigned integer: all-reduce it with MAX on int64), 1 = t, 2 = dt,
 * 3 = con2prim failure count (uint64). */
size_t echo_ctrl_offset(int what);

/* First and second half of RK stage `stage` (1 .. 3, or 1 .. 2 with SSP-RK2) of a block step; see above.  These are the
 * halves echo_step itself is made of (same kernels, same arguments), so a decomposed run repeats the undecomposed one
 * bit for bit.  No synchronisation.  ECHO_EINVAL on a uct = 0 handle. */
int echo_stage_sweeps(echo_ctx *ctx, int stage, double t_end);
int echo_stage_finish(echo_ctx *ctx, int stage);

/* Host only.  fields (HOST, 8 ints) = the workspace fields whose halos the NEXT half needs from the neighbouring
 * blocks once stage `stage` has finished: five cell fields then three face fields.  After stage 1 these are the rhs of
 * the cell fields (24..28: the update U1 = U^n + dt rhs is formed inside the INT + con2prim pass of stage 2, for every
 * cell of the padded block, from the refreshed rhs) and the stage B (13..15); after an inner stage the stage state
 * (8..15); after the last stage the state (0..7).  The five cell fields are final when echo_stage_sweeps returns, the
 * three face fields when echo_stage_finish does - so the exchange of the former can overlap the UCT kernels. */
int echo_stage_halo_fields(const echo_ctx *ctx, int stage, int *fields);

/* Packed halo messages of a block handle: ONE buffer per axis and side holds the slabs of 8 fields, [field][cell of the
 * slab, x fastest], each slab halo_d cells thick along `axis` and spanning the whole padded block along the other two
 * axes (edges and corners travel with the later axes when the axes are exchanged in the order x, y, z).
 * echo_halo_doubles: doubles per message (0 if the axis is not decomposed).  echo_halo_pack gathers the INTERIOR slab
 * next to side (0 = low, 1 = high) - what the neighbour on that side needs - into buf; echo_halo_unpack scatters buf
 * into the HALO on that side.  fields: HOST array of 8 field indices (echo_stage_halo_fields; -1 = leave that slot
 * of the message alone, so that the cell fields and the face fields of a stage can travel separately); buf: DEVICE;
 * cuda_stream: the stream to run on (NULL = the bound stream).  One kernel per call, no synchronisation. */
size_t echo_halo_doubles(const echo_ctx *ctx, int axis);
int echo_halo_pack(echo_ctx *ctx, const int *fields, int axis, int side, double *buf, void *cuda_stream);
int echo_halo_unpack(echo_ctx *ctx, const int *fields, int axis, int side, const double *buf, void *cuda_stream);

/* Host only (needs the device of the bound workspace for the occupancy query).  The launch configuration in force
 * for this handle, for tests that place samples across tile seams: out (HOST, 8 ints) = {cells per chunk of the
 * x-, y-, z-sweep (an axis longer than 512 cells is cut into chunks; 1 for a one-cell axis), planes per z-chunk of
 * the plane-marching INT+con2prim, UCT and curl+update kernels (0: that kernel is not used by this handle;
 * negative: -(y-tiles per chunk) of the n_z = 1 variants marching along y), tile width, tile height of those
 * kernels}. */
int echo_get_tiling(echo_ctx *ctx, int *out);

/* ---- measurement aids (used by bench.py; not part of the numerical path) -------------------- */

#define ECHO_NKCLASS 8
/* Kernel classes of the per-kernel timers: 0 k_prim (INT+con2prim), 1..3 k_flux<x,y,z> (REC+HLL+DER+
 * divergence), 4 k_uct, 5 k_update (curl+RK), 6 control kernels, 7 everything else. */

/* Host only.  echo_step replays ONE captured step (its 21 kernels as a CUDA graph, captured at the first call on an
 * internal stream and launched into the bound stream), which removes the gaps between dependent launches that cost
 * about a tenth of a step on grids of 32^3-64^3 cells.  enable = 0 makes echo_step launch its kernels one by one
 * (same kernels, same arguments, bit-identical results); 1 (default) restores the replay.  Plain launches are also
 * used while echo_timing is on and for the stage-wise entry points. */
int echo_use_graph(echo_ctx *ctx, int enable);

/* enable != 0: from now on every kernel launch of this handle is bracketed by a CUDA-event pair on
 * the bound stream (no synchronisation, no change to the launch order); also clears the timers and
 * the launch counters.  enable == 0: stops bracketing. */
int echo_timing(echo_ctx *ctx, int enable);

/* Synchronises the stream; ms_total[c] (HOST, ECHO_NKCLASS doubles) = summed device time of class c
 * since echo_timing(ctx, 1), launches[c] (HOST, ECHO_NKCLASS longs) = number of launches (counted
 * whether or not timing is enabled, since the last echo_timing call or echo_bind). */
int echo_get_timing(echo_ctx *ctx, double *ms_total, long *launches);

/* FP64 vector-pipe peak of the current device, measured: `reps` launches of a register-resident
 * kernel of independent DFMA chains (148 x 8 blocks x 256 threads), each timed with CUDA events on
 * `cuda_stream`.  tflops_host[0] = best launch (burst), tflops_host[1] = all launches together
 * (sustained).  Synchronises. */
int echo_fp64_peak(int reps, double *tflops_host, void *cuda_stream);

#ifdef __cplusplus
}
#endif
#endif /* ECHO_B200_H */
