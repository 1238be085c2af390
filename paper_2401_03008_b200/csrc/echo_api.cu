// echo_api.cu — C-ABI layer of libecho_b200 (see include/echo.h): argument checks, workspace
// carving, kernel launches on the bound stream.  No arithmetic of the method lives here.
#include <cuda.h>   // CUtensorMap and its enums only: the encoder is fetched through cudaGetDriverEntryPoint

#include <cmath>
#include <cstddef>
#include <cstdio>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "../../include/echo.h"
#include "echo_kernels.cuh"

using namespace echo;

struct echo_ctx {
    Grid g;
    double gamma, cfl, gg, hmin;
    char *ws = nullptr;
    size_t ws_bytes = 0;
    cudaStream_t stream = nullptr;
    Ctrl *ctrl = nullptr;
    double *part = nullptr;
    double *field[NFIELD] = {nullptr};
    long long npad = 0;
    bool bound = false, has_state = false;
    int rk = 3;              // SSP-RK3 or SSP-RK2 (echo_set_order)
    bool block = false;      // echo_create_block: explicit spacing, halos refreshed by the caller between stages
    int bc[3][2] = {{0, 0}, {0, 0}, {0, 0}};   // physical boundary per (axis, side) of a padded block: 0 none, 1 reflecting, 2 outflow
    bool gate_active = false;   // inside echo_step / echo_stage_*: con2prim failures count only while ctrl->active
    // one full step captured as a CUDA graph (echo_step replays it)
    cudaStream_t cap_stream = nullptr;    // capture target (the legacy default stream cannot be captured)
    cudaGraph_t graph = nullptr;
    cudaGraphExec_t gexec = nullptr;
    bool capturing = false, graph_failed = false;
    long graph_launches[ECHO_NKCLASS] = {0};
    int use_graph = 1;
    UctMaps uct_maps[2];     // TMA descriptors of the fields k_uct3 stages; [1]: staggered B in the stage buffers
    int device = -1;         // device the bound workspace lives on (echo_bind); every launching call runs there
    // launch configuration of the marching kernels (ensure_tiling; reported by echo_get_tiling)
    struct Tiling { bool ready = false; int cz_prim = 0, cz_uct = 0, cz_bupd = 0, cy_uct_flat = 0, cy_bupd_flat = 0; } til;
    std::string err;
    // measurement aids (echo_timing / echo_get_timing)
    bool timing = false;
    long launches[ECHO_NKCLASS] = {0};
    std::vector<cudaEvent_t> ev_pool;
    size_t ev_used = 0;
    struct Span { int cls; size_t e0, e1; };
    std::vector<Span> spans;
    void drop_graph() {
        if (gexec) cudaGraphExecDestroy(gexec);
        if (graph) cudaGraphDestroy(graph);
        gexec = nullptr; graph = nullptr; graph_failed = false;
    }
    ~echo_ctx() {
        for (cudaEvent_t e : ev_pool) cudaEventDestroy(e);
        drop_graph();
        if (cap_stream) cudaStreamDestroy(cap_stream);
    }
};

namespace {

enum { F_U = 0, F_BF = 5, F_U1 = 8, F_BF1 = 13, F_P = 16, F_BC = 21, F_R = 24, F_AP = 29, F_AM = 32, F_VB = 35, F_E = 41 };

int fail(echo_ctx *c, int code, const std::string &msg) {
    if (c) c->err = msg;
    return code;
}
int cuda_fail(echo_ctx *c, cudaError_t e, const char *where) {
    return fail(c, ECHO_ECUDA, std::string(where) + ": " + cudaGetErrorString(e));
}
#define CU(call)                                                   \
    do {                                                           \
        cudaError_t e_ = (call);                                   \
        if (e_ != cudaSuccess) return cuda_fail(ctx, e_, #call);   \
    } while (0)
#define LAUNCH_CHECK(name)                                         \
    do {                                                           \
        cudaError_t e_ = cudaGetLastError();                       \
        if (e_ != cudaSuccess) return cuda_fail(ctx, e_, name);    \
    } while (0)

// flux-sweep tiling: threads per block, transverse width, max tile length
// threads per block of the y/z sweeps and of the x-sweep (x marches 32 / 16 rows per round with 128 / 64 threads: a
// 256-cell row costs 10 rounds of 32 or 18 of 16, i.e. 320 or 288 row slots for its 261 faces: 0.74 -> 0.71 ms)
constexpr int FLUX_NT = 128, FLUX_NT_X = 64, FLUX_CMAX = 512;

// Length CZ of the z-chunks of a plane-marching kernel (k_uct3, k_bupd): tiles x chunks blocks run in waves of
// `slots` resident blocks, and every chunk pays about `fill` planes of pipeline fill (window prologue, first copies).
// Picks the chunk count with the best  (blocks / (waves * slots)) * CZ / (CZ + fill); at 256^3 this is 6 chunks of 43
// planes for the UCT kernel (3072 blocks = 6.9 waves of 444) instead of 3 of 86 (3.5 waves): 1.15 -> 1.08 ms.
int pick_chunk_planes(int tiles, int nz, int slots, int fill) {
    int best_cz = nz;
    double best = -1.0;
    for (int nchunk = 1; nchunk <= std::max(1, nz / 8); ++nchunk) {
        const int cz = (nz + nchunk - 1) / nchunk;
        const long blocks = (long)tiles * ((nz + cz - 1) / cz);
        const long waves = (blocks + slots - 1) / slots;
        const double eff = (double)blocks / (double)(waves * slots) * cz / (double)(cz + fill);
        if (eff > best * 1.0005) { best = eff; best_cz = cz; }
    }
    return best_cz;
}
template <typename K>
int resident_slots(K kernel, int threads, size_t dyn_smem = 0) {
    int per_sm = 0, sms = 0, dev = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (dyn_smem > 48 * 1024) cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)dyn_smem);
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel, threads, dyn_smem);
    return std::max(1, per_sm) * std::max(1, sms);
}
// ---- TMA descriptors (k_uct3).  A field is a 3-D tensor (nx, ny, nz) of doubles, x fastest; a box is {bx, by, 1}.
// Encoding needs 16-byte multiples for the row pitch (n_x even) and for the box rows (bx even).
static_assert(sizeof(TmaDesc) == sizeof(CUtensorMap) && alignof(TmaDesc) >= alignof(CUtensorMap), "TmaDesc mirrors CUtensorMap");
typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                                  const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
EncodeTiledFn encode_tiled_fn() {
    static EncodeTiledFn fn = [] {
        void *p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) != cudaSuccess || q != cudaDriverEntryPointSuccess)
            p = nullptr;
        cudaGetLastError();
        return reinterpret_cast<EncodeTiledFn>(p);
    }();
    return fn;
}
bool encode_box(const Grid &g, double *field, int bx, int by, TmaDesc *out) {
    EncodeTiledFn enc = encode_tiled_fn();
    if (!enc) return false;
    const cuuint64_t dims[3] = {(cuuint64_t)g.n[0], (cuuint64_t)g.n[1], (cuuint64_t)g.n[2]};
    const cuuint64_t strides[2] = {sizeof(double) * (cuuint64_t)g.n[0], sizeof(double) * (cuuint64_t)g.n[0] * g.n[1]};
    const cuuint32_t box[3] = {(cuuint32_t)bx, (cuuint32_t)by, 1u}, estr[3] = {1u, 1u, 1u};
    return enc(reinterpret_cast<CUtensorMap *>(out), CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3, field, dims, strides, box, estr,
               CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE,
               CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}
// maps of stage set `which` (0: staggered B of U^n, 1: of the stage buffers); ok = 0 if the grid has no interior tile
// or cannot be described (odd n_x): k_uct3 then fills every tile by cp.async
void build_uct_maps(echo_ctx *c, int which);

enum { KC_PRIM = 0, KC_FLUX = 1, KC_UCT = 4, KC_UPDATE = 5, KC_CTRL = 6, KC_OTHER = 7 };

// chunk lengths of the plane-marching kernels for this handle's grid on this handle's device (once per handle)
void ensure_tiling(echo_ctx *c) {
    if (c->til.ready) return;
    const Grid &g = c->g;
    const int tx = (g.n[0] + UCT_TX - 1) / UCT_TX, ty = (g.n[1] + UCT_TY - 1) / UCT_TY;
    c->til.cz_prim = pick_chunk_planes(tx * ty, g.n[2], resident_slots(k_prim_march<true>, UCT_NT), 2);
    const int ty3 = (g.n[1] + U3_TY - 1) / U3_TY;
    c->til.cz_uct = pick_chunk_planes(tx * ty3, g.n[2], resident_slots(k_uct3<false, U3_TY>, U3<U3_TY>::NT, U3<U3_TY>::SMEM), 3);
    resident_slots(k_uct3<true, U3_TY>, U3<U3_TY>::NT, U3<U3_TY>::SMEM);   // (opts the linear-REC instantiation into its shared memory too)
    c->til.cz_bupd = pick_chunk_planes(tx * ty, g.n[2], resident_slots(k_bupd, UCT_NT), 2);
    c->til.cy_uct_flat = pick_chunk_planes(tx, ty, resident_slots(k_uct2_flat<false>, UCT_NT), 3);
    c->til.cy_bupd_flat = pick_chunk_planes(tx, ty, resident_slots(k_bupd_flat, UCT_NT), 2);
    c->til.ready = true;
}
// chunk length of the flux sweep along D: one chunk per column unless the axis is long
int flux_chunk_cells(const Grid &g, int D) {
    const int nchunk = (g.n[D] + FLUX_CMAX - 1) / FLUX_CMAX;
    return (g.n[D] + nchunk - 1) / nchunk;
}

size_t next_event(echo_ctx *c) {
    if (c->ev_used == c->ev_pool.size()) {
        cudaEvent_t e;
        cudaEventCreate(&e);
        c->ev_pool.push_back(e);
    }
    cudaEventRecord(c->ev_pool[c->ev_used], c->stream);
    return c->ev_used++;
}
void tbegin(echo_ctx *c, int cls) {
    (c->capturing ? c->graph_launches : c->launches)[cls]++;   // a captured launch runs (and counts) at every replay
    if (c->timing) c->spans.push_back({cls, next_event(c), 0});
}
void tend(echo_ctx *c) {
    if (c->timing) c->spans.back().e1 = next_event(c);
}
// launch of one kernel of class `cls`: counted, optionally bracketed by events, checked
#define KL(cls, name, ...)        \
    do {                          \
        tbegin(ctx, cls);         \
        __VA_ARGS__;              \
        tend(ctx);                \
        LAUNCH_CHECK(name);       \
    } while (0)

dim3 cell_block() { return dim3(64, 4, 1); }
dim3 cell_grid(const Grid &g) { return dim3((g.n[0] + 63) / 64, (g.n[1] + 3) / 4, g.n[2]); }

// which[0] -> fields of the state L is applied to (0 = U^n at F_U, 1 = stage state at F_U1)
Stage make_stage(const echo_ctx *c, int which) {
    Stage st;
    const int u0 = which ? F_U1 : F_U, b0 = which ? F_BF1 : F_BF;
    for (int v = 0; v < 5; ++v) { st.U[v] = c->field[u0 + v]; st.P[v] = c->field[F_P + v]; st.R[v] = c->field[F_R + v]; }
    for (int d = 0; d < 3; ++d) {
        st.Bf[d] = c->field[b0 + d];
        st.Bc[d] = c->field[F_BC + d];
        st.ap[d] = c->field[F_AP + d];
        st.am[d] = c->field[F_AM + d];
        st.vb[d][0] = c->field[F_VB + 2 * d];
        st.vb[d][1] = c->field[F_VB + 2 * d + 1];
        st.E[d] = c->field[F_E + d];
    }
    return st;
}

void build_uct_maps(echo_ctx *c, int which) {
    const Grid &g = c->g;
    UctMaps &m = c->uct_maps[which];
    std::memset(&m, 0, sizeof(m));
    if (g.n[0] % 2 || g.n[0] < 3 * UCT_TX || g.n[1] < 3 * U3_TY || g.n[2] < 2) return;   // no interior tile / unaligned rows
    const Stage st = make_stage(c, which);
    double *xr[4] = {st.vb[1][1], const_cast<double *>(st.Bf[1]), st.vb[2][0], const_cast<double *>(st.Bf[2])};
    double *yr[4] = {st.vb[0][0], const_cast<double *>(st.Bf[0]), st.vb[2][1], const_cast<double *>(st.Bf[2])};
    bool ok = true;
    for (int f = 0; f < 4; ++f) {
        ok = ok && encode_box(g, xr[f], U3_XRP, U3_TY, &m.xr[f]);
        ok = ok && encode_box(g, yr[f], UCT_TX, U3_TY + 5, &m.yr[f]);
    }
    double *sp[3][2] = {{st.ap[0], st.am[0]}, {st.ap[1], st.am[1]}, {st.ap[2], st.am[2]}};
    for (int f = 0; f < 2; ++f) {
        ok = ok && encode_box(g, sp[2][f], U3_AP, U3_TY + 1, &m.az[f]);
        ok = ok && encode_box(g, sp[0][f], UCT_TX, U3_TY + 1, &m.ax[f]);
        ok = ok && encode_box(g, sp[1][f], U3_AP, U3_TY, &m.ay[f]);
    }
    m.ok = ok ? 1 : 0;
}

// fuse: 0 = plain operator (rhs written), 1 = the z-sweep applies the RK combination of the 5 cell fields
template <int D, int MODE, int NT>
int launch_flux_nt(echo_ctx *ctx, const Stage &st, int want_amax, const FluxUpd &fu) {
    constexpr int T = (D == 0) ? 4 : 16;
    constexpr int TD = (D == 0) ? 1 : 0, OD = 3 - D - TD;
    const Grid &g = ctx->g;
    if (g.n[D] == 1) {   // a one-cell axis: no stencil work left, only the face quantities (k_flux_flat)
        if (g.rec == 2 && g.uct)
            KL(KC_FLUX + D, "k_flux_flat", k_flux_flat<D, MODE, true, 2><<<cell_grid(g), cell_block(), 0, ctx->stream>>>(
                   g, st, ctx->gamma, ctx->gg, ctx->ctrl, want_amax, fu));
        else if (g.rec == 2)
            KL(KC_FLUX + D, "k_flux_flat", k_flux_flat<D, MODE, false, 2><<<cell_grid(g), cell_block(), 0, ctx->stream>>>(
                   g, st, ctx->gamma, ctx->gg, ctx->ctrl, want_amax, fu));
        else if (g.uct)
            KL(KC_FLUX + D, "k_flux_flat", k_flux_flat<D, MODE><<<cell_grid(g), cell_block(), 0, ctx->stream>>>(
                   g, st, ctx->gamma, ctx->gg, ctx->ctrl, want_amax, fu));
        else
            KL(KC_FLUX + D, "k_flux_flat", k_flux_flat<D, MODE, false><<<cell_grid(g), cell_block(), 0, ctx->stream>>>(
                   g, st, ctx->gamma, ctx->gg, ctx->ctrl, want_amax, fu));
        return ECHO_OK;
    }
    // chunks along D: one chunk per column unless the axis is long (5 halo faces per chunk are recomputed)
    const int C = flux_chunk_cells(g, D);
    const int nchunk = (g.n[D] + C - 1) / C;
    dim3 grid((g.n[TD] + T - 1) / T, nchunk, g.n[OD]);
    if (!g.uct) {   // UCT = NO: 8 flux components, rings of 49 KB in dynamic shared memory
        constexpr int R = NT / T, RL = 3 * R, SB = RL + 4;   // as in k_flux
        constexpr size_t smem = sizeof(double) * ((D == 0) ? (8 + 8) * T * SB : RL * (8 + 8) * T);
        if (g.rec == 2) {   // linear REC is wired with the second-order INT/DER only (echo_set_order)
            auto kern = k_flux<D, NT, MODE, false, false, 2>;
            CU(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
            KL(KC_FLUX + D, "k_flux_cc", kern<<<grid, NT, smem, ctx->stream>>>(g, st, C, ctx->gamma, ctx->gg, ctx->ctrl, want_amax, fu));
        } else if (g.ho) {
            auto kern = k_flux<D, NT, MODE, true, false>;
            CU(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
            KL(KC_FLUX + D, "k_flux_cc", kern<<<grid, NT, smem, ctx->stream>>>(g, st, C, ctx->gamma, ctx->gg, ctx->ctrl, want_amax, fu));
        } else {
            auto kern = k_flux<D, NT, MODE, false, false>;
            CU(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
            KL(KC_FLUX + D, "k_flux_cc", kern<<<grid, NT, smem, ctx->stream>>>(g, st, C, ctx->gamma, ctx->gg, ctx->ctrl, want_amax, fu));
        }
        return ECHO_OK;
    }
    if (g.rec == 2)
        KL(KC_FLUX + D, "k_flux", k_flux<D, NT, MODE, false, true, 2><<<grid, NT, 0, ctx->stream>>>(g, st, C, ctx->gamma, ctx->gg, ctx->ctrl, want_amax, fu));
    else if (g.ho)
        KL(KC_FLUX + D, "k_flux", k_flux<D, NT, MODE, true><<<grid, NT, 0, ctx->stream>>>(g, st, C, ctx->gamma, ctx->gg, ctx->ctrl, want_amax, fu));
    else
        KL(KC_FLUX + D, "k_flux", k_flux<D, NT, MODE, false><<<grid, NT, 0, ctx->stream>>>(g, st, C, ctx->gamma, ctx->gg, ctx->ctrl, want_amax, fu));
    return ECHO_OK;
}

template <int D, int MODE>
int launch_flux(echo_ctx *ctx, const Stage &st, int want_amax, const FluxUpd &fu) {
    // the x-sweep of the MP5 scheme runs 64-thread blocks; with the cheap linear REC the larger block is the faster one
    if (D == 0 && ctx->g.rec != 2) return launch_flux_nt<D, MODE, (D == 0) ? FLUX_NT_X : FLUX_NT>(ctx, st, want_amax, fu);
    return launch_flux_nt<D, MODE, FLUX_NT>(ctx, st, want_amax, fu);
}

// RK bookkeeping of one stage inside echo_step: which buffers hold what
struct StagePlan {
    bool prim_upd;      // k_prim first forms U1 = U^n + dt*R (the deferred stage-1 update) and stores it
    bool fuse_z;        // the z-sweep applies out = c0*U^n + c1*(cur + dt*rhs) to the 5 cell fields
    int cur, out;       // 0 = U^n buffers, 1 = stage buffers
    double c0, c1;
};

// points 1-3 of a sub-step (INT + con2prim, the three sweeps) on the given stage pointers
int launch_sweeps(echo_ctx *ctx, const Stage &st, int want_amax, const StagePlan *pl = nullptr) {
    const Grid &g = ctx->g;
    PrimUpd pu;
    for (int v = 0; v < 8; ++v) pu.uout[v] = ctx->field[F_U1 + v];
    for (int d = 0; d < 3; ++d) pu.bin[d] = ctx->field[F_BF + d];
    const int *gate = ctx->gate_active ? &ctx->ctrl->active : &ctx->ctrl->one;
    if (!g.uct) {
        if (pl && pl->prim_upd)
            KL(KC_PRIM, "k_prim_cc", k_prim<false, true, false><<<cell_grid(g), cell_block(), 0, ctx->stream>>>(g, st, ctx->gamma, ctx->ctrl, pu, gate));
        else
            KL(KC_PRIM, "k_prim_cc", k_prim<false, false, false><<<cell_grid(g), cell_block(), 0, ctx->stream>>>(g, st, ctx->gamma, ctx->ctrl, pu, gate));
    } else if (g.n[2] < 8) {   // a thin grid (2.5-D runs): nothing to march along, the thread-per-cell kernel is faster
        if (pl && pl->prim_upd)
            KL(KC_PRIM, "k_prim", k_prim<false, true><<<cell_grid(g), cell_block(), 0, ctx->stream>>>(g, st, ctx->gamma, ctx->ctrl, pu, gate));
        else
            KL(KC_PRIM, "k_prim", k_prim<false, false><<<cell_grid(g), cell_block(), 0, ctx->stream>>>(g, st, ctx->gamma, ctx->ctrl, pu, gate));
    } else {   // plane-marching INT + con2prim (k_prim_march), tiles and z-chunks as for k_bupd
        ensure_tiling(ctx);
        const int CZ = ctx->til.cz_prim;
        dim3 grid((g.n[0] + UCT_TX - 1) / UCT_TX, (g.n[1] + UCT_TY - 1) / UCT_TY, (g.n[2] + CZ - 1) / CZ);
        if (pl && pl->prim_upd)
            KL(KC_PRIM, "k_prim_march", k_prim_march<true><<<grid, UCT_NT, 0, ctx->stream>>>(g, st, ctx->gamma, ctx->ctrl, pu, CZ, gate));
        else
            KL(KC_PRIM, "k_prim_march", k_prim_march<false><<<grid, UCT_NT, 0, ctx->stream>>>(g, st, ctx->gamma, ctx->ctrl, pu, CZ, gate));
    }
    FluxUpd fu;
    for (int v = 0; v < 8; ++v) {
        fu.base[v] = ctx->field[F_U + v];
        fu.cur[v] = ctx->field[((pl && pl->cur) ? F_U1 : F_U) + v];
        fu.out[v] = ctx->field[((pl && pl->out) ? F_U1 : F_U) + v];
    }
    fu.c0 = pl ? pl->c0 : 0.0;
    fu.c1 = pl ? pl->c1 : 1.0;
    int rc;
    if ((rc = launch_flux<0, 0>(ctx, st, want_amax, fu))) return rc;
    if ((rc = launch_flux<1, 0>(ctx, st, want_amax, fu))) return rc;
    if (pl && pl->fuse_z) { if ((rc = launch_flux<2, 1>(ctx, st, want_amax, fu))) return rc; }
    else                  { if ((rc = launch_flux<2, 0>(ctx, st, want_amax, fu))) return rc; }
    return ECHO_OK;
}

// k_set_dt (stage 1 only) + point 4 (UCT)
int launch_uct(echo_ctx *ctx, const Stage &st, bool set_dt) {
    const Grid &g = ctx->g;
    if (set_dt) {   // stage 1 of a step: dt must exist before any update (S9)
        KL(KC_CTRL, "k_set_dt", k_set_dt<<<1, 1, 0, ctx->stream>>>(ctx->ctrl, ctx->cfl * ctx->hmin));
    }
    {   // plane-marching UCT: 16 x 8 tiles of (x, y), chunks of planes along z sized by pick_chunk_planes
        if (g.n[2] == 1) {   // 2.5-D: the same kernel marching along y (k_uct2_flat)
            const int tx = (g.n[0] + UCT_TX - 1) / UCT_TX, ty = (g.n[1] + UCT_TY - 1) / UCT_TY;
            ensure_tiling(ctx);
            const int CY = ctx->til.cy_uct_flat;
            dim3 grid(tx, (ty + CY - 1) / CY, 1);
            if (g.rec == 2) KL(KC_UCT, "k_uct2_flat", k_uct2_flat<true><<<grid, UCT_NT, 0, ctx->stream>>>(g, st, CY));
            else KL(KC_UCT, "k_uct2_flat", k_uct2_flat<false><<<grid, UCT_NT, 0, ctx->stream>>>(g, st, CY));
            return ECHO_OK;
        }
        ensure_tiling(ctx);
        const int CZ = ctx->til.cz_uct;
        dim3 grid((g.n[0] + UCT_TX - 1) / UCT_TX, (g.n[1] + UCT_TY - 1) / UCT_TY, (g.n[2] + CZ - 1) / CZ);
        // tiles by TMA where their boxes lie inside the grid, by cp.async along the periodic seams (k_uct3)
        const UctMaps &maps = ctx->uct_maps[st.Bf[0] == ctx->field[F_BF1] ? 1 : 0];
        grid.y = (g.n[1] + U3_TY - 1) / U3_TY;
        if (g.rec == 2) KL(KC_UCT, "k_uct3", k_uct3<true, U3_TY><<<grid, U3<U3_TY>::NT, U3<U3_TY>::SMEM, ctx->stream>>>(g, st, CZ, maps));
        else KL(KC_UCT, "k_uct3", k_uct3<false, U3_TY><<<grid, U3<U3_TY>::NT, U3<U3_TY>::SMEM, ctx->stream>>>(g, st, CZ, maps));
    }
    return ECHO_OK;
}

// points 1-4 of a sub-step on the given stage pointers
int launch_operator(echo_ctx *ctx, const Stage &st, int want_amax, const StagePlan *pl = nullptr) {
    int rc;
    if ((rc = launch_sweeps(ctx, st, want_amax, pl))) return rc;
    if (!ctx->g.uct) {   // UCT = NO: the sweeps already hold the rhs of B; only dt is left (stage 1)
        if (want_amax == 2) KL(KC_CTRL, "k_set_dt", k_set_dt<<<1, 1, 0, ctx->stream>>>(ctx->ctrl, ctx->cfl * ctx->hmin));
        return ECHO_OK;
    }
    return launch_uct(ctx, st, want_amax == 2);
}

// curl + RK combination of the staggered B (and, with_u, of the 5 cell fields as well)
int launch_update(echo_ctx *ctx, const Stage &st, int cur_which, int out_which, double c0, double c1, bool with_u) {
    Update up;
    for (int v = 0; v < 8; ++v) {
        up.base[v] = ctx->field[F_U + v];
        up.cur[v] = ctx->field[(cur_which ? F_U1 : F_U) + v];
        up.out[v] = ctx->field[(out_which ? F_U1 : F_U) + v];
    }
    up.c0 = c0;
    up.c1 = c1;
    const Grid &g = ctx->g;
    if (with_u) {
        KL(KC_UPDATE, "k_update", k_update<true><<<cell_grid(g), cell_block(), 0, ctx->stream>>>(g, st.E[0], st.E[1], st.E[2], st.R[0], st.R[1],
                                                                              st.R[2], st.R[3], st.R[4], up, ctx->ctrl, 1));
    } else if (g.n[2] == 1) {   // 2.5-D: curl + update marching along y (k_bupd_flat)
        const int tx = (g.n[0] + UCT_TX - 1) / UCT_TX, ty = (g.n[1] + UCT_TY - 1) / UCT_TY;
        ensure_tiling(ctx);
        const int CY = ctx->til.cy_bupd_flat;
        dim3 grid(tx, (ty + CY - 1) / CY, 1);
        KL(KC_UPDATE, "k_bupd_flat", k_bupd_flat<<<grid, UCT_NT, 0, ctx->stream>>>(g, st.E[0], st.E[1], st.E[2], up, ctx->ctrl, CY));
    } else {   // staggered B only: plane-marching curl + update
        ensure_tiling(ctx);
        const int CZ = ctx->til.cz_bupd;
        dim3 grid((g.n[0] + UCT_TX - 1) / UCT_TX, (g.n[1] + UCT_TY - 1) / UCT_TY, (g.n[2] + CZ - 1) / CZ);
        KL(KC_UPDATE, "k_bupd", k_bupd<<<grid, UCT_NT, 0, ctx->stream>>>(g, st.E[0], st.E[1], st.E[2], up, ctx->ctrl, CZ));
    }
    return ECHO_OK;
}

// ghost fill of the 8 given workspace fields (slots as in stage_halo_fields; -1 skipped) on every bounded side, axes in
// the order x, y, z (row f4)
int fill_boundaries(echo_ctx *ctx, const int *fields) {
    const Grid &g = ctx->g;
    HaloFields hf;
    for (int v = 0; v < 8; ++v) hf.f[v] = fields[v] < 0 ? nullptr : ctx->field[fields[v]];
    for (int a = 0; a < 3; ++a)
        for (int side = 0; side < 2; ++side) {
            const int kind = ctx->bc[a][side];
            if (!kind) continue;
            const int h = side == 0 ? g.lo[a] : g.n[a] - g.hi[a];
            const long long per_field = (long long)h * (g.N / g.n[a]);
            const int blocks = (int)std::min<long long>((per_field + 255) / 256, 148LL * 16);
            if (kind == 1) KL(KC_OTHER, "k_fill_ghost", k_fill_ghost<1><<<dim3(blocks, 8), 256, 0, ctx->stream>>>(g, hf, a, side, per_field));
            else KL(KC_OTHER, "k_fill_ghost", k_fill_ghost<2><<<dim3(blocks, 8), 256, 0, ctx->stream>>>(g, hf, a, side, per_field));
        }
    return ECHO_OK;
}
// true if no side of the padded block is left to the caller to refresh (plain periodic boxes included)
bool self_contained(const echo_ctx *ctx) {
    const Grid &g = ctx->g;
    for (int a = 0; a < 3; ++a) {
        if (g.lo[a] > 0 && !ctx->bc[a][0]) return false;
        if (g.hi[a] < g.n[a] && !ctx->bc[a][1]) return false;
    }
    return true;
}

// Every launching call runs on the device of the bound workspace, whatever the calling thread's current device is,
// and leaves the caller's current device as it found it.
struct DevGuard {
    int prev = -1;
    bool switched = false;
    explicit DevGuard(const echo_ctx *c) {
        if (c && c->device >= 0 && cudaGetDevice(&prev) == cudaSuccess && prev != c->device)
            switched = cudaSetDevice(c->device) == cudaSuccess;
    }
    ~DevGuard() { if (switched) cudaSetDevice(prev); }
};

struct GateScope {   // echo_step / echo_stage_sweeps: see echo_ctx::gate_active
    echo_ctx *c;
    explicit GateScope(echo_ctx *ctx) : c(ctx) { c->gate_active = true; }
    ~GateScope() { c->gate_active = false; }
};

int check_ready(echo_ctx *ctx, bool need_state) {
    if (!ctx) return ECHO_EINVAL;
    if (!ctx->bound) return fail(ctx, ECHO_ESTATE, "echo_bind has not been called");
    if (need_state && !ctx->has_state) return fail(ctx, ECHO_ESTATE, "echo_set_primitives has not been called");
    return ECHO_OK;
}

}  // namespace

extern "C" {

echo_ctx *echo_create(int nx, int ny, int nz, double gamma, double cfl) {
    if (nx < 1 || ny < 1 || nz < 1 || !(gamma > 1.0) || !(cfl > 0.0) || !std::isfinite(gamma) || !std::isfinite(cfl))
        return nullptr;
    // 32-bit cell indices; grid-dimension limits of the launches (the z-sweep puts y on gridDim.z when nz > 1)
    if ((long long)nx * ny * nz >= (1LL << 31) - 64 || nz > 65535 || ny > 4 * 65535 || (nz > 1 && ny > 65535)) return nullptr;
    echo_ctx *c = new (std::nothrow) echo_ctx();
    if (!c) return nullptr;
    Grid &g = c->g;
    g.n[0] = nx; g.n[1] = ny; g.n[2] = nz;
    g.s[0] = 1; g.s[1] = nx; g.s[2] = nx * ny;
    g.N = (long long)nx * ny * nz;
    for (int d = 0; d < 3; ++d) { g.h[d] = 1.0 / g.n[d]; g.rh[d] = (double)g.n[d]; g.lo[d] = 0; g.hi[d] = g.n[d]; }
    g.ho = 1;
    g.uct = 1;
    g.rec = 5;
    c->gamma = gamma;
    c->cfl = cfl;
    c->gg = gamma / (gamma - 1.0);
    c->hmin = std::fmin(g.h[0], std::fmin(g.h[1], g.h[2]));
    c->npad = (g.N + 31) / 32 * 32;
    return c;
}

void echo_destroy(echo_ctx *ctx) { delete ctx; }

size_t echo_workspace_bytes(const echo_ctx *ctx) {
    if (!ctx) return 0;
    return CTRL_BYTES + PART_BYTES + sizeof(double) * (size_t)ctx->npad * NFIELD;
}

const char *echo_last_error(const echo_ctx *ctx) { return ctx ? ctx->err.c_str() : "null handle"; }

int echo_bind(echo_ctx *ctx, void *dev_workspace, size_t bytes, void *cuda_stream) {
    if (!ctx) return ECHO_EINVAL;
    if (!dev_workspace || bytes < echo_workspace_bytes(ctx) || ((size_t)dev_workspace & 255))
        return fail(ctx, ECHO_ENOMEM, "workspace missing, misaligned or smaller than echo_workspace_bytes");
    cudaPointerAttributes attr;
    if (cudaPointerGetAttributes(&attr, dev_workspace) != cudaSuccess || attr.type != cudaMemoryTypeDevice) {
        cudaGetLastError();
        return fail(ctx, ECHO_EINVAL, "the workspace is not device memory");
    }
    ctx->device = attr.device;
    DevGuard dev_guard_(ctx);
    ctx->til.ready = false;
    ctx->drop_graph();
    ctx->ws = static_cast<char *>(dev_workspace);
    ctx->ws_bytes = bytes;
    ctx->stream = static_cast<cudaStream_t>(cuda_stream);
    ctx->ctrl = reinterpret_cast<Ctrl *>(ctx->ws);
    ctx->part = reinterpret_cast<double *>(ctx->ws + CTRL_BYTES);
    double *f0 = reinterpret_cast<double *>(ctx->ws + CTRL_BYTES + PART_BYTES);
    for (int f = 0; f < NFIELD; ++f) ctx->field[f] = f0 + (size_t)f * ctx->npad;
    build_uct_maps(ctx, 0);
    build_uct_maps(ctx, 1);
    Ctrl h;
    std::memset(&h, 0, sizeof(h));
    h.one = 1;
    CU(cudaMemcpyAsync(ctx->ctrl, &h, sizeof(h), cudaMemcpyHostToDevice, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));   // h is a stack object
    ctx->bound = true;
    ctx->has_state = false;
    return ECHO_OK;
}

int echo_set_primitives(echo_ctx *ctx, const double *rho, const double *vx, const double *vy, const double *vz,
                        const double *p, const double *bxf, const double *byf, const double *bzf) {
    int rc = check_ready(ctx, false);
    if (rc) return rc;
    DevGuard dev_guard_(ctx);
    if (!rho || !vx || !vy || !vz || !p || !bxf || !byf || !bzf) return fail(ctx, ECHO_EINVAL, "null array");
    const Grid &g = ctx->g;
    const double *bf[3] = {bxf, byf, bzf};
    for (int d = 0; d < 3; ++d)
        if (bf[d] != ctx->field[F_BF + d])
            CU(cudaMemcpyAsync(ctx->field[F_BF + d], bf[d], sizeof(double) * g.N, cudaMemcpyDeviceToDevice, ctx->stream));
    const int fB[8] = {-1, -1, -1, -1, -1, F_BF, F_BF + 1, F_BF + 2}, fU[8] = {F_U, F_U + 1, F_U + 2, F_U + 3, F_U + 4, -1, -1, -1};
    if (ctx->block && (rc = fill_boundaries(ctx, fB))) return rc;   // bounded block: ghost faces before INT reads them
    KL(KC_OTHER, "k_init", k_init<<<cell_grid(g), cell_block(), 0, ctx->stream>>>(g, rho, vx, vy, vz, p, ctx->field[F_BF], ctx->field[F_BF + 1],
                                                           ctx->field[F_BF + 2], ctx->field[F_U], ctx->field[F_U + 1],
                                                           ctx->field[F_U + 2], ctx->field[F_U + 3], ctx->field[F_U + 4],
                                                           ctx->gg));
    if (ctx->block && (rc = fill_boundaries(ctx, fU))) return rc;   // ... and the ghost cells of the conserved fields
    // the stage buffers are read (never trusted) by the passes of a step enqueued past t_end: give them defined contents
    CU(cudaMemsetAsync(ctx->field[F_U1], 0, sizeof(double) * (size_t)ctx->npad * 8, ctx->stream));
    Ctrl h;
    std::memset(&h, 0, sizeof(h));
    h.one = 1;
    // pageable source: the runtime stages the copy before returning, so the stack object is safe
    CU(cudaMemcpyAsync(ctx->ctrl, &h, sizeof(h), cudaMemcpyHostToDevice, ctx->stream));
    ctx->has_state = true;
    return ECHO_OK;
}

int echo_set_primitives_host(echo_ctx *ctx, const double *rho, const double *vx, const double *vy, const double *vz,
                             const double *p, const double *bxf, const double *byf, const double *bzf) {
    int rc = check_ready(ctx, false);
    if (rc) return rc;
    DevGuard dev_guard_(ctx);
    if (!rho || !vx || !vy || !vz || !p || !bxf || !byf || !bzf) return fail(ctx, ECHO_EINVAL, "null array");
    const size_t nb = sizeof(double) * ctx->g.N;
    const double *src[8] = {rho, vx, vy, vz, p, bxf, byf, bzf};
    double *dst[8];
    for (int v = 0; v < 5; ++v) dst[v] = ctx->field[F_P + v];       // scratch: the primitive fields
    for (int d = 0; d < 3; ++d) dst[5 + d] = ctx->field[F_BF + d];  // faces go straight into the state
    for (int v = 0; v < 8; ++v) CU(cudaMemcpyAsync(dst[v], src[v], nb, cudaMemcpyHostToDevice, ctx->stream));
    return echo_set_primitives(ctx, dst[0], dst[1], dst[2], dst[3], dst[4], dst[5], dst[6], dst[7]);
}

int echo_faces_from_potential(echo_ctx *ctx, const double *ax, const double *ay, const double *az, double b0x,
                              double b0y, double b0z, double *bxf, double *byf, double *bzf) {
    int rc = check_ready(ctx, false);
    if (rc) return rc;
    DevGuard dev_guard_(ctx);
    if (!ax || !ay || !az || !bxf || !byf || !bzf) return fail(ctx, ECHO_EINVAL, "null array");
    const Grid &g = ctx->g;
    KL(KC_OTHER, "k_curl", k_curl<<<cell_grid(g), cell_block(), 0, ctx->stream>>>(g, ax, ay, az, bxf, byf, bzf, -1.0, b0x, b0y, b0z));
    return ECHO_OK;
}

// The UCT = YES step as six halves: stage_sweeps(s) = points 1-3 of sub-step s, stage_finish(s) = point 4
// + the staggered part of point 5.  echo_step runs them back to back; a domain-decomposed run
// (echo_stage_sweeps / echo_stage_finish) runs the SAME halves with a halo refresh after each finish, so the two
// execute the same kernels with the same arguments.  rk2: SSP-RK2 (O3b) ends after stage 2 with weights 1/2, 1/2.
//   stage 1: L(U^n), dt from its speeds (S9); B1 = B^n + dt rhs_B now, U1 = U^n + dt rhs_U DEFERRED into the k_prim of
//            stage 2 (st.U = U^n, st.R = rhs, result stored to the stage buffers) - so what the next stage needs
//            from the neighbours after stage 1 is the rhs of the cell fields and B1 (stage_halo_fields)
//   stage 2: U2 = 3/4 U^n + 1/4 (U1 + dt L(U1)); the cell fields are combined inside the z-sweep
//   stage 3: U^{n+1} = 1/3 U^n + 2/3 (U2 + dt L(U2))
static int stage_sweeps_impl(echo_ctx *ctx, int stage) {
    const Stage s0 = make_stage(ctx, 0), s1 = make_stage(ctx, 1);
    const bool rk2 = ctx->rk == 2;
    if (stage == 1) {
        KL(KC_CTRL, "k_begin_step", k_begin_step<<<1, 1, 0, ctx->stream>>>(ctx->ctrl));
        return launch_sweeps(ctx, s0, 2);
    }
    if (stage == 2) {
        Stage s12 = s1;                                   // operator state: faces from the stage buffers ...
        for (int v = 0; v < 5; ++v) s12.U[v] = s0.U[v];   // ... cell fields = U^n (+ dt R inside k_prim)
        const StagePlan pl = {true, true, 1, rk2 ? 0 : 1, rk2 ? 0.5 : 0.75, rk2 ? 0.5 : 0.25};
        return launch_sweeps(ctx, s12, 0, &pl);
    }
    const StagePlan pl = {false, true, 1, 0, 1.0 / 3.0, 2.0 / 3.0};
    return launch_sweeps(ctx, s1, 0, &pl);
}
static int stage_finish_impl(echo_ctx *ctx, int stage) {
    int rc;
    const Stage s0 = make_stage(ctx, 0), s1 = make_stage(ctx, 1);
    const bool rk2 = ctx->rk == 2;
    if (stage == 1) {
        if ((rc = launch_uct(ctx, s0, true))) return rc;
        return launch_update(ctx, s0, 0, 1, 0.0, 1.0, false);
    }
    if ((rc = launch_uct(ctx, s1, false))) return rc;
    if (stage == 2) rc = launch_update(ctx, s1, 1, rk2 ? 0 : 1, rk2 ? 0.5 : 0.75, rk2 ? 0.5 : 0.25, false);
    else rc = launch_update(ctx, s1, 1, 0, 1.0 / 3.0, 2.0 / 3.0, false);
    if (rc) return rc;
    if (stage == ctx->rk) KL(KC_CTRL, "k_end_step", k_end_step<<<1, 1, 0, ctx->stream>>>(ctx->ctrl));
    return ECHO_OK;
}
// the fields whose halos the next half needs from the neighbouring blocks after stage `stage` (8 field indices)
static void stage_halo_fields(const echo_ctx *ctx, int stage, int *f) {
    const bool last = stage == ctx->rk;
    for (int v = 0; v < 5; ++v) f[v] = (stage == 1 ? F_R : last ? F_U : F_U1) + v;
    for (int d = 0; d < 3; ++d) f[5 + d] = (last ? F_BF : F_BF1) + d;
}

// the launches of one full step (t_end comes from the control block)
static int enqueue_step(echo_ctx *ctx) {
    int rc;
    if (!ctx->g.uct) {
        // UCT = NO: all 8 fields are cell fields.  Stage 1 writes rhs only; its update is formed by the
        // k_prim of stage 2 (U and B); stages 2 and 3 combine all 8 fields inside their z-sweep.  10 launches.
        const Stage s0 = make_stage(ctx, 0), s1 = make_stage(ctx, 1);
        const bool rk2 = ctx->rk == 2;
        KL(KC_CTRL, "k_begin_step", k_begin_step<<<1, 1, 0, ctx->stream>>>(ctx->ctrl));
        if ((rc = launch_operator(ctx, s0, 2))) return rc;
        Stage s12 = s1;
        for (int v = 0; v < 5; ++v) s12.U[v] = s0.U[v];
        const StagePlan p2 = {true, true, 1, rk2 ? 0 : 1, rk2 ? 0.5 : 0.75, rk2 ? 0.5 : 0.25};
        if ((rc = launch_operator(ctx, s12, 0, &p2))) return rc;
        if (!rk2) {
            const StagePlan p3 = {false, true, 1, 0, 1.0 / 3.0, 2.0 / 3.0};
            if ((rc = launch_operator(ctx, s1, 0, &p3))) return rc;
        }
        KL(KC_CTRL, "k_end_step", k_end_step<<<1, 1, 0, ctx->stream>>>(ctx->ctrl));
        return ECHO_OK;
    }
    for (int stage = 1; stage <= ctx->rk; ++stage) {
        if ((rc = stage_sweeps_impl(ctx, stage))) return rc;
        if ((rc = stage_finish_impl(ctx, stage))) return rc;
        if (ctx->block) {   // a bounded block: refill the ghost layers of what the next half reads (row f4)
            int f[8];
            stage_halo_fields(ctx, stage, f);
            if ((rc = fill_boundaries(ctx, f))) return rc;
        }
    }
    return ECHO_OK;
}

// Captures enqueue_step once (on an internal stream: the legacy default stream PyTorch hands over cannot be captured)
// and instantiates it; the executable graph is then launched into the bound stream.  Any failure falls back to plain
// launches for the rest of the handle's life (graph_failed).
static bool ensure_graph(echo_ctx *ctx) {
    if (ctx->gexec) return true;
    if (ctx->graph_failed) return false;
    ensure_tiling(ctx);                      // occupancy queries and attribute calls happen before the capture
    if (!ctx->cap_stream && cudaStreamCreateWithFlags(&ctx->cap_stream, cudaStreamNonBlocking) != cudaSuccess) {
        cudaGetLastError();
        ctx->graph_failed = true;
        return false;
    }
    cudaStream_t user = ctx->stream;
    for (int c = 0; c < ECHO_NKCLASS; ++c) ctx->graph_launches[c] = 0;
    bool ok = cudaStreamBeginCapture(ctx->cap_stream, cudaStreamCaptureModeThreadLocal) == cudaSuccess;
    if (ok) {
        ctx->stream = ctx->cap_stream;
        ctx->capturing = true;
        const int rc = enqueue_step(ctx);
        ctx->capturing = false;
        ctx->stream = user;
        ok = cudaStreamEndCapture(ctx->cap_stream, &ctx->graph) == cudaSuccess && rc == ECHO_OK && ctx->graph;
    }
    ok = ok && cudaGraphInstantiate(&ctx->gexec, ctx->graph, 0) == cudaSuccess;
    if (!ok) {
        cudaGetLastError();
        ctx->drop_graph();
        ctx->graph_failed = true;
    }
    return ok;
}

int echo_step(echo_ctx *ctx, int nsteps, double t_end) {
    int rc = check_ready(ctx, true);
    if (rc) return rc;
    DevGuard dev_guard_(ctx);
    if (nsteps < 0 || std::isnan(t_end)) return fail(ctx, ECHO_EINVAL, "nsteps < 0 or t_end is NaN");
    if (ctx->block && !self_contained(ctx))
        return fail(ctx, ECHO_EINVAL, "a block with halos is stepped stage by stage (echo_stage_sweeps / echo_stage_finish) by its owner, "
                                      "unless every padded side has a physical boundary (echo_set_boundaries)");
    if (ctx->block && !ctx->g.uct && (ctx->g.lo[0] || ctx->g.lo[1] || ctx->g.lo[2]))
        return fail(ctx, ECHO_EINVAL, "padded blocks are built for UCT=YES only");
    GateScope gate_scope_(ctx);
    if (nsteps == 0) return ECHO_OK;
    KL(KC_CTRL, "k_set_t_end", k_set_t_end<<<1, 1, 0, ctx->stream>>>(ctx->ctrl, t_end));
    // one captured step replayed nsteps times (no launch gaps between its 21 kernels); plain launches while the
    // per-kernel timers are on (their event records do not belong in a graph) or if capture is unavailable
    if (ctx->use_graph && !ctx->timing && ensure_graph(ctx)) {
        for (int n = 0; n < nsteps; ++n) {
            CU(cudaGraphLaunch(ctx->gexec, ctx->stream));
            for (int c = 0; c < ECHO_NKCLASS; ++c) ctx->launches[c] += ctx->graph_launches[c];
        }
        return ECHO_OK;
    }
    for (int n = 0; n < nsteps; ++n)
        if ((rc = enqueue_step(ctx))) return rc;
    return ECHO_OK;
}

int echo_run_until(echo_ctx *ctx, double t_end, long max_steps, long *steps_taken_host) {
    int rc = check_ready(ctx, true);
    if (rc) return rc;
    DevGuard dev_guard_(ctx);
    if (std::isnan(t_end) || max_steps < 0) return fail(ctx, ECHO_EINVAL, "t_end is NaN or max_steps < 0");
    if (ctx->block && !self_contained(ctx)) return fail(ctx, ECHO_EINVAL, "block handles are stepped stage by stage by their owner");
    Ctrl h;
    CU(cudaMemcpyAsync(&h, ctx->ctrl, sizeof(h), cudaMemcpyDeviceToHost, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));
    const long long steps0 = h.steps;
    const unsigned long long fails0 = h.c2p_fail_total;
    while (h.t < t_end && h.steps - steps0 < max_steps && h.c2p_fail_total == fails0) {
        // echo_step enqueues exactly the steps it is given (those past t_end are device-side no-ops that still
        // cost their kernels), so the count comes from the current speed: a little more than needed, then look
        long k = 8;
        if (h.amax > 0.0 && std::isfinite(t_end)) {
            const double est = (t_end - h.t) / (ctx->cfl * ctx->hmin / h.amax) * 1.02 + 1.0;
            k = est < 2048.0 ? (long)std::ceil(est) : 2048;
        } else if (h.amax > 0.0) {
            k = 2048;
        }
        k = std::max(1L, std::min(k, max_steps - (long)(h.steps - steps0)));
        if ((rc = echo_step(ctx, (int)k, t_end))) return rc;
        CU(cudaMemcpyAsync(&h, ctx->ctrl, sizeof(h), cudaMemcpyDeviceToHost, ctx->stream));
        CU(cudaStreamSynchronize(ctx->stream));
    }
    if (steps_taken_host) *steps_taken_host = (long)(h.steps - steps0);
    return h.c2p_fail_total == fails0 ? ECHO_OK : ECHO_EC2P;
}

int echo_get_primitives(echo_ctx *ctx, double *rho, double *vx, double *vy, double *vz, double *p, double *bxc,
                        double *byc, double *bzc, double *bxf, double *byf, double *bzf) {
    int rc = check_ready(ctx, true);
    if (rc) return rc;
    DevGuard dev_guard_(ctx);
    if (!rho || !vx || !vy || !vz || !p || !bxc || !byc || !bzc) return fail(ctx, ECHO_EINVAL, "null array");
    const Grid &g = ctx->g;
    Stage st = make_stage(ctx, 0);
    double *out[8] = {rho, vx, vy, vz, p, bxc, byc, bzc};
    for (int v = 0; v < 5; ++v) st.P[v] = out[v];
    for (int d = 0; d < 3; ++d) st.Bc[d] = out[5 + d];
    if (g.uct) KL(KC_PRIM, "k_prim", k_prim<true, false><<<cell_grid(g), cell_block(), 0, ctx->stream>>>(g, st, ctx->gamma, ctx->ctrl, PrimUpd(), &ctx->ctrl->one));
    else KL(KC_PRIM, "k_prim_cc", k_prim<true, false, false><<<cell_grid(g), cell_block(), 0, ctx->stream>>>(g, st, ctx->gamma, ctx->ctrl, PrimUpd(), &ctx->ctrl->one));
    double *bf[3] = {bxf, byf, bzf};
    for (int d = 0; d < 3; ++d)
        if (bf[d]) CU(cudaMemcpyAsync(bf[d], ctx->field[F_BF + d], sizeof(double) * g.N, cudaMemcpyDeviceToDevice, ctx->stream));
    return ECHO_OK;
}

static int get_primitives_host_impl(echo_ctx *ctx, double *rho, double *vx, double *vy, double *vz, double *p,
                                    double *bxc, double *byc, double *bzc, double *bxf, double *byf, double *bzf,
                                    bool sync) {
    int rc = check_ready(ctx, true);
    if (rc) return rc;
    DevGuard dev_guard_(ctx);
    if (!rho || !vx || !vy || !vz || !p || !bxc || !byc || !bzc) return fail(ctx, ECHO_EINVAL, "null array");
    const Grid &g = ctx->g;
    const size_t nb = sizeof(double) * g.N;
    Stage st = make_stage(ctx, 0);
    if (g.uct) KL(KC_PRIM, "k_prim", k_prim<true, false><<<cell_grid(g), cell_block(), 0, ctx->stream>>>(g, st, ctx->gamma, ctx->ctrl, PrimUpd(), &ctx->ctrl->one));
    else KL(KC_PRIM, "k_prim_cc", k_prim<true, false, false><<<cell_grid(g), cell_block(), 0, ctx->stream>>>(g, st, ctx->gamma, ctx->ctrl, PrimUpd(), &ctx->ctrl->one));
    double *out[8] = {rho, vx, vy, vz, p, bxc, byc, bzc};
    for (int v = 0; v < 8; ++v) CU(cudaMemcpyAsync(out[v], ctx->field[F_P + v], nb, cudaMemcpyDeviceToHost, ctx->stream));
    double *bf[3] = {bxf, byf, bzf};
    for (int d = 0; d < 3; ++d)
        if (bf[d]) CU(cudaMemcpyAsync(bf[d], ctx->field[F_BF + d], nb, cudaMemcpyDeviceToHost, ctx->stream));
    if (sync) CU(cudaStreamSynchronize(ctx->stream));
    return ECHO_OK;
}

int echo_get_primitives_host(echo_ctx *ctx, double *rho, double *vx, double *vy, double *vz, double *p, double *bxc,
                             double *byc, double *bzc, double *bxf, double *byf, double *bzf) {
    return get_primitives_host_impl(ctx, rho, vx, vy, vz, p, bxc, byc, bzc, bxf, byf, bzf, true);
}

int echo_get_primitives_host_async(echo_ctx *ctx, double *rho, double *vx, double *vy, double *vz, double *p,
                                   double *bxc, double *byc, double *bzc, double *bxf, double *byf, double *bzf) {
    return get_primitives_host_impl(ctx, rho, vx, vy, vz, p, bxc, byc, bzc, bxf, byf, bzf, false);
}

int echo_synchronize(echo_ctx *ctx) {
    int rc = check_ready(ctx, false);
    if (rc) return rc;
    DevGuard dev_guard_(ctx);
    CU(cudaStreamSynchronize(ctx->stream));
    return ECHO_OK;
}

int echo_get_conserved(echo_ctx *ctx, double *D, double *Sx, double *Sy, double *Sz, double *U) {
    int rc = check_ready(ctx, true);
    if (rc) return rc;
    DevGuard dev_guard_(ctx);
    double *out[5] = {D, Sx, Sy, Sz, U};
    for (int v = 0; v < 5; ++v) {
        if (!out[v]) return fail(ctx, ECHO_EINVAL, "null array");
        CU(cudaMemcpyAsync(out[v], ctx->field[F_U + v], sizeof(double) * ctx->g.N, cudaMemcpyDeviceToDevice, ctx->stream));
    }
    return ECHO_OK;
}

int echo_rhs(echo_ctx *ctx, double *const *rhsU, double *const *rhsB, double *const *E, double *amax_host) {
    int rc = check_ready(ctx, true);
    if (rc) return rc;
    DevGuard dev_guard_(ctx);
    const Grid &g = ctx->g;
    const size_t nb = sizeof(double) * g.N;
    const Stage st = make_stage(ctx, 0);
    CU(cudaMemsetAsync(&ctx->ctrl->amax_bits, 0, sizeof(unsigned long long), ctx->stream));
    if ((rc = launch_operator(ctx, st, 1))) return rc;
    if (rhsU)
        for (int v = 0; v < 5; ++v) CU(cudaMemcpyAsync(rhsU[v], st.R[v], nb, cudaMemcpyDeviceToDevice, ctx->stream));
    if (E && !g.uct)
        for (int d = 0; d < 3; ++d) CU(cudaMemsetAsync(E[d], 0, nb, ctx->stream));
    else if (E)
        for (int d = 0; d < 3; ++d) CU(cudaMemcpyAsync(E[d], st.E[d], nb, cudaMemcpyDeviceToDevice, ctx->stream));
    if (rhsB && !g.uct) {   // UCT = NO: the sweeps left the rhs of the cell-centred B in the E fields; no EMFs
        for (int d = 0; d < 3; ++d) CU(cudaMemcpyAsync(rhsB[d], st.E[d], nb, cudaMemcpyDeviceToDevice, ctx->stream));
    } else if (rhsB) {
        KL(KC_OTHER, "k_curl", k_curl<<<cell_grid(g), cell_block(), 0, ctx->stream>>>(g, st.E[0], st.E[1], st.E[2], rhsB[0], rhsB[1], rhsB[2],
                                                               1.0, 0.0, 0.0, 0.0));
    }
    if (amax_host) {
        unsigned long long bits = 0;
        CU(cudaMemcpyAsync(&bits, &ctx->ctrl->amax_bits, sizeof(bits), cudaMemcpyDeviceToHost, ctx->stream));
        CU(cudaStreamSynchronize(ctx->stream));
        std::memcpy(amax_host, &bits, sizeof(double));
    }
    return ECHO_OK;
}

int echo_con2prim(double gamma, long n, const double *D, const double *Sx, const double *Sy, const double *Sz,
                  const double *U, const double *Bx, const double *By, const double *Bz, double *rho, double *vx,
                  double *vy, double *vz, double *p, int *iters, void *cuda_stream) {
    if (n < 0 || !(gamma > 1.0)) return ECHO_EINVAL;
    if (n == 0) return ECHO_OK;
    if (!D || !Sx || !Sy || !Sz || !U || !Bx || !By || !Bz || !rho || !vx || !vy || !vz || !p) return ECHO_EINVAL;
    const int blocks = (int)std::min<long long>((n + 255) / 256, 148LL * 16);
    k_c2p_batch<<<blocks, 256, 0, static_cast<cudaStream_t>(cuda_stream)>>>(gamma, n, D, Sx, Sy, Sz, U, Bx, By, Bz, rho,
                                                                          vx, vy, vz, p, iters);
    return cudaGetLastError() == cudaSuccess ? ECHO_OK : ECHO_ECUDA;
}

int echo_prim2cons(double gamma, long n, const double *rho, const double *vx, const double *vy, const double *vz,
                   const double *p, const double *Bx, const double *By, const double *Bz, double *D, double *Sx,
                   double *Sy, double *Sz, double *U, void *cuda_stream) {
    if (n < 0 || !(gamma > 1.0)) return ECHO_EINVAL;
    if (n == 0) return ECHO_OK;
    if (!D || !Sx || !Sy || !Sz || !U || !Bx || !By || !Bz || !rho || !vx || !vy || !vz || !p) return ECHO_EINVAL;
    const int blocks = (int)std::min<long long>((n + 255) / 256, 148LL * 16);
    k_p2c_batch<<<blocks, 256, 0, static_cast<cudaStream_t>(cuda_stream)>>>(gamma / (gamma - 1.0), n, rho, vx, vy, vz, p,
                                                                          Bx, By, Bz, D, Sx, Sy, Sz, U);
    return cudaGetLastError() == cudaSuccess ? ECHO_OK : ECHO_ECUDA;
}

int echo_div_b(echo_ctx *ctx, double *div_field, double *max_abs_host) {
    int rc = check_ready(ctx, true);
    if (rc) return rc;
    DevGuard dev_guard_(ctx);
    const Grid &g = ctx->g;
    double *slot = ctx->part + 15 * NPART;   // spare partial row: one double for the max
    CU(cudaMemsetAsync(slot, 0, sizeof(double), ctx->stream));
    KL(KC_OTHER, "k_divb", k_divb<<<cell_grid(g), cell_block(), 0, ctx->stream>>>(g, ctx->field[F_BF], ctx->field[F_BF + 1],
                                                                                  ctx->field[F_BF + 2], div_field, slot));
    double m = 0.0;
    CU(cudaMemcpyAsync(&m, slot, sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));
    if (max_abs_host) *max_abs_host = m;
    return ECHO_OK;
}

int echo_diagnostics(echo_ctx *ctx, double *out) {
    int rc = check_ready(ctx, true);
    if (rc) return rc;
    DevGuard dev_guard_(ctx);
    if (!out) return fail(ctx, ECHO_EINVAL, "null output");
    const Grid &g = ctx->g;
    for (int m = 0; m < ECHO_NDIAG; ++m) out[m] = 0.0;
    double *f = ctx->field[F_U];
    const long long np = ctx->npad;
    KL(KC_OTHER, "k_sums", k_sums<<<NPART, 256, 0, ctx->stream>>>(g, f, f + np, f + 2 * np, f + 3 * np, f + 4 * np, f + 5 * np, f + 6 * np,
                                           f + 7 * np, ctx->part));
    Stage st = make_stage(ctx, 0);
    KL(KC_CTRL, "k_c2p_stats_reset", k_c2p_stats_reset<<<1, 1, 0, ctx->stream>>>(ctx->ctrl));
    if (g.uct) KL(KC_PRIM, "k_prim", k_prim<true, false><<<cell_grid(g), cell_block(), 0, ctx->stream>>>(g, st, ctx->gamma, ctx->ctrl, PrimUpd(), &ctx->ctrl->one));
    else KL(KC_PRIM, "k_prim_cc", k_prim<true, false, false><<<cell_grid(g), cell_block(), 0, ctx->stream>>>(g, st, ctx->gamma, ctx->ctrl, PrimUpd(), &ctx->ctrl->one));
    KL(KC_OTHER, "k_extrema", k_extrema<<<NPART, 256, 0, ctx->stream>>>(g.N, st.P[0], st.P[1], st.P[2], st.P[3], st.P[4], ctx->part));
    double dmax = 0.0;
    if ((rc = echo_div_b(ctx, nullptr, &dmax))) return rc;   // synchronises
    std::vector<double> part((size_t)NPART * 11);
    Ctrl h;
    CU(cudaMemcpy(part.data(), ctx->part, sizeof(double) * part.size(), cudaMemcpyDeviceToHost));
    CU(cudaMemcpy(&h, ctx->ctrl, sizeof(h), cudaMemcpyDeviceToHost));
    const double vol = g.h[0] * g.h[1] * g.h[2];
    out[0] = h.t; out[1] = h.dt_last; out[2] = (double)h.steps; out[3] = h.amax;
    for (int v = 0; v < 8; ++v) {
        long double s = 0.0L;
        for (int b = 0; b < NPART; ++b) s += part[(size_t)v * NPART + b];
        out[4 + v] = (double)(s * vol);
    }
    out[12] = dmax;
    double v2m = 0.0, rmin = INFINITY, pmin = INFINITY;
    for (int b = 0; b < NPART; ++b) {
        if ((long long)b * ((g.N + NPART - 1) / NPART) >= g.N) break;   // empty chunks hold no data
        v2m = std::fmax(v2m, part[8 * (size_t)NPART + b]);
        rmin = std::fmin(rmin, part[9 * (size_t)NPART + b]);
        pmin = std::fmin(pmin, part[10 * (size_t)NPART + b]);
    }
    out[13] = 1.0 / std::sqrt(1.0 - v2m);
    out[14] = rmin;
    out[15] = pmin;
    out[16] = (double)h.c2p_maxit;
    out[17] = h.c2p_calls ? (double)h.c2p_sumit / (double)h.c2p_calls : 0.0;
    out[18] = (double)h.c2p_fail_total;
    return h.c2p_fail_total ? fail(ctx, ECHO_EC2P, "con2prim failed in at least one cell") : ECHO_OK;
}

// ---- domain-decomposition blocks
echo_ctx *echo_create_block(int nx, int ny, int nz, double gamma, double cfl, int gnx, int gny, int gnz, int halo_x,
                            int halo_y, int halo_z) {
    const int n[3] = {nx, ny, nz}, gn[3] = {gnx, gny, gnz}, hl[3] = {halo_x, halo_y, halo_z};
    for (int d = 0; d < 3; ++d)
        if (gn[d] < 1 || hl[d] < 0 || n[d] - 2 * hl[d] < 1 || (hl[d] > 0 && n[d] - 2 * hl[d] < hl[d])) return nullptr;
    echo_ctx *c = echo_create(nx, ny, nz, gamma, cfl);
    if (!c) return nullptr;
    Grid &g = c->g;
    for (int d = 0; d < 3; ++d) {
        g.h[d] = 1.0 / gn[d];           // the spacing of the GLOBAL unit box, same arithmetic as echo_create
        g.rh[d] = (double)gn[d];
        g.lo[d] = hl[d];
        g.hi[d] = n[d] - hl[d];
    }
    c->hmin = std::fmin(g.h[0], std::fmin(g.h[1], g.h[2]));
    c->block = true;
    return c;
}

int echo_set_order(echo_ctx *ctx, int rec, int rk) {
    if (!ctx) return ECHO_EINVAL;
    if (ctx->has_state) return fail(ctx, ECHO_ESTATE, "echo_set_order must precede echo_set_primitives");
    if ((rec != 5 && rec != 2) || (rk != 3 && rk != 2)) return fail(ctx, ECHO_EINVAL, "rec must be 5 or 2, rk 3 or 2");
    if (rec == 2 && ctx->g.ho)
        return fail(ctx, ECHO_EINVAL, "linear reconstruction is built with the second-order INT/DER: echo_set_scheme(ctx, uct, 0) first");
    ctx->g.rec = rec;
    ctx->rk = rk;
    return ECHO_OK;
}

int echo_set_scheme(echo_ctx *ctx, int uct, int ho) {
    if (!ctx) return ECHO_EINVAL;
    if (ctx->has_state) return fail(ctx, ECHO_ESTATE, "echo_set_scheme must precede echo_set_primitives");
    if (ho && ctx->g.rec == 2) return fail(ctx, ECHO_EINVAL, "HO=YES with linear reconstruction is not built (echo_set_order)");
    if (!uct && ctx->block) return fail(ctx, ECHO_EINVAL, "UCT=NO is not built for block handles (echo_create_block)");
    ctx->g.uct = uct ? 1 : 0;
    ctx->g.ho = ho ? 1 : 0;
    return ECHO_OK;
}

size_t echo_field_offset(const echo_ctx *ctx, int field) {
    if (!ctx || field < 0 || field >= NFIELD) return 0;
    return CTRL_BYTES + PART_BYTES + sizeof(double) * (size_t)ctx->npad * field;
}

size_t echo_ctrl_offset(int what) {
    switch (what) {
        case 0: return offsetof(Ctrl, amax_bits);
        case 1: return offsetof(Ctrl, t);
        case 2: return offsetof(Ctrl, dt);
        case 3: return offsetof(Ctrl, c2p_fail_total);
        default: return (size_t)-1;
    }
}

int echo_stage_sweeps(echo_ctx *ctx, int stage, double t_end) {
    int rc = check_ready(ctx, true);
    if (rc) return rc;
    DevGuard dev_guard_(ctx);
    if (!ctx->g.uct) return fail(ctx, ECHO_EINVAL, "the stage-wise entry points are built for UCT=YES only");
    if (stage < 1 || stage > ctx->rk) return fail(ctx, ECHO_EINVAL, "stage must be 1 .. number of RK stages");
    GateScope gate_scope_(ctx);
    if (stage == 1) KL(KC_CTRL, "k_set_t_end", k_set_t_end<<<1, 1, 0, ctx->stream>>>(ctx->ctrl, t_end));
    return stage_sweeps_impl(ctx, stage);
}

int echo_stage_finish(echo_ctx *ctx, int stage) {
    int rc = check_ready(ctx, true);
    if (rc) return rc;
    DevGuard dev_guard_(ctx);
    if (!ctx->g.uct) return fail(ctx, ECHO_EINVAL, "the stage-wise entry points are built for UCT=YES only");
    if (stage < 1 || stage > ctx->rk) return fail(ctx, ECHO_EINVAL, "stage must be 1 .. number of RK stages");
    GateScope gate_scope_(ctx);
    return stage_finish_impl(ctx, stage);
}

int echo_set_boundaries(echo_ctx *ctx, const int *kinds) {
    if (!ctx) return ECHO_EINVAL;
    if (!kinds) return fail(ctx, ECHO_EINVAL, "null argument");
    if (ctx->has_state) return fail(ctx, ECHO_ESTATE, "echo_set_boundaries must precede echo_set_primitives");
    const Grid &g = ctx->g;
    for (int a = 0; a < 3; ++a)
        for (int side = 0; side < 2; ++side) {
            const int k = kinds[2 * a + side], h = side == 0 ? g.lo[a] : g.n[a] - g.hi[a];
            if (k < 0 || k > 2) return fail(ctx, ECHO_EINVAL, "boundary kind must be 0 (none), 1 (reflecting) or 2 (outflow)");
            if (k && h < 8) return fail(ctx, ECHO_EINVAL, "a physical boundary needs 8 ghost layers on that axis (echo_create_block with halo 8)");
            if (k && !g.uct) return fail(ctx, ECHO_EINVAL, "physical boundaries are built for UCT=YES only");
        }
    for (int a = 0; a < 3; ++a) { ctx->bc[a][0] = kinds[2 * a]; ctx->bc[a][1] = kinds[2 * a + 1]; }
    ctx->drop_graph();
    return ECHO_OK;
}

int echo_fill_boundaries(echo_ctx *ctx, const int *fields) {
    int rc = check_ready(ctx, false);
    if (rc) return rc;
    DevGuard dev_guard_(ctx);
    if (!fields) return fail(ctx, ECHO_EINVAL, "null argument");
    for (int v = 0; v < 8; ++v)
        if (fields[v] < -1 || fields[v] >= NFIELD) return fail(ctx, ECHO_EINVAL, "field index out of range");
    return fill_boundaries(ctx, fields);
}

int echo_stage_halo_fields(const echo_ctx *ctx, int stage, int *fields) {
    if (!ctx || !fields || stage < 1 || stage > ctx->rk || !ctx->g.uct) return ECHO_EINVAL;
    stage_halo_fields(ctx, stage, fields);
    return ECHO_OK;
}

// ---- packed halo slabs: all 8 fields of one side of one axis in ONE message
static int halo_slab(const echo_ctx *ctx, int axis, int side, bool interior, int *start, int *width) {
    if (axis < 0 || axis > 2 || side < 0 || side > 1) return ECHO_EINVAL;
    const Grid &g = ctx->g;
    const int h = g.lo[axis];
    if (h <= 0) return ECHO_EINVAL;                       // this axis is not decomposed
    *width = h;
    // interior slab next to `side` (what the neighbour on that side needs) or the halo on that side
    *start = side == 0 ? (interior ? h : 0) : (interior ? g.n[axis] - 2 * h : g.n[axis] - h);
    return ECHO_OK;
}

size_t echo_halo_doubles(const echo_ctx *ctx, int axis) {
    if (!ctx || axis < 0 || axis > 2 || ctx->g.lo[axis] <= 0) return 0;
    return (size_t)8 * ctx->g.lo[axis] * (size_t)(ctx->g.N / ctx->g.n[axis]);
}

static int halo_copy(echo_ctx *ctx, const int *fields, int axis, int side, double *buf, void *cuda_stream, bool pack) {
    int rc = check_ready(ctx, false);
    if (rc) return rc;
    DevGuard dev_guard_(ctx);
    if (!fields || !buf) return fail(ctx, ECHO_EINVAL, "null argument");
    int start = 0, width = 0;
    if ((rc = halo_slab(ctx, axis, side, pack, &start, &width))) return fail(ctx, rc, "axis is not decomposed or bad axis / side");
    HaloFields hf;
    for (int v = 0; v < 8; ++v) {
        if (fields[v] < -1 || fields[v] >= NFIELD) return fail(ctx, ECHO_EINVAL, "field index out of range");
        hf.f[v] = fields[v] < 0 ? nullptr : ctx->field[fields[v]];   // -1: this slot of the message is skipped
    }
    const Grid &g = ctx->g;
    const long long per_field = (long long)width * (g.N / g.n[axis]);
    cudaStream_t st = cuda_stream ? static_cast<cudaStream_t>(cuda_stream) : ctx->stream;
    const int blocks = (int)std::min<long long>((per_field + 255) / 256, 148LL * 32);
    cudaStream_t bound = ctx->stream;
    ctx->stream = st;                                     // (the timers, if on, bracket on the stream that runs the copy)
    if (pack) KL(KC_OTHER, "k_halo_pack", k_halo_copy<true><<<dim3(blocks, 8), 256, 0, st>>>(g, hf, buf, axis, start, width, per_field));
    else KL(KC_OTHER, "k_halo_unpack", k_halo_copy<false><<<dim3(blocks, 8), 256, 0, st>>>(g, hf, buf, axis, start, width, per_field));
    ctx->stream = bound;
    return ECHO_OK;
}

int echo_halo_pack(echo_ctx *ctx, const int *fields, int axis, int side, double *buf, void *cuda_stream) {
    return halo_copy(ctx, fields, axis, side, buf, cuda_stream, true);
}
int echo_halo_unpack(echo_ctx *ctx, const int *fields, int axis, int side, const double *buf, void *cuda_stream) {
    return halo_copy(ctx, fields, axis, side, const_cast<double *>(buf), cuda_stream, false);
}

int echo_get_tiling(echo_ctx *ctx, int *out) {
    int rc = check_ready(ctx, false);
    if (rc) return rc;
    DevGuard dev_guard_(ctx);
    if (!out) return fail(ctx, ECHO_EINVAL, "null output");
    ensure_tiling(ctx);
    const Grid &g = ctx->g;
    for (int d = 0; d < 3; ++d) out[d] = g.n[d] == 1 ? 1 : flux_chunk_cells(g, d);
    const bool march = g.n[2] >= 8;        // thin grids keep the thread-per-cell k_prim
    out[3] = (g.uct && march) ? ctx->til.cz_prim : 0;
    out[4] = !g.uct ? 0 : (g.n[2] == 1 ? -ctx->til.cy_uct_flat : ctx->til.cz_uct);
    out[5] = !g.uct ? 0 : (g.n[2] == 1 ? -ctx->til.cy_bupd_flat : ctx->til.cz_bupd);
    out[6] = UCT_TX;
    out[7] = UCT_TY;
    return ECHO_OK;
}

int echo_use_graph(echo_ctx *ctx, int enable) {
    if (!ctx) return ECHO_EINVAL;
    ctx->use_graph = enable ? 1 : 0;
    return ECHO_OK;
}

int echo_timing(echo_ctx *ctx, int enable) {
    int rc = check_ready(ctx, false);
    if (rc) return rc;
    DevGuard dev_guard_(ctx);
    CU(cudaStreamSynchronize(ctx->stream));
    ctx->timing = enable != 0;
    ctx->spans.clear();
    ctx->ev_used = 0;
    for (int c = 0; c < ECHO_NKCLASS; ++c) ctx->launches[c] = 0;
    return ECHO_OK;
}

int echo_get_timing(echo_ctx *ctx, double *ms_total, long *launches) {
    int rc = check_ready(ctx, false);
    if (rc) return rc;
    DevGuard dev_guard_(ctx);
    CU(cudaStreamSynchronize(ctx->stream));
    if (ms_total) {
        for (int c = 0; c < ECHO_NKCLASS; ++c) ms_total[c] = 0.0;
        for (const echo_ctx::Span &s : ctx->spans) {
            float ms = 0.f;
            CU(cudaEventElapsedTime(&ms, ctx->ev_pool[s.e0], ctx->ev_pool[s.e1]));
            ms_total[s.cls] += ms;
        }
    }
    if (launches)
        for (int c = 0; c < ECHO_NKCLASS; ++c) launches[c] = ctx->launches[c];
    return ECHO_OK;
}

int echo_fp64_peak(int reps, double *tflops_host, void *cuda_stream) {
    if (reps < 1 || !tflops_host) return ECHO_EINVAL;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    const int blocks = 148 * 8, threads = 256, iters = 4096;
    double *sink = nullptr;
    if (cudaMalloc(&sink, sizeof(double)) != cudaSuccess) return ECHO_ECUDA;
    std::vector<cudaEvent_t> ev(reps + 1);
    for (auto &e : ev) cudaEventCreate(&e);
    k_dfma_peak<<<blocks, threads, 0, st>>>(iters, 1.0000001, sink);   // warm-up
    cudaEventRecord(ev[0], st);
    for (int r = 0; r < reps; ++r) {
        k_dfma_peak<<<blocks, threads, 0, st>>>(iters, 1.0000001, sink);
        cudaEventRecord(ev[r + 1], st);
    }
    cudaError_t e = cudaStreamSynchronize(st);
    const double flop = 2.0 * DFMA_CHAINS * (double)iters * blocks * threads;
    double best = 0.0;
    float ms = 0.f;
    for (int r = 0; r < reps && e == cudaSuccess; ++r) {
        cudaEventElapsedTime(&ms, ev[r], ev[r + 1]);
        best = std::fmax(best, flop / (ms * 1e-3) * 1e-12);
    }
    cudaEventElapsedTime(&ms, ev[0], ev[reps]);
    tflops_host[0] = best;
    tflops_host[1] = flop * reps / (ms * 1e-3) * 1e-12;
    for (auto &x : ev) cudaEventDestroy(x);
    cudaFree(sink);
    return e == cudaSuccess ? ECHO_OK : ECHO_ECUDA;
}

}  // extern "C"

// ------------------------------------------------------------------ allocation-free div B (echo_div_b_static)
// For callers that may not allocate (code under stream capture, tight serving loops): the high-order div B of
// echo_div_b, stateless, with its scratch -- one partial maximum per 64 x 4 x 1 tile of cells -- in a file-scope device
// array instead of a workspace the caller would have had to cudaMalloc.  Every GPU that loads the library holds the
// ECHO_DIV_B_STATIC_MAX_TILES * 8 bytes (512 KiB) until the process exits.  In HOST code the name g_divb_static is only
// a stand-in for the symbol, not a device address: the address is looked up once per device with that device current
// (cudaGetSymbolAddress) and handed to the kernels as a plain pointer.
static __device__ __align__(256) double g_divb_static[ECHO_DIV_B_STATIC_MAX_TILES];

namespace {

constexpr int DIVB_TX = 64, DIVB_TY = 4;       // the tile of cell_block()
constexpr int DIVB_MAX_DEVICES = 64;
double *g_divb_static_ptr[DIVB_MAX_DEVICES] = {nullptr};   // device address of g_divb_static, per device ordinal
thread_local char g_divb_static_err[192] = "";

int divb_static_fail(int rc, const char *msg) {
    std::snprintf(g_divb_static_err, sizeof(g_divb_static_err), "%s", msg);
    return rc;
}

// Variant of k_divb: same stencil and the same order of operations per cell; the block's maximum of |div B| goes to
// partial[linear tile index] (every slot the finishing kernel reads is written by this launch, so nothing has to be
// cleared between calls).  1-D grid of tiles: blockIdx.x = tx + ntx * (ty + nty * k).
__global__ void __launch_bounds__(256) k_divb_static(Grid g, int ntx, int nty, const double *B0, const double *B1,
                                                     const double *B2, double *div, double *partial) {
    const int tile = blockIdx.x;
    const int i = (tile % ntx) * DIVB_TX + threadIdx.x;
    const int j = ((tile / ntx) % nty) * DIVB_TY + threadIdx.y;
    const int k = tile / (ntx * nty);
    double v = 0.0;
    if (i < g.n[0] && j < g.n[1]) {
        const int c3[3] = {i, j, k};
        const int c = i + g.s[1] * j + g.s[2] * k;
        const double *B[3] = {B0, B1, B2};
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            const int base = c - g.s[d] * c3[d];
            double f[6];
#pragma unroll
            for (int m = 0; m < 6; ++m) f[m] = __ldg(B[d] + (base + g.s[d] * wrapi(c3[d] + m - 3, g.n[d])));
            v += g.rh[d] * der_diff_ho(g.ho, f[0], f[1], f[2], f[3], f[4], f[5]);
        }
        if (div) div[c] = v;
        v = fabs(v);
    }
    __shared__ double sm[256];
    const int tid = threadIdx.y * blockDim.x + threadIdx.x;
    sm[tid] = v;
    __syncthreads();
    for (int s = 128; s > 0; s >>= 1) {
        if (tid < s) sm[tid] = fmax(sm[tid], sm[tid + s]);
        __syncthreads();
    }
    if (tid == 0) partial[tile] = sm[0];
}

// one block: maximum of the first ntiles partials -> *out
__global__ void __launch_bounds__(256) k_divb_static_finish(int ntiles, const double *partial, double *out) {
    double v = 0.0;
    for (int t = threadIdx.x; t < ntiles; t += 256) v = fmax(v, partial[t]);
    __shared__ double sm[256];
    sm[threadIdx.x] = v;
    __syncthreads();
    for (int s = 128; s > 0; s >>= 1) {
        if (threadIdx.x < s) sm[threadIdx.x] = fmax(sm[threadIdx.x], sm[threadIdx.x + s]);
        __syncthreads();
    }
    if (threadIdx.x == 0) *out = sm[0];
}

}  // namespace

extern "C" {

const char *echo_div_b_static_error(void) { return g_divb_static_err; }

int echo_div_b_static_setup(void) {
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) return divb_static_fail(ECHO_ECUDA, "echo_div_b_static: no current CUDA device");
    if (dev < 0 || dev >= DIVB_MAX_DEVICES) return divb_static_fail(ECHO_EINVAL, "echo_div_b_static: device ordinal beyond 63");
    if (g_divb_static_ptr[dev]) return ECHO_OK;
    double *ptr = nullptr;
    const cudaError_t e = cudaGetSymbolAddress((void **)&ptr, g_divb_static);
    if (e != cudaSuccess || !ptr) {
        char msg[160];
        std::snprintf(msg, sizeof(msg), "echo_div_b_static: cudaGetSymbolAddress failed: %s", cudaGetErrorString(e));
        return divb_static_fail(ECHO_ECUDA, msg);
    }
    g_divb_static_ptr[dev] = ptr;     // idempotent: two threads racing here store the same address
    return ECHO_OK;
}

int echo_div_b_static(int nx, int ny, int nz, int ho, const double *bx_face, const double *by_face,
                      const double *bz_face, double *div_field, double *max_abs_dev, void *cuda_stream) {
    if (nx < 1 || ny < 1 || nz < 1) return divb_static_fail(ECHO_EINVAL, "echo_div_b_static: nx, ny, nz must be >= 1");
    if (!bx_face || !by_face || !bz_face) return divb_static_fail(ECHO_EINVAL, "echo_div_b_static: null face array");
    if (!div_field && !max_abs_dev) return divb_static_fail(ECHO_EINVAL, "echo_div_b_static: both outputs are null");
    const long long ntx = (nx + DIVB_TX - 1) / DIVB_TX, nty = (ny + DIVB_TY - 1) / DIVB_TY;
    const long long ntiles = ntx * nty * (long long)nz;
    if (ntiles > ECHO_DIV_B_STATIC_MAX_TILES) {
        char msg[192];
        std::snprintf(msg, sizeof(msg),
                      "echo_div_b_static: grid %d x %d x %d needs %lld tiles of 64 x 4 x 1 cells, the static scratch holds %d "
                      "(e.g. 256^3); use echo_div_b",
                      nx, ny, nz, ntiles, ECHO_DIV_B_STATIC_MAX_TILES);
        return divb_static_fail(ECHO_EINVAL, msg);
    }
    int rc = echo_div_b_static_setup();
    if (rc) return rc;
    int dev = 0;
    cudaGetDevice(&dev);
    double *partial = g_divb_static_ptr[dev];
    Grid g;
    g.n[0] = nx; g.n[1] = ny; g.n[2] = nz;
    g.s[0] = 1; g.s[1] = nx; g.s[2] = nx * ny;          // ntiles <= 65536 bounds N by 2^24
    g.N = (long long)nx * ny * nz;
    for (int d = 0; d < 3; ++d) { g.h[d] = 1.0 / g.n[d]; g.rh[d] = (double)g.n[d]; g.lo[d] = 0; g.hi[d] = g.n[d]; }
    g.ho = ho ? 1 : 0;
    g.uct = 1;
    g.rec = 5;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    k_divb_static<<<(unsigned)ntiles, cell_block(), 0, st>>>(g, (int)ntx, (int)nty, bx_face, by_face, bz_face, div_field, partial);
    if (max_abs_dev) k_divb_static_finish<<<1, 256, 0, st>>>((int)ntiles, partial, max_abs_dev);
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) {
        char msg[160];
        std::snprintf(msg, sizeof(msg), "echo_div_b_static: launch failed: %s", cudaGetErrorString(e));
        return divb_static_fail(ECHO_ECUDA, msg);
    }
    return ECHO_OK;
}

}  // extern "C"
