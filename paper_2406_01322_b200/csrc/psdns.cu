// libpsdns host side: C ABI of include/psdns.h, workspace carving, kernel sequencing.
// One time step = rows a1..a11 of DESIGN.md, enqueued on the caller's stream
// and replayed as a CUDA graph.
#include "../../include/psdns.h"

#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <string>
#include <vector>

#include "kernels_spectral.cuh"
#include "kernels_transform.cuh"
#include "kernels_xfused.cuh"
#include "kernels_xfused_visc.cuh"
#include "kernels_diag.cuh"
#include "kernels_ztma.cuh"
#include "kernels_zgemm.cuh"
#include "kernels_raycast.cuh"

#include <cudaTypedefs.h>

using namespace psdns;

namespace {

constexpr size_t ALIGN = 256;
inline size_t align_up(size_t x) { return (x + ALIGN - 1) / ALIGN * ALIGN; }
inline int round_up8(int x) { return (x + 7) / 8 * 8; }
inline bool is_pow2(int x) { return x > 0 && (x & (x - 1)) == 0; }

enum KClass { KC_ZBWD, KC_YBWD, KC_XBWD, KC_PW, KC_XFWD, KC_YFWD, KC_ZFWD, KC_RHS, KC_SOLVE, KC_MISC, KC_XFUSED, KC_COUNT };
const char *kclass_names[KC_COUNT] = {"zbwd", "ybwd", "xbwd", "pointwise", "xfwd", "yfwd", "zfwd", "rhs", "solve", "misc", "xfused"};

struct Dims {
    int nx, ny, nz, N;
    int nkx, nky, nkz, jpos, kxp;      // retained (dealiased) set
    int nkxf, kxpf;                    // full set (round trip): nkxf = nx/2+1
    size_t ncols;                      // nky * kxp
    size_t s_ret;                      // cplx per retained spectrum with all nz planes
    size_t s_low;                      // cplx per retained spectrum with nkz planes
    size_t s_y;                        // cplx per Y array: nz * ny * kxp
    size_t s_p;                        // doubles per physical field
    size_t s_full;                     // cplx per full padded spectrum nz * ny * kxpf
    size_t s_bspec;                    // cplx per boundary spectral field nz * ny * nkxf
};

struct Layout {
    size_t tw_x, tw_y, tw_z, tw_zn;    // tw_zn: exp(-2 pi i k / N), k < N (the z passes' FFT length)
    size_t ctab_z;                     // c_k of the half-length Chebyshev transform, k <= N/2
    size_t zg_b, zg_f;                 // GEMM-form Chebyshev matrices [ZG_MP][ZG_KP] (N <= 64 only)
    size_t znodes;                     // z_k = cos(pi k / N) (ray-caster), nz doubles
    size_t ccw;                        // Clenshaw-Curtis weights on z_k (diagnostics), nz doubles
    size_t state[5];                   // u v w phi theta
    size_t hist[3];
    size_t dinv[3];                    // NS (beta^2), PO (k^2), CH (k^2 + lambda)
    size_t thh, wh;                    // real homogeneous solutions [nz][ncols]
    size_t hw, coef;                   // [2][ncols] doubles / cplx
    size_t tab_phi;                    // (c^_k, e^_k) of the phi solve's upward elimination, [nz][ncols] double2 (phase field)
    size_t tab_w;                      // the same for the w solve (sigma = k^2)
    size_t xom;
    size_t derived[8];                 // phz [exx eyy exy exz eyz]
    size_t prod[10];                   // txx-tzz txy txz tyy-tzz tyz q c [fx fy fz: force form of the surface tension]
    size_t zb[MAXF], yb[MAXF], ph[MAXF];
    size_t small;                      // ab[2] doubles + counter
    size_t stage[4];                   // host-staging device buffers (boundary layout): inputs of psdns_run_host
    size_t stage_b[4];                 // second set of input staging buffers: the upload of call k + 1 overlaps the compute of call k
    size_t stage_out[4];               // outputs of psdns_run_host (copied back on the side stream while the next call runs)
    size_t total, total_unfused;
};

}  // namespace

struct psdns_handle {
    psdns_grid g;
    psdns_params p;
    cudaStream_t st;
    Dims d;
    Layout L;
    char *ws;
    bool has_state;
    cudaGraphExec_t graph;
    bool graph_ready;
    bool use_graph;
    std::string err;
    long long launches, per_step;
    int timed_class;
    std::vector<std::pair<cudaEvent_t, cudaEvent_t>> tevents;
    int nf_in, nf_out;
    bool use_xfused, has_unfused_ws;
    cudaStream_t copy_st;        // side stream of psdns_run_host's device -> host copies
    cudaStream_t copy_in_st;     // side stream of its host -> device copies
    cudaEvent_t ev_out_ready, ev_d2h_done, ev_in_ready, ev_in_free[2];
    bool d2h_pending, in_used[2];
    long long host_calls;
    int xf_occ, xfv_occ, n_sm;
    int occ_z[2], occ_y[2];     // resident CTAs per SM of the persistent z / y passes, [fwd]
    int use_zgemm;              // psdns_set_option("zgemm"): GEMM-form Chebyshev on the FP64 tensor cores for N <= 64
    int use_ztma;               // psdns_set_option("ztma"): z passes with TMA tensor loads (k_zpass_tma) / register-fed (k_zpass)
    int occ_zt[2][2];           // resident CTAs per SM of k_zpass_tma, [fwd][full-length input]
    PFN_cuTensorMapEncodeTiled encode_tiled;
    int grid_cap;               // psdns_set_option("grid_cap"): upper bound on the grid of every persistent kernel (0 = none)
    int pf, pf_rhs;             // L2 prefetch distances of the column sweeps, in rows
    bool phi3 = true;           // phi problem in three sweeps (ElimUpNeu)
    bool lazy = true;           // with w3: theta^ stays theta_p, corrected where the next step reads it
    bool th_pending = false;    // theta^ in memory lacks the influence-matrix correction of the last step (coef holds it)
    bool w3 = true;             // w problem in three sweeps (ElimUpDir2; needs phi3 with a phase field)
    long long last_grid[KC_COUNT], last_items[KC_COUNT];   // grid / work items of the last launch of each persistent class

    int persistent_grid(int kc, long long items, int occ) {
        long long g = std::min<long long>(items, (long long)n_sm * std::max(occ, 1));
        if (grid_cap > 0) g = std::min<long long>(g, grid_cap);
        last_grid[kc] = g; last_items[kc] = items;
        return (int)g;
    }

    template <class T> T *at(size_t off) const { return reinterpret_cast<T *>(ws + off); }
};

namespace {

bool validate(const psdns_grid *g, const psdns_params *p) {
    if (!g || !p) return false;
    if (!is_pow2(g->nx) || !is_pow2(g->ny) || g->nx < 16 || g->ny < 16 || g->nx > 1024 || g->ny > 1024) return false;
    const int N = g->nz - 1;
    if (!is_pow2(N) || N < 8 || N > 512) return false;
    if (!(g->lx > 0) || !(g->ly > 0)) return false;
    if (!(p->re > 0) || !(p->dt > 0)) return false;
    if (p->phase_field != 0 && p->phase_field != 1) return false;
    if (p->surface_tension_form != 0 && p->surface_tension_form != 1) return false;
    if (p->surface_tension_form == 1 && (!p->phase_field || p->visc_ratio != 1.0)) return false;   // force form: matched viscosity only
    if (p->convection_form != 0 && p->convection_form != 1) return false;
    if (p->convection_form == 1 && p->phase_field && p->visc_ratio != 1.0) return false;
    if ((p->wall_top != 0 && p->wall_top != 1) || (p->wall_bottom != 0 && p->wall_bottom != 1)) return false;
    if (p->phase_field && (!(p->pe > 0) || !(p->ch > 0) || !(p->we > 0) || !(p->visc_ratio > 0))) return false;
    return true;
}

Dims make_dims(const psdns_grid &g) {
    Dims d;
    d.nx = g.nx; d.ny = g.ny; d.nz = g.nz; d.N = g.nz - 1;
    const int I = g.nx / 3, J = g.ny / 3, K = (2 * d.N) / 3;   // reading S3
    d.nkx = I + 1; d.nky = 2 * J + 1; d.nkz = K + 1; d.jpos = J + 1;
    d.kxp = round_up8(d.nkx);
    d.nkxf = g.nx / 2 + 1;
    d.kxpf = round_up8(d.nkxf);
    d.ncols = (size_t)d.nky * d.kxp;
    d.s_ret = (size_t)d.nz * d.ncols;
    d.s_low = (size_t)d.nkz * d.ncols;
    d.s_y = (size_t)d.nz * d.ny * d.kxp;
    d.s_p = (size_t)d.nz * d.ny * d.nx;
    d.s_full = (size_t)d.nz * d.ny * d.kxpf;
    d.s_bspec = (size_t)d.nz * d.ny * d.nkxf;
    return d;
}

Layout make_layout(const Dims &d, const psdns_params &p) {
    Layout L;
    size_t o = 0;
    auto take = [&](size_t bytes) { size_t r = o; o = align_up(o + bytes); return r; };
    const size_t C = sizeof(cplx);
    L.tw_x = take(d.nx * C);
    L.tw_y = take(d.ny * C);
    L.tw_z = take(2 * d.N * C);
    L.tw_zn = take(d.N * C);
    L.ctab_z = take((d.N / 2 + 1) * C);
    L.ccw = take(d.nz * sizeof(double));
    L.znodes = take(d.nz * sizeof(double));
    L.zg_b = L.zg_f = 0;
    if (d.N <= 64) { L.zg_b = take(ZG_MP * ZG_KP * sizeof(double)); L.zg_f = take(ZG_MP * ZG_KP * sizeof(double)); }
    for (int i = 0; i < 5; ++i) L.state[i] = take(d.s_ret * C);
    for (int i = 0; i < 3; ++i) L.hist[i] = take(d.s_low * C);
    for (int i = 0; i < 3; ++i) L.dinv[i] = take(d.s_ret * sizeof(double));
    L.thh = take(d.s_ret * sizeof(double));
    L.wh = take(d.s_ret * sizeof(double));
    L.hw = take(4 * d.ncols * sizeof(double));
    L.coef = take(2 * d.ncols * C);
    L.tab_phi = p.phase_field ? take(d.s_ret * sizeof(double2)) : 0;
    L.tab_w = take(d.s_ret * sizeof(double2));
    L.xom = take(d.s_ret * C);
    const bool visc_l = p.phase_field && p.visc_ratio != 1.0;
    for (int i = 0; i < 8; ++i) L.derived[i] = 0;
    const bool force_l = (p.phase_field && p.surface_tension_form == 1) || p.convection_form == 1;   // a force vector next to T
    for (int i = 0; i < (visc_l ? 6 : (force_l ? 5 : 1)); ++i) L.derived[i] = take(d.s_low * C);   // phz [+ 5 strains | + lap phi, 3 vorticity]
    for (int i = 0; i < 10; ++i) L.prod[i] = 0;
    for (int i = 0; i < (force_l ? 10 : 7); ++i) L.prod[i] = take(d.s_low * C);
    const int nf = (visc_l || force_l) ? 12 : 7;
    // Z / Y arrays double as the full-size round-trip scratch (3 arrays of s_full each)
    size_t zy_bytes = 0;
    for (int i = 0; i < MAXF; ++i) { L.zb[i] = 0; L.yb[i] = 0; L.ph[i] = 0; }
    for (int i = 0; i < nf; ++i) { L.zb[i] = take(d.s_ret * C); zy_bytes += align_up(d.s_ret * C); }
    for (int i = 0; i < nf; ++i) { L.yb[i] = take(d.s_y * C); zy_bytes += align_up(d.s_y * C); }
    const size_t need_full = 3 * align_up(d.s_full * C);
    if (zy_bytes < need_full) take(need_full - zy_bytes);
    L.small = take(64);
    const size_t stage_bytes = std::max(d.s_p * sizeof(double), d.s_bspec * C);
    for (int i = 0; i < 4; ++i) L.stage[i] = take(stage_bytes);
    for (int i = 0; i < 4; ++i) L.stage_b[i] = take(stage_bytes);
    for (int i = 0; i < 4; ++i) L.stage_out[i] = take(stage_bytes);
    // the force form of the surface tension runs the three-kernel x path: its physical arrays are product state
    if (force_l) for (int i = 0; i < nf; ++i) L.ph[i] = take(d.s_p * sizeof(double));
    L.total = o;
    // physical-space arrays of the UNFUSED x path (psdns_set_option "xfuse" 0, a cross-check): behind the product's
    // workspace, present only when the caller passed psdns_workspace_bytes_unfused() bytes to psdns_init
    if (!force_l) for (int i = 0; i < nf; ++i) L.ph[i] = take(d.s_p * sizeof(double));
    L.total_unfused = o;
    return L;
}

#define CUDA_TRY(h, expr)                                                                          \
    do {                                                                                           \
        cudaError_t e__ = (expr);                                                                  \
        if (e__ != cudaSuccess) {                                                                  \
            (h)->err = std::string(#expr) + ": " + cudaGetErrorString(e__);                        \
            return PSDNS_ECUDA;                                                                    \
        }                                                                                          \
    } while (0)

struct LaunchScope {   // optional CUDA-event bracket around launches of the timed class
    psdns_handle *h;
    bool on;
    cudaEvent_t e0, e1;
    LaunchScope(psdns_handle *h_, int kc) : h(h_), on(h_->timed_class == kc) {
        if (on) {
            cudaEventCreate(&e0); cudaEventCreate(&e1);
            cudaEventRecord(e0, h->st);
        }
    }
    ~LaunchScope() {
        if (on) {
            cudaEventRecord(e1, h->st);
            h->tevents.push_back({e0, e1});
        }
        h->launches++;
    }
};

inline int col_grid(const Dims &d) { return (int)((d.ncols + NT_COL - 1) / NT_COL); }

ColGeom geom(const psdns_handle *h) {
    ColGeom g;
    const Dims &d = h->d;
    g.ncols = (int)d.ncols; g.kxp = d.kxp; g.nkx = d.nkx; g.nky = d.nky; g.jpos = d.jpos;
    g.N = d.N; g.nkz = d.nkz;
    g.kxf = 2.0 * M_PI / h->g.lx; g.kyf = 2.0 * M_PI / h->g.ly;
    // L2 prefetch distances in rows (kernels_spectral.cuh).  Measured on B200: 2 (4 for k_rhs_elim) is best at 117 k
    // columns, where 6 thrashed the L2, and longer distances do not help the latency-bound small grids either
    // (256x256x257: solve 0.82 ms at 2 rows, 0.84 at 12, 0.90 at 24).
    g.pf = h->pf;
    g.pf_rhs = h->pf_rhs;
    return g;
}

// ---- transform pass launchers ------------------------------------------------------------------
template <int L>
size_t fft_smem() { return (size_t)(L * TILE_LINES + L) * sizeof(cplx); }

template <int L>
size_t xfusedv_smem(int nkx) { return (size_t)((L / 2) * XV_SLOTS + XV_NST * xf_spitch(nkx)) * sizeof(cplx) + 16; }

template <int L>
size_t xfusedw_smem(int nkx, int nst) {
    return (size_t)(xfw_lpi<L>() * ((L / 2) * TILE_LINES + nst * xf_spitch(nkx))) * sizeof(cplx) + 32;
}

template <class K>
cudaError_t set_smem(K kern, size_t bytes) {
    if (bytes > 48 * 1024) return cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
    return cudaSuccess;
}

#define DISPATCH_L(Lval, MACRO)            \
    switch (Lval) {                        \
        case 16: MACRO(16); break;         \
        case 32: MACRO(32); break;         \
        case 64: MACRO(64); break;         \
        case 128: MACRO(128); break;       \
        case 256: MACRO(256); break;       \
        case 512: MACRO(512); break;       \
        case 1024: MACRO(1024); break;     \
        default: return cudaErrorInvalidValue; \
    }

template <int N, bool FWD>
size_t zpass_smem() { return (size_t)zpass_smem_cplx<N, FWD>() * sizeof(cplx); }

#define DISPATCH_N(Nval, MACRO)            \
    switch (Nval) {                        \
        case 8: MACRO(8); break;           \
        case 16: MACRO(16); break;         \
        case 32: MACRO(32); break;         \
        case 64: MACRO(64); break;         \
        case 128: MACRO(128); break;       \
        case 256: MACRO(256); break;       \
        case 512: MACRO(512); break;       \
        default: return cudaErrorInvalidValue; \
    }

// derived outputs of the backward z pass (row a1): i kx X and / or i ky X of field dfield
struct ZDerived {
    int dfield = -1;
    cplx *out_dx = nullptr, *out_dy = nullptr;
};

// input rows of a z-pass tile -> (number of TMA boxes, rows per box); a box has at most 256 rows
inline std::pair<int, int> ztma_rows(int nin) {
    const int nb = (nin + 255) / 256;
    return {nb, (nin + nb - 1) / nb};
}

cudaError_t launch_zpass_tma(psdns_handle *h, bool fwd, const FieldPtrs &f, int nf, size_t ncols, int nk, int kxp, int nky,
                             int jpos, const ZDerived &zd) {
    ZTArgs a;
    const int N = h->d.N;
    const int nin = fwd ? N + 1 : nk;
    const auto rb = ztma_rows(nin);
    a.nf = nf; a.ncols = (int)ncols; a.nk = nk; a.nboxes = rb.first; a.box_rows = rb.second;
    a.dfield = fwd ? -1 : zd.dfield; a.out_dx = zd.out_dx; a.out_dy = zd.out_dy;
    a.kxp = kxp; a.nky = nky; a.jpos = jpos;
    a.kxf = 2.0 * M_PI / h->g.lx; a.kyf = 2.0 * M_PI / h->g.ly;
    for (int i = 0; i < nf; ++i) {
        a.out[i] = f.out[i];
        const cuuint64_t gdim[2] = {(cuuint64_t)(2 * ncols), (cuuint64_t)nin};
        const cuuint64_t gstr[1] = {(cuuint64_t)(ncols * sizeof(cplx))};
        const cuuint32_t box[2] = {16u, (cuuint32_t)rb.second};
        const cuuint32_t estr[2] = {1u, 1u};
        const CUresult r = h->encode_tiled(&a.in_map[i], CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, const_cast<void *>(f.in[i]), gdim, gstr,
                                           box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                                           CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (r != CUDA_SUCCESS) return cudaErrorInvalidValue;
    }
    const cplx *tw = h->at<cplx>(h->L.tw_zn);
    const cplx *ct = h->at<cplx>(h->L.ctab_z);
    const long long ntiles = (long long)(ncols / 8) * nf;
    const int srows = rb.first * rb.second;
    const int grid = h->persistent_grid(fwd ? KC_ZFWD : KC_ZBWD, ntiles, h->occ_zt[fwd][nin == N + 1]);
    LaunchScope ls(h, fwd ? KC_ZFWD : KC_ZBWD);
#define ZT(NN)                                                                                                         \
    {                                                                                                                  \
        if (fwd) k_zpass_tma<NN, true><<<grid, ztma_threads<NN>(), ztma_smem_bytes<NN>(srows), h->st>>>(a, tw, ct);    \
        else k_zpass_tma<NN, false><<<grid, ztma_threads<NN>(), ztma_smem_bytes<NN>(srows), h->st>>>(a, tw, ct);       \
    }
    DISPATCH_N(N, ZT)
#undef ZT
    return cudaGetLastError();
}

cudaError_t launch_zpass(psdns_handle *h, bool fwd, const FieldPtrs &f, int nf, size_t ncols, int nk, int kxp, int nky,
                         int jpos, const ZDerived &zd = ZDerived()) {
    if (h->use_zgemm && h->d.N <= 64 && !(zd.dfield >= 0 && zd.out_dx)) {
        // GEMM form on the FP64 tensor cores (kernels_zgemm.cuh), short columns only
        ZGArgs g; g.f = f; g.nf = nf; g.ncols = (int)ncols;
        g.nrow_in = fwd ? h->d.N + 1 : nk; g.nrow_out = fwd ? nk : h->d.N + 1;
        g.mat = h->at<double>(fwd ? h->L.zg_f : h->L.zg_b);
        g.dfield = fwd ? -1 : zd.dfield; g.out_dy = zd.out_dy; g.kxp = kxp; g.nky = nky; g.jpos = jpos;
        g.kyf = 2.0 * M_PI / h->g.ly;
        const long long nblk = ((2 * (long long)ncols + ZG_COLS - 1) / ZG_COLS) * nf;
        const int grid = h->persistent_grid(fwd ? KC_ZFWD : KC_ZBWD, nblk, 2);
        LaunchScope ls(h, fwd ? KC_ZFWD : KC_ZBWD);
        k_zgemm<<<grid, ZG_NT, ZG_SMEM, h->st>>>(g);
        return cudaGetLastError();
    }
    if (h->use_ztma && h->encode_tiled) return launch_zpass_tma(h, fwd, f, nf, ncols, nk, kxp, nky, jpos, zd);
    ZArgs a; a.f = f; a.nf = nf; a.ncols = (int)ncols; a.nk = nk;
    a.dfield = fwd ? -1 : zd.dfield; a.out_dx = zd.out_dx; a.out_dy = zd.out_dy;
    a.kxp = kxp; a.nky = nky; a.jpos = jpos;
    a.kxf = 2.0 * M_PI / h->g.lx; a.kyf = 2.0 * M_PI / h->g.ly;
    const cplx *tw = h->at<cplx>(h->L.tw_z);
    const cplx *ct = h->at<cplx>(h->L.ctab_z);
    const long long ntiles = (long long)(ncols / 8) * nf;
    const int grid = h->persistent_grid(fwd ? KC_ZFWD : KC_ZBWD, ntiles, h->occ_z[fwd]);
    LaunchScope ls(h, fwd ? KC_ZFWD : KC_ZBWD);
#define ZH(NN)                                                                                           \
    {                                                                                                    \
        if (fwd) k_zpass<NN, true><<<grid, zpass_threads<NN, true>(), zpass_smem<NN, true>(), h->st>>>(a, tw, ct);   \
        else k_zpass<NN, false><<<grid, zpass_threads<NN, false>(), zpass_smem<NN, false>(), h->st>>>(a, tw, ct);      \
    }
    DISPATCH_N(h->d.N, ZH)
#undef ZH
    return cudaGetLastError();
}

cudaError_t launch_ypass(psdns_handle *h, bool fwd, const FieldPtrs &f, int nf, int kxp, int nky, int jpos, int nplanes = -1) {
    if (nplanes < 0) nplanes = h->d.nz;
    YArgs a; a.f = f; a.nf = nf; a.nz = nplanes; a.kxp = kxp; a.nky = nky; a.jpos = jpos;
    const cplx *tw = h->at<cplx>(h->L.tw_y);
    const long long ntiles = (long long)(kxp / 8) * nplanes * nf;
    const int grid = h->persistent_grid(fwd ? KC_YFWD : KC_YBWD, ntiles, h->occ_y[fwd]);
    LaunchScope ls(h, fwd ? KC_YFWD : KC_YBWD);
#define YL(LL)                                                                                          \
    {                                                                                                   \
        if (fwd) k_ypass<LL, true><<<grid, fused_threads<LL>(), fft_smem<LL>(), h->st>>>(a, tw);        \
        else k_ypass<LL, false><<<grid, fused_threads<LL>(), fft_smem<LL>(), h->st>>>(a, tw);           \
    }
    DISPATCH_L(h->d.ny, YL)
#undef YL
    return cudaGetLastError();
}

cudaError_t launch_xpass(psdns_handle *h, bool fwd, const FieldPtrs &f, int nf, int kxp, int nkx) {
    XArgs a; a.f = f; a.kxp = kxp; a.nkx = nkx;
    const cplx *tw = h->at<cplx>(h->L.tw_x);
    dim3 grid((unsigned)((size_t)h->d.nz * h->d.ny / 16), nf);
    LaunchScope ls(h, fwd ? KC_XFWD : KC_XBWD);
#define XL(LL)                                                                                          \
    {                                                                                                   \
        if (fwd) k_xpass<LL, true><<<grid, tile_threads<LL>(), fft_smem<LL>(), h->st>>>(a, tw);                     \
        else k_xpass<LL, false><<<grid, tile_threads<LL>(), fft_smem<LL>(), h->st>>>(a, tw);                        \
    }
    DISPATCH_L(h->d.nx, XL)
#undef XL
    return cudaGetLastError();
}

// fused x kernel of one line length: the single-line warp-per-field kernel where a pass fills a warp (nx = 1024), the
// multi-line one below that.  Templates, so that only the kernel actually used for a line length is instantiated.
template <int LL>
cudaError_t setup_xfused_L(psdns_handle *h) {
    const size_t sm = xfusedw_smem<LL>(h->d.nkx, h->p.phase_field ? 7 : 3);
    int occ = 0;
    cudaError_t e = cudaSuccess;
    auto prep = [&](auto kern) {
        e = set_smem(kern, sm);
        if (e == cudaSuccess) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, XFW_THREADS, sm);
    };
    if constexpr (xfw_lpi<LL>() == 1) {
        if (h->p.phase_field) prep(k_xfusedw<LL, true>); else prep(k_xfusedw<LL, false>);
    } else {
        if (h->p.phase_field) prep(k_xfusedwm<LL, true>); else prep(k_xfusedwm<LL, false>);
    }
    h->xf_occ = occ;
    return e;
}

template <int LL>
cudaError_t launch_xfused_L(psdns_handle *h, const XFArgs &a, const cplx *tw, int grid) {
    const size_t sm = xfusedw_smem<LL>(h->d.nkx, h->p.phase_field ? 7 : 3);
    if (a.nkx != LL / 3 + 1 || a.kxp != round_up8(a.nkx)) return cudaErrorInvalidValue;   // the kernels' compile-time cut-offs
    if constexpr (xfw_lpi<LL>() == 1) {
        if (h->p.phase_field) k_xfusedw<LL, true><<<grid, XFW_THREADS, sm, h->st>>>(a, tw);
        else k_xfusedw<LL, false><<<grid, XFW_THREADS, sm, h->st>>>(a, tw);
    } else {
        if (h->p.phase_field) k_xfusedwm<LL, true><<<grid, XFW_THREADS, sm, h->st>>>(a, tw);
        else k_xfusedwm<LL, false><<<grid, XFW_THREADS, sm, h->st>>>(a, tw);
    }
    return cudaSuccess;
}

// opt-in to > 48 KB dynamic shared memory once, at init (not inside graph capture), and size the persistent grids
cudaError_t setup_attrs(psdns_handle *h) {
#define CU0(expr) do { cudaError_t e__ = (expr); if (e__ != cudaSuccess) return e__; } while (0)
#define ZA(NN)                                                                                                         \
    {                                                                                                                  \
        CU0(set_smem(k_zpass<NN, true>, zpass_smem<NN, true>())); CU0(set_smem(k_zpass<NN, false>, zpass_smem<NN, false>()));        \
        CU0(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&h->occ_z[1], k_zpass<NN, true>, zpass_threads<NN, true>(), zpass_smem<NN, true>()));  \
        CU0(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&h->occ_z[0], k_zpass<NN, false>, zpass_threads<NN, false>(), zpass_smem<NN, false>())); \
    }
#define YA(LL)                                                                                                         \
    {                                                                                                                  \
        CU0(set_smem(k_ypass<LL, true>, fft_smem<LL>())); CU0(set_smem(k_ypass<LL, false>, fft_smem<LL>()));            \
        CU0(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&h->occ_y[1], k_ypass<LL, true>, fused_threads<LL>(), fft_smem<LL>()));    \
        CU0(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&h->occ_y[0], k_ypass<LL, false>, fused_threads<LL>(), fft_smem<LL>()));   \
    }
#define XA(LL) { CU0(set_smem(k_xpass<LL, true>, fft_smem<LL>())); CU0(set_smem(k_xpass<LL, false>, fft_smem<LL>())); }
    DISPATCH_N(h->d.N, ZA)
#define ZTA(NN)                                                                                                        \
    {                                                                                                                  \
        const auto rf = ztma_rows(NN + 1);                                                                             \
        const size_t big = ztma_smem_bytes<NN>(rf.first * rf.second);                                                  \
        CU0(set_smem(k_zpass_tma<NN, true>, big)); CU0(set_smem(k_zpass_tma<NN, false>, big));                          \
        for (int full = 0; full < 2; ++full) {                                                                         \
            const auto rb = ztma_rows(full ? NN + 1 : h->d.nkz);                                                       \
            CU0(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&h->occ_zt[0][full], k_zpass_tma<NN, false>, ztma_threads<NN>(), ztma_smem_bytes<NN>(rb.first * rb.second))); \
            CU0(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&h->occ_zt[1][full], k_zpass_tma<NN, true>, ztma_threads<NN>(), big)); \
        }                                                                                                              \
    }
    DISPATCH_N(h->d.N, ZTA)
    CU0(set_smem(k_zgemm, ZG_SMEM));
#undef ZTA
    DISPATCH_L(h->d.ny, YA)
    DISPATCH_L(h->d.nx, XA)
#define XFA(LL) { CU0(setup_xfused_L<LL>(h)); }
    if (h->nf_in <= 7) { DISPATCH_L(h->d.nx, XFA) }
#undef XFA
#define XFVA(LL)                                                                                             \
    {                                                                                                        \
        const size_t sm = xfusedv_smem<LL>(h->d.nkx);                                                        \
        int occ = 0;                                                                                         \
        CU0(set_smem(k_xfusedv<LL>, sm));                                                                    \
        CU0(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_xfusedv<LL>, xv_threads<LL>(), sm));       \
        h->xfv_occ = occ;                                                                                    \
    }
    if (h->nf_in > 7) { DISPATCH_L(h->d.nx, XFVA) }
#undef XFVA
#undef ZA
#undef YA
#undef XA
#undef CU0
    return cudaSuccess;
}

cudaError_t launch_xfused(psdns_handle *h, const XFArgs &a) {
    const cplx *tw = h->at<cplx>(h->L.tw_x);
    const int grid = h->persistent_grid(KC_XFUSED, a.nlines, h->xf_occ);   // persistent: one wave
    LaunchScope ls(h, KC_XFUSED);
#define XF(LL) { const cudaError_t e = launch_xfused_L<LL>(h, a, tw, grid); if (e != cudaSuccess) return e; }
    DISPATCH_L(h->d.nx, XF)
#undef XF
    return cudaGetLastError();
}

cudaError_t launch_xfusedv(psdns_handle *h, const XFVArgs &a) {
    const cplx *tw = h->at<cplx>(h->L.tw_x);
    const int grid = h->persistent_grid(KC_XFUSED, a.nlines, h->xfv_occ);   // persistent: one wave
    if (a.nkx != h->d.nx / 3 + 1 || a.kxp != round_up8(a.nkx)) return cudaErrorInvalidValue;   // the kernel's compile-time cut-offs
    LaunchScope ls(h, KC_XFUSED);
#define XFV(LL) k_xfusedv<LL><<<grid, xv_threads<LL>(), xfusedv_smem<LL>(h->d.nkx), h->st>>>(a, tw);
    DISPATCH_L(h->d.nx, XFV)
#undef XFV
    return cudaGetLastError();
}

cudaError_t launch_relayout(psdns_handle *h, cplx *dst, const cplx *src, SpecSide ds, SpecSide ss, int nplanes) {
    const size_t total = (size_t)nplanes * ds.rows * ds.pitch;
    const int blocks = (int)std::min<size_t>((total + 255) / 256, (size_t)h->n_sm * 16);
    LaunchScope ls(h, KC_MISC);
    k_relayout<<<blocks, 256, 0, h->st>>>(dst, src, ds, ss, nplanes);
    return cudaGetLastError();
}

SpecSide side_boundary(const Dims &d) { return SpecSide{d.ny, d.nkxf, d.ny / 2 + 1, d.nkxf}; }
SpecSide side_ret(const Dims &d) { return SpecSide{d.nky, d.kxp, d.jpos, d.nkx}; }
SpecSide side_full(const Dims &d) { return SpecSide{d.ny, d.kxpf, d.ny / 2 + 1, d.nkxf}; }

cudaError_t launch_helm(psdns_handle *h, const cplx *in, cplx *out, int type, double shift, double scale, int bc,
                        double te, double to) {
    HelmArgs a;
    a.g = geom(h); a.in = in; a.out = out; a.dinv = h->at<double>(h->L.dinv[type]);
    a.shift = shift; a.scale = scale; a.bc = bc; a.tgt_e = te; a.tgt_o = to;
    LaunchScope ls(h, KC_SOLVE);
    k_helm<<<col_grid(h->d), NT_COL, 0, h->st>>>(a);
    return cudaGetLastError();
}

struct Coefs {
    double gamma, lam_phi, gam_phi, s_coef, cs;
};
Coefs coefs(const psdns_params &p) {
    Coefs c;
    c.gamma = p.dt / (2.0 * p.re);
    if (p.phase_field) {
        c.lam_phi = std::sqrt(p.pe / (p.dt * p.ch * p.ch));      // reading S8: s/2
        c.gam_phi = p.dt * p.ch * p.ch / p.pe;
        c.s_coef = 2.0 * c.lam_phi;
        c.cs = 3.0 / std::sqrt(8.0) * p.ch / p.we;              // Eq. 8
    } else {
        c.lam_phi = 1.0; c.gam_phi = 1.0; c.s_coef = 0.0; c.cs = 0.0;
    }
    return c;
}

#define CU(expr)                                  \
    do {                                          \
        cudaError_t e__ = (expr);                 \
        if (e__ != cudaSuccess) return e__;       \
    } while (0)

// ---- one time step (rows a1-a11) ------------------------------------------------------------------
// Field bookkeeping (matched viscosity, phase field on):
//   backward: 5 z transforms (u, v, w, phi, D phi) whose epilogue also emits i ky phi (row a1), 6 y
//             transforms, and the fused x kernel forms i kx phi from the staged phi row: 7 physical fields.
//   forward : 7 product fields Txx - Tzz, Txy, Txz, Tyy - Tzz, Tyz, Q, C.  Only the deviatoric part of T
//             enters Eqs. 14-15 (the isotropic part g delta_ij gives S = grad g, which the curl and the
//             k^2 S_z + D(ikx S_x + iky S_y) combination annihilate identically in the discrete operators), so
//             T_zz is subtracted pointwise instead of being transformed on its own.
cudaError_t enqueue_step(psdns_handle *h) {
    const Dims &d = h->d;
    const Layout &L = h->L;
    const psdns_params &p = h->p;
    const Coefs c = coefs(p);
    const bool phase = p.phase_field != 0;
    const bool visc = phase && p.visc_ratio != 1.0;
    const bool st_force = phase && p.surface_tension_form == 1;   // surface tension as a force vector
    const bool rot = p.convection_form == 1;                     // convection as u x omega
    const bool force = st_force || rot;                          // a force vector F next to the flux tensor (row f4)
    const int nout = h->nf_out;
    cplx *U = h->at<cplx>(L.state[0]), *V = h->at<cplx>(L.state[1]), *W = h->at<cplx>(L.state[2]);
    cplx *PHI = h->at<cplx>(L.state[3]), *TH = h->at<cplx>(L.state[4]), *OM = h->at<cplx>(L.xom);
    cplx *PHZ = h->at<cplx>(L.derived[0]);
    double *ab = h->at<double>(L.small);
    int *counter = reinterpret_cast<int *>(ab + 2);
    { LaunchScope ls(h, KC_MISC); k_begin_step<<<1, 1, 0, h->st>>>(ab, counter); CU(cudaGetLastError()); }

    // a1 (variable viscosity only): strain spectra
    if (visc) {
        PrepArgs a{};
        a.g = geom(h); a.u = U; a.v = V; a.w = W; a.phi = PHI; a.phz = PHZ;
        a.exx = h->at<cplx>(L.derived[1]); a.eyy = h->at<cplx>(L.derived[2]); a.exy = h->at<cplx>(L.derived[3]);
        a.exz = h->at<cplx>(L.derived[4]); a.eyz = h->at<cplx>(L.derived[5]);
        a.do_phz = 0; a.visc = 1;
        LaunchScope ls(h, KC_RHS);
        k_prep<<<col_grid(d), NT_COL, 0, h->st>>>(a);
        CU(cudaGetLastError());
    }
    if (force) {   // row a1, alternative forms: lap(phi)^ = (D^2 - k^2) P phi^ and / or the vorticity spectra of P u^
        PrepArgs a{};
        a.g = geom(h); a.u = U; a.v = V; a.w = W; a.phi = PHI; a.lap = h->at<cplx>(L.derived[1]);
        a.wx = h->at<cplx>(L.derived[2]); a.wy = h->at<cplx>(L.derived[3]); a.wz = h->at<cplx>(L.derived[4]);
        a.do_lap = st_force; a.do_vort = rot;
        LaunchScope ls(h, KC_RHS);
        k_prep<<<col_grid(d), NT_COL, 0, h->st>>>(a);
        CU(cudaGetLastError());
    }
    // a2-a3: backward z and y transforms
    FieldPtrs fz{}, fy{};
    ZDerived zd;
    int nz_f = 3, ny_f = 3;   // fields through the z pass / the y pass
    const cplx *src[MAXF] = {U, V, W, PHI, PHZ};
    if (!phase && rot) {   // single-phase, rotational form: u v w wx wy wz
        for (int i = 0; i < 3; ++i) src[3 + i] = h->at<cplx>(L.derived[2 + i]);
        nz_f = 6; ny_f = 6;
    }
    if (phase) {
        nz_f = 5;
        if (visc) {
            for (int i = 0; i < 5; ++i) src[5 + i] = h->at<cplx>(L.derived[1 + i]);
            nz_f = 10;
            if (h->use_xfused) {   // fused: i kx phi is derived in the x kernel's stage; Z / Y array 10 = i ky phi
                zd.dfield = 3; zd.out_dx = nullptr; zd.out_dy = h->at<cplx>(L.zb[10]);
                ny_f = 11;
            } else {
                zd.dfield = 3; zd.out_dx = h->at<cplx>(L.zb[10]); zd.out_dy = h->at<cplx>(L.zb[11]);
                ny_f = 12;
            }
        } else if (force) {   // Z arrays: u v w phi phz [lap] [wx wy wz] | i ky phi | i kx phi
            nz_f = 5;
            if (st_force) src[nz_f++] = h->at<cplx>(L.derived[1]);
            if (rot) for (int i = 0; i < 3; ++i) src[nz_f++] = h->at<cplx>(L.derived[2 + i]);
            zd.dfield = 3; zd.out_dy = h->at<cplx>(L.zb[nz_f]); zd.out_dx = h->at<cplx>(L.zb[nz_f + 1]);
            ny_f = nz_f + 2;
        } else {
            const bool fused = h->use_xfused;
            zd.dfield = 3; zd.out_dx = fused ? nullptr : h->at<cplx>(L.zb[6]); zd.out_dy = h->at<cplx>(L.zb[5]);
            ny_f = fused ? 6 : 7;
        }
    }
    for (int i = 0; i < nz_f; ++i) { fz.in[i] = src[i]; fz.out[i] = h->at<cplx>(L.zb[i]); }
    for (int i = 0; i < ny_f; ++i) { fy.in[i] = h->at<cplx>(L.zb[i]); fy.out[i] = h->at<cplx>(L.yb[i]); }
    CU(launch_zpass(h, false, fz, nz_f, d.ncols, d.nkz, d.kxp, d.nky, d.jpos, zd));
    CU(launch_ypass(h, false, fy, ny_f, d.kxp, d.nky, d.jpos));
    FieldPtrs gy{}, gz{};
    for (int i = 0; i < nout; ++i) {
        gy.in[i] = h->at<cplx>(L.yb[i]); gy.out[i] = h->at<cplx>(L.zb[i]);
        gz.in[i] = gy.out[i]; gz.out[i] = h->at<cplx>(L.prod[i]);
    }
    if (h->use_xfused && visc) {
        // a4 + a5 + a6 fused, 16-slot tile (kernels_xfused_visc.cuh); Y arrays: u v w phi phz exx eyy exy exz eyz phy
        XFVArgs a;
        const int stage_src[XV_NTMA] = {0, 1, 2, 3, 10, 4, 5, 6, 7, 8, 9};   // u v w phi phy phz exx eyy exy exz eyz
        for (int i = 0; i < XV_NTMA; ++i) a.in[i] = h->at<cplx>(L.yb[stage_src[i]]);
        for (int i = 0; i < XV_NOUT; ++i) a.out[i] = h->at<cplx>(L.yb[i]);
        a.kxp = d.kxp; a.nkx = d.nkx; a.nlines = d.nz * d.ny;
        a.cs = c.cs; a.kxf = 2.0 * M_PI / h->g.lx; a.eta_c = (p.visc_ratio - 1.0) / (2.0 * p.re);
        CU(launch_xfusedv(h, a));
    } else if (h->use_xfused && !visc) {
        // a4 + a5 + a6 fused: physical space never leaves the SM; in place on the Y arrays
        XFArgs a;
        const int stage_src[6] = {0, 1, 2, 3, 5, 4};   // u v w phi phy phz  <-  Y arrays u v w phi phz phy
        for (int i = 0; i < 6; ++i) a.in[i] = h->at<cplx>(L.yb[phase ? stage_src[i] : (i < 3 ? i : 0)]);
        for (int i = 0; i < 8; ++i) a.out[i] = h->at<cplx>(L.yb[i < nout ? i : 0]);
        a.kxp = d.kxp; a.nkx = d.nkx; a.nlines = d.nz * d.ny;
        a.cs = c.cs; a.kxf = 2.0 * M_PI / h->g.lx;
        CU(launch_xfused(h, a));
    } else {
        // unfused cross-check path (psdns_set_option "xfuse" 0): a4, a5, a6 as separate kernels
        FieldPtrs fx{}, gx{};
        const int nx_f = ny_f;
        for (int i = 0; i < nx_f; ++i) { fx.in[i] = h->at<cplx>(L.yb[i]); fx.out[i] = h->at<double>(L.ph[i]); }
        CU(launch_xpass(h, false, fx, nx_f, d.kxp, d.nkx));
        {
            PwArgs a;
            // pointwise order: u v w phi phx phy phz exx eyy exy exz eyz  <-  buffers 0 1 2 3 10 11 4 5 6 7 8 9
            //                                                            (matched viscosity: 0 1 2 3 6 5 4)
            const int order_v[MAXF] = {0, 1, 2, 3, 10, 11, 4, 5, 6, 7, 8, 9};
            const int order_m[MAXF] = {0, 1, 2, 3, 6, 5, 4, 0, 0, 0, 0, 0};
            // alternative forms: u v w phi phx phy phz lap wx wy wz  <-  Z/Y/physical buffers as laid out above
            int order_f[MAXF] = {0, 1, 2, 3, 0, 0, 4, 0, 0, 0, 0, 0};
            if (force) {
                if (phase) {
                    int nb = 5;
                    if (st_force) order_f[7] = nb++;
                    if (rot) for (int i = 0; i < 3; ++i) order_f[8 + i] = nb++;
                    order_f[5] = nb; order_f[4] = nb + 1;       // i ky phi, i kx phi
                } else {
                    for (int i = 0; i < 3; ++i) order_f[8 + i] = 3 + i;
                }
            }
            for (int i = 0; i < MAXF; ++i)
                a.b[i] = h->at<double>(L.ph[force ? order_f[i] : (phase ? (visc ? order_v[i] : order_m[i]) : (i < 3 ? i : 0))]);
            for (int i = 0; i < 10; ++i) a.o[i] = h->at<double>(L.ph[i < nout ? i : 0]);
            a.n = d.s_p; a.cs = c.cs; a.eta_c = (p.visc_ratio - 1.0) / (2.0 * p.re);
            a.phase = phase; a.visc = visc; a.force = force; a.st_force = st_force; a.rot = rot;
            LaunchScope ls(h, KC_PW);
            k_pointwise<<<h->n_sm * 8, 256, 0, h->st>>>(a);
            CU(cudaGetLastError());
        }
        for (int i = 0; i < nout; ++i) { gx.in[i] = h->at<double>(L.ph[i]); gx.out[i] = h->at<cplx>(L.yb[i]); }
        CU(launch_xpass(h, true, gx, nout, d.kxp, d.nkx));
    }
    // a7-a8: forward y, z with truncation
    CU(launch_ypass(h, true, gy, nout, d.kxp, d.nky, d.jpos));
    CU(launch_zpass(h, true, gz, nout, d.ncols, d.nkz, d.kxp, d.nky, d.jpos));
    // a9 + first elimination (K_A), substitution (K_B), second elimination (K_C), substitution +
    // influence-matrix correction (K_D), velocity recovery (a11)
    const double inv_g = 1.0 / c.gamma;
    const bool la2 = d.ncols > 60000;   // register look-ahead depth of the solver sweeps (kernels_spectral.cuh)
    const bool walls_gen = p.wall_top != 0 || p.wall_bottom != 0;   // free-slip or mixed walls (row f3)
    // phi problem in three sweeps: its second solve is eliminated upwards inside the first substitution (psi never stored)
    // and back-substituted by k_finish on its way down (ElimUpNeu); phi3 = 0 keeps the five-sweep form for cross-checks
    const bool phi3 = phase && h->phi3;
    // w problem likewise (ElimUpDir2): the solver stage is then three launches - k_rhs_elim (down),
    // k_subst3 (up), k_finish (down) - instead of five
    const bool w3 = h->w3 && (!phase || phi3);
    const bool lazy = w3 && h->lazy;   // theta^'s influence-matrix correction deferred to the next step's k_rhs_elim
    const double *dNS = h->at<double>(L.dinv[0]), *dPO = h->at<double>(L.dinv[1]), *dCH = h->at<double>(L.dinv[2]);
    {
        RhsElimArgs a;
        a.g = geom(h);
        a.txx = h->at<cplx>(L.prod[0]); a.txy = h->at<cplx>(L.prod[1]); a.txz = h->at<cplx>(L.prod[2]);
        a.tyy = h->at<cplx>(L.prod[3]); a.tyz = h->at<cplx>(L.prod[4]);
        a.q = h->at<cplx>(L.prod[5]); a.c = h->at<cplx>(L.prod[6]);
        a.fx = force ? h->at<cplx>(L.prod[7]) : nullptr; a.fy = force ? h->at<cplx>(L.prod[8]) : nullptr;
        a.fz = force ? h->at<cplx>(L.prod[9]) : nullptr;
        a.om = OM; a.th = TH; a.phi = PHI;
        a.h_om = h->at<cplx>(L.hist[0]); a.h_w = h->at<cplx>(L.hist[1]); a.h_phi = h->at<cplx>(L.hist[2]);
        a.dinv_ns = dNS; a.dinv_ch = dCH;
        a.ab = ab; a.dt = p.dt; a.gamma = c.gamma; a.inv_pe = phase ? 1.0 / p.pe : 0.0;
        a.e_phi = 1.0 + c.s_coef * p.ch * p.ch;
        a.gradp = p.gradp_x; a.lam_phi = c.lam_phi; a.gam_phi = c.gam_phi; a.phase = phase;
        a.wall_top = p.wall_top; a.wall_bot = p.wall_bottom;
        a.thh = h->at<double>(L.thh); a.coef = h->at<cplx>(L.coef);
        const int grid = (int)((d.ncols + RHS_COLS - 1) / RHS_COLS);
        LaunchScope ls(h, KC_RHS);
        const int nt = 32 * (phase ? 3 : 2);
        // lazy: theta^n is still the particular solution of the last step; its influence-matrix correction is applied here
        if (lazy) {
            if (force) { if (walls_gen) k_rhs_elim<true, true, true><<<grid, nt, 0, h->st>>>(a); else k_rhs_elim<false, true, true><<<grid, nt, 0, h->st>>>(a); }
            else if (walls_gen) k_rhs_elim<true, false, true><<<grid, nt, 0, h->st>>>(a);
            else k_rhs_elim<false, false, true><<<grid, nt, 0, h->st>>>(a);
        }
        else if (force) { if (walls_gen) k_rhs_elim<true, true><<<grid, nt, 0, h->st>>>(a); else k_rhs_elim<false, true><<<grid, nt, 0, h->st>>>(a); }
        else if (walls_gen) k_rhs_elim<true, false><<<grid, nt, 0, h->st>>>(a);
        else k_rhs_elim<false, false><<<grid, nt, 0, h->st>>>(a);
        CU(cudaGetLastError());
    }
    {
        SubstArgs a;
        a.g = geom(h);
        a.x[0] = OM; a.x[1] = TH; a.x[2] = PHI;
        a.dinv[0] = dNS; a.dinv[1] = dNS; a.dinv[2] = dCH;
        a.shift[0] = inv_g; a.shift[1] = inv_g; a.shift[2] = c.lam_phi;
        a.nchains = phase ? 3 : 2;
        a.pair01 = 1;
        a.coef = nullptr; a.wh = nullptr; a.thh = nullptr; a.th = nullptr;
        a.w3_out = W; a.w3_hw = h->at<double>(L.hw); a.w3_coef = h->at<cplx>(L.coef);
        a.wall_top = p.wall_top; a.wall_bot = p.wall_bottom;
        LaunchScope ls(h, KC_SOLVE);
        const dim3 g1(col_grid(d), phi3 ? 1 : a.nchains - 1);
        if (w3) {
            const dim3 g3(col_grid(d), phase ? 2 : 1);
            if (walls_gen) { if (la2) k_subst3<2, true><<<g3, NT_COL, 0, h->st>>>(a); else k_subst3<4, true><<<g3, NT_COL, 0, h->st>>>(a); }
            else if (la2) k_subst3<2><<<g3, NT_COL, 0, h->st>>>(a); else k_subst3<4><<<g3, NT_COL, 0, h->st>>>(a);
        }
        else if (la2) k_subst<2><<<g1, NT_COL, 0, h->st>>>(a);
        else k_subst<4><<<g1, NT_COL, 0, h->st>>>(a);
        CU(cudaGetLastError());

    }
    if (!w3) {
        Elim2Args a;
        a.g = geom(h); a.th = TH; a.w = W; a.phi = PHI; a.dinv_po = dPO; a.dinv_ch = dCH;
        a.hw = h->at<double>(L.hw); a.coef = h->at<cplx>(L.coef); a.lam_phi = c.lam_phi; a.phase = phase;
        a.wall_top = p.wall_top; a.wall_bot = p.wall_bottom;
        LaunchScope ls(h, KC_SOLVE);
        const dim3 g2(col_grid(d), phase ? 2 : 1);
        if (phi3) {   // block row 1: the psi chain's up sweep feeding the upward elimination of the phi solve
            SubstArgs b;
            b.g = a.g;
            b.x[0] = nullptr; b.x[1] = nullptr; b.x[2] = PHI;
            b.dinv[0] = nullptr; b.dinv[1] = nullptr; b.dinv[2] = dCH;
            b.shift[0] = 0.0; b.shift[1] = 0.0; b.shift[2] = c.lam_phi;
            b.nchains = 3; b.pair01 = 1;
            b.coef = nullptr; b.wh = nullptr; b.thh = nullptr; b.th = nullptr;
            b.w3_out = nullptr; b.w3_hw = nullptr; b.w3_coef = nullptr; b.wall_top = 0; b.wall_bot = 0;
            if (walls_gen) { if (la2) k_elim2up<2, true><<<g2, NT_COL, 0, h->st>>>(a, b); else k_elim2up<4, true><<<g2, NT_COL, 0, h->st>>>(a, b); }
            else if (la2) k_elim2up<2, false><<<g2, NT_COL, 0, h->st>>>(a, b);
            else k_elim2up<4, false><<<g2, NT_COL, 0, h->st>>>(a, b);
        }
        else if (walls_gen) { if (la2) k_elim2<2, true><<<g2, NT_COL, 0, h->st>>>(a); else k_elim2<4, true><<<g2, NT_COL, 0, h->st>>>(a); }
        else if (la2) k_elim2<2, false><<<g2, NT_COL, 0, h->st>>>(a);
        else k_elim2<4, false><<<g2, NT_COL, 0, h->st>>>(a);
        CU(cudaGetLastError());
    }
    if (!w3) {
        SubstArgs a;
        a.g = geom(h);
        a.x[0] = W; a.x[1] = PHI; a.x[2] = nullptr;
        a.dinv[0] = dPO; a.dinv[1] = dCH; a.dinv[2] = nullptr;
        a.shift[0] = 0.0; a.shift[1] = c.lam_phi; a.shift[2] = 0.0;
        a.nchains = (phase && !phi3) ? 2 : 1;
        a.pair01 = 0;
        a.coef = h->at<cplx>(L.coef); a.wh = h->at<double>(L.wh); a.thh = h->at<double>(L.thh); a.th = TH;
        a.w3_out = nullptr; a.w3_hw = nullptr; a.w3_coef = nullptr; a.wall_top = 0; a.wall_bot = 0;
        LaunchScope ls(h, KC_SOLVE);
        if (la2) k_subst<2><<<dim3(col_grid(d), a.nchains), NT_COL, 0, h->st>>>(a);
        else k_subst<4><<<dim3(col_grid(d), a.nchains), NT_COL, 0, h->st>>>(a);
        CU(cudaGetLastError());
    }
    // a11: u^, v^ (and D phi^ for the next step)
    {
        FinishArgs a;
        a.g = geom(h); a.om = OM; a.th = TH; a.u = U; a.v = V; a.w = W;
        a.phi = phase ? PHI : nullptr; a.phz = PHZ;
        a.tab_phi = phi3 ? h->at<double2>(L.tab_phi) : nullptr;
        a.tab_w = h->at<double2>(L.tab_w); a.wh = h->at<double>(L.wh); a.thh = h->at<double>(L.thh);
        a.coef = h->at<cplx>(L.coef); a.th_rw = TH;
        LaunchScope ls(h, KC_SOLVE);
        // look-ahead 2 at every size: 4 rows of this kernel's eleven operand streams do not fit in registers (measured at
        // 1024x512x513 / 256x256x257, solve stage: depth 1 3.85-3.91 / 0.29-0.30 ms, depth 2 3.74-3.77 / 0.25 ms)
        if (w3 && lazy) k_finish<2, true, true><<<col_grid(d), NT_COL, 0, h->st>>>(a);
        else if (w3) k_finish<2, true><<<col_grid(d), NT_COL, 0, h->st>>>(a);
        else if (la2) k_finish<2><<<col_grid(d), NT_COL, 0, h->st>>>(a);
        else k_finish<4><<<col_grid(d), NT_COL, 0, h->st>>>(a);
        CU(cudaGetLastError());
    }
    return cudaSuccess;
}

cudaError_t build_tables(psdns_handle *h) {
    const Dims &d = h->d;
    const Layout &L = h->L;
    // twiddles exp(-2 pi i k / L) in long double on the host
    auto fill = [&](size_t off, int n) -> cudaError_t {
        std::vector<cplx> t(n);
        for (int k = 0; k < n; ++k) {
            const long double ang = -2.0L * 3.14159265358979323846264338327950288L * (long double)k / (long double)n;
            t[k] = make_double2((double)cosl(ang), (double)sinl(ang));
        }
        // exact values on the axes
        t[0] = make_double2(1.0, 0.0);
        if (n % 4 == 0) { t[n / 4] = make_double2(0.0, -1.0); t[n / 2] = make_double2(-1.0, 0.0); t[3 * n / 4] = make_double2(0.0, 1.0); }
        cudaError_t e = cudaMemcpyAsync(h->ws + off, t.data(), n * sizeof(cplx), cudaMemcpyHostToDevice, h->st);
        if (e != cudaSuccess) return e;
        return cudaStreamSynchronize(h->st);   // t goes out of scope
    };
    CU(fill(L.tw_x, d.nx));
    CU(fill(L.tw_y, d.ny));
    CU(fill(L.tw_z, 2 * d.N));
    CU(fill(L.tw_zn, d.N));
    {   // c_k = -(1 + sin t)/(2 sin t) + i cos t/(2 sin t), t = pi k / N  (kernels_transform.cuh, k_zpass_h)
        std::vector<cplx> t(d.N / 2 + 1);
        t[0] = make_double2(0.0, 0.0);
        for (int k = 1; k <= d.N / 2; ++k) {
            const long double th = 3.14159265358979323846264338327950288L * (long double)k / (long double)d.N;
            const long double sn = sinl(th), cs = cosl(th);
            t[k] = make_double2((double)(-(1.0L + sn) / (2.0L * sn)), (double)(cs / (2.0L * sn)));
        }
        CU(cudaMemcpyAsync(h->ws + L.ctab_z, t.data(), t.size() * sizeof(cplx), cudaMemcpyHostToDevice, h->st));
        CU(cudaStreamSynchronize(h->st));
    }
    if (d.N <= 64) {   // GEMM-form Chebyshev matrices (kernels_zgemm.cuh), long double on the host
        std::vector<double> mb(ZG_MP * ZG_KP, 0.0), mf(ZG_MP * ZG_KP, 0.0);
        const long double pi = 3.14159265358979323846264338327950288L;
        for (int k = 0; k <= d.N; ++k)
            for (int n = 0; n <= d.N; ++n) {
                const long double cs = cosl(pi * (long double)((long long)n * k % (2 * d.N)) / (long double)d.N);
                mb[k * ZG_KP + n] = (double)cs;                                              // f_k = sum_n a_n cos(pi n k / N)
                const long double cn = (n == 0 || n == d.N) ? 2.0L : 1.0L, ck = (k == 0 || k == d.N) ? 2.0L : 1.0L;
                mf[n * ZG_KP + k] = (double)(2.0L * cs / ((long double)d.N * cn * ck));      // a_n = 2/(N c_n) sum_k f_k cos / c_k
            }
        CU(cudaMemcpyAsync(h->ws + L.zg_b, mb.data(), mb.size() * sizeof(double), cudaMemcpyHostToDevice, h->st));
        CU(cudaMemcpyAsync(h->ws + L.zg_f, mf.data(), mf.size() * sizeof(double), cudaMemcpyHostToDevice, h->st));
        CU(cudaStreamSynchronize(h->st));
    }
    {   // Gauss-Lobatto points z_k = cos(pi k / N) (ray-caster)
        std::vector<double> t(d.nz);
        for (int k = 0; k <= d.N; ++k) t[k] = (double)cosl(3.14159265358979323846264338327950288L * (long double)k / (long double)d.N);
        t[0] = 1.0; t[d.N] = -1.0; t[d.N / 2] = 0.0;
        CU(cudaMemcpyAsync(h->ws + L.znodes, t.data(), t.size() * sizeof(double), cudaMemcpyHostToDevice, h->st));
        CU(cudaStreamSynchronize(h->st));
    }
    {   // Clenshaw-Curtis weights w_k = (c_k / N) [1 - sum_{j=1}^{N/2} b_j cos(2 j k pi / N) / (4 j^2 - 1)], b_{N/2} = 1 else 2,
        // c_0 = c_N = 1 else 2 (N even): exact for polynomials of degree <= N on the Gauss-Lobatto points
        std::vector<double> t(d.nz);
        const long double pi = 3.14159265358979323846264338327950288L;
        for (int k = 0; k <= d.N; ++k) {
            long double acc = 1.0L;
            for (int j = 1; j <= d.N / 2; ++j)
                acc -= (j == d.N / 2 ? 1.0L : 2.0L) * cosl(2.0L * pi * (long double)j * (long double)k / (long double)d.N) /
                       (4.0L * (long double)j * (long double)j - 1.0L);
            t[k] = (double)(((k == 0 || k == d.N) ? 1.0L : 2.0L) * acc / (long double)d.N);
        }
        CU(cudaMemcpyAsync(h->ws + L.ccw, t.data(), t.size() * sizeof(double), cudaMemcpyHostToDevice, h->st));
        CU(cudaStreamSynchronize(h->st));
    }
    {   // p_k, q_k, r_k of the quasi-tridiagonal recurrence (kernels_spectral.cuh), k-only: constant memory
        static double hp[HELM_KMAX + 1], hq[HELM_KMAX + 1], hr[HELM_KMAX + 1];
        for (int k = 0; k <= HELM_KMAX; ++k) { hp[k] = helm_p_host(k); hq[k] = helm_q_host(k); hr[k] = helm_r_host(k); }
        CU(cudaMemcpyToSymbolAsync(c_helm_p, hp, sizeof(hp), 0, cudaMemcpyHostToDevice, h->st));
        CU(cudaMemcpyToSymbolAsync(c_helm_q, hq, sizeof(hq), 0, cudaMemcpyHostToDevice, h->st));
        CU(cudaMemcpyToSymbolAsync(c_helm_r, hr, sizeof(hr), 0, cudaMemcpyHostToDevice, h->st));
        CU(cudaStreamSynchronize(h->st));
    }
    const Coefs c = coefs(h->p);
    const double shifts[3] = {1.0 / c.gamma, 0.0, c.lam_phi};
    for (int t = 0; t < 3; ++t) {
        HelmSetupArgs a;
        a.g = geom(h); a.dinv = h->at<double>(L.dinv[t]); a.shift = shifts[t];
        LaunchScope ls(h, KC_MISC);
        k_helm_setup<<<col_grid(d), NT_COL, 0, h->st>>>(a);
        CU(cudaGetLastError());
    }
    for (int t = 0; t < 2; ++t) {   // down-sweep tables of the upward eliminations (kernels_spectral.cuh, ElimUpNeu / ElimUpDir2)
        if (t == 0 && !h->p.phase_field) continue;
        ElimUpSetupArgs a;
        a.g = geom(h); a.tab = h->at<double2>(t == 0 ? L.tab_phi : L.tab_w); a.shift = t == 0 ? c.lam_phi : 0.0;
        LaunchScope ls(h, KC_MISC);
        k_elimup_setup<<<col_grid(d), NT_COL, 0, h->st>>>(a);
        CU(cudaGetLastError());
    }
    // homogeneous solutions of the w problem: theta_h = Helmholtz(beta^2) with zero rhs and unit boundary
    // targets in both parities; w_h = Poisson(k^2) of theta_h with w_h(+-1) = 0.  Solved as complex in
    // scratch, then kept as real tables together with sum k^2 w_h per parity.
    cplx *thh_c = h->at<cplx>(L.zb[0]), *wh_c = h->at<cplx>(L.zb[1]);
    CU(cudaMemsetAsync(thh_c, 0, d.s_ret * sizeof(cplx), h->st));
    CU(launch_helm(h, thh_c, thh_c, 0, shifts[0], 1.0, BC_DIRICHLET, 1.0, 1.0));
    CU(launch_helm(h, thh_c, wh_c, 1, 0.0, 1.0, BC_DIRICHLET, 0.0, 0.0));
    {
        LaunchScope ls(h, KC_MISC);
        k_hom_tables<<<col_grid(d), NT_COL, 0, h->st>>>(geom(h), thh_c, wh_c, h->at<double>(L.thh), h->at<double>(L.wh),
                                                        h->at<double>(L.hw));
        CU(cudaGetLastError());
    }
    return cudaSuccess;
}

int finish_set_state(psdns_handle *h) {
    const Dims &d = h->d;
    const Layout &L = h->L;
    {
        LaunchScope ls(h, KC_MISC);
        k_hidden_state<<<col_grid(d), NT_COL, 0, h->st>>>(geom(h), h->at<cplx>(L.state[0]), h->at<cplx>(L.state[1]),
                                                          h->at<cplx>(L.state[2]), h->at<cplx>(L.state[4]),
                                                          h->at<cplx>(L.xom));
        CUDA_TRY(h, cudaGetLastError());
    }
    if (h->p.phase_field) {   // D phi^ for the first step (k_finish maintains it afterwards)
        PrepArgs a{};
        a.g = geom(h); a.phi = h->at<cplx>(L.state[3]); a.phz = h->at<cplx>(L.derived[0]);
        a.do_phz = 1; a.visc = 0;
        LaunchScope ls(h, KC_MISC);
        k_prep<<<col_grid(d), NT_COL, 0, h->st>>>(a);
        CUDA_TRY(h, cudaGetLastError());
    }
    for (int i = 0; i < 3; ++i) CUDA_TRY(h, cudaMemsetAsync(h->ws + L.hist[i], 0, d.s_low * sizeof(cplx), h->st));
    CUDA_TRY(h, cudaMemsetAsync(h->ws + L.small, 0, 64, h->st));
    CUDA_TRY(h, cudaMemsetAsync(h->ws + L.coef, 0, 2 * d.ncols * sizeof(cplx), h->st));   // no pending theta correction
    h->th_pending = false;
    h->has_state = true;
    return PSDNS_OK;
}

// theta^ of the three-sweep form is corrected lazily (k_rhs_elim<., ., true>); whoever needs the array itself calls this
int materialise_theta(psdns_handle *h) {
    if (!h->th_pending) return PSDNS_OK;
    LaunchScope ls(h, KC_MISC);
    k_theta_apply<<<col_grid(h->d), NT_COL, 0, h->st>>>(geom(h), h->at<cplx>(h->L.state[4]), h->at<double>(h->L.thh),
                                                      h->at<cplx>(h->L.coef));
    CUDA_TRY(h, cudaGetLastError());
    h->th_pending = false;
    return PSDNS_OK;
}

}  // namespace

// ================================================================================================
// C ABI
// ================================================================================================
extern "C" {

size_t psdns_workspace_bytes(const psdns_grid *grid, const psdns_params *params) {
    if (!validate(grid, params)) return 0;
    return make_layout(make_dims(*grid), *params).total;
}

size_t psdns_workspace_bytes_unfused(const psdns_grid *grid, const psdns_params *params) {
    if (!validate(grid, params)) return 0;
    return make_layout(make_dims(*grid), *params).total_unfused;
}

int psdns_init(const psdns_grid *grid, const psdns_params *params, void *d_workspace, size_t bytes, void *cuda_stream,
               psdns_handle **out) {
    if (!out) return PSDNS_EINVAL;
    *out = nullptr;
    if (!validate(grid, params) || !d_workspace) return PSDNS_EINVAL;
    psdns_handle *h = new (std::nothrow) psdns_handle();
    if (!h) return PSDNS_ENOMEM;
    h->g = *grid; h->p = *params; h->st = (cudaStream_t)cuda_stream;
    h->d = make_dims(*grid);
    h->L = make_layout(h->d, *params);
    h->ws = (char *)d_workspace;
    h->has_state = false; h->graph = nullptr; h->graph_ready = false;
    h->use_graph = true;
    h->use_xfused = true;
    h->copy_st = nullptr; h->copy_in_st = nullptr; h->ev_out_ready = nullptr; h->ev_d2h_done = nullptr; h->d2h_pending = false;
    h->ev_in_ready = nullptr; h->ev_in_free[0] = h->ev_in_free[1] = nullptr; h->in_used[0] = h->in_used[1] = false; h->host_calls = 0;
    h->grid_cap = 0; h->pf = 2; h->pf_rhs = 4;
    h->use_ztma = 1; h->encode_tiled = nullptr; h->use_zgemm = 0;
    for (int i = 0; i < 4; ++i) (&h->occ_zt[0][0])[i] = 1;
    {   // driver entry point of the tensor-map encoder (no link-time dependency on libcuda)
        void *fn = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) == cudaSuccess &&
            qres == cudaDriverEntryPointSuccess)
            h->encode_tiled = reinterpret_cast<PFN_cuTensorMapEncodeTiled>(fn);
        else
            cudaGetLastError();
    }
    for (int i = 0; i < KC_COUNT; ++i) { h->last_grid[i] = 0; h->last_items[i] = 0; }
    h->launches = 0; h->per_step = 0; h->timed_class = -1;
    const bool phase = params->phase_field != 0;
    const bool visc = phase && params->visc_ratio != 1.0;
    const bool force = (phase && params->surface_tension_form == 1) || params->convection_form == 1;
    h->nf_in = phase ? (visc ? 12 : (force ? 11 : 7)) : (force ? 6 : 3);
    h->nf_out = phase ? (force ? 10 : 7) : (force ? 10 : 5);
    if (force) h->use_xfused = false;   // three-kernel x path (k_xpass, k_pointwise, k_xpass): 10 forward fields exceed the fused tile
    h->xf_occ = 1; h->xfv_occ = 1; h->n_sm = 148;
    h->occ_z[0] = h->occ_z[1] = h->occ_y[0] = h->occ_y[1] = 1;
    {
        int dev = 0, nsm = 0;
        if (cudaGetDevice(&dev) == cudaSuccess && cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess && nsm > 0)
            h->n_sm = nsm;
    }
    if (bytes < h->L.total || ((uintptr_t)d_workspace % ALIGN) != 0) { delete h; return PSDNS_ENOMEM; }
    h->has_unfused_ws = bytes >= h->L.total_unfused || force;
    cudaError_t e = setup_attrs(h);
    if (e == cudaSuccess) e = build_tables(h);
    if (e != cudaSuccess) {
        // the handle is returned so that the caller can read the error text, then destroy it
        h->err = std::string("psdns_init: ") + cudaGetErrorString(e);
        *out = h;
        return PSDNS_ECUDA;
    }
    *out = h;
    return PSDNS_OK;
}

int psdns_set_state(psdns_handle *h, int space, const void *d_u, const void *d_v, const void *d_w, const void *d_phi) {
    if (!h) return PSDNS_EINVAL;
    const bool phase = h->p.phase_field != 0;
    if (!d_u || !d_v || !d_w || (phase && !d_phi) || (space != PSDNS_PHYSICAL && space != PSDNS_SPECTRAL)) {
        h->err = "psdns_set_state: null field pointer or bad space";
        return PSDNS_EINVAL;
    }
    const Dims &d = h->d;
    const Layout &L = h->L;
    const void *src[4] = {d_u, d_v, d_w, d_phi};
    const int nf = phase ? 4 : 3;
    if (!phase) CUDA_TRY(h, cudaMemsetAsync(h->ws + L.state[3], 0, d.s_ret * sizeof(cplx), h->st));
    if (space == PSDNS_SPECTRAL) {
        for (int i = 0; i < nf; ++i)
            CUDA_TRY(h, launch_relayout(h, h->at<cplx>(L.state[i]), (const cplx *)src[i], side_ret(d), side_boundary(d), d.nz));
    } else {
        // step i) (L138): forward transform x -> y -> z, keeping retained (kx, ky) and all nz Chebyshev modes
        FieldPtrs fx{}, fy{}, fz{};
        for (int i = 0; i < nf; ++i) {
            fx.in[i] = src[i]; fx.out[i] = h->at<cplx>(L.yb[i]);
            fy.in[i] = fx.out[i]; fy.out[i] = h->at<cplx>(L.zb[i]);
            fz.in[i] = fy.out[i]; fz.out[i] = h->at<cplx>(L.state[i]);
        }
        CUDA_TRY(h, launch_xpass(h, true, fx, nf, d.kxp, d.nkx));
        CUDA_TRY(h, launch_ypass(h, true, fy, nf, d.kxp, d.nky, d.jpos));
        CUDA_TRY(h, launch_zpass(h, true, fz, nf, d.ncols, d.nz, d.kxp, d.nky, d.jpos));
    }
    return finish_set_state(h);
}

int psdns_get_state(psdns_handle *h, int space, void *d_u, void *d_v, void *d_w, void *d_phi) {
    if (!h) return PSDNS_EINVAL;
    const bool phase = h->p.phase_field != 0;
    if (!d_u || !d_v || !d_w || (phase && !d_phi) || (space != PSDNS_PHYSICAL && space != PSDNS_SPECTRAL)) {
        h->err = "psdns_get_state: null field pointer or bad space";
        return PSDNS_EINVAL;
    }
    if (!h->has_state) { h->err = "psdns_get_state: no state set"; return PSDNS_ESTATE; }
    const Dims &d = h->d;
    const Layout &L = h->L;
    void *dst[4] = {d_u, d_v, d_w, d_phi};
    const int nf = phase ? 4 : 3;
    if (space == PSDNS_SPECTRAL) {
        for (int i = 0; i < nf; ++i)
            CUDA_TRY(h, launch_relayout(h, (cplx *)dst[i], h->at<cplx>(L.state[i]), side_boundary(d), side_ret(d), d.nz));
    } else {
        FieldPtrs fz{}, fy{}, fx{};
        for (int i = 0; i < nf; ++i) {
            fz.in[i] = h->at<cplx>(L.state[i]); fz.out[i] = h->at<cplx>(L.zb[i]);
            fy.in[i] = fz.out[i]; fy.out[i] = h->at<cplx>(L.yb[i]);
            fx.in[i] = fy.out[i]; fx.out[i] = dst[i];
        }
        CUDA_TRY(h, launch_zpass(h, false, fz, nf, d.ncols, d.nz, d.kxp, d.nky, d.jpos));
        CUDA_TRY(h, launch_ypass(h, false, fy, nf, d.kxp, d.nky, d.jpos));
        CUDA_TRY(h, launch_xpass(h, false, fx, nf, d.kxp, d.nkx));
    }
    return PSDNS_OK;
}

int psdns_step(psdns_handle *h, int nsteps) {
    if (!h) return PSDNS_EINVAL;
    if (nsteps < 0) { h->err = "psdns_step: nsteps < 0"; return PSDNS_EINVAL; }
    if (!h->p.dealias) { h->err = "psdns_step: dealias must be 1 (2/3 rule, reading S3)"; return PSDNS_EINVAL; }
    if (!h->has_state) { h->err = "psdns_step: no state set"; return PSDNS_ESTATE; }
    // the three-sweep solver with the lazy correction leaves theta^ as theta_p + (its coefficients): see materialise_theta
    if (nsteps > 0 && h->lazy && h->w3 && (!h->p.phase_field || h->phi3)) h->th_pending = true;
    const bool direct = !h->use_graph || h->timed_class >= 0;
    if (direct) {
        for (int i = 0; i < nsteps; ++i) CUDA_TRY(h, enqueue_step(h));
        return PSDNS_OK;
    }
    if (!h->graph_ready) {
        // run one un-captured step's worth of attribute setup first (cudaFuncSetAttribute is not capturable
        // on every driver): do the capture on a private stream so a failure leaves the user's stream clean
        cudaStream_t user = h->st, cap;
        CUDA_TRY(h, cudaStreamCreateWithFlags(&cap, cudaStreamNonBlocking));
        cudaGraph_t graph = nullptr;
        h->st = cap;
        const long long before = h->launches;
        cudaError_t e = cudaStreamBeginCapture(cap, cudaStreamCaptureModeThreadLocal);
        if (e == cudaSuccess) e = enqueue_step(h);
        cudaError_t e2 = cudaStreamEndCapture(cap, &graph);
        h->st = user;
        h->per_step = h->launches - before;
        h->launches = before;
        if (e == cudaSuccess) e = e2;
        if (e == cudaSuccess) e = cudaGraphInstantiate(&h->graph, graph, 0);
        if (graph) cudaGraphDestroy(graph);
        cudaStreamDestroy(cap);
        if (e != cudaSuccess) {
            cudaGetLastError();
            h->use_graph = false;   // fall back to direct launches (same kernels)
            for (int i = 0; i < nsteps; ++i) CUDA_TRY(h, enqueue_step(h));
            return PSDNS_OK;
        }
        h->graph_ready = true;
    }
    for (int i = 0; i < nsteps; ++i) {
        CUDA_TRY(h, cudaGraphLaunch(h->graph, h->st));
        h->launches += h->per_step;
    }
    return PSDNS_OK;
}

int psdns_transform_roundtrip(psdns_handle *h, int start_space, const void *d_in, void *d_out, void *d_mid) {
    if (!h) return PSDNS_EINVAL;
    if (!d_in || !d_out || (start_space != PSDNS_PHYSICAL && start_space != PSDNS_SPECTRAL)) {
        h->err = "psdns_transform_roundtrip: null pointer or bad space";
        return PSDNS_EINVAL;
    }
    const Dims &d = h->d;
    const Layout &L = h->L;
    // full-size scratch aliases the Z/Y transform buffers
    cplx *A = h->at<cplx>(L.zb[0]);
    cplx *B = reinterpret_cast<cplx *>(reinterpret_cast<char *>(A) + align_up(d.s_full * sizeof(cplx)));
    cplx *C = reinterpret_cast<cplx *>(reinterpret_cast<char *>(B) + align_up(d.s_full * sizeof(cplx)));
    const size_t ncols_f = (size_t)d.ny * d.kxpf;
    auto forward = [&](const double *phys, cplx *spec_boundary) -> int {
        FieldPtrs f{};
        f.in[0] = phys; f.out[0] = A;
        CUDA_TRY(h, launch_xpass(h, true, f, 1, d.kxpf, d.nkxf));
        f.in[0] = A; f.out[0] = B;
        CUDA_TRY(h, launch_ypass(h, true, f, 1, d.kxpf, d.ny, d.ny));
        f.in[0] = B; f.out[0] = C;
        CUDA_TRY(h, launch_zpass(h, true, f, 1, ncols_f, d.nz, d.kxpf, d.ny, d.ny));
        // the boundary-layout copy of the spectrum is only made when somebody looks at it (d_mid / spectral output)
        if (spec_boundary) CUDA_TRY(h, launch_relayout(h, spec_boundary, C, side_boundary(d), side_full(d), d.nz));
        return PSDNS_OK;
    };
    auto backward = [&](const cplx *spec_boundary, double *phys) -> int {
        if (spec_boundary) CUDA_TRY(h, launch_relayout(h, C, spec_boundary, side_full(d), side_boundary(d), d.nz));
        FieldPtrs f{};
        f.in[0] = C; f.out[0] = B;
        CUDA_TRY(h, launch_zpass(h, false, f, 1, ncols_f, d.nz, d.kxpf, d.ny, d.ny));
        f.in[0] = B; f.out[0] = A;
        CUDA_TRY(h, launch_ypass(h, false, f, 1, d.kxpf, d.ny, d.ny));
        f.in[0] = A; f.out[0] = phys;
        CUDA_TRY(h, launch_xpass(h, false, f, 1, d.kxpf, d.nkxf));
        return PSDNS_OK;
    };
    int rc;
    if (start_space == PSDNS_PHYSICAL) {
        // without d_mid the spectrum stays in the private layout between the two transforms (same values, two copies less)
        cplx *mid = (cplx *)d_mid;
        if ((rc = forward((const double *)d_in, mid)) != PSDNS_OK) return rc;
        if ((rc = backward(mid, (double *)d_out)) != PSDNS_OK) return rc;
    } else {
        double *mid = d_mid ? (double *)d_mid : h->at<double>(L.stage[0]);
        if ((rc = backward((const cplx *)d_in, mid)) != PSDNS_OK) return rc;
        if ((rc = forward(mid, (cplx *)d_out)) != PSDNS_OK) return rc;
    }
    return PSDNS_OK;
}

// hidden-state blob: theta | omega_z | D phi | N_omega | N_w | S_phi | (ab[2], counter) - each piece 256-byte aligned
namespace {
struct HistPiece { size_t off, bytes; };
int hist_pieces(const psdns_handle *h, HistPiece *pc) {
    const Dims &d = h->d;
    const Layout &L = h->L;
    int n = 0;
    pc[n++] = {L.state[4], d.s_ret * sizeof(cplx)};
    pc[n++] = {L.xom, d.s_ret * sizeof(cplx)};
    pc[n++] = {L.derived[0], d.s_low * sizeof(cplx)};
    for (int i = 0; i < 3; ++i) pc[n++] = {L.hist[i], d.s_low * sizeof(cplx)};
    pc[n++] = {L.small, 64};
    return n;
}
}  // namespace

size_t psdns_history_bytes(const psdns_handle *h) {
    if (!h) return 0;
    HistPiece pc[8];
    const int n = hist_pieces(h, pc);
    size_t tot = 0;
    for (int i = 0; i < n; ++i) tot += align_up(pc[i].bytes);
    return tot;
}

int psdns_get_history(psdns_handle *h, void *d_blob, size_t bytes) {
    if (!h) return PSDNS_EINVAL;
    if (!d_blob || bytes != psdns_history_bytes(h)) { h->err = "psdns_get_history: null blob or size mismatch"; return PSDNS_EINVAL; }
    if (!h->has_state) { h->err = "psdns_get_history: no state set"; return PSDNS_ESTATE; }
    { const int rc = materialise_theta(h); if (rc != PSDNS_OK) return rc; }
    HistPiece pc[8];
    const int n = hist_pieces(h, pc);
    size_t o = 0;
    for (int i = 0; i < n; ++i) {
        CUDA_TRY(h, cudaMemcpyAsync((char *)d_blob + o, h->ws + pc[i].off, pc[i].bytes, cudaMemcpyDeviceToDevice, h->st));
        o += align_up(pc[i].bytes);
    }
    return PSDNS_OK;
}

int psdns_set_history(psdns_handle *h, const void *d_blob, size_t bytes) {
    if (!h) return PSDNS_EINVAL;
    if (!d_blob || bytes != psdns_history_bytes(h)) { h->err = "psdns_set_history: null blob or size mismatch"; return PSDNS_EINVAL; }
    if (!h->has_state) { h->err = "psdns_set_history: call psdns_set_state first"; return PSDNS_ESTATE; }
    HistPiece pc[8];
    const int n = hist_pieces(h, pc);
    size_t o = 0;
    for (int i = 0; i < n; ++i) {
        CUDA_TRY(h, cudaMemcpyAsync(h->ws + pc[i].off, (const char *)d_blob + o, pc[i].bytes, cudaMemcpyDeviceToDevice, h->st));
        o += align_up(pc[i].bytes);
    }
    CUDA_TRY(h, cudaMemsetAsync(h->ws + h->L.coef, 0, 2 * h->d.ncols * sizeof(cplx), h->st));   // the blob's theta^ is complete
    h->th_pending = false;
    return PSDNS_OK;
}

int psdns_run_host(psdns_handle *h, int space, int nsteps, const void *h_in_u, const void *h_in_v, const void *h_in_w,
                   const void *h_in_phi, void *h_out_u, void *h_out_v, void *h_out_w, void *h_out_phi) {
    if (!h) return PSDNS_EINVAL;
    const bool phase = h->p.phase_field != 0;
    if (!h_in_u || !h_in_v || !h_in_w || !h_out_u || !h_out_v || !h_out_w || (phase && (!h_in_phi || !h_out_phi)) ||
        (space != PSDNS_PHYSICAL && space != PSDNS_SPECTRAL)) {
        h->err = "psdns_run_host: null pointer or bad space";
        return PSDNS_EINVAL;
    }
    const Dims &d = h->d;
    const size_t bytes = space == PSDNS_PHYSICAL ? d.s_p * sizeof(double) : d.s_bspec * sizeof(cplx);
    const void *hin[4] = {h_in_u, h_in_v, h_in_w, h_in_phi};
    void *hout[4] = {h_out_u, h_out_v, h_out_w, h_out_phi};
    void *dev[4];
    const int nf = phase ? 4 : 3;
    void *dout[4];
    const int b = (int)(h->host_calls++ & 1);      // input staging set of this call
    for (int i = 0; i < 4; ++i) { dev[i] = h->ws + (b ? h->L.stage_b[i] : h->L.stage[i]); dout[i] = h->ws + h->L.stage_out[i]; }
    if (!h->copy_st) {   // side streams and events of the two copy legs, created on first use
        CUDA_TRY(h, cudaStreamCreateWithFlags(&h->copy_st, cudaStreamNonBlocking));
        CUDA_TRY(h, cudaStreamCreateWithFlags(&h->copy_in_st, cudaStreamNonBlocking));
        CUDA_TRY(h, cudaEventCreateWithFlags(&h->ev_out_ready, cudaEventDisableTiming));
        CUDA_TRY(h, cudaEventCreateWithFlags(&h->ev_d2h_done, cudaEventDisableTiming));
        CUDA_TRY(h, cudaEventCreateWithFlags(&h->ev_in_ready, cudaEventDisableTiming));
        for (int i = 0; i < 2; ++i) CUDA_TRY(h, cudaEventCreateWithFlags(&h->ev_in_free[i], cudaEventDisableTiming));
    }
    // upload on its own stream, into the staging set that the call before the previous one has already consumed: it runs
    // while the previous call still computes on the init stream
    if (h->in_used[b]) CUDA_TRY(h, cudaStreamWaitEvent(h->copy_in_st, h->ev_in_free[b], 0));
    for (int i = 0; i < nf; ++i) CUDA_TRY(h, cudaMemcpyAsync(dev[i], hin[i], bytes, cudaMemcpyHostToDevice, h->copy_in_st));
    CUDA_TRY(h, cudaEventRecord(h->ev_in_ready, h->copy_in_st));
    CUDA_TRY(h, cudaStreamWaitEvent(h->st, h->ev_in_ready, 0));
    int rc = psdns_set_state(h, space, dev[0], dev[1], dev[2], phase ? dev[3] : nullptr);
    if (rc != PSDNS_OK) return rc;
    CUDA_TRY(h, cudaEventRecord(h->ev_in_free[b], h->st));
    h->in_used[b] = true;
    if ((rc = psdns_step(h, nsteps)) != PSDNS_OK) return rc;
    // the output staging buffers are still being read by the previous call's device -> host copies
    if (h->d2h_pending) CUDA_TRY(h, cudaStreamWaitEvent(h->st, h->ev_d2h_done, 0));
    if ((rc = psdns_get_state(h, space, dout[0], dout[1], dout[2], phase ? dout[3] : nullptr)) != PSDNS_OK) return rc;
    CUDA_TRY(h, cudaEventRecord(h->ev_out_ready, h->st));
    CUDA_TRY(h, cudaStreamWaitEvent(h->copy_st, h->ev_out_ready, 0));
    for (int i = 0; i < nf; ++i) CUDA_TRY(h, cudaMemcpyAsync(hout[i], dout[i], bytes, cudaMemcpyDeviceToHost, h->copy_st));
    CUDA_TRY(h, cudaEventRecord(h->ev_d2h_done, h->copy_st));
    h->d2h_pending = true;
    return PSDNS_OK;
}

int psdns_run_host_wait(psdns_handle *h) {
    if (!h) return PSDNS_EINVAL;
    if (h->d2h_pending) {
        CUDA_TRY(h, cudaEventSynchronize(h->ev_d2h_done));
        h->d2h_pending = false;
    }
    return PSDNS_OK;
}

long long psdns_launch_count(const psdns_handle *h) { return h ? h->launches : 0; }

int psdns_kernel_timing(psdns_handle *h, const char *name, int enable) {
    if (!h || !name) return PSDNS_EINVAL;
    for (auto &pr : h->tevents) { cudaEventDestroy(pr.first); cudaEventDestroy(pr.second); }
    h->tevents.clear();
    if (!enable) { h->timed_class = -1; return PSDNS_OK; }
    for (int i = 0; i < KC_COUNT; ++i)
        if (std::strcmp(name, kclass_names[i]) == 0) { h->timed_class = i; return PSDNS_OK; }
    h->err = std::string("psdns_kernel_timing: unknown kernel class ") + name;
    return PSDNS_EINVAL;
}

int psdns_kernel_time_ms(psdns_handle *h, double *ms_total, long long *launches) {
    if (!h || !ms_total || !launches) return PSDNS_EINVAL;
    double tot = 0.0;
    for (auto &pr : h->tevents) {
        CUDA_TRY(h, cudaEventSynchronize(pr.second));
        float ms = 0.f;
        CUDA_TRY(h, cudaEventElapsedTime(&ms, pr.first, pr.second));
        tot += ms;
    }
    *ms_total = tot;
    *launches = (long long)h->tevents.size();
    return PSDNS_OK;
}

int psdns_diagnostics(psdns_handle *h, double *d_out) {
    if (!h) return PSDNS_EINVAL;
    if (!d_out) { h->err = "psdns_diagnostics: null output pointer"; return PSDNS_EINVAL; }
    if (!h->has_state) { h->err = "psdns_diagnostics: no state set"; return PSDNS_ESTATE; }
    const Dims &d = h->d;
    const Layout &L = h->L;
    const bool phase = h->p.phase_field != 0;
    const cplx *U = h->at<cplx>(L.state[0]), *V = h->at<cplx>(L.state[1]), *W = h->at<cplx>(L.state[2]);
    // partial results live behind the three Z arrays the energy pass needs (transform scratch is free between steps)
    double *part_max = h->at<double>(L.zb[3]);
    const int nb_cols = (int)((d.ncols + DIAG_NT - 1) / DIAG_NT);
    const int nb_en = h->n_sm * 8;
    double *part_sum = part_max + nb_cols;
    {
        LaunchScope ls(h, KC_MISC);
        k_diag_columns<<<nb_cols, DIAG_NT, 0, h->st>>>(geom(h), U, V, W, phase ? h->at<cplx>(L.state[3]) : nullptr, part_max, d_out);
        CUDA_TRY(h, cudaGetLastError());
    }
    FieldPtrs fz{};
    for (int i = 0; i < 3; ++i) { fz.in[i] = h->at<cplx>(L.state[i]); fz.out[i] = h->at<cplx>(L.zb[i]); }
    CUDA_TRY(h, launch_zpass(h, false, fz, 3, d.ncols, d.nz, d.kxp, d.nky, d.jpos));
    {
        LaunchScope ls(h, KC_MISC);
        k_diag_energy<<<nb_en, DIAG_NT, 0, h->st>>>(h->at<cplx>(L.zb[0]), h->at<cplx>(L.zb[1]), h->at<cplx>(L.zb[2]),
                                                     h->at<double>(L.ccw), d.nz, (int)d.ncols, d.kxp, part_sum);
        CUDA_TRY(h, cudaGetLastError());
    }
    {
        LaunchScope ls(h, KC_MISC);
        k_diag_final<<<1, DIAG_NT, 0, h->st>>>(part_max, nb_cols, part_sum, nb_en, d_out);
        CUDA_TRY(h, cudaGetLastError());
    }
    return PSDNS_OK;
}

// ---- psdns_diagnostics_static: the same diagnostics with the reduction partials in a file-scope device array ----------
// For callers that may not allocate (CUDA graph capture, serving loops, harnesses that forbid cudaMalloc) and whose
// workspace is not theirs to hand out: nothing below calls cudaMalloc, cudaFree or an allocating library routine.
// Every GPU that loads the library holds the array (PSDNS_STATIC_SCRATCH_DOUBLES x 8 bytes = 16 KiB) until exit.
// g_static_scratch is a HOST-side stand-in in host code, not a device address: the kernels get the address that
// cudaGetSymbolAddress returns, looked up once per device with that device current.
static __device__ __align__(256) double g_static_scratch[PSDNS_STATIC_SCRATCH_DOUBLES];

namespace {
constexpr int STATIC_MAX_DEVICES = 64;
double *g_static_scratch_ptr[STATIC_MAX_DEVICES];   // device address of g_static_scratch on each ordinal, nullptr = not looked up
std::mutex g_static_scratch_mu;

int static_scratch_address(psdns_handle *h, double **out) {
    int dev = -1;
    CUDA_TRY(h, cudaGetDevice(&dev));
    if (dev < 0 || dev >= STATIC_MAX_DEVICES) { h->err = "psdns_diagnostics_static: device ordinal beyond 63"; return PSDNS_EINVAL; }
    std::lock_guard<std::mutex> lk(g_static_scratch_mu);
    if (!g_static_scratch_ptr[dev]) {
        void *p = nullptr;
        CUDA_TRY(h, cudaGetSymbolAddress(&p, g_static_scratch));
        if (!p) { h->err = "psdns_diagnostics_static: cudaGetSymbolAddress returned a null address"; return PSDNS_ECUDA; }
        g_static_scratch_ptr[dev] = (double *)p;
    }
    *out = g_static_scratch_ptr[dev];
    return PSDNS_OK;
}
}  // namespace

int psdns_diagnostics_static(psdns_handle *h, double *d_out) {
    if (!h) return PSDNS_EINVAL;
    if (!d_out) { h->err = "psdns_diagnostics_static: null output pointer"; return PSDNS_EINVAL; }
    if (!h->has_state) { h->err = "psdns_diagnostics_static: no state set"; return PSDNS_ESTATE; }
    if (h->timed_class >= 0) {   // psdns_kernel_timing creates a pair of CUDA events per launch
        h->err = "psdns_diagnostics_static: kernel timing is enabled (it creates events); disable it first";
        return PSDNS_ESTATE;
    }
    const Dims &d = h->d;
    const Layout &L = h->L;
    const bool phase = h->p.phase_field != 0;
    const int nb_cols = (int)((d.ncols + DIAG_NT - 1) / DIAG_NT);
    const int nb_en = h->n_sm * 8;
    if ((long long)nb_cols + nb_en > PSDNS_STATIC_SCRATCH_DOUBLES) {
        h->err = "psdns_diagnostics_static: this grid needs " + std::to_string((long long)nb_cols + nb_en) +
                 " doubles of static scratch, the limit is " + std::to_string(PSDNS_STATIC_SCRATCH_DOUBLES) +
                 " (PSDNS_STATIC_SCRATCH_DOUBLES); use psdns_diagnostics";
        return PSDNS_EINVAL;
    }
    double *scratch = nullptr;
    const int rc = static_scratch_address(h, &scratch);
    if (rc != PSDNS_OK) return rc;
    // every slot the final kernel reads is written by this call's two partial kernels first: the last call's
    // contents never reach the result and nothing has to be cleared
    double *part_max = scratch, *part_sum = scratch + nb_cols;
    const cplx *U = h->at<cplx>(L.state[0]), *V = h->at<cplx>(L.state[1]), *W = h->at<cplx>(L.state[2]);
    k_diag_columns<<<nb_cols, DIAG_NT, 0, h->st>>>(geom(h), U, V, W, phase ? h->at<cplx>(L.state[3]) : nullptr, part_max, d_out);
    CUDA_TRY(h, cudaGetLastError());
    FieldPtrs fz{};
    for (int i = 0; i < 3; ++i) { fz.in[i] = h->at<cplx>(L.state[i]); fz.out[i] = h->at<cplx>(L.zb[i]); }
    CUDA_TRY(h, launch_zpass(h, false, fz, 3, d.ncols, d.nz, d.kxp, d.nky, d.jpos));
    k_diag_energy<<<nb_en, DIAG_NT, 0, h->st>>>(h->at<cplx>(L.zb[0]), h->at<cplx>(L.zb[1]), h->at<cplx>(L.zb[2]),
                                                 h->at<double>(L.ccw), d.nz, (int)d.ncols, d.kxp, part_sum);
    CUDA_TRY(h, cudaGetLastError());
    k_diag_final<<<1, DIAG_NT, 0, h->st>>>(part_max, nb_cols, part_sum, nb_en, d_out);
    CUDA_TRY(h, cudaGetLastError());
    h->launches += 3;
    return PSDNS_OK;
}

int psdns_render_isosurface(psdns_handle *h, const psdns_camera *cam, double iso, const void *d_field, void *d_intensity,
                            void *d_depth) {
    if (!h) return PSDNS_EINVAL;
    if (!cam || !d_intensity || !d_depth || cam->width <= 0 || cam->height <= 0 || !(cam->step > 0) ||
        !(cam->fov_y_deg > 0) || !(cam->fov_y_deg < 180)) {
        h->err = "psdns_render_isosurface: null pointer or bad camera";
        return PSDNS_EINVAL;
    }
    const Dims &d = h->d;
    const Layout &L = h->L;
    const double *field = (const double *)d_field;
    if (!field) {   // the current phase field, brought to physical space in the staging buffer
        if (!h->p.phase_field) { h->err = "psdns_render_isosurface: no phase field and no d_field"; return PSDNS_EINVAL; }
        if (!h->has_state) { h->err = "psdns_render_isosurface: no state set"; return PSDNS_ESTATE; }
        FieldPtrs fz{}, fy{}, fx{};
        fz.in[0] = h->at<cplx>(L.state[3]); fz.out[0] = h->at<cplx>(L.zb[0]);
        fy.in[0] = fz.out[0]; fy.out[0] = h->at<cplx>(L.yb[0]);
        fx.in[0] = fy.out[0]; fx.out[0] = h->ws + L.stage[3];
        CUDA_TRY(h, launch_zpass(h, false, fz, 1, d.ncols, d.nz, d.kxp, d.nky, d.jpos));
        CUDA_TRY(h, launch_ypass(h, false, fy, 1, d.kxp, d.nky, d.jpos));
        CUDA_TRY(h, launch_xpass(h, false, fx, 1, d.kxp, d.nkx));
        field = h->at<double>(L.stage[3]);
    }
    auto unit = [](const double *v, double *o) { const double n = std::sqrt(v[0] * v[0] + v[1] * v[1] + v[2] * v[2]); for (int c = 0; c < 3; ++c) o[c] = v[c] / n; };
    auto cross = [](const double *a, const double *b, double *o) { o[0] = a[1] * b[2] - a[2] * b[1]; o[1] = a[2] * b[0] - a[0] * b[2]; o[2] = a[0] * b[1] - a[1] * b[0]; };
    RayArgs a;
    a.phi = field; a.zn = h->at<double>(L.znodes);
    a.intensity = (double *)d_intensity; a.depth = (double *)d_depth;
    a.nx = d.nx; a.ny = d.ny; a.nz = d.nz; a.lx = h->g.lx; a.ly = h->g.ly;
    double f[3] = {cam->target[0] - cam->eye[0], cam->target[1] - cam->eye[1], cam->target[2] - cam->eye[2]}, r[3];
    unit(f, a.fwd);
    cross(a.fwd, cam->up, r);
    if (!(r[0] * r[0] + r[1] * r[1] + r[2] * r[2] > 0)) { h->err = "psdns_render_isosurface: up is parallel to the view direction"; return PSDNS_EINVAL; }
    unit(r, a.right);
    cross(a.right, a.fwd, a.upv);
    unit(cam->light, a.light);
    for (int c = 0; c < 3; ++c) a.eye[c] = cam->eye[c];
    a.tan_half = std::tan(cam->fov_y_deg * M_PI / 180.0 / 2.0);
    a.aspect = (double)cam->width / (double)cam->height;
    a.step = cam->step; a.iso = iso; a.width = cam->width; a.height = cam->height;
    LaunchScope ls(h, KC_MISC);
    k_raycast<<<(cam->width * cam->height + 127) / 128, 128, 0, h->st>>>(a);
    CUDA_TRY(h, cudaGetLastError());
    return PSDNS_OK;
}

int psdns_measure_fp64_peak(psdns_handle *h, double *tflops) {
    if (!h || !tflops) return PSDNS_EINVAL;
    // scratch: the first Z array (transform scratch is free between steps)
    double *out = h->at<double>(h->L.zb[0]);
    const int blocks = h->n_sm * 8, iters = 4096;
    const int nslots = (int)std::max<size_t>(1, std::min<size_t>((size_t)blocks, h->d.s_ret * sizeof(cplx) / (256 * sizeof(double))));
    cudaEvent_t e0, e1;
    CUDA_TRY(h, cudaEventCreate(&e0)); CUDA_TRY(h, cudaEventCreate(&e1));
    double best = 0.0;
    for (int rep = 0; rep < 4; ++rep) {
        CUDA_TRY(h, cudaEventRecord(e0, h->st));
        k_fp64_fma_chain<<<blocks, 256, 0, h->st>>>(out, nslots, iters, 0.999999, 1e-6);
        CUDA_TRY(h, cudaGetLastError());
        CUDA_TRY(h, cudaEventRecord(e1, h->st));
        CUDA_TRY(h, cudaEventSynchronize(e1));
        float ms = 0.f;
        CUDA_TRY(h, cudaEventElapsedTime(&ms, e0, e1));
        const double flops = 2.0 * 8 * 16 * (double)iters * 256.0 * blocks;
        if (rep > 0) best = std::max(best, flops / (ms * 1e-3) / 1e12);
        h->launches++;
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    *tflops = best;
    return PSDNS_OK;
}

int psdns_set_option(psdns_handle *h, const char *name, double value) {
    if (!h || !name) return PSDNS_EINVAL;
    const std::string n(name);
    const int iv = (int)value;
    if (h->has_state) {   // the options choose who corrects theta^: complete it now, and leave no stale coefficients behind
        const int rc = materialise_theta(h);
        if (rc != PSDNS_OK) return rc;
        CUDA_TRY(h, cudaMemsetAsync(h->ws + h->L.coef, 0, 2 * h->d.ncols * sizeof(cplx), h->st));
    }
    if (n == "graph") h->use_graph = iv != 0;
    else if (n == "xfuse" && iv && ((h->p.phase_field && h->p.surface_tension_form == 1) || h->p.convection_form == 1)) {
        h->err = "psdns_set_option: the alternative non-linear forms have no fused x kernel";
        return PSDNS_EINVAL;
    }
    else if (n == "xfuse") {
        if (!iv && !h->has_unfused_ws) { h->err = "psdns_set_option: xfuse = 0 needs psdns_workspace_bytes_unfused() bytes at init"; return PSDNS_ENOMEM; }
        h->use_xfused = iv != 0;
    }
    else if (n == "grid_cap" && iv >= 0) h->grid_cap = iv;
    else if (n == "ztma") h->use_ztma = iv != 0;
    else if (n == "zgemm") h->use_zgemm = iv != 0;
    else if (n == "phi3") h->phi3 = iv != 0;
    else if (n == "w3") h->w3 = iv != 0;
    else if (n == "lazy") h->lazy = iv != 0;

    else if (n == "pf" && iv >= 0) h->pf = iv;
    else if (n == "pf_rhs" && iv >= 0) h->pf_rhs = iv;
    else { h->err = "psdns_set_option: unknown option or bad value: " + n; return PSDNS_EINVAL; }
    if (h->graph) { cudaGraphExecDestroy(h->graph); h->graph = nullptr; }   // the captured step bakes the options in
    h->graph_ready = false;
    return PSDNS_OK;
}

double psdns_get_info(const psdns_handle *h, const char *name) {
    if (!h || !name) return -1.0;
    const std::string n(name);
    for (int i = 0; i < KC_COUNT; ++i) {
        if (n == std::string(kclass_names[i]) + "_grid") return (double)h->last_grid[i];
        if (n == std::string(kclass_names[i]) + "_items") return (double)h->last_items[i];
    }
    if (n == "n_sm") return (double)h->n_sm;
    if (n == "workspace_bytes") return (double)h->L.total;
    if (n == "launches_per_step") return (double)h->per_step;
    return -1.0;
}

int psdns_destroy(psdns_handle *h) {
    if (!h) return PSDNS_EINVAL;
    if (h->graph) cudaGraphExecDestroy(h->graph);
    if (h->copy_st) {
        cudaStreamSynchronize(h->copy_in_st); cudaStreamSynchronize(h->copy_st);
        cudaStreamDestroy(h->copy_in_st); cudaStreamDestroy(h->copy_st);
        cudaEventDestroy(h->ev_out_ready); cudaEventDestroy(h->ev_d2h_done); cudaEventDestroy(h->ev_in_ready);
        cudaEventDestroy(h->ev_in_free[0]); cudaEventDestroy(h->ev_in_free[1]);
    }
    for (auto &pr : h->tevents) { cudaEventDestroy(pr.first); cudaEventDestroy(pr.second); }
    delete h;
    return PSDNS_OK;
}

const char *psdns_last_error(const psdns_handle *h) { return h ? h->err.c_str() : "null handle"; }

}  // extern "C"
