// Spectral-space kernels: one thread per retained (kx, ky) column, sweeping the Chebyshev index
// n sequentially; consecutive threads own consecutive columns so every access is coalesced.
//   k_relayout      boundary <-> private spectral layouts
//   k_hidden_state  theta = (D^2 - k^2) w, omega_z = i kx v - i ky u            (hidden state, reading S13)
//   k_prep          row a1: grad(phi) spectra [+ strain spectra]
//   k_helm_setup / k_helm / k_elimup_setup / k_hom_tables   init: pivot tables, homogeneous solutions
//   The solver stage of a step is three sweeps over the columns (rows a9-a11):
//   k_rhs_elim      DOWN: S = div T, N_omega (Eq. 14), N_w (Eq. 15), S_phi (Eq. 17), AB2, CN/IE right-hand sides, all
//                   derivative recurrences, streamed into the Gauss elimination of the omega_z, theta, psi problems
//   k_subst3        UP:   their substitution; theta_p and psi feed the UPWARD elimination of the w and phi solves
//   k_finish        DOWN: back substitution of w and phi, influence-matrix correction (Dw(+-1) = 0), u^, v^ from
//                   continuity (Eq. 6) and the vorticity definition (Eq. 16), D phi^
//   k_subst / k_elim2 / k_elim2up   the five-sweep forms of the same solves (options "w3", "phi3": cross-checks)
#pragma once
#include "fft_tile.cuh"

namespace psdns {

constexpr int NT_COL = 128;

struct ColGeom {
    int ncols;   // nky * kxp
    int kxp, nkx, nky, jpos;
    int N;       // nz - 1
    int nkz;     // retained Chebyshev planes (K + 1)
    double kxf, kyf;  // 2 pi / Lx, 2 pi / Ly
    int pf, pf_rhs;   // L2 prefetch distances in rows
};

__device__ __forceinline__ void col_wavenumbers(const ColGeom &g, int col, double &kx, double &ky) {
    const int ir = col % g.kxp, jr = col / g.kxp;
    kx = g.kxf * (double)ir;   // pad columns (ir >= nkx) carry zeros; their k is irrelevant
    ky = g.kyf * (double)(jr < g.jpos ? jr : jr - g.nky);
}

__device__ __forceinline__ cplx cz() { return make_double2(0.0, 0.0); }
__device__ __forceinline__ cplx ci(cplx a) { return make_double2(-a.y, a.x); }           // i * a
__device__ __forceinline__ cplx cfma(double s, cplx a, cplx b) {                          // s*a + b
    return make_double2(fma(s, a.x, b.x), fma(s, a.y, b.y));
}

// L2 prefetch of the cache line that holds p: the column sweeps below touch one 16-byte element per array
// per row, so the rows PF_ROWS ahead are requested early and the demand loads become L2 hits.
__device__ __forceinline__ void pf_l2(const void *p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }
// Distances measured on B200 at 1024x512x513: the substitution / second-elimination / finish kernels keep every column
// resident at once, so rows x arrays x 1.9 MB of prefetched data must stay well inside the 126 MB L2 (6 rows ahead thrashed
// it: +2 GB of re-reads per kernel); k_rhs_elim has 12 % of the columns resident and likes a longer distance.
// The distance is a run-time number in ColGeom (pf for the sweeps that keep every column resident, pf_rhs for
// k_rhs_elim), set by the host (psdns.cu geom()): 2 / 4 rows.

// ---- layout conversion ---------------------------------------------------------------------
// Both sides are cplx [n][rows][pitch]; a side is described by (rows, pitch, jpos, nkx):
// row r < jpos holds j' = r, row r >= jpos holds j' = r - rows; columns i < nkx are valid.
struct SpecSide {
    int rows, pitch, jpos, nkx;
};

__global__ void __launch_bounds__(256) k_relayout(cplx *__restrict__ dst, const cplx *__restrict__ src,
                                                  SpecSide d, SpecSide s, int nplanes) {
    const size_t total = (size_t)nplanes * d.rows * d.pitch;
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    for (size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x; e < total; e += stride) {
        const int i = (int)(e % d.pitch);
        const size_t t = e / d.pitch;
        const int r = (int)(t % d.rows);
        const int n = (int)(t / d.rows);
        cplx v = cz();
        if (i < d.nkx && i < s.nkx) {
            const int jp = r < d.jpos ? r : r - d.rows;
            int rs = -1;
            if (jp >= 0) { if (jp < s.jpos) rs = jp; }
            else { if (s.rows + jp >= s.jpos) rs = s.rows + jp; }
            if (rs >= 0) v = src[((size_t)n * s.rows + rs) * s.pitch + i];
        }
        dst[e] = v;
    }
}

// ---- hidden state: theta = (D^2 - k^2) w (reading S13), omega_z = i kx v - i ky u (Eq. 16) ------------
// Chebyshev derivative recurrence: ct_n b_n = b_{n+2} + 2 (n+1) a_{n+1}, ct_0 = 2.
// Column (0,0) carries the mean flow instead: the omega slot holds u-bar, the theta slot v-bar (reading S12).
__global__ void __launch_bounds__(NT_COL) k_hidden_state(const __grid_constant__ ColGeom g, const cplx *__restrict__ u,
                                                         const cplx *__restrict__ v, const cplx *__restrict__ w,
                                                         cplx *__restrict__ th, cplx *__restrict__ om) {
    const int col = blockIdx.x * blockDim.x + threadIdx.x;
    if (col >= g.ncols) return;
    double kx, ky;
    col_wavenumbers(g, col, kx, ky);
    const double k2 = kx * kx + ky * ky;
    const size_t st = g.ncols;
    cplx a1 = cz(), b1 = cz(), b2 = cz(), c1 = cz(), c2 = cz();
    for (int n = g.N; n >= 0; --n) {
        const double f = 2.0 * (n + 1), h = (n == 0) ? 0.5 : 1.0;
        const size_t o = n * st + col;
        const cplx an = w[o], un = u[o], vn = v[o];
        cplx bn = cscale(cfma(f, a1, b2), h);
        cplx cn = cscale(cfma(f, b1, c2), h);
        if (col == 0) {
            th[o] = vn;
            om[o] = un;
        } else {
            th[o] = cfma(-k2, an, cn);
            om[o] = ci(csub(cscale(vn, kx), cscale(un, ky)));
        }
        a1 = an; b2 = b1; b1 = bn; c2 = c1; c1 = cn;
    }
}

// ---- derivative recurrences fed top-down (used by rows a1, a9, a11) ------------------------------------
struct Chain1 {  // first derivative of a sequence fed top-down
    cplx a1, b1, b2;
    __device__ __forceinline__ void init() { a1 = b1 = b2 = cz(); }
    __device__ __forceinline__ cplx step(cplx an, double f, double h) {
        cplx bn = cscale(cfma(f, a1, b2), h);
        a1 = an; b2 = b1; b1 = bn;
        return bn;
    }
};
struct Chain2 {  // second derivative
    cplx a1, b1, b2, c1, c2;
    __device__ __forceinline__ void init() { a1 = b1 = b2 = c1 = c2 = cz(); }
    __device__ __forceinline__ cplx step(cplx an, double f, double h) {
        cplx bn = cscale(cfma(f, a1, b2), h);
        cplx cn = cscale(cfma(f, b1, c2), h);
        a1 = an; b2 = b1; b1 = bn; c2 = c1; c1 = cn;
        return cn;
    }
};

// ---- row a1: derived spectra that need a z derivative ----------------------------------------------------
// phz = D phi^ (only at set_state: k_finish maintains it afterwards); the five strain spectra of the
// variable-viscosity term (config 4, reading S14).  i kx phi^ and i ky phi^ are formed inside the z pass.
struct PrepArgs {
    ColGeom g;
    const cplx *u, *v, *w, *phi;
    cplx *phz;
    cplx *exx, *eyy, *exy, *exz, *eyz;
    int do_phz, visc;
    cplx *lap;       // do_lap: (D^2 - k^2) of the truncated phi^ (force form of the surface tension)
    int do_lap;
    cplx *wx, *wy, *wz;   // do_vort: vorticity of the truncated velocity (rotational form of convection)
    int do_vort;
};

__global__ void __launch_bounds__(NT_COL) k_prep(const __grid_constant__ PrepArgs a) {
    const ColGeom &g = a.g;
    const int col = blockIdx.x * blockDim.x + threadIdx.x;
    if (col >= g.ncols) return;
    double kx, ky;
    col_wavenumbers(g, col, kx, ky);
    const size_t st = g.ncols;
    cplx p1 = cz(), dp1 = cz(), dp2 = cz();
    cplx u1 = cz(), du1 = cz(), du2 = cz(), v1 = cz(), dv1 = cz(), dv2 = cz();
    Chain2 cL;
    cL.init();
    const double k2 = kx * kx + ky * ky;
    // every derivative is taken of the TRUNCATED field (P first, then D)
    for (int n = g.nkz - 1; n >= 0; --n) {
        const double f = 2.0 * (n + 1), h = (n == 0) ? 0.5 : 1.0;
        const size_t o = n * st + col;
        if (a.do_lap) {
            const cplx pn = a.phi[o];
            a.lap[o] = cfma(-k2, pn, cL.step(pn, f, h));
        }
        if (a.do_vort) {   // omega = curl u: (i ky w - D v, D u - i kx w, i kx v - i ky u); column (0,0) included (omega_z = 0 there)
            const cplx un = a.u[o], vn = a.v[o], wn = a.w[o];
            const cplx dun = cscale(cfma(f, u1, du2), h);
            const cplx dvn = cscale(cfma(f, v1, dv2), h);
            a.wx[o] = csub(cscale(ci(wn), ky), dvn);
            a.wy[o] = csub(dun, cscale(ci(wn), kx));
            a.wz[o] = csub(cscale(ci(vn), kx), cscale(ci(un), ky));
            u1 = un; du2 = du1; du1 = dun;
            v1 = vn; dv2 = dv1; dv1 = dvn;
        }
        if (a.do_phz) {
            const cplx pn = a.phi[o];
            const cplx dpn = cscale(cfma(f, p1, dp2), h);
            a.phz[o] = dpn;
            p1 = pn; dp2 = dp1; dp1 = dpn;
        }
        if (a.visc) {
            const cplx un = a.u[o], vn = a.v[o], wn = a.w[o];
            const cplx dun = cscale(cfma(f, u1, du2), h);
            const cplx dvn = cscale(cfma(f, v1, dv2), h);
            a.exx[o] = cscale(ci(un), 2.0 * kx);
            a.eyy[o] = cscale(ci(vn), 2.0 * ky);
            a.exy[o] = cadd(cscale(ci(un), ky), cscale(ci(vn), kx));
            a.exz[o] = cadd(dun, cscale(ci(wn), kx));
            a.eyz[o] = cadd(dvn, cscale(ci(wn), ky));
            u1 = un; du2 = du1; du1 = dun;
            v1 = vn; dv2 = dv1; dv1 = dvn;
        }
    }
}

// ---- row a10: quasi-tridiagonal Chebyshev-tau Helmholtz solve ---------------------------------------
// (D^2 - sigma) u = f in rows 0..N-2 plus two boundary rows (reading S11).  In coefficient space,
// for k = 2..N (even and odd k decouple):
//   a_k u_{k-2} + d_k u_k + c_k u_{k+2} = p_k f_{k-2} + q_k f_k + r_k f_{k+2} =: g_k
//   p_k = ct_{k-2}/(4k(k-1)), q_k = -1/(2(k^2-1)), r_k = 1/(4k(k+1)), f_j := 0 for j > N-2,
//   a_k = -sigma p_k, d_k = 1 + sigma e_{k+2}/(2(k^2-1)), c_k = -sigma e_{k+4}/(4k(k+1)), e_j = [j <= N].
// Gauss elimination from k = N down removes c_k (pivots d'_k, stored as 1/d'_k by k_helm_setup);
// the remaining lower-bidiagonal rows give u_k = alpha_k + beta_k u_par (par = k & 1), and the
// boundary row of each parity fixes u_par.
// p_k, q_k, r_k depend on k only and every thread of a warp is at the same k: constant-memory tables (one broadcast
// read instead of an FP64 division each; filled once by psdns_init with the host versions of the same formulas,
// k <= HELM_KMAX = N_max + 2).
constexpr int HELM_KMAX = 516;
__constant__ double c_helm_p[HELM_KMAX + 1], c_helm_q[HELM_KMAX + 1], c_helm_r[HELM_KMAX + 1];
inline double helm_p_host(int k) { return k < 2 ? 0.0 : (k == 2 ? 2.0 : 1.0) / (4.0 * k * (double)(k - 1)); }
inline double helm_q_host(int k) { return k < 2 ? 0.0 : -1.0 / (2.0 * ((double)k * k - 1.0)); }
inline double helm_r_host(int k) { return k < 1 ? 0.0 : 1.0 / (4.0 * k * (double)(k + 1)); }
__device__ __forceinline__ double helm_p(int k) { return c_helm_p[k]; }
__device__ __forceinline__ double helm_q(int k) { return c_helm_q[k]; }
__device__ __forceinline__ double helm_r(int k) { return c_helm_r[k]; }

// Pivots of the downward elimination, d'_k = d_k - c_k a_{k+2} / d'_{k+2} (the recurrence of k_helm_setup), recomputed
// on the fly by the down sweeps instead of being read from the [N+1][ncols] table (the up sweeps, which need them in
// ascending order, still read the table): saves 0.48 GB of reads per down sweep at 1024x512x513.
struct PivotDown {
    double di1, di2;   // 1/d'_{k+1}, 1/d'_{k+2}
    __device__ __forceinline__ void init() { di1 = di2 = 0.0; }
    __device__ __forceinline__ double step(int k, int N, double sigma) {
        double d = 1.0 + ((k + 2 <= N) ? sigma * (-helm_q(k)) : 0.0);
        if (k + 4 <= N) {
            const double ck = -sigma * helm_r(k);
            const double ak2 = -sigma * helm_p(k + 2);
            d -= ck * ak2 * di2;
        }
        const double di = 1.0 / d;
        di2 = di1; di1 = di;
        return di;
    }
};

struct HelmSetupArgs {
    ColGeom g;
    double *dinv;   // [N+1][ncols]
    double shift;   // sigma = k^2 + shift
};

__global__ void __launch_bounds__(NT_COL) k_helm_setup(const __grid_constant__ HelmSetupArgs a) {
    const ColGeom &g = a.g;
    const int col = blockIdx.x * blockDim.x + threadIdx.x;
    if (col >= g.ncols) return;
    double kx, ky;
    col_wavenumbers(g, col, kx, ky);
    const double sigma = kx * kx + ky * ky + a.shift;
    const size_t st = g.ncols;
    const int N = g.N;
    PivotDown pv;
    pv.init();
    for (int k = N; k >= 2; --k) a.dinv[k * st + col] = pv.step(k, N, sigma);
    a.dinv[col] = 0.0;
    a.dinv[st + col] = 0.0;
}

enum { BC_DIRICHLET = 0, BC_NEUMANN = 1 };

struct HelmArgs {
    ColGeom g;
    const cplx *in;   // f (rows 0..N-2 used)
    cplx *out;        // solution (may alias in)
    const double *dinv;
    double shift, scale;   // sigma = k^2 + shift ; f is multiplied by scale
    int bc;
    double tgt_e, tgt_o;   // boundary-row targets of the even / odd parity (0 in the time step)
};

__global__ void __launch_bounds__(NT_COL) k_helm(const __grid_constant__ HelmArgs a) {
    const ColGeom &g = a.g;
    const int col = blockIdx.x * blockDim.x + threadIdx.x;
    if (col >= g.ncols) return;
    double kx, ky;
    col_wavenumbers(g, col, kx, ky);
    const double sigma = kx * kx + ky * ky + a.shift;
    const size_t st = g.ncols;
    const int N = g.N;
    const cplx *__restrict__ in = a.in + col;
    cplx *__restrict__ out = a.out + col;
    const double *__restrict__ dinv = a.dinv + col;
    const double sc = a.scale;
    // sweep 1 (down): g'_k = g_k - (c_k / d'_{k+2}) g'_{k+2}
    {
        cplx fp2 = cz(), fp1 = cz();
        cplx f0 = cz(), fm1 = cz();   // f_N = f_{N-1} := 0
        cplx gp2 = cz(), gp1 = cz();
        double dp2 = 0.0, dp1 = 0.0;
#pragma unroll 4
        for (int k = N; k >= 2; --k) {
            const cplx fm2 = cscale(in[(k - 2) * st], sc);
            const double di = dinv[k * st];
            cplx gk = cfma(helm_p(k), fm2, cfma(helm_q(k), f0, cscale(fp2, helm_r(k))));
            if (k + 4 <= N) {
                const double m = -sigma * helm_r(k) * dp2;
                gk = cfma(-m, gp2, gk);
            }
            out[k * st] = gk;
            gp2 = gp1; gp1 = gk;
            dp2 = dp1; dp1 = di;
            fp2 = fp1; fp1 = f0; f0 = fm1; fm1 = fm2;
        }
    }
    // sweep 2 (up): alpha_k, beta_k, boundary sums
    const bool neu = a.bc == BC_NEUMANN;
    cplx sa_e = cz(), sa_o = cz();
    double sb_e = neu ? 0.0 : 1.0, sb_o = 1.0;
    {
        cplx al2 = cz(), al1 = cz();   // alpha_{k-2}, alpha_{k-1}
        double be2 = 1.0, be1 = 1.0;
#pragma unroll 4
        for (int k = 2; k <= N; ++k) {
            const double ak = -sigma * helm_p(k);
            const double di = dinv[k * st];
            const cplx gk = out[k * st];
            const cplx al = cscale(cfma(-ak, al2, gk), di);
            const double be = -ak * be2 * di;
            out[k * st] = al;
            const double wk = neu ? (double)k * k : 1.0;
            if (k & 1) { sa_o = cfma(wk, al, sa_o); sb_o += wk * be; }
            else       { sa_e = cfma(wk, al, sa_e); sb_e += wk * be; }
            al2 = al1; al1 = al;
            be2 = be1; be1 = be;
        }
    }
    // Dirichlet: sum_even u = tgt_e, sum_odd u = tgt_o.  Neumann: sum_even k^2 u = tgt_e, sum_odd k^2 u = tgt_o.
    const cplx u0 = cscale(make_double2(a.tgt_e - sa_e.x, -sa_e.y), 1.0 / sb_e);
    const cplx u1 = cscale(make_double2(a.tgt_o - sa_o.x, -sa_o.y), 1.0 / sb_o);
    // sweep 3 (up): u_k = alpha_k + beta_k u_par
    {
        double be2 = 1.0, be1 = 1.0;
        out[0] = u0;
        out[st] = u1;
#pragma unroll 4
        for (int k = 2; k <= N; ++k) {
            const double ak = -sigma * helm_p(k);
            const double be = -ak * be2 * dinv[k * st];
            const cplx al = out[k * st];
            out[k * st] = cfma(be, (k & 1) ? u1 : u0, al);
            be2 = be1; be1 = be;
        }
    }
}

// ================================================================================================
// Two-sweep form of the same tau solve, used by the time step (k_helm above builds the init tables).
//
// Down sweep (rows k = N..2): Gauss elimination of c_k as in k_helm, PLUS the adjoint weights
//   z_k = (w_k - a_{k+2} z_{k+2}) / d'_k     (L^T z = w, L = reduced lower-bidiagonal system)
// so that the boundary functional of the particular solution is known without a substitution pass:
//   sum_{k>=2} w_k alpha_k = sum_k z_k g'_k =: J_par,   sum_{k>=2} w_k beta_k = -a_{par+2} z_{par+2}
//   u_par = (target - J_par) / (w_par - a_{par+2} z_{par+2}).
// The down sweep therefore ends knowing u_0, u_1 (stored in the two unused slots of the g' array) and ONE
// up sweep u_k = (g'_k - a_k u_{k-2}) / d'_k finishes the solve.  A second weight set (k^2) gives
// sum k^2 w_k of the Dirichlet solution for the influence-matrix coefficient of the w problem.
// ================================================================================================
struct ElimDown {
    cplx fp2, fp1, f0, fm1;   // F(k+2), F(k+1), F(k), F(k-1) of the next row k
    cplx gp2, gp1;            // g'_{k+2}, g'_{k+1}
    double dp2, dp1;          // 1/d'_{k+2}, 1/d'_{k+1}
    double zp2, zp1;          // boundary-row adjoint weights z_{k+2}, z_{k+1}
    double yp2, yp1;          // second functional (weights k^2)
    double xp2, xp1;          // third functional (weights k^2 (k^2 - 1) / 3: T_k''(+-1), free-slip walls)
    cplx Je, Jo, Ke, Ko, Me, Mo;
    __device__ __forceinline__ void init() {
        fp2 = fp1 = f0 = fm1 = gp2 = gp1 = Je = Jo = Ke = Ko = Me = Mo = cz();
        dp2 = dp1 = zp2 = zp1 = yp2 = yp1 = xp2 = xp1 = 0.0;
    }
    // row k (N >= k >= 2): fm2 = F(k-2) (scaled RHS, zero-extended above N-2), di = 1/d'_k.  Returns g'_k.
    template <bool NEU, bool SECOND, bool THIRD = false>
    __device__ __forceinline__ cplx row(int k, int N, double sigma, cplx fm2, double di) {
        cplx g = cfma(helm_p(k), fm2, cfma(helm_q(k), f0, cscale(fp2, helm_r(k))));
        if (k + 4 <= N) g = cfma(sigma * helm_r(k) * dp2, gp2, g);   // g - (c_k/d'_{k+2}) g'_{k+2}, c_k = -sigma r_k
        const double sp = (k + 2 <= N) ? sigma * helm_p(k + 2) : 0.0;   // -a_{k+2}
        const double wk = NEU ? (double)k * k : 1.0;
        const double z = (wk + sp * zp2) * di;
        if (k & 1) Jo = cfma(z, g, Jo); else Je = cfma(z, g, Je);
        if (SECOND) {
            const double y = ((double)k * k + sp * yp2) * di;
            if (k & 1) Ko = cfma(y, g, Ko); else Ke = cfma(y, g, Ke);
            yp2 = yp1; yp1 = y;
        }
        if (THIRD) {
            const double k2 = (double)k * k;
            const double x = (k2 * (k2 - 1.0) * (1.0 / 3.0) + sp * xp2) * di;
            if (k & 1) Mo = cfma(x, g, Mo); else Me = cfma(x, g, Me);
            xp2 = xp1; xp1 = x;
        }
        zp2 = zp1; zp1 = z;
        gp2 = gp1; gp1 = g;
        dp2 = dp1; dp1 = di;
        fp2 = fp1; fp1 = f0; f0 = fm1; fm1 = fm2;
        return g;
    }
    // after row 2: zp1 = z_2, zp2 = z_3.  Boundary rows: Dirichlet sum u = tgt; Neumann sum k^2 u = tgt.
    template <bool NEU>
    __device__ __forceinline__ void finish(double sigma, double tgt_e, double tgt_o, cplx &u0, cplx &u1) const {
        const double se = (NEU ? 0.0 : 1.0) + sigma * helm_p(2) * zp1;
        const double so = 1.0 + sigma * helm_p(3) * zp2;
        u0 = cscale(make_double2(tgt_e - Je.x, -Je.y), 1.0 / se);
        u1 = cscale(make_double2(tgt_o - Jo.x, -Jo.y), 1.0 / so);
    }
    // sum_{k in parity} k^2 u_k of the finished solution (needs SECOND)
    __device__ __forceinline__ void second(double sigma, cplx u0, cplx u1, cplx &de, cplx &dodd) const {
        de = cfma(sigma * helm_p(2) * yp1, u0, Ke);                    // 0^2 u_0 + K_e + u_0 sum k^2 beta_k
        dodd = cadd(u1, cfma(sigma * helm_p(3) * yp2, u1, Ko));          // 1^2 u_1 + K_o + u_1 sum k^2 beta_k
    }
    // sum_{k in parity} k^2 (k^2 - 1)/3 u_k of the finished solution (needs THIRD); the weights of k = 0, 1 vanish
    __device__ __forceinline__ void third(double sigma, cplx u0, cplx u1, cplx &me, cplx &mo) const {
        me = cfma(sigma * helm_p(2) * xp1, u0, Me);
        mo = cfma(sigma * helm_p(3) * xp2, u1, Mo);
    }
};

// Boundary closure of one Helmholtz solve for any pair of wall conditions (no-slip, free-slip or a
// combination; kind 0 = value prescribed (Dirichlet), 1 = first derivative (Neumann), homogeneous).  With
// u_k = alpha_k + beta_k u_par the four parity sums of the solution are
//   S_e = Sa_e + se u_0,  S_o = Sa_o + so u_1   (weights 1),      K_e = Ka_e + ke u_0,  K_o = Ka_o + ko u_1   (weights k^2)
// and T_k(+-1) = (+-1)^k, T_k'(+-1) = (+-1)^(k+1) k^2 give the value / derivative at z = +1 as S_e + S_o / K_e + K_o and
// at z = -1 as S_e - S_o / -K_e + K_o.  Equal kinds decouple by parity; mixed kinds leave a 2 x 2 system.
__device__ __forceinline__ void wall_closure(int top, int bot, double Sae, double Sao, double Kae, double Kao, double se,
                                             double so, double ke, double ko, double &u0, double &u1) {
    if (top == 0 && bot == 0) { u0 = -Sae / se; u1 = -Sao / so; return; }
    if (top == 1 && bot == 1) { u0 = -Kae / ke; u1 = -Kao / ko; return; }
    double a11, a12, b1, a21, a22, b2;
    if (top == 1) { a11 = ke; a12 = ko; b1 = -(Kae + Kao); a21 = se; a22 = -so; b2 = -(Sae - Sao); }     // N at +1, D at -1
    else          { a11 = se; a12 = so; b1 = -(Sae + Sao); a21 = -ke; a22 = ko; b2 = Kae - Kao; }        // D at +1, N at -1
    const double idet = 1.0 / (a11 * a22 - a12 * a21);
    u0 = (b1 * a22 - a12 * b2) * idet;
    u1 = (a11 * b2 - a21 * b1) * idet;
}

// Real-component form of ElimDown for TWO right-hand sides that share sigma, the pivots and the Dirichlet adjoint
// weights (the omega_z and theta problems of one column: both sigma = k^2 + 1/gamma).  The tau system has real
// coefficients, so the real and imaginary parts of a column are two independent real problems.
template <bool GEN = false>   // GEN: also the k^2-weighted functional, for walls that are not both no-slip
struct ElimDown2R {
    double fp2[2], fp1[2], f0[2], fm1[2];   // F(k+2), F(k+1), F(k), F(k-1) of the next row k, per right-hand side
    double gp2[2], gp1[2];                  // g'_{k+2}, g'_{k+1}
    double Je[2], Jo[2];
    double Ke[2], Ko[2];                    // GEN only
    double dp2, dp1, zp2, zp1;
    double yp2, yp1;                        // GEN only
    __device__ __forceinline__ void init() {
#pragma unroll
        for (int i = 0; i < 2; ++i) fp2[i] = fp1[i] = f0[i] = fm1[i] = gp2[i] = gp1[i] = Je[i] = Jo[i] = Ke[i] = Ko[i] = 0.0;
        dp2 = dp1 = zp2 = zp1 = yp2 = yp1 = 0.0;
    }
    __device__ __forceinline__ void row(int k, int N, double sigma, double fa, double fb, double di, double &ga, double &gb) {
        const double pk = helm_p(k), qk = helm_q(k), rk = helm_r(k);
        const double fm2[2] = {fa, fb};
        double g[2];
        const double m = (k + 4 <= N) ? sigma * rk * dp2 : 0.0;
        const double sp = (k + 2 <= N) ? sigma * helm_p(k + 2) : 0.0;
        const double z = (1.0 + sp * zp2) * di;
        const double y = GEN ? ((double)k * k + sp * yp2) * di : 0.0;
#pragma unroll
        for (int i = 0; i < 2; ++i) {
            g[i] = fma(pk, fm2[i], fma(qk, f0[i], fp2[i] * rk));
            g[i] = fma(m, gp2[i], g[i]);
            if (k & 1) Jo[i] = fma(z, g[i], Jo[i]); else Je[i] = fma(z, g[i], Je[i]);
            if (GEN) { if (k & 1) Ko[i] = fma(y, g[i], Ko[i]); else Ke[i] = fma(y, g[i], Ke[i]); }
            gp2[i] = gp1[i]; gp1[i] = g[i];
            fp2[i] = fp1[i]; fp1[i] = f0[i]; f0[i] = fm1[i]; fm1[i] = fm2[i];
        }
        if (GEN) { yp2 = yp1; yp1 = y; }
        zp2 = zp1; zp1 = z;
        dp2 = dp1; dp1 = di;
        ga = g[0]; gb = g[1];
    }
    // homogeneous Dirichlet rows: u_0 = -J_e / s_e, u_1 = -J_o / s_o
    __device__ __forceinline__ void finish(double sigma, int i, double &u0, double &u1) const {
        const double se = 1.0 + sigma * helm_p(2) * zp1;
        const double so = 1.0 + sigma * helm_p(3) * zp2;
        u0 = -Je[i] / se;
        u1 = -Jo[i] / so;
    }
    // any pair of homogeneous wall conditions (GEN): kinds 0 = value, 1 = derivative, at z = +1 / z = -1
    __device__ __forceinline__ void finish_walls(double sigma, int i, int top, int bot, double &u0, double &u1) const {
        const double se = 1.0 + sigma * helm_p(2) * zp1, so = 1.0 + sigma * helm_p(3) * zp2;
        const double ke = sigma * helm_p(2) * yp1, ko = 1.0 + sigma * helm_p(3) * yp2;
        wall_closure(top, bot, Je[i], Jo[i], Ke[i], Ko[i], se, so, ke, ko, u0, u1);
    }
};

// ================================================================================================
// UPWARD elimination of the same system, used for the SECOND solve of the phi problem ((D^2 - k^2 - lambda) phi = psi)
// so that it can ride on the up sweep that produces psi (k_subst) and finish in the down sweep that k_finish makes
// anyway: psi never reaches HBM and two sweeps over the phi column disappear (three sweeps instead of five for this
// problem).  Rows k = 2, 3, .. ascending, each parity on its own; u_par (par = k & 1) is carried symbolically:
//   d''_k u_k + c_k u_{k+2} = g''_k + e_k u_par,
//   first row of a parity (k = 2, 3):  d''_k = d_k, g''_k = g_k, e_k = -a_k,
//   then  m_k = a_k / d''_{k-2}:       d''_k = d_k - m_k c_{k-2}, g''_k = g_k - m_k g''_{k-2}, e_k = -m_k e_{k-2}.
// Back substitution (descending): u_k = g^_k + e^_k u_par - c^_k u_{k+2},  g^ = g''/d'', e^ = e/d'', c^ = c/d''.
// u_par comes from the boundary row BEFORE that sweep through the adjoint of the upper-bidiagonal system:
//   y_k = (w_k - c_{k-2} y_{k-2}) / d''_k   =>   sum_{k>=2} w_k u_k = sum_k y_k g''_k + u_par sum_k y_k e_k,
//   u_par = (target - sum y_k g''_k) / (w_par + sum y_k e_k)       (Neumann rows: w_k = k^2, target 0).
// d''_k and e_k depend on (k, sigma) only; the up sweep recomputes them, the down sweep reads (c^_k, e^_k) from a table
// (they obey an ascending recurrence, and the backward form d''_{k-2} = a_k c_{k-2} / (d_k - d''_k) cancels).
// The system is diagonally dominant in both directions (|a_k| + |c_k| < d_k - 1 + 1), so no pivoting either way.
// ================================================================================================
struct PivotUp {
    double dm1, dm2;   // 1/d''_{k-1}, 1/d''_{k-2}
    double em1, em2;   // e_{k-1}, e_{k-2}
    __device__ __forceinline__ void init() { dm1 = dm2 = em1 = em2 = 0.0; }
    // row k (2 <= k <= N): returns 1/d''_k; m = a_k / d''_{k-2} (0 in the first row of a parity), e = e_k, c = c_k,
    // cm2 = c_{k-2} (c_j = -sigma r_j for j + 4 <= N, else 0)
    __device__ __forceinline__ double step(int k, int N, double sigma, double &m, double &e, double &c, double &cm2) {
        const double ak = -sigma * helm_p(k);
        double d = 1.0 + ((k + 2 <= N) ? sigma * (-helm_q(k)) : 0.0);
        c = (k + 4 <= N) ? -sigma * helm_r(k) : 0.0;
        cm2 = (k >= 4 && k + 2 <= N) ? -sigma * helm_r(k - 2) : 0.0;
        if (k < 4) { m = 0.0; e = -ak; }
        else {
            m = ak * dm2;
            d -= m * cm2;
            e = -m * em2;
        }
        const double di = 1.0 / d;
        dm2 = dm1; dm1 = di;
        em2 = em1; em1 = e;
        return di;
    }
};

struct ElimUpNeu {   // Neumann rows (sum k^2 u_k = 0 per parity), complex right-hand side
    PivotUp pv;
    cplx gm2, gm1;            // g''_{k-2}, g''_{k-1}
    double ym2, ym1;          // adjoint weights y_{k-2}, y_{k-1}
    cplx Je, Jo;              // sum y_k g''_k per parity
    double Ee, Eo;            // sum y_k e_k per parity
    __device__ __forceinline__ void init() { pv.init(); gm2 = gm1 = Je = Jo = cz(); ym2 = ym1 = Ee = Eo = 0.0; }
    // row k: F(k-2), F(k), F(k+2) of the right-hand side (zero-extended above N-2).  Returns g^_k = g''_k / d''_k.
    __device__ __forceinline__ cplx row(int k, int N, double sigma, cplx fm2, cplx f0, cplx fp2) {
        double m, e, c, cm2;
        const double di = pv.step(k, N, sigma, m, e, c, cm2);
        cplx g = cfma(helm_p(k), fm2, cfma(helm_q(k), f0, cscale(fp2, helm_r(k))));
        g = cfma(-m, gm2, g);
        const double y = ((double)k * k - cm2 * ym2) * di;
        if (k & 1) { Jo = cfma(y, g, Jo); Eo = fma(y, e, Eo); } else { Je = cfma(y, g, Je); Ee = fma(y, e, Ee); }
        gm2 = gm1; gm1 = g;
        ym2 = ym1; ym1 = y;
        return cscale(g, di);
    }
    __device__ __forceinline__ void finish(cplx &u0, cplx &u1) const {
        u0 = cscale(Je, -1.0 / Ee);              // weight of u_0 itself: 0^2
        u1 = cscale(Jo, -1.0 / (1.0 + Eo));      // weight of u_1 itself: 1^2
    }
};

// Dirichlet rows (sum u_k = 0 per parity) plus the k^2-weighted functional of the solution: the w problem
// (D^2 - k^2) w = theta_p, whose influence-matrix coefficient needs sum k^2 w_p per parity (k_elim2 / ElimDown::second).
template <bool GEN = false>   // GEN: also the k^2 (k^2 - 1) / 3 functional (T_k''(+-1): free-slip walls, row f3)
struct ElimUpDir2 {
    PivotUp pv;
    cplx gm2, gm1;            // g''_{k-2}, g''_{k-1}
    double ym2, ym1;          // adjoint of the boundary row (weights 1)
    double sm2, sm1;          // adjoint of the second functional (weights k^2)
    double tm2, tm1;          // GEN: adjoint of the third functional (weights k^2 (k^2 - 1) / 3)
    cplx Je, Jo, Ke, Ko, Me, Mo;      // sum y_k g''_k, sum s_k g''_k, sum t_k g''_k per parity
    double Ee, Eo, Fe, Fo, Ge, Go;    // sum y_k e_k, sum s_k e_k, sum t_k e_k per parity
    __device__ __forceinline__ void init() {
        pv.init();
        gm2 = gm1 = Je = Jo = Ke = Ko = Me = Mo = cz();
        ym2 = ym1 = sm2 = sm1 = tm2 = tm1 = Ee = Eo = Fe = Fo = Ge = Go = 0.0;
    }
    __device__ __forceinline__ cplx row(int k, int N, double sigma, cplx fm2, cplx f0, cplx fp2) {
        double m, e, c, cm2;
        const double di = pv.step(k, N, sigma, m, e, c, cm2);
        cplx g = cfma(helm_p(k), fm2, cfma(helm_q(k), f0, cscale(fp2, helm_r(k))));
        g = cfma(-m, gm2, g);
        const double k2 = (double)k * k;
        const double y = (1.0 - cm2 * ym2) * di;
        const double sq = (k2 - cm2 * sm2) * di;
        if (k & 1) { Jo = cfma(y, g, Jo); Eo = fma(y, e, Eo); Ko = cfma(sq, g, Ko); Fo = fma(sq, e, Fo); }
        else       { Je = cfma(y, g, Je); Ee = fma(y, e, Ee); Ke = cfma(sq, g, Ke); Fe = fma(sq, e, Fe); }
        if (GEN) {
            const double t = (k2 * (k2 - 1.0) * (1.0 / 3.0) - cm2 * tm2) * di;
            if (k & 1) { Mo = cfma(t, g, Mo); Go = fma(t, e, Go); } else { Me = cfma(t, g, Me); Ge = fma(t, e, Ge); }
            tm2 = tm1; tm1 = t;
        }
        gm2 = gm1; gm1 = g;
        ym2 = ym1; ym1 = y;
        sm2 = sm1; sm1 = sq;
        return cscale(g, di);
    }
    // u_0, u_1 of the particular solution and its k^2-weighted parity sums
    __device__ __forceinline__ void finish(cplx &u0, cplx &u1, cplx &de, cplx &dodd) const {
        u0 = cscale(Je, -1.0 / (1.0 + Ee));
        u1 = cscale(Jo, -1.0 / (1.0 + Eo));
        de = cfma(Fe, u0, Ke);                   // 0^2 u_0 + K_e + u_0 F_e
        dodd = cadd(u1, cfma(Fo, u1, Ko));       // 1^2 u_1 + K_o + u_1 F_o
    }
    // GEN: its k^2 (k^2 - 1) / 3 - weighted parity sums (the weights of k = 0, 1 vanish)
    __device__ __forceinline__ void third(cplx u0, cplx u1, cplx &me, cplx &mo) const {
        me = cfma(Ge, u0, Me);
        mo = cfma(Go, u1, Mo);
    }
};

// table of the down sweep: tab[k] = (c^_k, e^_k) = (c_k, e_k) / d''_k, k = 2..N (rows 0, 1 unused)
struct ElimUpSetupArgs {
    ColGeom g;
    double2 *tab;   // [N+1][ncols]
    double shift;   // sigma = k^2 + shift
};

__global__ void __launch_bounds__(NT_COL) k_elimup_setup(const __grid_constant__ ElimUpSetupArgs a) {
    const ColGeom &g = a.g;
    const int col = blockIdx.x * blockDim.x + threadIdx.x;
    if (col >= g.ncols) return;
    double kx, ky;
    col_wavenumbers(g, col, kx, ky);
    const double sigma = kx * kx + ky * ky + a.shift;
    const size_t st = g.ncols;
    PivotUp pv;
    pv.init();
    a.tab[col] = make_double2(0.0, 0.0);
    a.tab[st + col] = make_double2(0.0, 0.0);
    for (int k = 2; k <= g.N; ++k) {
        double m, e, c, cm2;
        const double di = pv.step(k, g.N, sigma, m, e, c, cm2);
        a.tab[k * st + col] = make_double2(c * di, e * di);
    }
}

// ---- K_A: row a9 + first elimination ------------------------------------------------------------------
// CTA = 32 consecutive columns, three warps.  Warps 0 and 1: the omega_z AND theta chains of 16 columns each, one
// thread per (column, real / imaginary part) - both chains need the same five product rows and the same pivots,
// so these are fetched once (profiles/r1d: as separate warps the two chains read them twice, 3.7 GB per step).
// Warp 2: the psi chain of all 32 columns (complex).
// omega_z (column 0: u-bar)   f = -H_omega / gamma,  sigma = k^2 + 1/gamma, Dirichlet
// theta   (column 0: v-bar)   f = -H_w / gamma,      same sigma, Dirichlet (homogeneous part added later)
// chain 2: psi                         f = H_phi / gamma_phi, sigma = k^2 + lambda_phi, Neumann
// Every chain works in place: it reads x^n at row n going down and writes g' at row n + 2.
struct RhsElimArgs {
    ColGeom g;
    const cplx *txx, *txy, *txz, *tyy, *tyz, *q, *c;   // txx, tyy hold the deviatoric T_xx - T_zz, T_yy - T_zz
    const cplx *fx, *fy, *fz;         // FORCE only: the surface-tension force -c lap(phi) grad(phi), added to S = div T
    cplx *om, *th, *phi;              // in: omega^n, theta^n, phi^n; out: g' arrays (slots 0,1 = u_0, u_1)
    cplx *h_om, *h_w, *h_phi;
    const double *dinv_ns, *dinv_ch;
    const double *ab;
    double dt, gamma, inv_pe, e_phi, gradp, lam_phi, gam_phi;
    int phase;
    int wall_top, wall_bot;           // 0 = no-slip, 1 = free-slip
    const double *thh;                // LAZY: real homogeneous solution theta_h [nz][ncols]
    const cplx *coef;                 // LAZY: [2][ncols] influence-matrix coefficients of the last step (0 after set_state)
};

constexpr int RHS_COLS = 32;   // columns per CTA of k_rhs_elim (blockDim = 32 * number of chains)

#ifndef RHS_MINB
#define RHS_MINB 4
#endif
// GEN: walls that are not both no-slip (row f3).  FORCE: the surface tension enters as a force vector F next to the flux
// tensor: N_omega += i (kx F_y - ky F_x), N_w += -k^2 F_z - D (i kx F_x + i ky F_y), S-bar += F(0,0).
// <false, false> is the product path, unchanged.
// LAZY: theta^n in memory is the particular solution theta_p of the last step; its influence-matrix correction
// A_par theta_h (the coefficients are still in a.coef) is applied here, where theta^n is read anyway, instead of by a
// read-modify-write of the whole array in k_finish (three-sweep form).
template <bool GEN, bool FORCE, bool LAZY = false>
__global__ void __launch_bounds__(96, (FORCE ? 3 : RHS_MINB)) k_rhs_elim(const __grid_constant__ RhsElimArgs a) {
    const ColGeom &g = a.g;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const bool nschain = warp < 2;
    const int col = blockIdx.x * RHS_COLS + (nschain ? warp * 16 + (lane >> 1) : lane);
    if (col >= g.ncols) return;
    double kx, ky;
    col_wavenumbers(g, col, kx, ky);
    const double k2 = kx * kx + ky * ky;
    const bool mean = (col == 0);
    const size_t st = g.ncols;
    const int N = g.N, nkz = g.nkz;
    const double ab0 = a.ab[0], ab1 = a.ab[1];
    const double dt = a.dt, gam = a.gamma;
    // Software pipelining: the operands of row n - 1 are loaded into registers before row n is computed, so
    // each row costs one (prefetched, L2-hit) load latency instead of one per dependent load group
    // (profiles/r1c: 77 % of the stall samples were long-scoreboard waits).
    if (nschain) {
        const int c = lane & 1;                       // 0: real part, 1: imaginary part
        const double sg = c ? 1.0 : -1.0;             // (i z)_c = sg * z_{1-c}
        const double sigma = k2 + 1.0 / gam, fs = -1.0 / gam;
        const cplx *__restrict__ txx = a.txx + col, *__restrict__ txy = a.txy + col, *__restrict__ txz = a.txz + col;
        const cplx *__restrict__ tyy = a.tyy + col, *__restrict__ tyz = a.tyz + col;
        // component views: element (n, col) of a cplx array = doubles 2 (n st + col) + {0, 1}
        double *xo = reinterpret_cast<double *>(a.om + col) + c, *xt = reinterpret_cast<double *>(a.th + col) + c;
        double *ho = reinterpret_cast<double *>(a.h_om + col) + c, *hw = reinterpret_cast<double *>(a.h_w + col) + c;
        const size_t st2 = 2 * st;
        struct RowIn { double xo, xt, ho, hw, t0, t1, t3; cplx t2, t4; cplx f0, f1; double f2; double thh; };
        PivotDown pv;
        pv.init();
        double lazy_e = 0.0, lazy_o = 0.0;
        if (LAZY) {
            lazy_e = reinterpret_cast<const double *>(a.coef + col)[c];
            lazy_o = reinterpret_cast<const double *>(a.coef + st + col)[c];
        }
        auto load = [&](int n) {
            RowIn r;
            r.xo = xo[n * st2]; r.xt = xt[n * st2];
            if (LAZY) r.thh = a.thh[n * st + col];
            r.ho = r.hw = r.t0 = r.t1 = r.t3 = 0.0; r.t2 = r.t4 = cz();
            if (n < nkz) {
                const size_t o = n * st;
                r.ho = ho[n * st2]; r.hw = hw[n * st2];
                r.t0 = reinterpret_cast<const double *>(txx + o)[c];
                r.t1 = reinterpret_cast<const double *>(txy + o)[c];
                r.t3 = reinterpret_cast<const double *>(tyy + o)[c];
                r.t2 = txz[o]; r.t4 = tyz[o];
                if (FORCE) {
                    r.f0 = a.fx[col + o]; r.f1 = a.fy[col + o];
                    r.f2 = reinterpret_cast<const double *>(a.fz + col + o)[c];
                }
            }
            return r;
        };
        // derivative chains of real sequences (same recurrences as Chain1 / Chain2)
        double Ra1 = 0, Rb1 = 0, Rb2 = 0;                               // D R
        double Ba1 = 0, Bb1 = 0, Bb2 = 0;                               // D B
        double Aa1 = 0, Ab1 = 0, Ab2 = 0, Ac1 = 0, Ac2 = 0;             // D^2 A
        double Oa1 = 0, Ob1 = 0, Ob2 = 0, Oc1 = 0, Oc2 = 0;             // D^2 omega
        double Ta1 = 0, Tb1 = 0, Tb2 = 0, Tc1 = 0, Tc2 = 0;             // D^2 theta
        ElimDown2R<GEN> el;
        el.init();
        RowIn nx = load(N);
        for (int n = N; n >= 0; --n) {
            RowIn r = nx;
            if (n > 0) nx = load(n - 1);
            if (LAZY) r.xt = fma(r.thh, (n & 1) ? lazy_o : lazy_e, r.xt);     // theta^n = theta_p + A_par theta_h
            const int np = n - g.pf_rhs;
            if (np >= 0 && c == 0) {
                pf_l2(a.om + col + np * st); pf_l2(a.th + col + np * st);
                if (LAZY) pf_l2(a.thh + col + np * st);
                if (np < nkz) {
                    pf_l2(txz + np * st); pf_l2(txx + np * st); pf_l2(txy + np * st); pf_l2(tyy + np * st); pf_l2(tyz + np * st);
                    pf_l2(a.h_om + col + np * st); pf_l2(a.h_w + col + np * st);
                }
            }
            const double f = 2.0 * (n + 1), h = (n == 0) ? 0.5 : 1.0;
            const bool low = n < nkz;
            const double t2c = c ? r.t2.y : r.t2.x, t2o = c ? r.t2.x : r.t2.y;
            const double t4c = c ? r.t4.y : r.t4.x, t4o = c ? r.t4.x : r.t4.y;
            // N_omega = P + D R (Eq. 14 expanded); column 0: S-bar_x = D T_xz (+ G)
            // N_w = D B - D^2 A - k^2 A (Eq. 15 expanded); column 0: S-bar_y = D T_yz
            double P = 0.0, R = 0.0, A = 0.0, B = 0.0;
            if (low) {
                if (mean) { R = t2c; B = t4c; }
                else {
                    P = r.t1 * (ky * ky - kx * kx) + (r.t0 - r.t3) * (kx * ky);
                    R = sg * (kx * t4o - ky * t2o);
                    A = sg * (kx * t2o + ky * t4o);
                    // kx^2 Txx + 2 kx ky Txy + ky^2 Tyy - k^2 Tzz with the deviatoric inputs
                    B = r.t0 * (kx * kx) + r.t1 * (2.0 * kx * ky) + r.t3 * (ky * ky);
                }
            }
            double extra_w = 0.0;
            if (FORCE && low) {
                const double f0c = c ? r.f0.y : r.f0.x, f0o = c ? r.f0.x : r.f0.y;
                const double f1c = c ? r.f1.y : r.f1.x, f1o = c ? r.f1.x : r.f1.y;
                if (mean) { P = f0c; extra_w = f1c; }                     // S-bar_x += F_x(0,0), S-bar_y += F_y(0,0)
                else {
                    P += sg * (kx * f1o - ky * f0o);                      // i (kx F_y - ky F_x)
                    B -= sg * (kx * f0o + ky * f1o);                      // -D (i kx F_x + i ky F_y): B is differentiated once
                    extra_w = -k2 * r.f2;                                 // -k^2 F_z
                }
            }
            const double dR = fma(f, Ra1, Rb2) * h; Ra1 = R; Rb2 = Rb1; Rb1 = dR;
            const double dB = fma(f, Ba1, Bb2) * h; Ba1 = B; Bb2 = Bb1; Bb1 = dB;
            const double dA = fma(f, Aa1, Ab2) * h, ddA = fma(f, Ab1, Ac2) * h;
            Aa1 = A; Ab2 = Ab1; Ab1 = dA; Ac2 = Ac1; Ac1 = ddA;
            const double dO = fma(f, Oa1, Ob2) * h, ddO = fma(f, Ob1, Oc2) * h;
            Oa1 = r.xo; Ob2 = Ob1; Ob1 = dO; Oc2 = Oc1; Oc1 = ddO;
            const double dT = fma(f, Ta1, Tb2) * h, ddT = fma(f, Tb1, Tc2) * h;
            Ta1 = r.xt; Tb2 = Tb1; Tb1 = dT; Tc2 = Tc1; Tc1 = ddT;
            double nl_o = P + dR;
            if (mean && n == 0 && c == 0) nl_o += a.gradp;
            const double nl_w = (dB - ddA) + A * (-k2) + extra_w;
            double so = nl_o * ab0, sw = nl_w * ab0;
            if (low) {
                so = fma(ab1, r.ho, so); sw = fma(ab1, r.hw, sw);
                ho[n * st2] = nl_o; hw[n * st2] = nl_w;
            }
            const double Ho = fma(dt, so, fma(gam, fma(-k2, r.xo, ddO), r.xo));
            const double Hw = fma(dt, sw, fma(gam, fma(-k2, r.xt, ddT), r.xt));
            if (n <= N - 2) {
                const int k = n + 2;
                double go, gw;
                el.row(k, N, sigma, Ho * fs, Hw * fs, pv.step(k, N, sigma), go, gw);
                xo[k * st2] = go; xt[k * st2] = gw;
            }
        }
        double u0, u1;
        if (GEN) {
            // omega_z (column 0: u-bar): value at a no-slip wall, derivative at a free-slip wall.  theta_p: value at both
            // walls (the influence matrix closes the w problem); column 0 carries v-bar there, with u-bar's conditions
            el.finish_walls(sigma, 0, a.wall_top, a.wall_bot, u0, u1);
            xo[0] = u0; xo[st2] = u1;
            el.finish_walls(sigma, 1, mean ? a.wall_top : 0, mean ? a.wall_bot : 0, u0, u1);
            xt[0] = u0; xt[st2] = u1;
        } else {
            el.finish(sigma, 0, u0, u1);
            xo[0] = u0; xo[st2] = u1;
            el.finish(sigma, 1, u0, u1);
            xt[0] = u0; xt[st2] = u1;
        }
    } else {
        const double sigma = k2 + a.lam_phi, fs = 1.0 / a.gam_phi;
        const cplx *__restrict__ qq = a.q + col, *__restrict__ cc = a.c + col;
        cplx *x = a.phi + col, *hist = a.h_phi + col;
        struct RowIn { cplx x, h, t0, t1; };
        ElimDown el;
        el.init();
        PivotDown pv;
        pv.init();
        auto load = [&](int n) {
            RowIn r;
            const size_t o = n * st;
            r.x = x[o];
            r.h = r.t0 = r.t1 = cz();
            if (n < nkz) { r.h = hist[o]; r.t0 = qq[o]; r.t1 = cc[o]; }
            return r;
        };
        Chain2 cE;
        cE.init();
        RowIn nx = load(N);
        for (int n = N; n >= 0; --n) {
            const RowIn r = nx;
            if (n > 0) nx = load(n - 1);
            const int np = n - g.pf_rhs;
            if (np >= 0) {
                pf_l2(x + np * st);
                if (np < nkz) { pf_l2(qq + np * st); pf_l2(cc + np * st); pf_l2(hist + np * st); }
            }
            const double f = 2.0 * (n + 1), h = (n == 0) ? 0.5 : 1.0;
            const size_t o = n * st;
            const bool low = n < nkz;
            cplx E = cz(), Q = cz();
            if (low) {
                Q = r.t0;
                E = cscale(cfma(-a.e_phi, r.x, r.t1), a.inv_pe);
            }
            const cplx ddE = cE.step(E, f, h);
            const cplx s_phi = csub(cfma(-k2, E, ddE), Q);
            cplx nl = cscale(s_phi, ab0);
            if (low) { nl = cfma(ab1, r.h, nl); hist[o] = s_phi; }
            const cplx H = cfma(dt, nl, r.x);
            if (n <= N - 2) {
                const int k = n + 2;
                x[k * st] = el.row<true, false>(k, N, sigma, cscale(H, fs), pv.step(k, N, sigma));
            }
        }
        cplx u0, u1;
        el.finish<true>(sigma, 0.0, 0.0, u0, u1);
        x[0] = u0; x[st] = u1;
    }
}

// ---- K_B / K_D: up sweep u_k = (g'_k - a_k u_{k-2}) / d'_k, optional homogeneous correction ------------
struct SubstArgs {
    ColGeom g;
    cplx *x[3];                 // per chain: g' array in (slots 0,1 = u_0,u_1), solution out (in place)
    const double *dinv[3];
    double shift[3];
    int nchains;
    int pair01;                 // chains 0 and 1 share sigma and the pivot table: one thread does both (grid.y = nchains - 1)
    // influence-matrix correction (chain 0 only, when coef != nullptr): x += A_par * wh ; th += A_par * thh
    const cplx *coef;           // [2][ncols]: A_e, A_o
    const double *wh, *thh;     // real homogeneous solutions [nz][ncols]
    cplx *th;
    // W3 (three-sweep w problem): the pair's theta_p rows feed the upward elimination of (D^2 - k^2) w = theta_p
    cplx *w3_out;               // g^ of that elimination (slots 0, 1 = w_p,0, w_p,1)
    const double *w3_hw;        // [4][ncols]: sum k^2 w_h per parity, then sum k^2 (k^2 - 1)/3 w_h (k_hom_tables)
    cplx *w3_coef;              // [2][ncols] out: influence-matrix coefficients A_e, A_o
    int wall_top, wall_bot;     // GEN: 0 = no-slip (Dw = 0), 1 = free-slip (D^2 w = 0)
};

// The sweeps work in place, so the compiler cannot move the load of row k + 1 above the store of row k (same
// pointer, run-time stride): every row then costs a full memory latency, which dominates on small grids (few
// columns, little parallelism).  The loops below therefore load a GROUP of G rows into registers before the
// previous group's results are stored (different rows: no hazard).  G is a template parameter chosen by the host:
// 4 on small grids (latency-bound), 2 above 60 k columns (DRAM-bound: more resident threads win; measured at
// 1024x512x513: solve 4.23 ms with 2, 4.36 with 4, 4.51 with 8; at 256x256x257: 0.43 with 4, 0.42 with 8).

// UP: the psi chain (chain 2 of the first substitution) does not store psi but feeds it, row by row, into the upward
// elimination of the phi solve (ElimUpNeu) and stores g^_k of that solve instead; k_finish completes it on its way down.
template <int G, bool UP, bool W3 = false, bool GEN = false>
__device__ __forceinline__ void subst_body(const SubstArgs &a, int by) {
    const ColGeom &g = a.g;
    const int col = blockIdx.x * blockDim.x + threadIdx.x;
    if (col >= g.ncols) return;
    const int chain = UP ? 2 : (a.pair01 ? by + 1 : by);   // UP: the psi chain, in a block row of k_elim2up
    double kx, ky;
    col_wavenumbers(g, col, kx, ky);
    const size_t st = g.ncols;
    const int N = g.N;
    if (!UP && a.pair01 && by == 0) {      // omega_z and theta: same recurrence coefficients, two right-hand sides
        const double sigma = kx * kx + ky * ky + a.shift[0];
        cplx *x0 = a.x[0] + col, *x1 = a.x[1] + col;
        const double *__restrict__ dinv = a.dinv[0] + col;
        cplx um2 = x0[0], um1 = x0[st], vm2 = x1[0], vm1 = x1[st];
        ElimUpDir2<GEN> ew;
        cplx w4 = cz(), w3 = cz(), w2 = vm2, w1 = vm1;      // F(k-4) .. F(k-1) of the w solve's right-hand side theta_p
        const double k2w = kx * kx + ky * ky;
        cplx *wout = W3 ? a.w3_out + col : nullptr;
        if (W3) ew.init();
        cplx q0[G], q1[G];
        double dq[G];
        auto load = [&](int k0, cplx (&p0)[G], cplx (&p1)[G], double (&d)[G]) {
#pragma unroll
            for (int i = 0; i < G; ++i) {
                const int k = k0 + i;
                if (k <= N) { p0[i] = x0[k * st]; p1[i] = x1[k * st]; d[i] = dinv[k * st]; }
            }
        };
        load(2, q0, q1, dq);
        for (int k0 = 2; k0 <= N; k0 += G) {
            cplx n0[G], n1[G];
            double dn[G];
            load(k0 + G, n0, n1, dn);
            const int kp = k0 + 2 * G + g.pf;
#pragma unroll
            for (int i = 0; i < G; ++i)
                if (kp + i <= N) { pf_l2(x0 + (kp + i) * st); pf_l2(x1 + (kp + i) * st); pf_l2(dinv + (kp + i) * st); }
#pragma unroll
            for (int i = 0; i < G; ++i) {
                const int k = k0 + i;
                if (k <= N) {
                    const double ak = -sigma * helm_p(k);
                    const cplx u = cscale(cfma(-ak, um2, q0[i]), dq[i]);
                    const cplx v = cscale(cfma(-ak, vm2, q1[i]), dq[i]);
                    um2 = um1; um1 = u; vm2 = vm1; vm1 = v;
                    x0[k * st] = u; x1[k * st] = v;
                    if (W3) {
                        const cplx fk = (k <= N - 2) ? v : cz();    // the right-hand side is zero-extended above N - 2
                        if (k >= 4) wout[(k - 2) * st] = ew.row(k - 2, N, k2w, w4, w2, fk);
                        w4 = w3; w3 = w2; w2 = w1; w1 = fk;
                    }
                }
            }
#pragma unroll
            for (int i = 0; i < G; ++i) { q0[i] = n0[i]; q1[i] = n1[i]; dq[i] = dn[i]; }
        }
        if (W3) {       // rows N - 1 and N, boundary unknowns, influence-matrix coefficients (as k_elim2, no-slip walls)
            wout[(N - 1) * st] = ew.row(N - 1, N, k2w, w4, cz(), cz());
            wout[N * st] = ew.row(N, N, k2w, w3, cz(), cz());
            cplx u0, u1, de, dodd;
            ew.finish(u0, u1, de, dodd);
            wout[0] = u0; wout[st] = u1;
            const bool off = (col == 0);
            if (!GEN) {
                a.w3_coef[col] = off ? cz() : cscale(de, -1.0 / a.w3_hw[col]);
                a.w3_coef[st + col] = off ? cz() : cscale(dodd, -1.0 / a.w3_hw[st + col]);
            } else {     // per wall Dw = 0 (no-slip) or D^2 w = 0 (free-slip): the 2 x 2 closure of k_elim2<., true>
                cplx me, mo;
                ew.third(u0, u1, me, mo);
                const double Keh = a.w3_hw[col], Koh = a.w3_hw[st + col], Meh = a.w3_hw[2 * st + col], Moh = a.w3_hw[3 * st + col];
                cplx Ae, Ao;
                if (a.wall_top == 1 && a.wall_bot == 1) { Ae = cscale(me, -1.0 / Meh); Ao = cscale(mo, -1.0 / Moh); }
                else {
                    double a11, a12, a21, a22;
                    cplx b1, b2;
                    if (a.wall_top == 1) { a11 = Meh; a12 = Moh; b1 = cscale(cadd(me, mo), -1.0); a21 = -Keh; a22 = Koh; b2 = csub(de, dodd); }
                    else                 { a11 = Keh; a12 = Koh; b1 = cscale(cadd(de, dodd), -1.0); a21 = Meh; a22 = -Moh; b2 = cscale(csub(me, mo), -1.0); }
                    const double idet = 1.0 / (a11 * a22 - a12 * a21);
                    Ae = cscale(csub(cscale(b1, a22), cscale(b2, a12)), idet);
                    Ao = cscale(csub(cscale(b2, a11), cscale(b1, a21)), idet);
                }
                a.w3_coef[col] = off ? cz() : Ae;
                a.w3_coef[st + col] = off ? cz() : Ao;
            }
        }
        return;
    }
    const double sigma = kx * kx + ky * ky + a.shift[chain];
    cplx *x = a.x[chain] + col;
    const double *__restrict__ dinv = a.dinv[chain] + col;
    const bool corr = !UP && (chain == 0 && a.coef != nullptr);
    cplx Ae = cz(), Ao = cz();
    if (corr) { Ae = a.coef[col]; Ao = a.coef[st + col]; }
    cplx um2 = x[0], um1 = x[st];
    constexpr bool upel = UP;
    ElimUpNeu eu;
    cplx w4 = cz(), w3 = cz(), w2 = um2, w1 = um1;      // F(k-4) .. F(k-1) of the phi solve's right-hand side psi
    if (UP) eu.init();
    if (corr) {
        x[0] = cfma(a.wh[col], Ae, um2);
        x[st] = cfma(a.wh[st + col], Ao, um1);
        a.th[col] = cfma(a.thh[col], Ae, a.th[col]);
        a.th[st + col] = cfma(a.thh[st + col], Ao, a.th[st + col]);
    }
    struct Row { cplx x, th; double di, wh, thh; };
    auto load = [&](int k0, Row (&r)[G]) {
#pragma unroll
        for (int i = 0; i < G; ++i) {
            const int k = k0 + i;
            if (k <= N) {
                r[i].x = x[k * st]; r[i].di = dinv[k * st];
                if (corr) { const size_t o = k * st + col; r[i].wh = a.wh[o]; r[i].thh = a.thh[o]; r[i].th = a.th[o]; }
            }
        }
    };
    Row q[G];
    load(2, q);
    for (int k0 = 2; k0 <= N; k0 += G) {
        Row nx[G];
        load(k0 + G, nx);
        const int kp = k0 + 2 * G + g.pf;
#pragma unroll
        for (int i = 0; i < G; ++i)
            if (kp + i <= N) {
                pf_l2(x + (kp + i) * st); pf_l2(dinv + (kp + i) * st);
                if (corr) { pf_l2(a.wh + (kp + i) * st + col); pf_l2(a.thh + (kp + i) * st + col); pf_l2(a.th + (kp + i) * st + col); }
            }
#pragma unroll
        for (int i = 0; i < G; ++i) {
            const int k = k0 + i;
            if (k <= N) {
                const double ak = -sigma * helm_p(k);
                const cplx u = cscale(cfma(-ak, um2, q[i].x), q[i].di);
                um2 = um1; um1 = u;
                if (UP && upel) {
                    const cplx fk = (k <= N - 2) ? u : cz();        // the right-hand side is zero-extended above N - 2
                    if (k >= 4) x[(k - 2) * st] = eu.row(k - 2, N, sigma, w4, w2, fk);
                    w4 = w3; w3 = w2; w2 = w1; w1 = fk;
                } else if (corr) {
                    const size_t o = k * st + col;
                    const cplx A = (k & 1) ? Ao : Ae;
                    x[k * st] = cfma(q[i].wh, A, u);
                    a.th[o] = cfma(q[i].thh, A, q[i].th);
                } else {
                    x[k * st] = u;
                }
            }
        }
#pragma unroll
        for (int i = 0; i < G; ++i) q[i] = nx[i];
    }
    if (UP && upel) {       // rows N - 1 and N: F(k) = F(k + 2) = 0
        x[(N - 1) * st] = eu.row(N - 1, N, sigma, w4, cz(), cz());
        x[N * st] = eu.row(N, N, sigma, w3, cz(), cz());
        cplx u0, u1;
        eu.finish(u0, u1);
        x[0] = u0; x[st] = u1;
    }
}

template <int G>
__global__ void __launch_bounds__(NT_COL) k_subst(const __grid_constant__ SubstArgs a) { subst_body<G, false>(a, blockIdx.y); }

// Three-sweep form of both two-stage problems: block row 0 = the (omega_z, theta_p) pair, whose theta_p rows also feed the
// upward elimination of the w solve (ElimUpDir2); block row 1 (phase field) = the psi chain feeding the upward
// elimination of the phi solve (ElimUpNeu).  k_finish<., true> back-substitutes both on its way down.
template <int G, bool GEN = false>
__global__ void __launch_bounds__(NT_COL) k_subst3(const __grid_constant__ SubstArgs a) {
    if (blockIdx.y == 0) subst_body<G, false, true, GEN>(a, 0);
    else subst_body<G, true>(a, 0);
}

// ---- K_C: second elimination of the two-stage problems (RHS = the first stage's solution) ----------------
// chain 0: (D^2 - k^2) w = theta_p, Dirichlet, plus the influence coefficient A_par = -sum k^2 w_p / sum k^2 w_h
// chain 1: (D^2 - k^2 - lambda) phi = psi, Neumann (in place)
struct Elim2Args {
    ColGeom g;
    const cplx *th;   cplx *w;      // chain 0
    cplx *phi;                      // chain 1 (in place)
    const double *dinv_po, *dinv_ch;
    const double *hw;               // [4][ncols]: sum_{even}, sum_{odd} of k^2 w_h, then of k^2 (k^2 - 1)/3 w_h
    cplx *coef;                     // [2][ncols] out
    double lam_phi;
    int phase;
    int wall_top, wall_bot;         // 0 = no-slip (Dw = 0), 1 = free-slip (D^2 w = 0)
};

template <int G, bool GEN>
__device__ __forceinline__ void elim2_body(const Elim2Args &a, int chain) {
    const ColGeom &g = a.g;
    const int col = blockIdx.x * blockDim.x + threadIdx.x;
    if (col >= g.ncols) return;
    double kx, ky;
    col_wavenumbers(g, col, kx, ky);
    const double k2 = kx * kx + ky * ky;
    const size_t st = g.ncols;
    const int N = g.N;
    ElimDown el;
    el.init();
    if (chain == 0) {
        const cplx *__restrict__ in = a.th + col;
        cplx *__restrict__ out = a.w + col;
        PivotDown pv;
        pv.init();
            cplx q[G];
        auto load = [&](int k0, cplx (&r)[G]) {          // rows k0, k0 - 1, .. (descending)
#pragma unroll
            for (int i = 0; i < G; ++i) if (k0 - i >= 2) r[i] = in[(k0 - i - 2) * st];
        };
        load(N, q);
        for (int k0 = N; k0 >= 2; k0 -= G) {
            cplx nx[G];
            load(k0 - G, nx);
            const int kp = k0 - 2 * G - g.pf;
#pragma unroll
            for (int i = 0; i < G; ++i) if (kp - i >= 2) pf_l2(in + (kp - i - 2) * st);
#pragma unroll
            for (int i = 0; i < G; ++i) {
                const int k = k0 - i;
                if (k >= 2) out[k * st] = el.row<false, true, GEN>(k, N, k2, q[i], pv.step(k, N, k2));
            }
#pragma unroll
            for (int i = 0; i < G; ++i) q[i] = nx[i];
        }
        cplx u0, u1, de, dodd;
        el.finish<false>(k2, 0.0, 0.0, u0, u1);
        el.second(k2, u0, u1, de, dodd);
        out[0] = u0; out[st] = u1;
        const bool off = (col == 0);
        if (!GEN) {
            a.coef[col] = off ? cz() : cscale(de, -1.0 / a.hw[col]);
            a.coef[st + col] = off ? cz() : cscale(dodd, -1.0 / a.hw[st + col]);
        } else {
            // w = w_p + A_e w_h,e + A_o w_h,o with, per wall, Dw = 0 (no-slip) or D^2 w = 0 (free-slip):
            //   T_k'(+-1) = (+-1)^(k+1) k^2       -> Dw(+1) = K_e + K_o,    Dw(-1) = -K_e + K_o
            //   T_k''(+-1) = (+-1)^k k^2(k^2-1)/3 -> D^2 w(+1) = M_e + M_o, D^2 w(-1) = M_e - M_o
            cplx me, mo;
            el.third(k2, u0, u1, me, mo);
            const double Keh = a.hw[col], Koh = a.hw[st + col], Meh = a.hw[2 * st + col], Moh = a.hw[3 * st + col];
            cplx Ae, Ao;
            if (a.wall_top == 1 && a.wall_bot == 1) { Ae = cscale(me, -1.0 / Meh); Ao = cscale(mo, -1.0 / Moh); }
            else {
                double a11, a12, a21, a22;
                cplx b1, b2;
                if (a.wall_top == 1) { a11 = Meh; a12 = Moh; b1 = cscale(cadd(me, mo), -1.0); a21 = -Keh; a22 = Koh; b2 = csub(de, dodd); }
                else                 { a11 = Keh; a12 = Koh; b1 = cscale(cadd(de, dodd), -1.0); a21 = Meh; a22 = -Moh; b2 = cscale(csub(me, mo), -1.0); }
                const double idet = 1.0 / (a11 * a22 - a12 * a21);
                Ae = cscale(csub(cscale(b1, a22), cscale(b2, a12)), idet);
                Ao = cscale(csub(cscale(b2, a11), cscale(b1, a21)), idet);
            }
            a.coef[col] = off ? cz() : Ae;
            a.coef[st + col] = off ? cz() : Ao;
        }
    } else {
        if (!a.phase) return;
        const double sigma = k2 + a.lam_phi;
        cplx *x = a.phi + col;
        PivotDown pv;
        pv.init();
        // in place: row k - 2 is read (as the right-hand side of row k) before it is overwritten by row k - 2's result,
        // G >= 2 rows later in this loop order; the register look-ahead reads it even earlier
            cplx q[G];
        auto load = [&](int k0, cplx (&r)[G]) {
#pragma unroll
            for (int i = 0; i < G; ++i) if (k0 - i >= 2) r[i] = x[(k0 - i - 2) * st];
        };
        load(N, q);
        for (int k0 = N; k0 >= 2; k0 -= G) {
            cplx nx[G];
            load(k0 - G, nx);
            const int kp = k0 - 2 * G - g.pf;
#pragma unroll
            for (int i = 0; i < G; ++i) if (kp - i >= 2) pf_l2(x + (kp - i - 2) * st);
#pragma unroll
            for (int i = 0; i < G; ++i) {
                const int k = k0 - i;
                if (k >= 2) x[k * st] = el.row<true, false>(k, N, sigma, q[i], pv.step(k, N, sigma));
            }
#pragma unroll
            for (int i = 0; i < G; ++i) q[i] = nx[i];
        }
        cplx u0, u1;
        el.finish<true>(sigma, 0.0, 0.0, u0, u1);
        x[0] = u0; x[st] = u1;
    }
}

template <int G, bool GEN>
__global__ void __launch_bounds__(NT_COL, 3) k_elim2(const __grid_constant__ Elim2Args a) { elim2_body<G, GEN>(a, blockIdx.y); }

// Three-sweep form of the phi problem (ElimUpNeu): block row 0 = the w elimination of k_elim2, block row 1 = the up sweep of
// the psi chain feeding the upward elimination of the phi solve (psi is not stored).
template <int G, bool GEN>
__global__ void __launch_bounds__(NT_COL, 3) k_elim2up(const __grid_constant__ Elim2Args a, const __grid_constant__ SubstArgs b) {
    if (blockIdx.y == 0) elim2_body<G, GEN>(a, 0);
    else subst_body<G, true>(b, 0);
}

// ---- init helper: real copies of the homogeneous solutions and their k^2 sums --------------------------
__global__ void __launch_bounds__(NT_COL) k_hom_tables(const __grid_constant__ ColGeom g, const cplx *__restrict__ thh_c,
                                                       const cplx *__restrict__ wh_c, double *__restrict__ thh,
                                                       double *__restrict__ wh, double *__restrict__ hw) {
    const int col = blockIdx.x * blockDim.x + threadIdx.x;
    if (col >= g.ncols) return;
    const size_t st = g.ncols;
    double he = 0.0, ho = 0.0, me = 0.0, mo = 0.0;
    for (int k = 0; k <= g.N; ++k) {
        const size_t o = k * st + col;
        const double w = wh_c[o].x;
        thh[o] = thh_c[o].x;
        wh[o] = w;
        const double k2 = (double)k * k, m = k2 * (k2 - 1.0) * (1.0 / 3.0);
        if (k & 1) { ho += k2 * w; mo += m * w; } else { he += k2 * w; me += m * w; }
    }
    hw[col] = he;
    hw[st + col] = ho;
    hw[2 * st + col] = me;      // free-slip walls (row f3): sums of T_k''(1) w_h,k per parity
    hw[3 * st + col] = mo;
}

// ---- row a11: velocity recovery, plus D phi^ for the next step's grad(phi) (row a1) -----------------------
struct FinishArgs {
    ColGeom g;
    const cplx *om;    // omega_z^{n+1} (column 0: u-bar^{n+1})
    const cplx *th;    // column 0 only: v-bar^{n+1}
    cplx *u, *v, *w;
    cplx *phi;         // nullable (single-phase)
    cplx *phz;         // [nkz][ncols]: D phi^, truncated (operator P)
    const double2 *tab_phi;   // non-null: phi holds g^ of the upward elimination (k_subst<., true>); this sweep substitutes
    // W3: w holds g^ of the w solve's upward elimination (k_subst3); this sweep substitutes, adds the influence-matrix
    // correction w += A_par w_h, theta += A_par theta_h (what the second k_subst does in the five-sweep form)
    const double2 *tab_w;
    const double *wh, *thh;
    const cplx *coef;
    cplx *th_rw;
};

// LZ (with W3): theta^ is left as theta_p; the next step's k_rhs_elim<., ., true> applies A_par theta_h where it reads theta^.
template <int G, bool W3 = false, bool LZ = false>
__global__ void __launch_bounds__(NT_COL) k_finish(const __grid_constant__ FinishArgs a) {
    const ColGeom &g = a.g;
    const int col = blockIdx.x * blockDim.x + threadIdx.x;
    if (col >= g.ncols) return;
    const size_t st = g.ncols;
    double kx, ky;
    col_wavenumbers(g, col, kx, ky);
    const double k2 = kx * kx + ky * ky;
    const bool mean = (col == 0);
    const double ik2 = (!mean && col % g.kxp < g.nkx) ? 1.0 / k2 : 0.0;
    const bool phase = a.phi != nullptr;
    Chain1 cW, cP;
    cW.init(); cP.init();
    // phi_k = g^_k + e^_k phi_par - c^_k phi_{k+2} (back substitution of ElimUpNeu), in place
    const bool upphi = phase && a.tab_phi != nullptr;
    cplx pu0 = cz(), pu1 = cz(), pp2 = cz(), pp1 = cz();
    if (upphi) { pu0 = a.phi[col]; pu1 = a.phi[st + col]; }
    // w_p,k = g^_k + e^_k w_p,par - c^_k w_p,k+2 (back substitution of ElimUpDir2), then w = w_p + A_par w_h
    cplx wu0 = cz(), wu1 = cz(), wp2 = cz(), wp1 = cz(), Ae = cz(), Ao = cz();
    if (W3) { wu0 = a.w[col]; wu1 = a.w[st + col]; Ae = a.coef[col]; Ao = a.coef[st + col]; }
    struct Row { cplx w, om, phi, thv; double2 tb, tw; double whv, thhv; };
    auto load = [&](int n0, Row (&r)[G]) {               // rows n0, n0 - 1, .. (descending)
#pragma unroll
        for (int i = 0; i < G; ++i) {
            const int n = n0 - i;
            if (n >= 0) {
                const size_t o = n * st + col;
                r[i].w = a.w[o];
                r[i].om = a.om[o];
                if (phase && (upphi || n < g.nkz)) r[i].phi = a.phi[o];
                if (upphi && n >= 2) r[i].tb = a.tab_phi[o];
                if (W3) {
                    if (n >= 2) r[i].tw = a.tab_w[o];
                    r[i].whv = a.wh[o];
                    if (!LZ) { r[i].thhv = a.thh[o]; r[i].thv = a.th_rw[o]; }
                    else if (mean) r[i].thv = a.th_rw[o];
                } else if (mean) r[i].w = a.th[o];       // column (0,0): v-bar lives in the theta slot
            }
        }
    };
    Row q[G];
    load(g.N, q);
    for (int n0 = g.N; n0 >= 0; n0 -= G) {
        Row nx[G];
        load(n0 - G, nx);
        const int np0 = n0 - 2 * G - g.pf;
#pragma unroll
        for (int i = 0; i < G; ++i) {
            const int np = np0 - i;
            if (np >= 0) {
                const size_t op = np * st + col;
                pf_l2(a.w + op); pf_l2(a.om + op);
                if (phase && (upphi || np < g.nkz)) pf_l2(a.phi + op);
                if (upphi) pf_l2(a.tab_phi + op);
                if (W3) { pf_l2(a.tab_w + op); pf_l2(a.wh + op); if (!LZ) { pf_l2(a.thh + op); pf_l2(a.th_rw + op); } }
            }
        }
#pragma unroll
        for (int i = 0; i < G; ++i) {
            const int n = n0 - i;
            if (n < 0) continue;
            const size_t o = n * st + col;
            const double f = 2.0 * (n + 1), h = (n == 0) ? 0.5 : 1.0;
            cplx ph = q[i].phi;
            if (upphi) {
                if (n >= 2) {
                    ph = cfma(q[i].tb.y, (n & 1) ? pu1 : pu0, cfma(-q[i].tb.x, pp2, ph));
                    a.phi[o] = ph;
                }
                pp2 = pp1; pp1 = ph;
            }
            if (phase && n < g.nkz) a.phz[o] = cP.step(ph, f, h);   // D of the truncated phi^ (P first, then D)
            cplx wv = q[i].w;
            if (W3) {
                if (n >= 2) wv = cfma(q[i].tw.y, (n & 1) ? wu1 : wu0, cfma(-q[i].tw.x, wp2, wv));
                wp2 = wp1; wp1 = wv;
                const cplx A = (n & 1) ? Ao : Ae;
                wv = cfma(q[i].whv, A, wv);
                if (!mean) { a.w[o] = wv; if (!LZ) a.th_rw[o] = cfma(q[i].thhv, A, q[i].thv); }
                else wv = q[i].thv;                       // column (0,0): v-bar lives in the theta slot
            }
            if (mean) {   // mean flow: u-bar from the omega slot, v-bar from the theta slot, w = 0 (reading S12)
                a.u[o] = q[i].om;
                a.v[o] = wv;
                a.w[o] = cz();
            } else {
                const cplx dw = cW.step(wv, f, h);
                const cplx om = q[i].om;
                a.u[o] = cscale(ci(cadd(cscale(dw, kx), cscale(om, ky))), ik2);
                a.v[o] = cscale(ci(csub(cscale(dw, ky), cscale(om, kx))), ik2);
            }
        }
#pragma unroll
        for (int i = 0; i < G; ++i) q[i] = nx[i];
    }
}

// ---- pending influence-matrix correction of theta^ (three-sweep form with LZ): theta += A_par theta_h, then A := 0 --------
__global__ void __launch_bounds__(NT_COL) k_theta_apply(const __grid_constant__ ColGeom g, cplx *__restrict__ th,
                                                        const double *__restrict__ thh, cplx *__restrict__ coef) {
    const int col = blockIdx.x * blockDim.x + threadIdx.x;
    if (col >= g.ncols) return;
    const size_t st = g.ncols;
    const cplx Ae = coef[col], Ao = coef[st + col];
    for (int n = 0; n <= g.N; ++n) {
        const size_t o = n * st + col;
        th[o] = cfma(thh[o], (n & 1) ? Ao : Ae, th[o]);      // the same fma per component as k_rhs_elim<., ., true>
    }
    coef[col] = cz();
    coef[st + col] = cz();
}

// ---- per-step bookkeeping ---------------------------------------------------------------------------
__global__ void k_begin_step(double *ab, int *counter) {
    // reading S7: explicit Euler on the first step after set_state, AB2 afterwards
    if (*counter == 0) { ab[0] = 1.0; ab[1] = 0.0; }
    else               { ab[0] = 1.5; ab[1] = -0.5; }
    *counter += 1;
}

__global__ void k_set_real(cplx *dst, size_t n, double re) {
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) dst[i] = make_double2(re, 0.0);
}

}  // namespace psdns
