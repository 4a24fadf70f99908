// Fused x pass for the variable-viscosity step (BASELINE.json config 4, reading S14): rows a4 + a5 + a6 with
// 12 fields backward (u v w phi phx phy phz exx eyy exy exz eyz) and 7 forward, in a tile of SIXTEEN field slots.
// Same stages A-F as the matched-viscosity kernels of kernels_xfused.cuh (half-length real transform, TMA-staged
// spectra rows, DIF backward / DIT forward with the radix-2 + pointwise stage in the middle), here in the
// thread = (butterfly, field slot) organisation with CTA-wide barriers between the stages.
//   T_ij = -u_i u_j + cs (|grad phi|^2 delta_ij - phi_i phi_j) + eta1(phi) E_ij,  eta1 = eta_c (phi + 1),
//   eta_c = (lambda - 1) / (2 Re);  E_zz = -E_xx - E_yy;  only T_ij - T_zz delta_ij is transformed (see psdns.cu).
// Without it the variable-viscosity step runs three kernels with 19 physical-space arrays in HBM
// (k_xpass, k_pointwise, k_xpass): 4.5 ms of a 7.8 ms step at 512x256x257.
// The pointwise stage works on the real and imaginary parts in two sweeps (a thread owns rows 2t, 2t+1 of all
// fields = 4 grid points x 12 inputs; half of that fits the register budget without spills).
#pragma once
#include "kernels_xfused.cuh"

namespace psdns {

constexpr int XV_SLOTS = 16;
constexpr int XV_NIN = 12, XV_NOUT = 7, XV_NTMA = 11, XV_NST = 12;

struct XFVArgs {
    const cplx *in[XV_NTMA];   // Y arrays: u v w phi phy phz exx eyy exy exz eyz
    cplx *out[XV_NOUT];        // Y arrays: Txx-Tzz Txy Txz Tyy-Tzz Tyz Q C
    int kxp, nkx, nlines;
    double cs, kxf, eta_c;
};

template <int L> __host__ __device__ constexpr int xv_threads() {
    return (XV_SLOTS * (L / 2) / XPlan<L / 2>::R1) > 64 ? (XV_SLOTS * (L / 2) / XPlan<L / 2>::R1) : 64;
}

// tile index: slot rotated by row/2 (pointwise stage: 8 consecutive threads at one field hit 8 bank groups; butterfly
// stages: a quarter-warp covers 8 consecutive slots of one row = one 128-byte segment)
__device__ __forceinline__ int xvidx(int row, int f) { return row * XV_SLOTS + ((f + (row >> 1)) & (XV_SLOTS - 1)); }

template <int H, int R, int SIGN, int NT, bool DIT>
__device__ __forceinline__ void xvpass_mid(cplx *__restrict__ s, int tid) {
    tid = opaque(tid);
    constexpr int LS = 2 * R;
    constexpr int NBLK = H / LS;
    static_assert(NBLK % 2 == 0, "twiddle class must be uniform over a warp (2 butterflies x 16 slots)");
    const int f = tid & (XV_SLOTS - 1);
    for (int b = tid >> 4; b < 2 * NBLK; b += NT / XV_SLOTS) {
        const int j = b / NBLK, blk = b % NBLK;
        const int row0 = blk * LS + j;
        cplx v[R];
#pragma unroll
        for (int m = 0; m < R; ++m) v[m] = s[xvidx(row0 + 2 * m, f)];
        if (DIT && j) {
#pragma unroll
            for (int m = 1; m < R; ++m) v[m] = cmultw<SIGN>(v[m], make_double2(wc_re<LS>(m), wc_im<LS>(m)));
        }
        RegFFT<R, SIGN>::run(v);
        if (!DIT && j) {
#pragma unroll
            for (int q = 1; q < R; ++q) v[q] = cmultw<SIGN>(v[q], make_double2(wc_re<LS>(q), wc_im<LS>(q)));
        }
#pragma unroll
        for (int q = 0; q < R; ++q) s[xvidx(row0 + 2 * q, f)] = v[q];
    }
}

// the seven products at one grid point; in: u v w phi phx phy phz exx eyy exy exz eyz
__device__ __forceinline__ void nl_visc(const double (&in)[XV_NIN], double cs, double eta_c, double (&o)[XV_NOUT]) {
    const double u = in[0], v = in[1], w = in[2], ph = in[3], px = in[4], py = in[5], pz = in[6];
    const double e1 = eta_c * (ph + 1.0);
    o[0] = w * w - u * u + cs * (pz * pz - px * px) + e1 * (2.0 * in[7] + in[8]);   // (Txx - Tzz), Ezz = -Exx - Eyy
    o[1] = -u * v - cs * px * py + e1 * in[9];
    o[2] = -u * w - cs * px * pz + e1 * in[10];
    o[3] = w * w - v * v + cs * (pz * pz - py * py) + e1 * (in[7] + 2.0 * in[8]);
    o[4] = -v * w - cs * py * pz + e1 * in[11];
    o[5] = u * px + v * py + w * pz;
    o[6] = ph * ph * ph;
}

template <int L>
__global__ void __launch_bounds__(xv_threads<L>(), (L >= 1024 ? 1 : 2)) k_xfusedv(const __grid_constant__ XFVArgs a,
                                                                                const cplx *__restrict__ twx) {
    constexpr int H = L / 2;
    constexpr int R1 = XPlan<H>::R1, R2 = XPlan<H>::R2;
    constexpr int NT = xv_threads<L>();
    constexpr int S1 = H / R1;
    // compile-time cut-offs, as in k_xfusedw (the host checks a.nkx == NKX)
    constexpr int NKX = L / 3 + 1, KXP = (NKX + 7) & ~7;
    static_assert(R1 * R2 * 2 == H, "plan");
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cplx *s = reinterpret_cast<cplx *>(smem_raw);
    cplx *stage = s + H * XV_SLOTS;
    constexpr int kxp = KXP, nkx = NKX;
    constexpr int spitch = NKX | 1;
    unsigned long long *bar = reinterpret_cast<unsigned long long *>(stage + (size_t)XV_NST * spitch);
    const int tid = threadIdx.x, f = tid & (XV_SLOTS - 1), j = tid >> 4;
    const bool item = j < S1;
    cplx *outf = a.out[f < XV_NOUT ? f : 0];
    const double sc = 0.5 / L;
    constexpr unsigned row_bytes = (unsigned)(NKX * sizeof(cplx));
    auto issue = [&](int line) {
        mbar_expect_tx(bar, row_bytes * XV_NTMA);
#pragma unroll
        for (int q = 0; q < XV_NTMA; ++q) bulk_g2s(stage + (size_t)q * spitch, a.in[q] + (size_t)line * kxp, row_bytes, bar);
    };
    if (tid == 0) {
        mbar_init(bar, 1);
        if ((int)blockIdx.x < a.nlines) issue(blockIdx.x);
    }
    __syncthreads();
    cplx wj = twx[item ? j : 0];
    unsigned parity = 0;
    // field slot -> staged row: u v w phi | phx = derived row 11 | phy phz exx eyy exy exz eyz = rows 4..10
    const int srow = f < 4 ? f : (f == 4 ? 11 : (f < XV_NIN ? f - 1 : 0));
    const cplx *sf = stage + (size_t)srow * spitch;
    for (int line = blockIdx.x; line < a.nlines; line += gridDim.x) {
        const size_t base = (size_t)line * kxp;
        mbar_wait(bar, parity);
        parity ^= 1;
        for (int k = tid; k < nkx; k += NT) {            // row a1: phx^ = i kx phi^
            const cplx p = stage[3 * spitch + k];
            const double kk = a.kxf * (double)k;
            stage[11 * spitch + k] = make_double2(-kk * p.y, kk * p.x);
        }
        __syncthreads();
        asm volatile("" : "+d"(wj.x), "+d"(wj.y));
        // ---- A: pre-twiddle from the staged rows + DIF pass R1 (inverse transform, sign +) ----
        if (item) {
            const int jj = (opaque(tid) >> 4) & (S1 - 1);
            const bool live = f < XV_NIN;              // slots 12..15 carry zeros through the backward passes
            cplx v[R1];
            static_for<0, R1>([&](auto M) {
                constexpr int m = decltype(M)::value;
                if (m && (m & 3) == 0) asm volatile("" ::: "memory");
                // rows k = jj + S1 m of this m: X_k is retained for k < NKX, the partner X_{H-k} for k > H - NKX
                constexpr bool a_all = (S1 * m + S1 - 1 < NKX), a_none = (S1 * m >= NKX);
                constexpr bool b_all = (S1 * m > H - NKX), b_none = (S1 * m + S1 - 1 <= H - NKX);
                const int k = jj + S1 * m, kb = H - k;
                const cplx w = m ? cmul(wj, make_double2(wc_re<2 * R1>(m), wc_im<2 * R1>(m))) : wj;
                if constexpr (b_none) {
                    static_assert(a_all, "cut-offs");
                    cplx xa = make_double2(0.0, 0.0);
                    if (live) xa = sf[k];
                    if (m == 0 && k == 0) xa.y = 0.0;           // reading S20
                    v[m] = make_double2(fma(w.y, xa.x, fma(-w.x, xa.y, xa.x)), fma(w.y, xa.y, fma(w.x, xa.x, xa.y)));
                } else if constexpr (a_none) {
                    static_assert(b_all, "cut-offs");
                    cplx xb = make_double2(0.0, 0.0);
                    if (live) xb = sf[kb];                      // S = conj(xb), D = -conj(xb)
                    v[m] = make_double2(fma(-w.y, xb.x, fma(-w.x, xb.y, xb.x)), fma(w.y, xb.y, fma(-w.x, xb.x, -xb.y)));
                } else {
                    cplx xa = make_double2(0.0, 0.0), xb = xa;
                    if (live && (a_all || k < NKX)) xa = sf[k];
                    if (live && (b_all || kb < NKX)) xb = sf[kb];
                    if (m == 0 && k == 0) { xa.y = 0.0; xb.y = 0.0; }   // reading S20
                    const double Sx = xa.x + xb.x, Sy = xa.y - xb.y, Dx = xa.x - xb.x, Dy = xa.y + xb.y;
                    v[m] = make_double2(fma(w.y, Dx, fma(-w.x, Dy, Sx)), fma(w.y, Dy, fma(w.x, Dx, Sy)));
                }
            });
            RegFFT<R1, +1>::run(v);
            TwPow<R1> tp;
            tp.init(cmul(wj, wj));
            s[xvidx(jj, f)] = v[0];
            tp.each([&](int q, cplx wq) { s[xvidx(jj + S1 * q, f)] = cmultw<+1>(v[q], wq); });
        }
        __syncthreads();
        if (tid == 0 && line + (int)gridDim.x < a.nlines) {   // stage is free: prefetch the next line
            fence_proxy_async();
            issue(line + gridDim.x);
        }
        // ---- B: DIF pass R2 ----
        if constexpr (R2 > 1) {
            xvpass_mid<H, R2, +1, NT, false>(s, tid);
            __syncthreads();
        }
        // ---- C: last DIF radix 2, pointwise products, first DIT radix 2; real parts, then imaginary parts ----
        for (int t = opaque(tid); t < H / 2; t += NT) {
#pragma unroll
            for (int part = 0; part < 2; ++part) {
                double a0[XV_NIN], a1[XV_NIN];           // the two grid points (p + m), (p - m) of this part
#pragma unroll
                for (int q = 0; q < XV_NIN; ++q) {
                    const cplx p = s[xvidx(2 * t, q)], m = s[xvidx(2 * t + 1, q)];
                    const double pc = part ? p.y : p.x, mc = part ? m.y : m.x;
                    a0[q] = pc + mc; a1[q] = pc - mc;
                }
                double o0[XV_NOUT], o1[XV_NOUT];
                nl_visc(a0, a.cs, a.eta_c, o0);
                nl_visc(a1, a.cs, a.eta_c, o1);
                // only this part of the output rows is written: the other part of the INPUT fields in the same slots is
                // still needed by the second sweep
#pragma unroll
                for (int q = 0; q < XV_NOUT; ++q) {
                    reinterpret_cast<double *>(s + xvidx(2 * t, q))[part] = o0[q] + o1[q];
                    reinterpret_cast<double *>(s + xvidx(2 * t + 1, q))[part] = o0[q] - o1[q];
                }
            }
        }
        __syncthreads();
        // ---- D: DIT pass R2 (forward transform, sign -) ----
        if constexpr (R2 > 1) {
            xvpass_mid<H, R2, -1, NT, true>(s, tid);
            __syncthreads();
        }
        // ---- E: DIT pass R1; results stay in registers, only the rows some partner needs go to the tile ----
        asm volatile("" : "+d"(wj.x), "+d"(wj.y));
        cplx v[R1];
        if (item) {
            const int jj = (opaque(tid) >> 4) & (S1 - 1);
            TwPow<R1> tp;
            tp.init(cmul(wj, wj));
            v[0] = s[xvidx(jj, f)];
            tp.each([&](int m, cplx wq) { v[m] = cmultw<-1>(s[xvidx(jj + S1 * m, f)], wq); });
            RegFFT<R1, -1>::run(v);
#pragma unroll
            for (int q = 0; q < R1; ++q) {
                const int r = jj + S1 * q;
                if (S1 * q + S1 - 1 > H - NKX && (S1 * q > H - NKX || r > H - NKX)) s[xvidx(r, f)] = v[q];
            }
        }
        __syncthreads();
        // ---- F: post-twiddle of row k against the partner row H - k, truncated store ----
        if (item && f < XV_NOUT) {
            const int jj = (opaque(tid) >> 4) & (S1 - 1);
            cplx *o = outf + base + jj;
            static_for<0, R1 / 4>([&](auto Q0) {
                constexpr int q0 = 4 * decltype(Q0)::value;
                if constexpr (S1 * q0 < KXP) {
                    cplx zb[4];
#pragma unroll
                    for (int i = 0; i < 4; ++i) {
                        const int k = jj + S1 * (q0 + i);
                        zb[i] = make_double2(0.0, 0.0);
                        if (S1 * (q0 + i) < NKX) zb[i] = s[xvidx((H - k) & (H - 1), f)];
                    }
                    static_for<0, 4>([&](auto I) {
                        constexpr int i = decltype(I)::value, q = q0 + i;
                        if constexpr (S1 * q < KXP) {
                            constexpr bool all = (S1 * q + S1 - 1 < NKX);
                            const int k = jj + S1 * q;
                            const cplx za = v[q];
                            cplx zp = zb[i];
                            if (q == 0 && k == 0) zp = za;
                            const cplx w = q ? cmul(wj, make_double2(wc_re<2 * R1>(q), wc_im<2 * R1>(q))) : wj;
                            const double Sx = za.x + zp.x, Sy = za.y - zp.y, Dx = za.x - zp.x, Dy = za.y + zp.y;
                            cplx r = make_double2(sc * fma(w.y, Dx, fma(w.x, Dy, Sx)), sc * fma(w.y, Dy, fma(-w.x, Dx, Sy)));
                            if constexpr (all) {
                                stg_off<q * S1 * (int)sizeof(cplx)>(o, r);
                            } else {
                                if (k >= NKX) r = make_double2(0.0, 0.0);
                                if (k < KXP) stg_off<q * S1 * (int)sizeof(cplx)>(o, r);
                            }
                        }
                    });
                }
            });
        }
        __syncthreads();
    }
}

}  // namespace psdns
