// Diagnostics on the resident spectra (the quantities a run monitors without a host
// round trip): mean(phi), max |div u| over the spectrum, volume-averaged kinetic energy, wall shear of the mean flow,
// bulk velocity.  Deterministic two-stage reductions (per-block partials, one final block): no floating-point atomics.
#pragma once
#include "kernels_spectral.cuh"

namespace psdns {

constexpr int DIAG_NT = 256;

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
__device__ __forceinline__ double warp_max(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}

// One thread per retained (kx, ky) column, sweeping n downwards with the Chebyshev derivative recurrence:
//   max_n |i kx u^_n + i ky v^_n + (D w^)_n|  -> part_max[block]
// Column (0,0) also produces the one-column functionals:
//   out[0] mean(phi) = 1/2 sum_{n even} phi^_n 2/(1 - n^2);  out[5] bulk velocity (same functional of u-bar);
//   out[3], out[4] d u-bar/dz at z = +1, -1 = sum n^2 u_n, sum (-1)^(n+1) n^2 u_n.
__global__ void __launch_bounds__(DIAG_NT) k_diag_columns(const __grid_constant__ ColGeom g, const cplx *__restrict__ u,
                                                          const cplx *__restrict__ v, const cplx *__restrict__ w,
                                                          const cplx *__restrict__ phi, double *__restrict__ part_max,
                                                          double *__restrict__ out) {
    __shared__ double red[DIAG_NT / 32];
    const int col = blockIdx.x * blockDim.x + threadIdx.x;
    double m = 0.0;
    if (col < g.ncols) {
        double kx, ky;
        col_wavenumbers(g, col, kx, ky);
        const size_t st = g.ncols;
        Chain1 cW;
        cW.init();
        double mphi = 0.0, bulk = 0.0, sh_p = 0.0, sh_m = 0.0;
        for (int n = g.N; n >= 0; --n) {
            const size_t o = n * st + col;
            const double f = 2.0 * (n + 1), h = (n == 0) ? 0.5 : 1.0;
            const cplx un = u[o], vn = v[o];
            const cplx dw = cW.step(w[o], f, h);
            const double dr = -kx * un.y - ky * vn.y + dw.x, di = kx * un.x + ky * vn.x + dw.y;
            m = fmax(m, sqrt(dr * dr + di * di));
            if (col == 0) {
                const double n2 = (double)n * n;
                if ((n & 1) == 0) {
                    const double q = 1.0 / (1.0 - n2);
                    bulk += un.x * q;
                    if (phi) mphi += phi[o].x * q;
                    sh_m -= n2 * un.x;
                } else {
                    sh_m += n2 * un.x;
                }
                sh_p += n2 * un.x;
            }
        }
        if (col == 0) { out[0] = mphi; out[5] = bulk; out[3] = sh_p; out[4] = sh_m; }
    }
    m = warp_max(m);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = m;
    __syncthreads();
    if (threadIdx.x < 32) {
        double r = threadIdx.x < DIAG_NT / 32 ? red[threadIdx.x] : 0.0;
        r = warp_max(r);
        if (threadIdx.x == 0) part_max[blockIdx.x] = r;
    }
}

// Kinetic energy from the Z arrays (z physical, x and y spectral) of u, v, w: Parseval over the retained (kx, ky)
// (weight 2 for kx > 0: the half spectrum stands for its conjugate half), Clenshaw-Curtis weights over z_k:
//   E = 1/4 sum_k ccw_k sum_col mult |u|^2 + |v|^2 + |w|^2          -> part_sum[block]
__global__ void __launch_bounds__(DIAG_NT) k_diag_energy(const cplx *__restrict__ zu, const cplx *__restrict__ zv,
                                                         const cplx *__restrict__ zw, const double *__restrict__ ccw,
                                                         int nz, int ncols, int kxp, double *__restrict__ part_sum) {
    __shared__ double red[DIAG_NT / 32];
    const size_t total = (size_t)nz * ncols, stride = (size_t)gridDim.x * blockDim.x;
    double acc = 0.0;
    for (size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x; e < total; e += stride) {
        const int k = (int)(e / ncols), col = (int)(e - (size_t)k * ncols);
        const double mult = (col % kxp == 0) ? 1.0 : 2.0;
        const cplx a = zu[e], b = zv[e], c = zw[e];
        acc = fma(ccw[k] * mult, a.x * a.x + a.y * a.y + b.x * b.x + b.y * b.y + c.x * c.x + c.y * c.y, acc);
    }
    acc = warp_sum(acc);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x < 32) {
        double r = threadIdx.x < DIAG_NT / 32 ? red[threadIdx.x] : 0.0;
        r = warp_sum(r);
        if (threadIdx.x == 0) part_sum[blockIdx.x] = r;
    }
}

// final stage: one block folds the partials in a fixed order
__global__ void __launch_bounds__(DIAG_NT) k_diag_final(const double *__restrict__ part_max, int nmax,
                                                        const double *__restrict__ part_sum, int nsum,
                                                        double *__restrict__ out) {
    __shared__ double rm[DIAG_NT / 32], rs[DIAG_NT / 32];
    double m = 0.0, s = 0.0;
    for (int i = threadIdx.x; i < nmax; i += DIAG_NT) m = fmax(m, part_max[i]);
    for (int i = threadIdx.x; i < nsum; i += DIAG_NT) s += part_sum[i];
    m = warp_max(m); s = warp_sum(s);
    if ((threadIdx.x & 31) == 0) { rm[threadIdx.x >> 5] = m; rs[threadIdx.x >> 5] = s; }
    __syncthreads();
    if (threadIdx.x == 0) {
        double mm = 0.0, ss = 0.0;
        for (int i = 0; i < DIAG_NT / 32; ++i) { mm = fmax(mm, rm[i]); ss += rs[i]; }
        out[1] = mm;
        out[2] = 0.25 * ss;
        out[6] = 0.0; out[7] = 0.0;
    }
}

// FP64 FMA-chain microbenchmark ("the builder measures [the FP64 peak] with an FMA-chain microbenchmark"):
// every thread runs 8 independent chains of dependent DFMAs, `iters` x 8 x 16 FMAs per thread; the result is stored so that
// nothing is optimised away.
__global__ void __launch_bounds__(256) k_fp64_fma_chain(double *out, int nslots, int iters, double a, double b) {
    double x[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) x[i] = 1.0 + 1e-9 * (threadIdx.x + i);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < 16; ++r) {
#pragma unroll
            for (int i = 0; i < 8; ++i) x[i] = fma(x[i], a, b);
        }
    }
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < 8; ++i) s += x[i];
    out[(size_t)(blockIdx.x % nslots) * blockDim.x + threadIdx.x] = s;   // blocks may share a slot: the value is never read
}

}  // namespace psdns
