// Fused x pass (rows a4 + a5 + a6): for one (k, y) line at a time, C2R of the 7 input fields,
// pointwise non-linear terms, R2C of the 8 product fields - physical-space arrays never reach HBM
// ("physical-space arrays never leave the SM"; PAPER.md L166-176 for the transforms,
// L182-196 and Eqs. 1, 4, 7, 8 for the products).
//
// Tile: the 8 tile lines of fft_tile are the FIELDS; the FFT is the half-length real transform:
//   backward: Z_k = (X_k + conj X_{H-k}) + i conj(w_k) (X_k - conj X_{H-k}),  w_k = exp(-2 pi i k / L), H = L/2,
//             z = IFFT_H(Z) gives z_n = x_{2n} + i x_{2n+1}
//   forward : A_k = (Z_k + conj Z_{H-k})/2, B_k = (Z_k - conj Z_{H-k})/(2i), X_k = (A_k + w_k B_k)/L
// so one line of 8 fields at nx = 1024 is 64 KB of shared memory (3 CTAs per SM).  The backward FFT is
// decimation in frequency (digit-reversed output), the products are elementwise so order does not matter,
// and the forward FFT is decimation in time (digit-reversed input, natural output): no reordering at all.
// The swizzled tile layout makes both the butterflies and the per-row pointwise stage bank-conflict free.
#pragma once
#include "fft_tile.cuh"
#include "kernels_transform.cuh"

namespace psdns {

// ---- TMA (bulk async copy) + mbarrier helpers, sm_90+/sm_100a PTX ------------------------------------
__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long *bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long *bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long *bar, unsigned parity) {
    unsigned done = 0;
    while (!done) {
        asm volatile(
            "{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
            : "=r"(done)
            : "r"(smem_u32(bar)), "r"(parity)
            : "memory");
    }
}
// global -> shared bulk copy (1-D TMA, SASS UBLKCP); bytes multiple of 16, both addresses 16-byte aligned
__device__ __forceinline__ void bulk_g2s(void *dst_smem, const void *src_gmem, unsigned bytes, unsigned long long *bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst_smem)),
                 "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

struct XFArgs {
    const cplx *in[8];
    cplx *out[8];
    int kxp, nkx, nlines;
    int nin, nout;
    double cs;
    int phase;
};

// shared memory: tile [H][8] | twiddles [H] | stage [nin][kxp + 1] | mbarrier.  The stage receives the NEXT
// line's nin spectra rows by TMA bulk copies while the current line is transformed (pitch kxp + 1 keeps the
// 8 fields of one k in 8 different 16-byte bank groups).
template <int L>
__global__ void __launch_bounds__(NT_FFT, 2) k_xfused(const __grid_constant__ XFArgs a, const cplx *__restrict__ twx) {
    constexpr int H = L / 2;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cplx *s = reinterpret_cast<cplx *>(smem_raw);
    cplx *tw = s + H * TILE_LINES;
    cplx *stage = tw + H;
    const int spitch = a.kxp + 1;
    unsigned long long *bar = reinterpret_cast<unsigned long long *>(stage + (size_t)8 * spitch);
    const int tid = threadIdx.x, f = tid & 7, r0 = tid >> 3;
    constexpr int RSTEP = NT_FFT / TILE_LINES;
    const int kxp = a.kxp, nkx = a.nkx;
    for (int i = tid; i < H; i += NT_FFT) tw[i] = twx[2 * i];
    const cplx *inf = a.in[f < a.nin ? f : 0];   // may alias outf (in-place per line)
    cplx *outf = a.out[f < a.nout ? f : 0];
    const double sc = 1.0 / L;
    const unsigned row_bytes = (unsigned)(nkx * sizeof(cplx));
    auto issue = [&](int line) {   // one thread: arm the barrier and launch nin bulk copies
        mbar_expect_tx(bar, row_bytes * a.nin);
        for (int q = 0; q < a.nin; ++q) bulk_g2s(stage + (size_t)q * spitch, a.in[q] + (size_t)line * kxp, row_bytes, bar);
    };
    if (tid == 0) {
        mbar_init(bar, 1);
        if ((int)blockIdx.x < a.nlines) issue(blockIdx.x);
    }
    __syncthreads();
    unsigned parity = 0;
    const cplx *sf = stage + (size_t)(f < a.nin ? f : 0) * spitch;
    for (int line = blockIdx.x; line < a.nlines; line += gridDim.x) {
        const size_t base = (size_t)line * kxp;
        mbar_wait(bar, parity);
        parity ^= 1;
        // ---- pre-twiddle from the staged rows (pairs k, H-k) ----
        for (int k = r0; k <= H / 2; k += RSTEP) {
            const int kb = H - k;
            cplx xa = make_double2(0.0, 0.0), xb = xa;
            if (f < a.nin) {
                if (k < nkx) xa = sf[k];
                if (kb < nkx) xb = sf[kb];
            }
            if (k == 0) { xa.y = 0.0; xb.y = 0.0; }   // reading S20
            const cplx w = twx[k];
            const cplx S = make_double2(xa.x + xb.x, xa.y - xb.y);
            const cplx D = make_double2(xa.x - xb.x, xa.y + xb.y);
            // T = i * conj(w) * D
            const cplx T = make_double2(-(w.x * D.y - w.y * D.x), w.x * D.x + w.y * D.y);
            s[tile_idx<true>(k, f)] = cadd(S, T);
            if (k != 0 && kb != k) s[tile_idx<true>(kb, f)] = cconj(csub(S, T));
        }
        __syncthreads();
        if (tid == 0 && line + (int)gridDim.x < a.nlines) {   // stage is free: prefetch the next line
            fence_proxy_async();
            issue(line + gridDim.x);
        }
        fft_tile<H, +1, NT_FFT, true>(s, tw, tid);
        __syncthreads();
        // ---- pointwise: each thread owns whole rows (both packed points x_{2n}, x_{2n+1}) ----
        for (int r = tid; r < H; r += NT_FFT) {
            cplx v[8];
#pragma unroll
            for (int q = 0; q < 8; ++q) v[q] = s[tile_idx<true>(r, q)];
            cplx o[8];
#pragma unroll
            for (int c = 0; c < 2; ++c) {
                const double u = c ? v[0].y : v[0].x, vv = c ? v[1].y : v[1].x, w = c ? v[2].y : v[2].x;
                double txx = -u * u, txy = -u * vv, txz = -u * w, tyy = -vv * vv, tyz = -vv * w, tzz = -w * w;
                double qq = 0.0, cc = 0.0;
                if (a.phase) {
                    const double ph = c ? v[3].y : v[3].x, px = c ? v[4].y : v[4].x, py = c ? v[5].y : v[5].x,
                                 pz = c ? v[6].y : v[6].x;
                    const double g2 = px * px + py * py + pz * pz;
                    const double cs = a.cs;
                    txx += cs * (g2 - px * px);
                    tyy += cs * (g2 - py * py);
                    tzz += cs * (g2 - pz * pz);
                    txy -= cs * px * py;
                    txz -= cs * px * pz;
                    tyz -= cs * py * pz;
                    qq = u * px + vv * py + w * pz;
                    cc = ph * ph * ph;
                }
                if (c == 0) {
                    o[0].x = txx; o[1].x = txy; o[2].x = txz; o[3].x = tyy; o[4].x = tyz; o[5].x = tzz; o[6].x = qq; o[7].x = cc;
                } else {
                    o[0].y = txx; o[1].y = txy; o[2].y = txz; o[3].y = tyy; o[4].y = tyz; o[5].y = tzz; o[6].y = qq; o[7].y = cc;
                }
            }
#pragma unroll
            for (int q = 0; q < 8; ++q) s[tile_idx<true>(r, q)] = o[q];
        }
        __syncthreads();
        fft_tile_dit<H, -1, NT_FFT, true>(s, tw, tid);
        __syncthreads();
        // ---- post-twiddle + truncated store ----
        if (f < a.nout) {
            for (int k = r0; k <= H / 2; k += RSTEP) {
                const int kb = H - k;
                const cplx za = s[tile_idx<true>(k, f)];
                const cplx zb = s[tile_idx<true>(kb & (H - 1), f)];
                const cplx A = make_double2(0.5 * (za.x + zb.x), 0.5 * (za.y - zb.y));
                const cplx B = make_double2(0.5 * (za.y + zb.y), -0.5 * (za.x - zb.x));
                const cplx w = twx[k];
                const cplx wB = make_double2(w.x * B.x - w.y * B.y, w.x * B.y + w.y * B.x);
                if (k < nkx) outf[base + k] = cscale(cadd(A, wB), sc);
                if (k != kb && kb < nkx) outf[base + kb] = cscale(cconj(csub(A, wB)), sc);   // k = 0: X_H = A_0 - B_0
            }
            for (int i = nkx + r0; i < kxp; i += RSTEP) outf[base + i] = make_double2(0.0, 0.0);
        }
        __syncthreads();
    }
}

}  // namespace psdns
