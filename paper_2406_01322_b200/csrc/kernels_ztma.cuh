// z pass (Chebyshev transform = DCT-I) with TMA tensor loads: the strided column tile
// ([rows] x 8 columns = 128-byte inner extent, row stride = one spectral plane) is fetched by ONE thread as 2-D boxes
// (cp.async.bulk.tensor.2d, SASS UTMALDG) into a two-deep shared-memory stage guarded by mbarriers, while the CTA
// transforms the previous tile - the "TMA-staged pencil transposes replacing the MPI all-to-all" of north_star
// (PAPER.md L154-156).  This removes the limit of the register-fed form (k_zpass, kernels_transform.cuh): a thread
// cannot keep its 32 strided 16-byte loads in flight in 128 registers, so that kernel ran at the latency of its loads.
//
// Same arithmetic as k_zpass (half-length DCT-I, Makhoul re-ordering [32], see kernels_transform.cuh): the head pass
// reads its inputs from the stage instead of global memory; everything after it is identical, so both kernels give
// bit-identical results.
// Pipeline per CTA (persistent, tiles t = blockIdx.x + i gridDim.x):
//   prologue: thread 0 issues the boxes of tiles 0 and 1 into stage 0 and 1
//   tile i  : wait full[i & 1] -> head pass (stage -> registers -> FFT tile) -> barrier -> thread 0 re-arms the stage
//             with tile i + 2 (fence.proxy.async first: the stage was read through the generic proxy) -> remaining
//             passes, post-processing E_k = Z_k + c_k (Z_k - Z_{N-k}), stores.
#pragma once
#include <cuda.h>

#include "kernels_transform.cuh"
#include "kernels_xfused.cuh"   // mbarrier / proxy-fence helpers

namespace psdns {

struct ZTArgs {
    CUtensorMap in_map[MAXF];   // per field: 2-D tensor {2 ncols doubles, nin rows}, box {16 doubles, box_rows}
    void *out[MAXF];
    int nf, ncols, nk;
    int box_rows, nboxes;       // nboxes * box_rows >= input rows; rows beyond the tensor are zero-filled by TMA
    int dfield;
    cplx *out_dx, *out_dy;
    int kxp, nky, jpos;
    double kxf, kyf;
};

__device__ __forceinline__ void tma_load_2d(void *dst_smem, const CUtensorMap *map, int c0, int c1, unsigned long long *bar) {
    asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];" ::"r"(
                     smem_u32(dst_smem)),
                 "l"(map), "r"(c0), "r"(c1), "r"(smem_u32(bar))
                 : "memory");
}

// One CTA per SM (the two stages fill most of the shared memory), so both directions run the 512-thread radix-8 plan at
// N = 512 (PlanZB) for the warps to hide each other's shared-memory latency.
template <int N> __host__ __device__ constexpr int ztma_threads() { return fused_threads<N, PlanZB<N>>(); }

// shared memory (cplx units): 2 stages srows*8 | FFT tile N*8 | H_0 partials NW*8 | twiddles N | c_k table N/2+1 | 2 mbarriers
// Measured on B200 at N = 512 (1024x512x513, backward / forward pass, register-fed k_zpass = 2.57 / 2.89 ms):
//   this form, one CTA per SM                                                    2.10 / 2.70 ms
//   one stage, tables read from global memory, two CTAs per SM (backward only)   2.23 ms
//   in place (the stage IS the FFT tile, no prefetch), two CTAs per SM           2.31 / 3.02 ms
// and at N = 256 (512x256x257; two CTAs per SM fit with both stages): 0.322 -> 0.241 / 0.377 -> 0.284 ms.
template <int N> __host__ __device__ constexpr int ztma_fixed_cplx() {
    return N * TILE_LINES + (ztma_threads<N>() / 32) * 8 + N + (N / 2 + 1) + 1;
}
template <int N> inline size_t ztma_smem_bytes(int srows) {
    return ((size_t)ztma_fixed_cplx<N>() + 2 * (size_t)srows * TILE_LINES) * sizeof(cplx) + 32;
}

// Last FFT pass fused with the post-processing E_k = Z_k + c_k (Z_k - Z_{N-k}) (round 2; the kernel is bound by the
// shared-memory pipe, and this removes one tile write, one tile read and one CTA-wide barrier per tile).  The last pass
// has stride 1 and no twiddles: butterfly b reads tile rows b RL .. b RL + RL - 1 and produces the elements k0 + KS q
// (q < RL) with k0 = k0(b) < KS.  The partner N - k of element k0 + KS q is element (KS - k0) + KS (RL - 1 - q) of
// butterfly KS - k0.  Every thread runs ONE butterfly; the butterflies k0 and KS - k0 sit in lanes that differ in bit 3,
// so the partner value is one warp shuffle away; k0 = 0 and k0 = KS / 2 are their own partners (a register permutation).
// With c extended by c_{N-k} = conj(c_k), every element is E_k = Z_k + c_k (Z_k - Z_{N-k}), stored straight to global
// memory.  Used when the plan has one last-pass butterfly per thread and RL <= 8.
template <class ZP> __host__ __device__ constexpr int zplan_npass() { return ZP::R2 > 1 ? (ZP::R3 > 1 ? 3 : 2) : 1; }
template <class ZP> __host__ __device__ constexpr int zplan_rl() { return zplan_npass<ZP>() == 3 ? ZP::R3 : ZP::R2; }
template <int N, class ZP, int NT> __host__ __device__ constexpr bool z_fuse_last() {
    return zplan_npass<ZP>() >= 2 && zplan_rl<ZP>() <= 8 && (N / zplan_rl<ZP>()) == NT / TILE_LINES && (N / zplan_rl<ZP>()) >= 4;
}

template <int N, class ZP, bool FWD, int NT, class Emit>
__device__ __forceinline__ void z_last_pass_fused(const cplx *__restrict__ s, const cplx *__restrict__ ctab,
                                                  const cplx *__restrict__ red, int tid, int nout, double sc, Emit emit) {
    constexpr int R1 = ZP::R1, R2 = ZP::R2;
    constexpr int NPASS = zplan_npass<ZP>();
    constexpr int RL = zplan_rl<ZP>();
    constexpr int KS = NPASS == 3 ? R1 * R2 : R1;
    constexpr int NW = NT / 32;
    static_assert(KS * RL == N && KS == NT / TILE_LINES, "one last-pass butterfly per thread");
    const int line = tid & (TILE_LINES - 1);
    const int i = tid >> 3, p = i >> 1, h = i & 1;
    const int k0 = p == 0 ? (h ? KS / 2 : 0) : (h ? KS - p : p);
    const int b = NPASS == 3 ? (k0 % R1) * R2 + k0 / R1 : k0;
    cplx v[RL];
#pragma unroll
    for (int m = 0; m < RL; ++m) v[m] = s[(b * RL + m) * TILE_LINES + line];
    RegFFT<RL, -1>::run(v);
    cplx H0 = make_double2(0.0, 0.0);
    if (k0 == 0) {
#pragma unroll
        for (int w = 0; w < NW; ++w) H0 = cadd(H0, red[w * 8 + line]);
    }
#pragma unroll
    for (int q = 0; q < RL; ++q) {
        // partner value Z_{N-k}: lane ^ 8 holds butterfly KS - k0, element RL - 1 - q (all lanes shuffle, also the self-paired)
        cplx zp;
        zp.x = __shfl_xor_sync(0xffffffffu, v[RL - 1 - q].x, 8);
        zp.y = __shfl_xor_sync(0xffffffffu, v[RL - 1 - q].y, 8);
        if (p == 0) zp = h ? v[RL - 1 - q] : v[(RL - q) & (RL - 1)];     // k0 = KS/2: q <-> RL-1-q;  k0 = 0: q <-> RL-q
        const int k = k0 + KS * q;
        const cplx z = v[q];
        if (k == 0) {
            const cplx G0 = make_double2(z.x + H0.y, z.y - H0.x);          // Z_0 - i H_0
            emit(0, cscale(cadd(G0, H0), FWD ? 0.5 * sc : sc));
            if (N < nout) emit(N, cscale(csub(G0, H0), FWD ? 0.5 * sc : sc));
        } else if (k < nout) {
            cplx c = ctab[k <= N / 2 ? k : N - k];
            if (k > N / 2) c.y = -c.y;                                     // c_{N-k} = conj(c_k)
            const cplx d = csub(z, zp);
            emit(k, cscale(make_double2(z.x + (c.x * d.x - c.y * d.y), z.y + (c.x * d.y + c.y * d.x)), sc));
        }
    }
}

template <int N, bool FWD>
__global__ void __launch_bounds__(ztma_threads<N>()) k_zpass_tma(const __grid_constant__ ZTArgs a,
                                                                       const cplx *__restrict__ twn_g,
                                                                       const cplx *__restrict__ ctab_g) {
    typedef PlanZB<N> ZP;
    constexpr int NT = ztma_threads<N>();
    constexpr int NW = NT / 32;
    constexpr int NSTG = 2;
    extern __shared__ __align__(16) unsigned char smem_raw[];   // dynamic shared memory starts 1024-byte aligned (no static part)
    const int srows = a.nboxes * a.box_rows;
    cplx *stg0 = reinterpret_cast<cplx *>(smem_raw);                 // stages first: TMA destinations, 128-byte aligned
    cplx *stg1 = stg0 + (size_t)(NSTG - 1) * srows * TILE_LINES;
    cplx *s = stg1 + (size_t)srows * TILE_LINES;
    cplx *red = s + N * TILE_LINES;
    cplx *tw_s = red + NW * 8;
    cplx *ctab_s = tw_s + N;
    unsigned long long *bar = reinterpret_cast<unsigned long long *>(ctab_s + (N / 2 + 1) + 1);   // 2 barriers
    const cplx *__restrict__ tw = tw_s;
    const cplx *__restrict__ ctab = ctab_s;
    const int tid = threadIdx.x, line = tid & 7, r0 = tid >> 3;
    constexpr int RSTEP = NT / TILE_LINES;
    const size_t stride = (size_t)a.ncols;
    const int nin = FWD ? N + 1 : a.nk;
    const int nout = FWD ? a.nk : N + 1;
    const double sc = FWD ? 1.0 / N : 1.0;
    const int tiles_per_field = a.ncols / 8;
    const int ntiles = tiles_per_field * a.nf;
    const unsigned tile_bytes = (unsigned)((size_t)srows * TILE_LINES * sizeof(cplx));
    auto issue = [&](int t, int b) {          // thread 0 only
        const int fl = t / tiles_per_field, ct = t - fl * tiles_per_field;
        cplx *dst = b ? stg1 : stg0;
        mbar_expect_tx(bar + b, tile_bytes);
        for (int q = 0; q < a.nboxes; ++q)
            tma_load_2d(dst + (size_t)q * a.box_rows * TILE_LINES, &a.in_map[fl], ct * 16, q * a.box_rows, bar + b);
    };
    if (tid == 0) {
        mbar_init(bar, 1);
        mbar_init(bar + 1, 1);
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        if ((int)blockIdx.x < ntiles) issue(blockIdx.x, 0);
        if (NSTG > 1 && (int)(blockIdx.x + gridDim.x) < ntiles) issue(blockIdx.x + gridDim.x, 1);
    }
    for (int i = tid; i < N; i += NT) tw_s[i] = twn_g[i];
    for (int i = tid; i <= N / 2; i += NT) ctab_s[i] = ctab_g[i];
    __syncthreads();
    int it = 0;
    for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x, ++it) {
        const int b = it & (NSTG - 1);
        const unsigned parity = (unsigned)((NSTG > 1 ? it >> 1 : it) & 1);
        const int fld = tile / tiles_per_field, ct = tile - fld * tiles_per_field;
        const size_t col = (size_t)ct * 8 + line;
        cplx *__restrict__ out = reinterpret_cast<cplx *>(a.out[fld]) + col;
        const cplx *__restrict__ stg = b ? stg1 : stg0;
        mbar_wait(bar + b, parity);
        cplx h0 = make_double2(0.0, 0.0);
        fft_head_z<N, NT, ZP>(s, tw, tid, [&](int m) {
            const int ne = (m < N / 2) ? 2 * m : 2 * N - 2 * m;
            const int no = (m < N / 2) ? 2 * m + 1 : 2 * N - 2 * m - 1;
            cplx e0 = make_double2(0.0, 0.0), e1 = e0;
            if (ne < nin) e0 = stg[ne * TILE_LINES + line];
            if (no < nin) e1 = stg[no * TILE_LINES + line];
            if (!FWD) {
                if (ne > 0 && ne < N) e0 = cscale(e0, 0.5);
                e1 = cscale(e1, 0.5);
            }
            h0 = cadd(h0, e1);
            return make_double2(e0.x - e1.y, e0.y + e1.x);
        });
        h0.x += __shfl_xor_sync(0xffffffffu, h0.x, 8);  h0.y += __shfl_xor_sync(0xffffffffu, h0.y, 8);
        h0.x += __shfl_xor_sync(0xffffffffu, h0.x, 16); h0.y += __shfl_xor_sync(0xffffffffu, h0.y, 16);
        if ((tid & 31) < 8) red[(tid >> 5) * 8 + line] = h0;
        __syncthreads();                      // head pass done: stage b is free, the FFT tile is complete
        if (tid == 0 && tile + NSTG * (int)gridDim.x < ntiles) {
            fence_proxy_async();
            issue(tile + NSTG * gridDim.x, b);
        }
        const bool der = !FWD && fld == a.dfield;
        double kx = 0.0, ky = 0.0;
        cplx *odx = nullptr, *ody = nullptr;
        if (der) {
            const int ir = (int)(col % a.kxp), jr = (int)(col / a.kxp);
            kx = a.kxf * (double)ir;
            ky = a.kyf * (double)(jr < a.jpos ? jr : jr - a.nky);
            if (a.out_dx) odx = a.out_dx + col;
            if (a.out_dy) ody = a.out_dy + col;
        }
        auto emit = [&](int k, cplx v) {
            out[(size_t)k * stride] = v;
            if (der) {
                if (odx) odx[(size_t)k * stride] = make_double2(-kx * v.y, kx * v.x);
                if (ody) ody[(size_t)k * stride] = make_double2(-ky * v.y, ky * v.x);
            }
        };
        if constexpr (z_fuse_last<N, ZP, NT>()) {
            // middle pass (three-pass plans) in place, then the last pass fused with the post-processing
            if constexpr (zplan_npass<ZP>() == 3) {
                fft_pass<N, N / ZP::R1, ZP::R2, -1, NT>(s, tw, tid);
                __syncthreads();
            }
            z_last_pass_fused<N, ZP, FWD, NT>(s, ctab, red, tid, nout, sc, emit);
        } else {
            fft_rest_inplace_nb<N, -1, NT, ZP>(s, tw, tid);
            __syncthreads();
            for (int k = r0; k <= N / 2; k += RSTEP) {
                const int kb = N - k;
                if (k == 0) {
                    cplx H0 = make_double2(0.0, 0.0);
#pragma unroll
                    for (int w = 0; w < NW; ++w) H0 = cadd(H0, red[w * 8 + line]);
                    const cplx z0 = s[line];
                    const cplx G0 = make_double2(z0.x + H0.y, z0.y - H0.x);
                    emit(0, cscale(cadd(G0, H0), FWD ? 0.5 * sc : sc));
                    if (N < nout) emit(N, cscale(csub(G0, H0), FWD ? 0.5 * sc : sc));
                } else {
                    const cplx za = s[fft_pos_f<N, ZP>(k) * TILE_LINES + line];
                    const cplx zb = s[fft_pos_f<N, ZP>(kb) * TILE_LINES + line];
                    const cplx c = ctab[k];
                    const cplx d = csub(za, zb);
                    const cplx cd = make_double2(c.x * d.x - c.y * d.y, c.x * d.y + c.y * d.x);
                    const cplx ccd = make_double2(c.x * d.x + c.y * d.y, c.x * d.y - c.y * d.x);
                    if (k < nout) emit(k, cscale(cadd(za, cd), sc));
                    if (kb != k && kb < nout) emit(kb, cscale(csub(zb, ccd), sc));
                }
            }
        }
        __syncthreads();
    }
}


}  // namespace psdns
