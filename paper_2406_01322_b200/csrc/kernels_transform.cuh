// Batched 1-D transform passes over the private device layouts, and the pointwise kernel.
//
// Private layouts (x / kx fastest everywhere, never transposed):
//   spectral  S : cplx [n ][jr][ir]   n < nk planes, jr < nky retained ky rows, ir < kxp (padded pitch)
//   z-physical Z: cplx [k ][jr][ir]   k <= N wall-normal points
//   zy-physical Y: cplx [k ][y ][ir]
//   physical   P: double [k][y][x]
// A z- or y-pass CTA owns a tile of 8 consecutive ir (one aligned 128-byte segment per row) and
// the whole line in the transform direction; an x-pass CTA owns 16 consecutive (k,y) lines, two
// real lines packed into one complex FFT.  This replaces the paper's transposes (L178) and MPI
// pencil all-to-alls (L154) by strided 128-byte-row accesses of one resident array.
#pragma once
#include "fft_tile.cuh"
#include "fft_fused.cuh"

namespace psdns {

constexpr int MAXF = 12;      // max fields per batched launch
// the 147 KB tile (L = 1024) allows one CTA per SM: give it 16 warps instead of 8 to hide latency
template <int L> __host__ __device__ constexpr int tile_threads() { return L >= 1024 ? 512 : 256; }

struct FieldPtrs {
    const void *in[MAXF];
    void *out[MAXF];
};

// Ampere-style asynchronous copy (LDGSTS): 16 bytes global -> shared without passing through registers
__device__ __forceinline__ void cp_async16(void *dst_smem, const void *src) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"((unsigned)__cvta_generic_to_shared(dst_smem)), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

template <int L>
__device__ __forceinline__ void load_twiddles(cplx *tw, const cplx *__restrict__ twg, int tid, int nt) {
    for (int i = tid; i < L; i += nt) tw[i] = twg[i];
}

// ------------------------------------------------------------------------------------------
// z pass: Chebyshev transform = DCT-I ("FFT of a 2N even extension ... transposes"), in the
// half-length form that L178 attributes to Makhoul [32] ("does not require performing a transform of size 2N
// but only of size N by re-ordering the input signal"), Re and Im transformed together, no transposes.
//   backward (row a2): a_n, n < nk  ->  f_k = sum_n a_n cos(pi n k / N), k = 0..N
//   forward  (row a8): f_k          ->  a_n = 2/(N c_n) sum_k f_k cos(pi n k / N) / c_k, n < nk (truncation)
// With e = even extension (length 2N) of the (weighted) column, g_m = e_{2m}, h_m = e_{2m+1} (m < N):
//   E_k = DFT_2N(e)_k = G_k + w_2N^k H_k.  Pack z_m = g_m + i h_m (complex arithmetic), Z = FFT_N(z).
//   g is even (G_{N-k} = G_k) and h is half-sample symmetric (H_{N-k} = w_N^k H_k), so
//   Z_k - Z_{N-k} = i (1 - w_N^k) H_k and
//   E_k = Z_k + c_k (Z_k - Z_{N-k}),  c_k = -(1 + sin t)/(2 sin t) + i cos t/(2 sin t),  t = pi k / N,
//   c_{N-k} = conj(c_k); k = 0 and k = N need H_0 = sum_m h_m (reduced while loading):
//   G_0 = Z_0 - i H_0, E_0 = G_0 + H_0, E_N = G_0 - H_0.
// Rounding error is amplified by |c_k| <= ~N/(2 pi k) in the lowest/highest modes (<= 1e-14 relative at
// N = 512; tolerance 1e-11).
// Persistent CTAs loop over tiles of 8 consecutive columns; the first FFT pass is fed through registers
// (fft_fused.cuh): the even rows straight from global memory, the odd rows from a shared-memory stage that
// cp.async fills one tile ahead (a thread cannot keep all 32 of its 16-byte loads in flight in 128 registers;
// profiles/r1d: 35 % of the samples were long-scoreboard waits in the head pass).  Optional derived outputs i kx X and i ky X of one field (row a1:
// the x / y derivatives of phi commute with the z transform, so they cost no transform of their own).
// ------------------------------------------------------------------------------------------
// fft_head with an explicit plan (the load functor type is deduced)
template <int L, int NT, class P, class Load>
__device__ __forceinline__ void fft_head_z(cplx *__restrict__ s, const cplx *__restrict__ tw, int tid, Load load) {
    fft_head<L, -1, NT, Load, P>(s, tw, tid, load);
}

struct ZArgs {
    FieldPtrs f;
    int nf;     // fields
    int ncols;  // nky * kxp (multiple of 8) = plane stride in cplx
    int nk;     // coefficient planes read (backward) or written (forward)
    // derived outputs of field dfield (backward only; either pointer may be null; dfield < 0: none)
    int dfield;
    cplx *out_dx, *out_dy;
    int kxp, nky, jpos;
    double kxf, kyf;
};

template <int N, bool FWD> struct ZPlan { typedef PlanF<N> type; };
template <int N> struct ZPlan<N, false> { typedef PlanZB<N> type; };
template <int N, bool FWD> __host__ __device__ constexpr int zpass_threads() { return fused_threads<N, typename ZPlan<N, FWD>::type>(); }

template <int N, bool FWD> __host__ __device__ constexpr int zpass_smem_cplx() {
    return N * TILE_LINES + N + (zpass_threads<N, FWD>() / 32) * 8 + (N / 2 + 1) + (FWD ? 0 : (N / 2) * TILE_LINES);
}

template <int N, bool FWD>
__global__ void __launch_bounds__(zpass_threads<N, FWD>(), (N >= 512 ? 2 : 3)) k_zpass(const __grid_constant__ ZArgs a,
                                                                               const cplx *__restrict__ tw2n,
                                                                               const cplx *__restrict__ ctab_g) {
    typedef typename ZPlan<N, FWD>::type ZP;
    constexpr int NT = zpass_threads<N, FWD>();
    constexpr int NW = NT / 32;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cplx *s = reinterpret_cast<cplx *>(smem_raw);
    cplx *tw = s + N * TILE_LINES;
    cplx *red = tw + N;                       // [NW][8] partial sums of H_0
    cplx *ctab = red + NW * 8;                // c_k, k <= N/2
    cplx *stg = ctab + (N / 2 + 1);           // [N/2][8]: odd input rows 1, 3, .., N-1 of the next tile
    const int tid = threadIdx.x, line = tid & 7, r0 = tid >> 3;
    constexpr int RSTEP = NT / TILE_LINES;
    const size_t stride = (size_t)a.ncols;
    for (int i = tid; i < N; i += NT) tw[i] = tw2n[2 * i];
    for (int i = tid; i <= N / 2; i += NT) ctab[i] = ctab_g[i];
    const int nin = FWD ? N + 1 : a.nk;       // input rows that are not structurally zero
    const int nout = FWD ? a.nk : N + 1;      // output rows kept
    const double sc = FWD ? 1.0 / N : 1.0;
    const int tiles_per_field = a.ncols / 8;
    const int ntiles = tiles_per_field * a.nf;
    // measured (B200, N = 512): staging helps the backward pass (2/3 of the rows are structurally zero, so the
    // remaining direct loads all fit in flight: 3.03 -> 2.74 ms) and hurts the forward pass (3.0 -> 3.5 ms)
    constexpr bool STAGE = !FWD;
    auto prefetch = [&](int t) {              // odd rows of tile t -> stage (each thread: its line of rows r0, r0 + RSTEP, ..)
        if (STAGE && t < ntiles) {
            const int fl = t / tiles_per_field;
            const cplx *src = reinterpret_cast<const cplx *>(a.f.in[fl]) + (size_t)(t - fl * tiles_per_field) * 8 + line;
            for (int r = r0; 2 * r + 1 < nin && r < N / 2; r += RSTEP) cp_async16(stg + r * TILE_LINES + line, src + (size_t)(2 * r + 1) * stride);
        }
        cp_async_commit();
    };
    prefetch(blockIdx.x);
    for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
        const int fld = tile / tiles_per_field, ct = tile - fld * tiles_per_field;
        const size_t col = (size_t)ct * 8 + line;
        const cplx *__restrict__ in = reinterpret_cast<const cplx *>(a.f.in[fld]) + col;
        cplx *__restrict__ out = reinterpret_cast<cplx *>(a.f.out[fld]) + col;
        cp_async_wait_all();
        __syncthreads();                      // stage (and, first time, the tables) visible to all threads
        cplx h0 = make_double2(0.0, 0.0);
        // z_m = e_{2m} + i e_{2m+1}; for m >= N/2 the even extension folds back: e_j = a_{2N-j}
        fft_head_z<N, NT, ZP>(s, tw, tid, [&](int m) {
            const int ne = (m < N / 2) ? 2 * m : 2 * N - 2 * m;
            const int no = (m < N / 2) ? 2 * m + 1 : 2 * N - 2 * m - 1;
            cplx e0 = make_double2(0.0, 0.0), e1 = e0;
            if (ne < nin) e0 = __ldcg(in + ne * stride);
            if (no < nin) e1 = STAGE ? stg[(no >> 1) * TILE_LINES + line] : __ldcg(in + no * stride);
            if (!FWD) {                       // backward: interior coefficients enter with weight 1/2
                if (ne > 0 && ne < N) e0 = cscale(e0, 0.5);
                e1 = cscale(e1, 0.5);         // odd rows are always interior
            }
            h0 = cadd(h0, e1);
            return make_double2(e0.x - e1.y, e0.y + e1.x);
        });
        // reduce H_0 over the threads that share this line: lanes differ in bits 3, 4 within a warp
        h0.x += __shfl_xor_sync(0xffffffffu, h0.x, 8);  h0.y += __shfl_xor_sync(0xffffffffu, h0.y, 8);
        h0.x += __shfl_xor_sync(0xffffffffu, h0.x, 16); h0.y += __shfl_xor_sync(0xffffffffu, h0.y, 16);
        if ((tid & 31) < 8) red[(tid >> 5) * 8 + line] = h0;
        __syncthreads();                      // head pass done: the stage is free
        prefetch(tile + gridDim.x);
        fft_rest_inplace_nb<N, -1, NT, ZP>(s, tw, tid);
        __syncthreads();
        // derived outputs: i kx E, i ky E of this column
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
        for (int k = r0; k <= N / 2; k += RSTEP) {
            const int kb = N - k;
            if (k == 0) {
                cplx H0 = make_double2(0.0, 0.0);
#pragma unroll
                for (int w = 0; w < NW; ++w) H0 = cadd(H0, red[w * 8 + line]);
                const cplx z0 = s[line];          // fft_pos_f(0) = 0
                const cplx G0 = make_double2(z0.x + H0.y, z0.y - H0.x);   // Z_0 - i H_0
                emit(0, cscale(cadd(G0, H0), FWD ? 0.5 * sc : sc));
                if (N < nout) emit(N, cscale(csub(G0, H0), FWD ? 0.5 * sc : sc));
            } else {
                const cplx za = s[fft_pos_f<N, ZP>(k) * TILE_LINES + line];
                const cplx zb = s[fft_pos_f<N, ZP>(kb) * TILE_LINES + line];
                const cplx c = ctab[k];
                const cplx d = csub(za, zb);
                const cplx cd = make_double2(c.x * d.x - c.y * d.y, c.x * d.y + c.y * d.x);     // c_k d
                const cplx ccd = make_double2(c.x * d.x + c.y * d.y, c.x * d.y - c.y * d.x);    // conj(c_k) d
                if (k < nout) emit(k, cscale(cadd(za, cd), sc));
                if (kb != k && kb < nout) emit(kb, cscale(csub(zb, ccd), sc));
            }
        }
        __syncthreads();
    }
}

// ------------------------------------------------------------------------------------------
// y pass: complex <-> complex DFT of length ny per (ir, k) line (Z2Z).
//   backward (row a3): nky retained rows (FFT order compacted) -> ny points, e^{+i ky y}
//   forward  (row a7): ny points -> nky retained rows, e^{-i ky y} / ny
// Persistent CTAs loop over tiles (8 consecutive ir) x (one z plane) x (one field); first pass fed from
// global memory through registers, last pass drained to global memory (fft_fused.cuh).
// ------------------------------------------------------------------------------------------
struct YArgs {
    FieldPtrs f;
    int nf, nz;
    int kxp;   // row pitch in cplx (multiple of 8)
    int nky;   // retained ky rows
    int jpos;  // rows 0..jpos-1 are j' = jr >= 0; rows jpos.. are j' = jr - nky < 0
};

template <int L, bool FWD>
__global__ void __launch_bounds__(fused_threads<L>(), (L >= 512 ? 2 : 3)) k_ypass(const __grid_constant__ YArgs a,
                                                                               const cplx *__restrict__ twg) {
    constexpr int NT = fused_threads<L>();
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cplx *s = reinterpret_cast<cplx *>(smem_raw);
    cplx *tw = s + L * TILE_LINES;
    const int tid = threadIdx.x, line = tid & 7;
    const size_t pitch = (size_t)a.kxp;
    const int nky = a.nky, jpos = a.jpos;
    const int nneg = nky - jpos;              // retained rows with j' < 0
    load_twiddles<L>(tw, twg, tid, NT);
    __syncthreads();
    const int tiles_x = a.kxp / 8;
    const int ntiles = tiles_x * a.nz * a.nf;
    const double sc = 1.0 / L;
    for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
        const int cx = tile % tiles_x;
        const int t2 = tile / tiles_x;
        const int z = t2 % a.nz, fld = t2 / a.nz;
        const size_t zin = (size_t)z * (FWD ? L : nky) * pitch;
        const size_t zout = (size_t)z * (FWD ? nky : L) * pitch;
        const cplx *__restrict__ in = reinterpret_cast<const cplx *>(a.f.in[fld]) + zin + (size_t)cx * 8 + line;
        cplx *__restrict__ out = reinterpret_cast<cplx *>(a.f.out[fld]) + zout + (size_t)cx * 8 + line;
        if (!FWD) {
            // FFT-order row j holds j' = j (j < jpos) or j' = j - L (j >= L - nneg); the rest is zero
            fft_head<L, +1, NT>(s, tw, tid, [&](int j) {
                cplx v = make_double2(0.0, 0.0);
                if (j < jpos) v = __ldcg(in + j * pitch);
                else if (j >= L - nneg) v = __ldcg(in + (j - (L - nky)) * pitch);
                return v;
            });
            fft_rest_store<L, +1, NT>(s, tw, tid, [&](int y, cplx v) { out[y * pitch] = v; });
        } else {
            fft_head<L, -1, NT>(s, tw, tid, [&](int y) { return __ldcg(in + y * pitch); });
            fft_rest_store<L, -1, NT>(s, tw, tid, [&](int j, cplx v) {
                if (j < jpos) out[j * pitch] = cscale(v, sc);
                else if (j >= L - nneg) out[(j - (L - nky)) * pitch] = cscale(v, sc);
            });
        }
        __syncthreads();
    }
}

// ------------------------------------------------------------------------------------------
// x pass: real <-> half-complex DFT of length nx per (k, y) line (D2Z / Z2D).
// Two real lines A, B ride one complex FFT: z = a + i b.
//   backward (row a4): Z_i = A^_i + i B^_i, Z_{L-i} = conj(A^_i) + i conj(B^_i); the imaginary
//                      parts of the i = 0 and i = L/2 coefficients are dropped (reading S20)
//   forward  (row a6): A^_i = (Z_i + conj Z_{L-i})/2, B^_i = (Z_i - conj Z_{L-i})/(2i), times 1/nx,
//                      only i < nkx kept (truncation), pad columns written as zero
// grid = (nlines/16, nfields); L = nx; lines are the flattened (k, y) index.
// ------------------------------------------------------------------------------------------
struct XArgs {
    FieldPtrs f;
    int kxp;  // spectral row pitch
    int nkx;  // retained kx (<= L/2 + 1)
};

template <int L, bool FWD>
__global__ void __launch_bounds__(tile_threads<L>()) k_xpass(const __grid_constant__ XArgs a, const cplx *__restrict__ twg) {
    constexpr int NT = tile_threads<L>();
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cplx *s = reinterpret_cast<cplx *>(smem_raw);
    cplx *tw = s + L * TILE_LINES;
    const int tid = threadIdx.x, p = tid & 7, r0 = tid >> 3;
    constexpr int RSTEP = NT / TILE_LINES;
    const size_t lineA = (size_t)blockIdx.x * 16 + 2 * p;
    const int kxp = a.kxp, nkx = a.nkx;
    load_twiddles<L>(tw, twg, tid, NT);
    if (!FWD) {
        const cplx *__restrict__ inA = reinterpret_cast<const cplx *>(a.f.in[blockIdx.y]) + lineA * kxp;
        const cplx *__restrict__ inB = inA + kxp;
        // two consecutive coefficients per thread: 32 contiguous bytes per line (whole sectors)
        for (int i0 = 2 * r0; i0 <= L / 2; i0 += 2 * RSTEP) {
            cplx ca[2], cb[2];
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                ca[e] = cb[e] = make_double2(0.0, 0.0);
                if (i0 + e < nkx) { ca[e] = inA[i0 + e]; cb[e] = inB[i0 + e]; }
            }
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                const int i = i0 + e;
                if (i > L / 2) break;
                if (i == 0 || i == L / 2) {
                    s[i * TILE_LINES + p] = make_double2(ca[e].x, cb[e].x);
                } else {
                    s[i * TILE_LINES + p] = make_double2(ca[e].x - cb[e].y, ca[e].y + cb[e].x);
                    s[(L - i) * TILE_LINES + p] = make_double2(ca[e].x + cb[e].y, cb[e].x - ca[e].y);
                }
            }
        }
        __syncthreads();
        fft_tile<L, +1, NT>(s, tw, tid);
        __syncthreads();
        double *__restrict__ outA = reinterpret_cast<double *>(a.f.out[blockIdx.y]) + lineA * L;
        double *__restrict__ outB = outA + L;
        // a thread stores FOUR consecutive x of its line pair (32 contiguous bytes per line: whole sectors; the 4 threads of a
        // warp that share a line pair cover one 128-byte line) - one x per thread left every sector 3/4 unused per request
        for (int xb = r0 * 4; xb < L; xb += RSTEP * 4) {
            const cplx v0 = s[fft_pos<L>(xb) * TILE_LINES + p], v1 = s[fft_pos<L>(xb + 1) * TILE_LINES + p];
            const cplx v2 = s[fft_pos<L>(xb + 2) * TILE_LINES + p], v3 = s[fft_pos<L>(xb + 3) * TILE_LINES + p];
            *reinterpret_cast<double2 *>(outA + xb) = make_double2(v0.x, v1.x);
            *reinterpret_cast<double2 *>(outA + xb + 2) = make_double2(v2.x, v3.x);
            *reinterpret_cast<double2 *>(outB + xb) = make_double2(v0.y, v1.y);
            *reinterpret_cast<double2 *>(outB + xb + 2) = make_double2(v2.y, v3.y);
        }
    } else {
        const double *__restrict__ inA = reinterpret_cast<const double *>(a.f.in[blockIdx.y]) + lineA * L;
        const double *__restrict__ inB = inA + L;
        for (int xb = r0 * 4; xb < L; xb += RSTEP * 4) {      // four consecutive x per thread: whole 32-byte sectors per line
            const double2 a0 = *reinterpret_cast<const double2 *>(inA + xb), a1 = *reinterpret_cast<const double2 *>(inA + xb + 2);
            const double2 b0 = *reinterpret_cast<const double2 *>(inB + xb), b1 = *reinterpret_cast<const double2 *>(inB + xb + 2);
            s[xb * TILE_LINES + p] = make_double2(a0.x, b0.x);
            s[(xb + 1) * TILE_LINES + p] = make_double2(a0.y, b0.y);
            s[(xb + 2) * TILE_LINES + p] = make_double2(a1.x, b1.x);
            s[(xb + 3) * TILE_LINES + p] = make_double2(a1.y, b1.y);
        }
        __syncthreads();
        fft_tile<L, -1, NT>(s, tw, tid);
        __syncthreads();
        cplx *__restrict__ outA = reinterpret_cast<cplx *>(a.f.out[blockIdx.y]) + lineA * kxp;
        cplx *__restrict__ outB = outA + kxp;
        const double sc = 0.5 / L;
        for (int i0 = 2 * r0; i0 < kxp; i0 += 2 * RSTEP) {   // kxp is a multiple of 8: both coefficients of a pair are inside the row
            cplx ra[2], rb[2];
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                const int i = i0 + e;
                ra[e] = rb[e] = make_double2(0.0, 0.0);
                if (i < nkx) {
                    const cplx z1 = s[fft_pos<L>(i) * TILE_LINES + p];
                    const cplx z2 = s[fft_pos<L>((L - i) & (L - 1)) * TILE_LINES + p];
                    // A^ = (z1 + conj z2)/2 ; B^ = (z1 - conj z2)/(2i) = (-i/2)(z1 - conj z2)
                    ra[e] = make_double2((z1.x + z2.x) * sc, (z1.y - z2.y) * sc);
                    rb[e] = make_double2((z1.y + z2.y) * sc, (z2.x - z1.x) * sc);
                }
            }
            outA[i0] = ra[0]; outA[i0 + 1] = ra[1];
            outB[i0] = rb[0]; outB[i0 + 1] = rb[1];
        }
    }
}

// ------------------------------------------------------------------------------------------
// pointwise non-linear terms (row a5; Eqs. 1, 4, 7, 8 and L182-196), unfused form (variable
// viscosity, reading S14; the matched-viscosity step uses the fused x kernel):
//   in : u v w [phi phx phy phz [exx eyy exy exz eyz]]     (b[0..11])
//   out: Txx-Tzz Txy Txz Tyy-Tzz Tyz [Q C]                 (o[0..6]; may alias the inputs)
//   T_ij = -u_i u_j + cs (|grad phi|^2 delta_ij - phi_i phi_j) + eta1(phi) E_ij; only the deviatoric
//   combinations enter Eqs. 14-15, so T_zz is subtracted here instead of being transformed.
// ------------------------------------------------------------------------------------------
struct PwArgs {
    const double *b[MAXF];
    double *o[10];
    size_t n;
    double cs;        // 3/sqrt(8) Ch/We
    double eta_c;     // (lambda - 1) / (2 Re)
    int phase, visc;
    int force;        // a force vector F = o[7..9] next to the flux tensor (alternative non-linear forms):
    int st_force;     //   surface tension as -cs lap(phi) grad(phi) (b[7] = lap phi) instead of the Korteweg tensor
    int rot;          //   convection as u x omega (b[8..10] = omega) instead of -div(u u)
};

__global__ void __launch_bounds__(256) k_pointwise(const __grid_constant__ PwArgs a) {
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < a.n; i += stride) {
        const double u = a.b[0][i], v = a.b[1][i], w = a.b[2][i];
        double dxx = w * w - u * u, dyy = w * w - v * v, txy = -u * v, txz = -u * w, tyz = -v * w;
        double q = 0.0, c3 = 0.0;
        double fx = 0.0, fy = 0.0, fz = 0.0;
        if (a.rot) {
            const double ox = a.b[8][i], oy = a.b[9][i], oz = a.b[10][i];
            dxx = dyy = txy = txz = tyz = 0.0;
            fx = v * oz - w * oy; fy = w * ox - u * oz; fz = u * oy - v * ox;
        }
        if (a.phase) {
            const double ph = a.b[3][i], px = a.b[4][i], py = a.b[5][i], pz = a.b[6][i];
            const double cs = a.cs;
            if (a.st_force) {
                const double m = -cs * a.b[7][i];
                fx += m * px; fy += m * py; fz += m * pz;
            } else {
                dxx += cs * (pz * pz - px * px);
                dyy += cs * (pz * pz - py * py);
                txy -= cs * px * py;
                txz -= cs * px * pz;
                tyz -= cs * py * pz;
            }
            if (a.visc) {
                const double e1 = a.eta_c * (ph + 1.0);
                const double exx = a.b[7][i], eyy = a.b[8][i], exy = a.b[9][i], exz = a.b[10][i], eyz = a.b[11][i];
                dxx += e1 * (2.0 * exx + eyy);     // E_xx - E_zz, E_zz = -E_xx - E_yy
                dyy += e1 * (exx + 2.0 * eyy);
                txy += e1 * exy;
                txz += e1 * exz;
                tyz += e1 * eyz;
            }
            q = u * px + v * py + w * pz;
            c3 = ph * ph * ph;
        }
        a.o[0][i] = dxx; a.o[1][i] = txy; a.o[2][i] = txz; a.o[3][i] = dyy; a.o[4][i] = tyz;
        if (a.phase || a.force) { a.o[5][i] = q; a.o[6][i] = c3; }
        if (a.force) { a.o[7][i] = fx; a.o[8][i] = fy; a.o[9][i] = fz; }
    }
}

}  // namespace psdns
