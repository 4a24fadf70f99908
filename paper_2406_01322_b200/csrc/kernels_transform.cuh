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

namespace psdns {

constexpr int MAXF = 12;      // max fields per batched launch
constexpr int NT_FFT = 256;   // threads per transform CTA (tiles up to 74 KB, >= 3 CTAs per SM)
// the 147 KB tile (L = 1024) allows one CTA per SM: give it 16 warps instead of 8 to hide latency
template <int L> __host__ __device__ constexpr int tile_threads() { return L >= 1024 ? 512 : 256; }

struct FieldPtrs {
    const void *in[MAXF];
    void *out[MAXF];
};

template <int L>
__device__ __forceinline__ void load_twiddles(cplx *tw, const cplx *__restrict__ twg, int tid, int nt) {
    for (int i = tid; i < L; i += nt) tw[i] = twg[i];
}

// ------------------------------------------------------------------------------------------
// z pass: Chebyshev transform = DCT-I as the length-2N FFT of the even extension,
// Re and Im transformed together (the DFT of a real-even sequence is real).
//   backward (row a2): a_n, n < nk  ->  f_k = sum_n a_n cos(pi n k / N), k = 0..N
//   forward  (row a8): f_k          ->  a_n = 1/(N c_n) DFT_n(even ext), n < nk (truncation)
// grid = (ncols/8, nfields); L = 2N.
// ------------------------------------------------------------------------------------------
struct ZArgs {
    FieldPtrs f;
    int ncols;  // nky * kxp (multiple of 8) = plane stride in cplx
    int nk;     // coefficient planes read (backward) or written (forward)
};

template <int L, bool FWD>
__global__ void __launch_bounds__(tile_threads<L>()) k_zpass(const __grid_constant__ ZArgs a, const cplx *__restrict__ twg) {
    constexpr int NT = tile_threads<L>();
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cplx *s = reinterpret_cast<cplx *>(smem_raw);
    cplx *tw = s + L * TILE_LINES;
    constexpr int N = L / 2;
    const int tid = threadIdx.x, line = tid & 7, r0 = tid >> 3;
    constexpr int RSTEP = NT / TILE_LINES;
    const size_t stride = (size_t)a.ncols;
    const cplx *__restrict__ in = reinterpret_cast<const cplx *>(a.f.in[blockIdx.y]) + (size_t)blockIdx.x * 8 + line;
    cplx *__restrict__ out = reinterpret_cast<cplx *>(a.f.out[blockIdx.y]) + (size_t)blockIdx.x * 8 + line;
    load_twiddles<L>(tw, twg, tid, NT);
    if (!FWD) {
        const int nk = a.nk;
        for (int n = r0; n <= N; n += RSTEP) {
            cplx v = make_double2(0.0, 0.0);
            if (n < nk) v = in[n * stride];
            if (n > 0 && n < N) {
                v = cscale(v, 0.5);
                s[(L - n) * TILE_LINES + line] = v;
            }
            s[n * TILE_LINES + line] = v;
        }
    } else {
        for (int k = r0; k <= N; k += RSTEP) {
            cplx v = in[k * stride];
            if (k > 0 && k < N) s[(L - k) * TILE_LINES + line] = v;
            s[k * TILE_LINES + line] = v;
        }
    }
    __syncthreads();
    fft_tile<L, -1, NT>(s, tw, tid);
    __syncthreads();
    if (!FWD) {
        for (int k = r0; k <= N; k += RSTEP) out[k * stride] = s[fft_pos<L>(k) * TILE_LINES + line];
    } else {
        const int nk = a.nk;
        const double sc = 1.0 / N;
        for (int n = r0; n < nk; n += RSTEP) {
            cplx v = s[fft_pos<L>(n) * TILE_LINES + line];
            out[n * stride] = cscale(v, (n == 0 || n == N) ? 0.5 * sc : sc);
        }
    }
}

// ------------------------------------------------------------------------------------------
// z pass, half-length form (the optimisation PAPER.md L178 attributes to Makhoul [32]: "does not require
// performing a transform of size 2N but only of size N by re-ordering the input signal").
// With e = even extension (length 2N) of the complex column, g_m = e_{2m}, h_m = e_{2m+1} (m < N):
//   E_k = DFT_2N(e)_k = G_k + w_2N^k H_k.  Pack z_m = g_m + i h_m (complex arithmetic), Z = FFT_N(z).
//   g is even (G_{N-k} = G_k) and h is half-sample symmetric (H_{N-k} = w_N^k H_k), so
//   Z_k - Z_{N-k} = i (1 - w_N^k) H_k and
//   E_k = Z_k + c_k (Z_k - Z_{N-k}),  c_k = -(1 + sin t)/(2 sin t) + i cos t/(2 sin t),  t = pi k / N,
//   c_{N-k} = conj(c_k); k = 0 and k = N need H_0 = sum_m h_m (reduced while loading):
//   G_0 = Z_0 - i H_0, E_0 = G_0 + H_0, E_N = G_0 - H_0.
// One N-point complex FFT per complex column: half the flops and half the shared memory of the 2N form
// (64 KB tile at N = 512, three CTAs per SM).  Rounding error is amplified by |c_k| <= ~N/(2 pi k) in the
// lowest/highest modes (<= 1e-14 relative at N = 512; tolerance 1e-11).
//   grid = (ncols/8, nfields); template N = nz - 1.
// ------------------------------------------------------------------------------------------
template <int N, bool FWD>
__global__ void __launch_bounds__(NT_FFT) k_zpass_h(const __grid_constant__ ZArgs a, const cplx *__restrict__ tw2n,
                                                    const cplx *__restrict__ ctab) {
    constexpr int NT = NT_FFT;
    constexpr int NW = NT / 32;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cplx *s = reinterpret_cast<cplx *>(smem_raw);
    cplx *tw = s + N * TILE_LINES;
    cplx *red = tw + N;                       // [NW][8] partial sums of H_0
    const int tid = threadIdx.x, line = tid & 7, r0 = tid >> 3;
    constexpr int RSTEP = NT / TILE_LINES;
    const size_t stride = (size_t)a.ncols;
    const cplx *__restrict__ in = reinterpret_cast<const cplx *>(a.f.in[blockIdx.y]) + (size_t)blockIdx.x * 8 + line;
    cplx *__restrict__ out = reinterpret_cast<cplx *>(a.f.out[blockIdx.y]) + (size_t)blockIdx.x * 8 + line;
    for (int i = tid; i < N; i += NT) tw[i] = tw2n[2 * i];
    const int nin = FWD ? N + 1 : a.nk;       // input rows that are not structurally zero
    cplx h0 = make_double2(0.0, 0.0);
    for (int m = r0; m <= N / 2; m += RSTEP) {
        const int ne = 2 * m;
        cplx ev = make_double2(0.0, 0.0), op = ev, om = ev;
        if (ne < nin) ev = in[ne * stride];
        if (m < N / 2 && ne + 1 < nin) op = in[(ne + 1) * stride];
        if (m >= 1 && ne - 1 < nin) om = in[(ne - 1) * stride];
        if (!FWD) {                           // backward: interior coefficients enter with weight 1/2
            if (ne > 0 && ne < N) ev = cscale(ev, 0.5);
            op = cscale(op, 0.5);             // odd rows are always interior
            om = cscale(om, 0.5);
        }
        // z_m = e_{2m} + i e_{2m+1} ; z_{N-m} = e_{2m} + i e_{2m-1}
        if (m < N / 2) s[m * TILE_LINES + line] = make_double2(ev.x - op.y, ev.y + op.x);
        if (m >= 1) s[(N - m) * TILE_LINES + line] = make_double2(ev.x - om.y, ev.y + om.x);
        h0 = cadd(h0, cadd(op, om));
    }
    // reduce H_0 over the threads that share this line: lanes differ in bits 3, 4 within a warp
    h0.x += __shfl_xor_sync(0xffffffffu, h0.x, 8);  h0.y += __shfl_xor_sync(0xffffffffu, h0.y, 8);
    h0.x += __shfl_xor_sync(0xffffffffu, h0.x, 16); h0.y += __shfl_xor_sync(0xffffffffu, h0.y, 16);
    if ((tid & 31) < 8) red[(tid >> 5) * 8 + line] = h0;
    __syncthreads();
    fft_tile<N, -1, NT>(s, tw, tid);
    __syncthreads();
    const int nout = FWD ? a.nk : N + 1;      // output rows kept
    const double sc = FWD ? 1.0 / N : 1.0;
    for (int k = r0; k <= N / 2; k += RSTEP) {
        const int kb = N - k;
        if (k == 0) {
            cplx H0 = make_double2(0.0, 0.0);
#pragma unroll
            for (int w = 0; w < NW; ++w) H0 = cadd(H0, red[w * 8 + line]);
            const cplx z0 = s[line];          // fft_pos(0) = 0
            const cplx G0 = make_double2(z0.x + H0.y, z0.y - H0.x);   // Z_0 - i H_0
            out[0] = cscale(cadd(G0, H0), FWD ? 0.5 * sc : sc);
            if (N < nout) out[(size_t)N * stride] = cscale(csub(G0, H0), FWD ? 0.5 * sc : sc);
        } else {
            const cplx za = s[fft_pos<N>(k) * TILE_LINES + line];
            const cplx zb = s[fft_pos<N>(kb) * TILE_LINES + line];
            const cplx c = ctab[k];
            const cplx d = csub(za, zb);
            const cplx cd = make_double2(c.x * d.x - c.y * d.y, c.x * d.y + c.y * d.x);     // c_k d
            const cplx ccd = make_double2(c.x * d.x + c.y * d.y, c.x * d.y - c.y * d.x);    // conj(c_k) d
            if (k < nout) out[(size_t)k * stride] = cscale(cadd(za, cd), sc);
            if (kb != k && kb < nout) out[(size_t)kb * stride] = cscale(csub(zb, ccd), sc);
        }
    }
}

// ------------------------------------------------------------------------------------------
// y pass: complex <-> complex DFT of length ny per (ir, k) line (Z2Z).
//   backward (row a3): nky retained rows (FFT order compacted) -> ny points, e^{+i ky y}
//   forward  (row a7): ny points -> nky retained rows, e^{-i ky y} / ny
// grid = (kxp/8, nz, nfields); L = ny.
// ------------------------------------------------------------------------------------------
struct YArgs {
    FieldPtrs f;
    int kxp;   // row pitch in cplx (multiple of 8)
    int nky;   // retained ky rows
    int jpos;  // rows 0..jpos-1 are j' = jr >= 0; rows jpos.. are j' = jr - nky < 0
};

template <int L, bool FWD>
__global__ void __launch_bounds__(tile_threads<L>()) k_ypass(const __grid_constant__ YArgs a, const cplx *__restrict__ twg) {
    constexpr int NT = tile_threads<L>();
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cplx *s = reinterpret_cast<cplx *>(smem_raw);
    cplx *tw = s + L * TILE_LINES;
    const int tid = threadIdx.x, line = tid & 7, r0 = tid >> 3;
    constexpr int RSTEP = NT / TILE_LINES;
    const size_t pitch = (size_t)a.kxp;
    const int nky = a.nky, jpos = a.jpos;
    const size_t zin = (size_t)blockIdx.y * (FWD ? L : nky) * pitch;
    const size_t zout = (size_t)blockIdx.y * (FWD ? nky : L) * pitch;
    const cplx *__restrict__ in = reinterpret_cast<const cplx *>(a.f.in[blockIdx.z]) + zin + (size_t)blockIdx.x * 8 + line;
    cplx *__restrict__ out = reinterpret_cast<cplx *>(a.f.out[blockIdx.z]) + zout + (size_t)blockIdx.x * 8 + line;
    load_twiddles<L>(tw, twg, tid, NT);
    if (!FWD) {
        for (int j = r0; j < L; j += RSTEP) {
            // FFT-order row j holds j' = j (j < jpos) or j' = j - L (j >= L - (nky - jpos))
            cplx v = make_double2(0.0, 0.0);
            if (j < jpos) v = in[j * pitch];
            else if (j >= L - (nky - jpos)) v = in[(j - (L - nky)) * pitch];
            s[j * TILE_LINES + line] = v;
        }
    } else {
        for (int y = r0; y < L; y += RSTEP) s[y * TILE_LINES + line] = in[y * pitch];
    }
    __syncthreads();
    fft_tile<L, (FWD ? -1 : +1), NT>(s, tw, tid);
    __syncthreads();
    if (!FWD) {
        for (int y = r0; y < L; y += RSTEP) out[y * pitch] = s[fft_pos<L>(y) * TILE_LINES + line];
    } else {
        const double sc = 1.0 / L;
        for (int jr = r0; jr < nky; jr += RSTEP) {
            const int j = jr < jpos ? jr : jr + (L - nky);
            out[jr * pitch] = cscale(s[fft_pos<L>(j) * TILE_LINES + line], sc);
        }
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
        for (int i = r0; i <= L / 2; i += RSTEP) {
            cplx ca = make_double2(0.0, 0.0), cb = ca;
            if (i < nkx) { ca = inA[i]; cb = inB[i]; }
            if (i == 0 || i == L / 2) {
                s[i * TILE_LINES + p] = make_double2(ca.x, cb.x);
            } else {
                s[i * TILE_LINES + p] = make_double2(ca.x - cb.y, ca.y + cb.x);
                s[(L - i) * TILE_LINES + p] = make_double2(ca.x + cb.y, cb.x - ca.y);
            }
        }
        __syncthreads();
        fft_tile<L, +1, NT>(s, tw, tid);
        __syncthreads();
        double *__restrict__ outA = reinterpret_cast<double *>(a.f.out[blockIdx.y]) + lineA * L;
        double *__restrict__ outB = outA + L;
        for (int x = r0; x < L; x += RSTEP) {
            cplx v = s[fft_pos<L>(x) * TILE_LINES + p];
            outA[x] = v.x;
            outB[x] = v.y;
        }
    } else {
        const double *__restrict__ inA = reinterpret_cast<const double *>(a.f.in[blockIdx.y]) + lineA * L;
        const double *__restrict__ inB = inA + L;
        for (int x = r0; x < L; x += RSTEP) s[x * TILE_LINES + p] = make_double2(inA[x], inB[x]);
        __syncthreads();
        fft_tile<L, -1, NT>(s, tw, tid);
        __syncthreads();
        cplx *__restrict__ outA = reinterpret_cast<cplx *>(a.f.out[blockIdx.y]) + lineA * kxp;
        cplx *__restrict__ outB = outA + kxp;
        const double sc = 0.5 / L;
        for (int i = r0; i < kxp; i += RSTEP) {
            cplx ra = make_double2(0.0, 0.0), rb = ra;
            if (i < nkx) {
                cplx z1 = s[fft_pos<L>(i) * TILE_LINES + p];
                cplx z2 = s[fft_pos<L>((L - i) & (L - 1)) * TILE_LINES + p];
                // A^ = (z1 + conj z2)/2 ; B^ = (z1 - conj z2)/(2i) = (-i/2)(z1 - conj z2)
                ra = make_double2((z1.x + z2.x) * sc, (z1.y - z2.y) * sc);
                rb = make_double2((z1.y + z2.y) * sc, (z2.x - z1.x) * sc);
            }
            outA[i] = ra;
            outB[i] = rb;
        }
    }
}

// ------------------------------------------------------------------------------------------
// pointwise non-linear terms (row a5; Eqs. 1, 4, 7, 8 and L182-196), in place:
//   in : u v w [phi phx phy phz [exx eyy exy exz eyz]]     (buffers 0..11)
//   out: Txx Txy Txz Tyy Tyz Tzz [Q C]                     (buffers 0..7)
//   T_ij = -u_i u_j + cs (|grad phi|^2 delta_ij - phi_i phi_j) + eta1(phi) E_ij
// ------------------------------------------------------------------------------------------
struct PwArgs {
    double *b[MAXF];
    size_t n;
    double cs;        // 3/sqrt(8) Ch/We
    double eta_c;     // (lambda - 1) / (2 Re)
    int phase, visc;
};

__global__ void __launch_bounds__(256) k_pointwise(const __grid_constant__ PwArgs a) {
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < a.n; i += stride) {
        const double u = a.b[0][i], v = a.b[1][i], w = a.b[2][i];
        double txx = -u * u, txy = -u * v, txz = -u * w, tyy = -v * v, tyz = -v * w, tzz = -w * w;
        if (a.phase) {
            const double ph = a.b[3][i], px = a.b[4][i], py = a.b[5][i], pz = a.b[6][i];
            const double g2 = px * px + py * py + pz * pz;
            const double cs = a.cs;
            txx += cs * (g2 - px * px);
            tyy += cs * (g2 - py * py);
            tzz += cs * (g2 - pz * pz);
            txy -= cs * px * py;
            txz -= cs * px * pz;
            tyz -= cs * py * pz;
            if (a.visc) {
                const double e1 = a.eta_c * (ph + 1.0);
                const double exx = a.b[7][i], eyy = a.b[8][i], exy = a.b[9][i], exz = a.b[10][i], eyz = a.b[11][i];
                txx += e1 * exx;
                tyy += e1 * eyy;
                tzz += e1 * (-exx - eyy);
                txy += e1 * exy;
                txz += e1 * exz;
                tyz += e1 * eyz;
            }
            a.b[6][i] = u * px + v * py + w * pz;
            a.b[7][i] = ph * ph * ph;
        }
        a.b[0][i] = txx; a.b[1][i] = txy; a.b[2][i] = txz;
        a.b[3][i] = tyy; a.b[4][i] = tyz; a.b[5][i] = tzz;
    }
}

}  // namespace psdns
