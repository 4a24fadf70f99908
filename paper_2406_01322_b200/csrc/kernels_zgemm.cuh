// GEMM form of the Chebyshev transform for short columns (N <= 64, i.e. nz = 33, 65): the DCT-I written as a dense
// FP64 matrix product on the tensor cores (mma.sync.m8n8k4.f64, SASS DMMA) - SURVEY 8(f)-1 / north_star: "DCT-I via the
// FFT path, or a batched dense FP64 matrix transform on tensor cores, chosen by measurement".
//   backward: f_k = sum_{n < nk} a_n cos(pi n k / N)                       out [N+1] x cols = Mb [N+1 x nk] . in [nk x cols]
//   forward : a_n = 2/(N c_n) sum_k f_k cos(pi n k / N) / c_k, n < nk      out [nk]  x cols = Mf [nk x N+1] . in [N+1 x cols]
// A spectral array [row][ncols] of cplx is a real row-major matrix with 2 ncols columns (Re and Im of a column are two
// independent real sequences), so the whole pass is ONE skinny GEMM per field: M, K <= 65, N_gemm = 2 ncols.
// CTA = 4 warps, a block of ZG_COLS = 64 real columns, all rows.  The matrices come from a host long-double table
// (psdns.cu build_tables), zero-padded to [ZG_MP][ZG_KP].
#pragma once
#include "kernels_transform.cuh"

namespace psdns {

constexpr int ZG_MP = 72, ZG_KP = 68;      // padded rows (multiple of 8) / inner length (multiple of 4) for N <= 64
constexpr int ZG_COLS = 64;                // real columns per CTA (= 32 complex columns)
constexpr int ZG_NT = 128;
constexpr size_t ZG_SMEM = (size_t)(72 * 68 + 68 * 68) * sizeof(double);
constexpr int ZG_BP = ZG_COLS + 4;         // row pitch of the staged input = 8 banks mod 32: the 4 rows of a fragment hit disjoint banks

struct ZGArgs {
    FieldPtrs f;
    int nf, ncols;       // complex columns
    int nrow_in, nrow_out;
    const double *mat;   // [ZG_MP][ZG_KP], row = output index, column = input index
    int dfield;
    cplx *out_dy;
    int kxp, nky, jpos;
    double kyf;
};

__device__ __forceinline__ void dmma884(double &c0, double &c1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0, %1}, {%2}, {%3}, {%0, %1};" : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

__global__ void __launch_bounds__(ZG_NT) k_zgemm(const __grid_constant__ ZGArgs a) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double *sA = reinterpret_cast<double *>(smem_raw);      // [ZG_MP][ZG_KP]
    double *sB = sA + ZG_MP * ZG_KP;                        // [ZG_KP][ZG_BP]
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int ld = 2 * a.ncols;                         // doubles per row
    const int nblk = (ld + ZG_COLS - 1) / ZG_COLS;
    const int kp = (a.nrow_in + 3) & ~3;                // inner length rounded up to the MMA k = 4
    const int mt = (a.nrow_out + 7) >> 3;               // output row tiles of 8
    for (int i = tid; i < ZG_MP * ZG_KP; i += ZG_NT) sA[i] = a.mat[i];
    for (int blk = blockIdx.x; blk < nblk * a.nf; blk += gridDim.x) {
        const int fld = blk / nblk, c0 = (blk - fld * nblk) * ZG_COLS;
        const double *__restrict__ in = reinterpret_cast<const double *>(a.f.in[fld]);
        double *__restrict__ out = reinterpret_cast<double *>(a.f.out[fld]);
        __syncthreads();
        // stage the input block: rows k < nrow_in, 64 consecutive doubles (512 bytes) each; zero beyond
        for (int e = tid; e < kp * (ZG_COLS / 2); e += ZG_NT) {
            const int k = e / (ZG_COLS / 2), c = (e - k * (ZG_COLS / 2)) * 2;
            double2 v = make_double2(0.0, 0.0);
            if (k < a.nrow_in && c0 + c < ld) v = *reinterpret_cast<const double2 *>(in + (size_t)k * ld + c0 + c);
            *reinterpret_cast<double2 *>(sB + k * ZG_BP + c) = v;
        }
        __syncthreads();
        const int gq = lane >> 2, tq = lane & 3;        // fragment coordinates: group, thread-in-group
#pragma unroll
        for (int nt = 0; nt < 2; ++nt) {
            const int n0 = warp * 16 + nt * 8;          // column tile of this warp inside the block
            for (int m = 0; m < mt; ++m) {
                double acc0 = 0.0, acc1 = 0.0;
                for (int k0 = 0; k0 < kp; k0 += 4)
                    dmma884(acc0, acc1, sA[(m * 8 + gq) * ZG_KP + k0 + tq], sB[(k0 + tq) * ZG_BP + n0 + gq]);
                // C fragment: row m*8 + gq, columns n0 + 2 tq, + 1 = (Re, Im) of one complex column
                const int row = m * 8 + gq, cc = c0 + n0 + 2 * tq;
                if (row < a.nrow_out && cc < ld) {
                    *reinterpret_cast<double2 *>(out + (size_t)row * ld + cc) = make_double2(acc0, acc1);
                    if (fld == a.dfield && a.out_dy) {  // row a1: i ky phi of the same column
                        const int jr = (cc >> 1) / a.kxp;
                        const double ky = a.kyf * (double)(jr < a.jpos ? jr : jr - a.nky);
                        a.out_dy[(size_t)row * a.ncols + (cc >> 1)] = make_double2(-ky * acc1, ky * acc0);
                    }
                }
            }
        }
    }
}

}  // namespace psdns
