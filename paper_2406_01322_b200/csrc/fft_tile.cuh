// FP64 complex FFT of TILE_LINES (= 8) lines side by side in shared memory, sm_100a.
//
// Data layout: s[row * 8 + line], double2 (re, im); a "row" is one FFT element index shared
// by the 8 lines = 128 contiguous bytes.  Every global<->shared copy of a row is one aligned
// 128-byte segment, and every shared access by a quarter-warp (8 lanes x 16 B) covers exactly
// one row, so the layout is bank-conflict free for ANY row permutation / butterfly stride.
//
// Algorithm: in-place decimation-in-frequency with a mixed-radix plan (radix 16 / 8 / 4
// butterflies held in registers, one shared-memory read+write per pass).  Input rows are in
// natural order; output element k ends up at row fft_pos<L>(k) (mixed-radix digit reversal),
// which the caller folds into its store addressing - rows are independent 128-byte segments so
// the permutation is free.  Twiddles come from a table w[k] = exp(-2 pi i k / L) staged in
// shared memory (computed on the host in long double, so 0.5 ulp accurate).
//
// This implements the batched FFTs of PAPER.md section 3.2.1 (L164-178; there: cuFFT D2Z/Z2D,
// Z2Z and the DCT-I as the FFT of a 2N even extension).
#pragma once
#include <cuda_runtime.h>

namespace psdns {

typedef double2 cplx;
constexpr int TILE_LINES = 8;

__device__ __forceinline__ cplx cadd(cplx a, cplx b) { return make_double2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ cplx csub(cplx a, cplx b) { return make_double2(a.x - b.x, a.y - b.y); }
__device__ __forceinline__ cplx cscale(cplx a, double s) { return make_double2(a.x * s, a.y * s); }
__device__ __forceinline__ cplx cconj(cplx a) { return make_double2(a.x, -a.y); }
// a * (c + i s)
__device__ __forceinline__ cplx cmulcs(cplx a, double c, double s) {
    return make_double2(a.x * c - a.y * s, a.x * s + a.y * c);
}
// a * w (SIGN = -1) or a * conj(w) (SIGN = +1), w = exp(-2 pi i k / L) from the table
template <int SIGN>
__device__ __forceinline__ cplx cmultw(cplx a, cplx w) {
    if (SIGN < 0) return make_double2(a.x * w.x - a.y * w.y, a.x * w.y + a.y * w.x);
    return make_double2(a.x * w.x + a.y * w.y, a.y * w.x - a.x * w.y);
}
// a * (SIGN * i)
template <int SIGN>
__device__ __forceinline__ cplx cmuli(cplx a) {
    return SIGN > 0 ? make_double2(-a.y, a.x) : make_double2(a.y, -a.x);
}

// ---- register butterflies: natural order in, natural order out -------------------------
// X_k = sum_n x_n exp(SIGN * 2 pi i n k / R)

template <int SIGN>
__device__ __forceinline__ void fft2(cplx &a, cplx &b) {
    cplx t = csub(a, b);
    a = cadd(a, b);
    b = t;
}

template <int SIGN>
__device__ __forceinline__ void fft4(cplx &x0, cplx &x1, cplx &x2, cplx &x3) {
    cplx s02 = cadd(x0, x2), d02 = csub(x0, x2);
    cplx s13 = cadd(x1, x3), d13 = cmuli<SIGN>(csub(x1, x3));
    x0 = cadd(s02, s13);
    x2 = csub(s02, s13);
    x1 = cadd(d02, d13);
    x3 = csub(d02, d13);
}

template <int SIGN>
__device__ __forceinline__ void fft8(cplx (&v)[8]) {
    constexpr double h = 0.70710678118654752440;
    cplx t0 = cadd(v[0], v[4]), t1 = cadd(v[1], v[5]), t2 = cadd(v[2], v[6]), t3 = cadd(v[3], v[7]);
    cplx u0 = csub(v[0], v[4]);
    cplx u1 = cmulcs(csub(v[1], v[5]), h, SIGN * h);
    cplx u2 = cmuli<SIGN>(csub(v[2], v[6]));
    cplx u3 = cmulcs(csub(v[3], v[7]), -h, SIGN * h);
    fft4<SIGN>(t0, t1, t2, t3);
    fft4<SIGN>(u0, u1, u2, u3);
    v[0] = t0; v[2] = t1; v[4] = t2; v[6] = t3;
    v[1] = u0; v[3] = u1; v[5] = u2; v[7] = u3;
}

template <int SIGN>
__device__ __forceinline__ void fft16(cplx (&v)[16]) {
    constexpr double c1 = 0.92387953251128673848;  // cos(pi/8)
    constexpr double c2 = 0.70710678118654752440;  // cos(pi/4)
    constexpr double c3 = 0.38268343236508977173;  // cos(3pi/8)
    cplx t[8], u[8];
#pragma unroll
    for (int m = 0; m < 8; ++m) {
        t[m] = cadd(v[m], v[m + 8]);
        u[m] = csub(v[m], v[m + 8]);
    }
    u[1] = cmulcs(u[1], c1, SIGN * c3);
    u[2] = cmulcs(u[2], c2, SIGN * c2);
    u[3] = cmulcs(u[3], c3, SIGN * c1);
    u[4] = cmuli<SIGN>(u[4]);
    u[5] = cmulcs(u[5], -c3, SIGN * c1);
    u[6] = cmulcs(u[6], -c2, SIGN * c2);
    u[7] = cmulcs(u[7], -c1, SIGN * c3);
    fft8<SIGN>(t);
    fft8<SIGN>(u);
#pragma unroll
    for (int m = 0; m < 8; ++m) {
        v[2 * m] = t[m];
        v[2 * m + 1] = u[m];
    }
}

template <int R, int SIGN>
struct RegFFT;
template <int SIGN>
struct RegFFT<2, SIGN> {
    static __device__ __forceinline__ void run(cplx (&v)[2]) { fft2<SIGN>(v[0], v[1]); }
};
template <int SIGN>
struct RegFFT<4, SIGN> {
    static __device__ __forceinline__ void run(cplx (&v)[4]) { fft4<SIGN>(v[0], v[1], v[2], v[3]); }
};
template <int SIGN>
struct RegFFT<8, SIGN> {
    static __device__ __forceinline__ void run(cplx (&v)[8]) { fft8<SIGN>(v); }
};
template <int SIGN>
struct RegFFT<16, SIGN> {
    static __device__ __forceinline__ void run(cplx (&v)[16]) { fft16<SIGN>(v); }
};

// ---- mixed-radix plans ----------------------------------------------------------------------
// Plan<L>: R1, R2, R3 (R = 1 means "no pass").
template <int L> struct Plan;
template <> struct Plan<8>    { static constexpr int R1 = 8,  R2 = 1,  R3 = 1; };
template <> struct Plan<16>   { static constexpr int R1 = 16, R2 = 1,  R3 = 1; };
template <> struct Plan<32>   { static constexpr int R1 = 8,  R2 = 4,  R3 = 1; };
template <> struct Plan<64>   { static constexpr int R1 = 8,  R2 = 8,  R3 = 1; };
template <> struct Plan<128>  { static constexpr int R1 = 16, R2 = 8,  R3 = 1; };
template <> struct Plan<256>  { static constexpr int R1 = 16, R2 = 16, R3 = 1; };
template <> struct Plan<512>  { static constexpr int R1 = 8,  R2 = 8,  R3 = 8; };
template <> struct Plan<1024> { static constexpr int R1 = 16, R2 = 8,  R3 = 8; };

// row that holds output element k after fft_tile<L>
template <int L>
__device__ __forceinline__ int fft_pos(int k) {
    constexpr int R1 = Plan<L>::R1, R2 = Plan<L>::R2, R3 = Plan<L>::R3;
    int q1 = k % R1;
    int r = k / R1;
    int pos = q1 * (L / R1);
    if (R2 > 1) {
        int q2 = r % R2;
        r /= R2;
        pos += q2 * (L / (R1 * R2));
        if (R3 > 1) pos += r;  // q3 * (L/(R1 R2 R3)) = q3
    }
    return pos;
}

// shared-memory index of (row, line).  SWZ = false: s[row*8 + line].  SWZ = true: the line index is
// rotated by the row, s[row*8 + ((line + row) & 7)], which keeps the butterfly accesses conflict free
// (a quarter-warp still covers one whole row) AND makes "one thread reads all 8 lines of its own row"
// conflict free when consecutive threads own consecutive rows (used by the fused x kernel's pointwise stage).
template <bool SWZ>
__device__ __forceinline__ int tile_idx(int row, int line) {
    return SWZ ? row * TILE_LINES + ((line + row) & (TILE_LINES - 1)) : row * TILE_LINES + line;
}

// one DIF pass: sub-length LS, radix R, over all L/R butterflies of each of the 8 lines
template <int L, int LS, int R, int SIGN, int NT, bool SWZ = false>
__device__ __forceinline__ void fft_pass(cplx *__restrict__ s, const cplx *__restrict__ tw, int tid) {
    constexpr int STRIDE = LS / R;
    constexpr int NBF = L / R;
    const int line = tid & (TILE_LINES - 1);
    for (int b = tid >> 3; b < NBF; b += NT / TILE_LINES) {
        const int blk = b / STRIDE, j = b % STRIDE;
        const int row0 = blk * LS + j;
        cplx v[R];
#pragma unroll
        for (int m = 0; m < R; ++m) v[m] = s[tile_idx<SWZ>(row0 + m * STRIDE, line)];
        RegFFT<R, SIGN>::run(v);
#pragma unroll
        for (int q = 0; q < R; ++q) {
            cplx o = v[q];
            if (LS > R && q > 0) o = cmultw<SIGN>(o, tw[(L / LS) * j * q]);
            s[tile_idx<SWZ>(row0 + q * STRIDE, line)] = o;
        }
    }
}

// one DIT pass (inverse data flow of fft_pass): twiddle the inputs, then butterfly
template <int L, int LS, int R, int SIGN, int NT, bool SWZ = false>
__device__ __forceinline__ void fft_pass_dit(cplx *__restrict__ s, const cplx *__restrict__ tw, int tid) {
    constexpr int STRIDE = LS / R;
    constexpr int NBF = L / R;
    const int line = tid & (TILE_LINES - 1);
    for (int b = tid >> 3; b < NBF; b += NT / TILE_LINES) {
        const int blk = b / STRIDE, j = b % STRIDE;
        const int row0 = blk * LS + j;
        cplx v[R];
#pragma unroll
        for (int m = 0; m < R; ++m) {
            cplx x = s[tile_idx<SWZ>(row0 + m * STRIDE, line)];
            if (LS > R && m > 0) x = cmultw<SIGN>(x, tw[(L / LS) * j * m]);
            v[m] = x;
        }
        RegFFT<R, SIGN>::run(v);
#pragma unroll
        for (int q = 0; q < R; ++q) s[tile_idx<SWZ>(row0 + q * STRIDE, line)] = v[q];
    }
}

// Full in-place DIF FFT of the 8-line tile: natural-order rows in, element k at row fft_pos<L>(k) out.
// Caller must __syncthreads() before (data + twiddles visible) and after (before reading results).
template <int L, int SIGN, int NT, bool SWZ = false>
__device__ __forceinline__ void fft_tile(cplx *__restrict__ s, const cplx *__restrict__ tw, int tid) {
    constexpr int R1 = Plan<L>::R1, R2 = Plan<L>::R2, R3 = Plan<L>::R3;
    fft_pass<L, L, R1, SIGN, NT, SWZ>(s, tw, tid);
    if constexpr (R2 > 1) {
        __syncthreads();
        fft_pass<L, L / R1, R2, SIGN, NT, SWZ>(s, tw, tid);
    }
    if constexpr (R3 > 1) {
        __syncthreads();
        fft_pass<L, L / (R1 * R2), R3, SIGN, NT, SWZ>(s, tw, tid);
    }
}

// Full in-place DIT FFT: element n at row fft_pos<L>(n) in (exactly the order fft_tile leaves),
// natural-order rows out.  Lets backward-FFT -> pointwise -> forward-FFT run without any reordering.
template <int L, int SIGN, int NT, bool SWZ = false>
__device__ __forceinline__ void fft_tile_dit(cplx *__restrict__ s, const cplx *__restrict__ tw, int tid) {
    constexpr int R1 = Plan<L>::R1, R2 = Plan<L>::R2, R3 = Plan<L>::R3;
    if constexpr (R3 > 1) {
        fft_pass_dit<L, R3, R3, SIGN, NT, SWZ>(s, tw, tid);
        __syncthreads();
        fft_pass_dit<L, R3 * R2, R2, SIGN, NT, SWZ>(s, tw, tid);
        __syncthreads();
    } else if constexpr (R2 > 1) {
        fft_pass_dit<L, R2, R2, SIGN, NT, SWZ>(s, tw, tid);
        __syncthreads();
    }
    fft_pass_dit<L, L, R1, SIGN, NT, SWZ>(s, tw, tid);
}

}  // namespace psdns
