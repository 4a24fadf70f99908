// FP64 complex FFT of 8 lines side by side with the FIRST pass fed straight from a load functor
// (global memory -> registers -> butterfly) and, optionally, the LAST pass drained straight into a
// store functor (butterfly -> registers -> global memory).  Only the exchanges BETWEEN passes go
// through the shared-memory tile, so a 3-pass FFT costs 2 tile round trips instead of 4:
// shared-memory bandwidth (128 B/clk/SM) is the co-limit of every transform pass next to HBM
// (profiles/r1b: l1tex 60-68 % busy at 38 % DRAM with the load -> tile -> FFT -> tile -> store form).
//
// Decimation in frequency, plan L = R1 * R2 * R3 (PlanF), natural-order input rows:
//   pass 1: rows j + (L/R1) m                     -> tile rows j + (L/R1) q, twiddled
//   pass 2: in place on the tile
//   pass 3: tile rows (q1 R2 + q2) R3 + q         -> element k = q1 + R1 q2 + R1 R2 q
// Tile layout s[row * 8 + line]; a quarter-warp always touches one whole 128-byte row (conflict free).
// Implements the batched FFTs of PAPER.md section 3.2.1 (L164-178).
#pragma once
#include "fft_tile.cuh"

namespace psdns {

template <int L> struct PlanF;
template <> struct PlanF<8>    { static constexpr int R1 = 8,  R2 = 1,  R3 = 1; };
template <> struct PlanF<16>   { static constexpr int R1 = 16, R2 = 1,  R3 = 1; };
template <> struct PlanF<32>   { static constexpr int R1 = 8,  R2 = 4,  R3 = 1; };
template <> struct PlanF<64>   { static constexpr int R1 = 8,  R2 = 8,  R3 = 1; };
template <> struct PlanF<128>  { static constexpr int R1 = 16, R2 = 8,  R3 = 1; };
template <> struct PlanF<256>  { static constexpr int R1 = 16, R2 = 16, R3 = 1; };
template <> struct PlanF<512>  { static constexpr int R1 = 16, R2 = 8,  R3 = 4; };
template <> struct PlanF<1024> { static constexpr int R1 = 16, R2 = 8,  R3 = 8; };

// Plan of the backward z pass: radix 8 throughout at L = 512 (512 threads of 64 registers instead of 256 of 128:
// measured on B200 2.74 -> 2.57 ms; the forward z pass and both y passes are faster with the radix-16 head).
template <int L> struct PlanZB : PlanF<L> {};
template <> struct PlanZB<512> { static constexpr int R1 = 8, R2 = 8, R3 = 8; };

template <int L> __host__ __device__ constexpr int planf_npass() {
    return PlanF<L>::R2 > 1 ? (PlanF<L>::R3 > 1 ? 3 : 2) : 1;
}

// threads per CTA: one (butterfly, line) item of the first pass per thread, at least two warps
template <int L, class P = PlanF<L>> __host__ __device__ constexpr int fused_threads() {
    return (8 * L / P::R1) > 64 ? (8 * L / P::R1) : 64;
}

// tile row that holds element k after all passes ran in place
template <int L, class P = PlanF<L>>
__device__ __forceinline__ int fft_pos_f(int k) {
    constexpr int R1 = P::R1, R2 = P::R2, R3 = P::R3;
    int q1 = k % R1;
    int r = k / R1;
    int pos = q1 * (L / R1);
    if (R2 > 1) {
        int q2 = r % R2;
        r /= R2;
        pos += q2 * (L / (R1 * R2));
        if (R3 > 1) pos += r;
    }
    return pos;
}

// Pass 1: Load = cplx operator()(int row) for the natural input row of this thread's line (tid & 7).
// Writes the tile.  The twiddle table tw[k] = exp(-2 pi i k / L) must be visible to the CTA.
template <int L, int SIGN, int NT, class Load, class P = PlanF<L>>
__device__ __forceinline__ void fft_head(cplx *__restrict__ s, const cplx *__restrict__ tw, int tid, Load load) {
    constexpr int R1 = P::R1;
    constexpr int STRIDE = L / R1, NBF = L / R1;
    const int line = tid & (TILE_LINES - 1);
    for (int j = tid >> 3; j < NBF; j += NT / TILE_LINES) {
        cplx v[R1];
#pragma unroll
        for (int m = 0; m < R1; ++m) v[m] = load(j + m * STRIDE);
        RegFFT<R1, SIGN>::run(v);
#pragma unroll
        for (int q = 0; q < R1; ++q) {
            cplx o = v[q];
            if (STRIDE > 1 && q > 0) o = cmultw<SIGN>(o, tw[j * q]);
            s[(j + q * STRIDE) * TILE_LINES + line] = o;
        }
    }
}

// Remaining passes in place; afterwards element k sits at row fft_pos_f<L>(k).  Starts with a barrier;
// the caller adds one before reading the results.
template <int L, int SIGN, int NT>
__device__ __forceinline__ void fft_rest_inplace(cplx *__restrict__ s, const cplx *__restrict__ tw, int tid) {
    constexpr int R1 = PlanF<L>::R1, R2 = PlanF<L>::R2, R3 = PlanF<L>::R3;
    if constexpr (R2 > 1) {
        __syncthreads();
        fft_pass<L, L / R1, R2, SIGN, NT>(s, tw, tid);
    }
    if constexpr (R3 > 1) {
        __syncthreads();
        fft_pass<L, L / (R1 * R2), R3, SIGN, NT>(s, tw, tid);
    }
}

// Same without the leading barrier (the caller has already synchronised after the head pass).
template <int L, int SIGN, int NT, class P = PlanF<L>>
__device__ __forceinline__ void fft_rest_inplace_nb(cplx *__restrict__ s, const cplx *__restrict__ tw, int tid) {
    constexpr int R1 = P::R1, R2 = P::R2, R3 = P::R3;
    if constexpr (R2 > 1) fft_pass<L, L / R1, R2, SIGN, NT>(s, tw, tid);
    if constexpr (R3 > 1) {
        __syncthreads();
        fft_pass<L, L / (R1 * R2), R3, SIGN, NT>(s, tw, tid);
    }
}

// Remaining passes with the last one drained into Store = void operator()(int k, cplx v), k natural.
template <int L, int SIGN, int NT, class Store>
__device__ __forceinline__ void fft_rest_store(cplx *__restrict__ s, const cplx *__restrict__ tw, int tid, Store store) {
    constexpr int R1 = PlanF<L>::R1, R2 = PlanF<L>::R2, R3 = PlanF<L>::R3;
    constexpr int NPASS = planf_npass<L>();
    const int line = tid & (TILE_LINES - 1);
    if constexpr (NPASS == 3) {
        __syncthreads();
        fft_pass<L, L / R1, R2, SIGN, NT>(s, tw, tid);
    }
    __syncthreads();
    if constexpr (NPASS == 1) {
        for (int k = tid >> 3; k < L; k += NT / TILE_LINES) store(k, s[k * TILE_LINES + line]);
    } else {
        constexpr int RL = (NPASS == 3 ? R3 : R2);       // radix of the last pass, stride 1
        constexpr int NBF = L / RL;
        constexpr int KS = (NPASS == 3 ? R1 * R2 : R1);
        for (int b = tid >> 3; b < NBF; b += NT / TILE_LINES) {
            cplx v[RL];
#pragma unroll
            for (int m = 0; m < RL; ++m) v[m] = s[(b * RL + m) * TILE_LINES + line];
            RegFFT<RL, SIGN>::run(v);
            const int k0 = (NPASS == 3) ? (b / R2 + R1 * (b % R2)) : b;
#pragma unroll
            for (int q = 0; q < RL; ++q) store(k0 + KS * q, v[q]);
        }
    }
}

}  // namespace psdns
