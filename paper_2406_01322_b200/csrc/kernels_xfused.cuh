// Fused x pass (rows a4 + a5 + a6): for one (k, y) line at a time, C2R of the input fields,
// pointwise non-linear terms, R2C of the product fields - physical-space arrays never reach HBM
// ("physical-space arrays never leave the SM"; PAPER.md L166-176 for the transforms,
// L182-196 and Eqs. 1, 4, 7, 8 for the products).
//
// Tile: 8 FIELDS side by side, s[row][field]; the FFT is the half-length real transform (H = L/2):
//   backward: Z_k = (X_k + conj X_{H-k}) + i conj(w_k) (X_k - conj X_{H-k}),  w_k = exp(-2 pi i k / L),
//             z = IFFT_H(Z) gives z_n = x_{2n} + i x_{2n+1}
//   forward : A_k = (Z_k + conj Z_{H-k})/2, B_k = (Z_k - conj Z_{H-k})/(2i), X_k = (A_k + w_k B_k)/L
// with H = R1 * R2 * 2.  Shared-memory traffic is what bounds this kernel (128 B/clk/SM), so every stage
// that can stay in registers does:
//   A  pre-twiddle straight from the TMA-staged spectra + DIF pass R1            -> tile
//   B  DIF pass R2                                                   tile -> tile
//   C  DIF radix 2 + pointwise products + DIT radix 2 (a thread owns two rows x all 8 fields)
//   D  DIT pass R2                                                   tile -> tile
//   E  DIT pass R1, results kept in registers
//   F  post-twiddle against the partner row H-k (a register of another lane: warp shuffle), truncated store
// i.e. 4 tile exchanges per line instead of 9.  The backward FFT is decimation in frequency, the
// products are elementwise, the forward FFT is decimation in time: no reordering anywhere.
#pragma once
#include <type_traits>
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

// An opaque copy of a loop-invariant index: address arithmetic derived from it is redone where it is used
// instead of being hoisted out of the line loop and spilled (profiles/r1d: 30 hoisted shared-memory addresses
// were spilled and re-read from local memory for every line).
__device__ __forceinline__ int opaque(int v) { asm volatile("" : "+r"(v)); return v; }
// global store that the compiler may move shared-memory loads across (a store through a generic pointer may not)
__device__ __forceinline__ void stg(cplx *p, cplx v) {
    asm volatile("st.global.v2.f64 [%0], {%1, %2};" ::"l"(__cvta_generic_to_global(p)), "d"(v.x), "d"(v.y));
}

// ---- plan of the half-length FFT: H = R1 * R2 * 2 ---------------------------------------------------
template <int H> struct XPlan;
template <> struct XPlan<8>   { static constexpr int R1 = 4,  R2 = 1; };
template <> struct XPlan<16>  { static constexpr int R1 = 8,  R2 = 1; };
template <> struct XPlan<32>  { static constexpr int R1 = 16, R2 = 1; };
template <> struct XPlan<64>  { static constexpr int R1 = 8,  R2 = 4; };
template <> struct XPlan<128> { static constexpr int R1 = 8,  R2 = 8; };
template <> struct XPlan<256> { static constexpr int R1 = 16, R2 = 8; };
template <> struct XPlan<512> { static constexpr int R1 = 16, R2 = 16; };

// compile-time twiddle w_LS^q = exp(-2 pi i q / LS) for LS in {4, 8, 16, 32}, 0 <= q < LS/2
__device__ __forceinline__ constexpr double cos32(int i) {   // cos(2 pi i / 32), 0 <= i <= 16
    constexpr double C[9] = {1.0, 0.98078528040323044913, 0.92387953251128675613, 0.83146961230254523708,
                             0.70710678118654752440, 0.55557023301960222474, 0.38268343236508977173,
                             0.19509032201612826785, 0.0};
    return i <= 8 ? C[i] : -C[16 - i];
}
template <int LS>
__device__ __forceinline__ constexpr double wc_re(int q) { return cos32(q * (32 / LS)); }
template <int LS>
__device__ __forceinline__ constexpr double wc_im(int q) {   // -sin(2 pi q / LS)
    return q * (32 / LS) <= 8 ? -cos32(8 - q * (32 / LS)) : -cos32(q * (32 / LS) - 8);
}

// Powers w^1 .. w^{R-1} of a per-thread base twiddle from the loop-invariant set {w, w^2, w^4, w^8}:
// the R1-pass twiddles w_H^{j q} depend on the thread (j) only, so they live in registers instead of
// being re-read from shared memory for every line.
__device__ __forceinline__ cplx cmul(cplx a, cplx b) { return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
template <int R>
struct TwPow {
    cplx w1, w2, w4, w8;
    __device__ __forceinline__ void init(cplx w) {
        w1 = w; w2 = cmul(w, w); w4 = cmul(w2, w2); w8 = cmul(w4, w4);
    }
    // visits fn(q, w^q) for q = 1 .. R-1 in an order that needs at most two temporaries besides {w, w^2, w^4, w^8}
    // (an array of all R-1 powers next to the R butterfly values does not fit in 128 registers)
    template <class Fn>
    __device__ __forceinline__ void each(Fn fn) const {
        fn(1, w1);
        if (R > 2) { fn(2, w2); fn(3, cmul(w2, w1)); }
        if (R > 4) {
            fn(4, w4); fn(5, cmul(w4, w1));
            const cplx w6 = cmul(w4, w2);
            fn(6, w6); fn(7, cmul(w6, w1));
        }
        if (R > 8) {
            fn(8, w8); fn(9, cmul(w8, w1));
            const cplx w10 = cmul(w8, w2);
            fn(10, w10); fn(11, cmul(w10, w1));
            const cplx w12 = cmul(w8, w4);
            fn(12, w12); fn(13, cmul(w12, w1));
            const cplx w14 = cmul(w12, w2);
            fn(14, w14); fn(15, cmul(w14, w1));
        }
    }
};

// ---- pointwise products at one grid point (row a5; Eqs. 1, 4, 7, 8) --------------------------
//   in : u v w [phi phx phy phz]      out: Txx-Tzz Txy Txz Tyy-Tzz Tyz [Q C]
//   T_ij = -u_i u_j + cs (|grad phi|^2 delta_ij - phi_i phi_j),  Q = u . grad phi,  C = phi^3.
//   Only the deviatoric combinations enter Eqs. 14-15 (see enqueue_step), so T_zz is subtracted here.
template <int Q, bool PHASE>
__device__ __forceinline__ double nl_out(const double (&in)[8], double cs) {
    const double u = in[0], v = in[1], w = in[2];
    const double px = in[4], py = in[5], pz = in[6];
    if (Q == 0) { double r = w * w - u * u; if (PHASE) r += cs * (pz * pz - px * px); return r; }
    if (Q == 1) { double r = -u * v; if (PHASE) r -= cs * px * py; return r; }
    if (Q == 2) { double r = -u * w; if (PHASE) r -= cs * px * pz; return r; }
    if (Q == 3) { double r = w * w - v * v; if (PHASE) r += cs * (pz * pz - py * py); return r; }
    if (Q == 4) { double r = -v * w; if (PHASE) r -= cs * py * pz; return r; }
    if (Q == 5) return u * px + v * py + w * pz;
    return in[3] * in[3] * in[3];
}

// the four products of output field q at the four points of a row pair (q is a compile-time constant after unrolling)
template <bool PHASE>
__device__ __forceinline__ void nl_quad(int q, const double (&p00)[8], const double (&p01)[8], const double (&p10)[8],
                                        const double (&p11)[8], double cs, double &o00, double &o01, double &o10, double &o11) {
#define NLQ(Q) case Q: o00 = nl_out<Q, PHASE>(p00, cs); o01 = nl_out<Q, PHASE>(p01, cs); o10 = nl_out<Q, PHASE>(p10, cs); o11 = nl_out<Q, PHASE>(p11, cs); break;
    switch (q) { NLQ(0) NLQ(1) NLQ(2) NLQ(3) NLQ(4) NLQ(5) default: NLQ(6) }
#undef NLQ
}

struct XFArgs {
    const cplx *in[6];      // Y arrays: u v w [phi phy phz]
    cplx *out[8];           // Y arrays: Txx-Tzz Txy Txz Tyy-Tzz Tyz [Q C]
    int kxp, nkx, nlines;
    double cs;
    double kxf;             // 2 pi / Lx: the phx row is i kx times the staged phi row (row a1)
};

// stage pitch (cplx): odd, so that the 8 fields of one k sit in 8 different 16-byte bank groups
__host__ __device__ inline int xf_spitch(int nkx) { return nkx | 1; }

// shared memory: tile [LPI H][8] | stage [LPI][NST][spitch] | mbarriers.  The stage receives the NEXT iteration's
// spectra rows by TMA bulk copies while the current lines are transformed; with the phase field its last row is
// derived in place: i kx phi^ (row a1).
// Register budget (128 at 2 CTAs/SM): only the thread's base twiddle w_L^j is carried across the line loop;
// its powers are re-derived per stage (profiles/r1c: an earlier form spilled 456 B/thread, 8 GB of extra DRAM
// writes per step and 15 % of the time in local-memory waits).
#ifndef XF_MINB
#define XF_MINB 2
#endif
template <bool PHASE> __host__ __device__ constexpr int xf_nstage() { return PHASE ? 7 : 3; }

// ====================================================================================================
// Warp-per-field organisation of the stages above (k_xfusedw: nx = 1024, where a pass has 32 butterflies per field =
// one per lane; k_xfusedwm further down: smaller nx, several lines per iteration fill the warp).
//
// Every stage except the pointwise one is independent per field, so a WARP owns one field: its 32 lanes are
// the (up to) 32 butterflies of a pass.  Consequences (profiles/r1e: an earlier field-interleaved form (thread = (butterfly, field)) ran its
// FP64 pipe 48 % and its shared-memory pipe 73 % busy, in lockstep between eight CTA-wide barriers per line):
//   * stages A -> B and D -> E -> F need only __syncwarp: three CTA-wide barriers per line (stage ready,
//     before and after the pointwise stage), so the field warps drift apart and FP64 work of one overlaps
//     the shared-memory traffic of another;
//   * 7 fields = 7 working warps: the eighth field slot costs no work any more (it was 1/8 of all lanes); the
//     eighth warp is a service warp (derives the i kx phi row, issues the TMA copies of the next line);
//   * the j = 1 twiddles of the inner radix-R2 passes move into the pointwise stage (a thread there owns
//     rows 2t, 2t+1 of all fields and needs ONE loop-invariant twiddle), so the inner passes have none and
//     no lane diverges.
// Tile index: the field slot is XOR-swizzled with row bits chosen so that a quarter-warp is conflict free in
// every stage: 8 consecutive rows of one field (A, E: bits 0-2), 4 blocks x 2 classes of the inner pass
// (B, D: bit 0 and the two bits above log2(2 R2)), 8 consecutive row pairs (pointwise: bits 1-3).
// ====================================================================================================
template <int LOG2LS>
__device__ __forceinline__ int widx(int row, int f) {
    const int sw = (row & 7) ^ ((row >> 3) & 1) ^ (((row >> LOG2LS) & 3) << 1);
    return row * TILE_LINES + ((f ^ sw) & (TILE_LINES - 1));
}
__host__ __device__ constexpr int ilog2(int x) { return x <= 1 ? 0 : 1 + ilog2(x / 2); }

__device__ __forceinline__ void mbar_arrive(unsigned long long *bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}

constexpr int XFW_THREADS = 256;   // 8 warps: one per field slot
// lines per CTA iteration: a warp's 32 lanes = LPI lines x S1 butterflies of its field (1 at nx = 1024, 2 at nx = 512 ..)
template <int L> __host__ __device__ constexpr int xfw_lpi() {
    return ((L / 2) / XPlan<L / 2>::R1) >= 32 ? 1 : 32 / ((L / 2) / XPlan<L / 2>::R1);
}

// compile-time loop: f(std::integral_constant<int, I>) for I = 0 .. N-1 (the body can use `if constexpr` on I)
template <int I, int N, class F>
__device__ __forceinline__ void static_for(F &&f) {
    if constexpr (I < N) {
        f(std::integral_constant<int, I>{});
        static_for<I + 1, N>(f);
    }
}
// global store with a compile-time byte offset folded into the instruction
template <int OFF>
__device__ __forceinline__ void stg_off(cplx *p, cplx v) {
    asm volatile("st.global.v2.f64 [%0+%3], {%1, %2};" ::"l"(__cvta_generic_to_global(p)), "d"(v.x), "d"(v.y), "n"(OFF));
}

// nx = 1024 (S1 = 32: one butterfly per lane).  The retained k_x of the step are functions of L alone (reading S3), so the
// cut-offs are compile-time constants here: which rows of stage A have a partner, which rows of stage F are stored, every
// stage address.  Measured against the run-time form of the same kernel (profiles/r2c_experiments.md): 4.76e9 -> 4.0e9
// warp instructions per launch (no predicated zero loads, no per-row branches, 40 DADD less per line), 8.2-8.4 -> 7.4-7.6 ms.
template <int L, bool PHASE>
__global__ void __launch_bounds__(XFW_THREADS, XF_MINB) k_xfusedw(const __grid_constant__ XFArgs a, const cplx *__restrict__ twx) {
    constexpr int H = L / 2;
    constexpr int R1 = XPlan<H>::R1, R2 = XPlan<H>::R2;
    constexpr int NT = XFW_THREADS;
    constexpr int S1 = H / R1;              // butterflies per field of pass R1
    constexpr int LS = 2 * R2;              // sub-length of the inner pass
    constexpr int NB2 = H / R2;             // butterflies per field of the inner pass
    constexpr int LG = ilog2(LS) < 3 ? 3 : ilog2(LS);
    constexpr int NIN = PHASE ? 7 : 3, NOUT = PHASE ? 7 : 5;
    constexpr int NTMA = PHASE ? 6 : 3;
    constexpr int NST = xf_nstage<PHASE>();
    // the step's retained k_x (reading S3) are functions of L alone: compile-time cut-offs (the host checks a.nkx == NKX)
    constexpr int NKX = L / 3 + 1, KXP = (NKX + 7) & ~7;
    constexpr int SP = NKX | 1;
    static_assert(R1 * R2 * 2 == H && S1 == 32 && NB2 == 32, "plan");
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cplx *s = reinterpret_cast<cplx *>(smem_raw);
    cplx *stage = s + H * TILE_LINES;
    unsigned long long *bar = reinterpret_cast<unsigned long long *>(stage + (size_t)NST * SP);
    unsigned long long *bar_free = bar + 1;         // stage consumed by every input-field warp
    const int tid = threadIdx.x, f = tid >> 5, lane = tid & 31;
    const bool service = (f == TILE_LINES - 1);
    cplx *outf = a.out[f < NOUT ? f : 0];
    const double sc = 0.5 / L;
    constexpr unsigned row_bytes = (unsigned)(NKX * sizeof(cplx));
    auto issue = [&](int line) {
        mbar_expect_tx(bar, row_bytes * NTMA);
#pragma unroll
        for (int q = 0; q < NTMA; ++q) bulk_g2s(stage + (size_t)q * SP, a.in[q] + (size_t)line * KXP, row_bytes, bar);
    };
    unsigned long long *bar_drv = bar + 2;          // i kx phi^ row of the staged line derived (service warp -> phx warp)
    if (tid == 0) {
        mbar_init(bar, 1);
        mbar_init(bar_free, NIN);
        mbar_init(bar_drv, 1);
        if ((int)blockIdx.x < a.nlines) issue(blockIdx.x);
    }
    __syncthreads();
    // row a1: phx^ = i kx phi^, formed in the stage by the service warp as soon as the line's rows have landed - for the
    // first line here, for every later line while the field warps run stages D-F of the line before
    auto derive = [&](unsigned par) {
        mbar_wait(bar, par);
        for (int k = lane; k < NKX; k += 32) {
            const cplx p = stage[3 * SP + k];
            const double kk = a.kxf * (double)k;
            stage[6 * SP + k] = make_double2(-kk * p.y, kk * p.x);
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(bar_drv);
    };
    if constexpr (PHASE) {
        if (service && (int)blockIdx.x < a.nlines) derive(0);
    }
    const int j = lane;                             // butterfly of passes A, E, F
    cplx wj = twx[j];                               // w_L^j
    // pointwise-stage twiddle of this thread's row pair: w_LS^(t mod R2) = w_L^((t mod R2) L / LS)
    cplx wc = twx[(tid % R2) * (L / LS)];
    unsigned parity = 0;
    // field -> staged row: u v w phi phx phy phz  <-  0 1 2 3 6 4 5
    const int srow = !PHASE ? (f < NST ? f : 0) : (f < 4 ? f : (f == 4 ? 6 : (f < NIN ? f - 1 : 0)));
    const cplx *sf = stage + (size_t)srow * SP;
    for (int line = blockIdx.x; line < a.nlines; line += gridDim.x) {
        const size_t base = (size_t)line * KXP;
        if (f < NIN) mbar_wait(bar, parity);
        if constexpr (PHASE) {
            if (srow == 6) mbar_wait(bar_drv, parity);
        }
        asm volatile("" : "+d"(wj.x), "+d"(wj.y), "+d"(wc.x), "+d"(wc.y));
        if (f < NIN) {
            // ---- A: pre-twiddle from the staged rows + DIF pass R1 (inverse transform, sign +) ----
            {
                const int jj = opaque(j) & (S1 - 1);
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
                        cplx xa = sf[k];
                        if (m == 0 && k == 0) xa.y = 0.0;           // reading S20
                        v[m] = make_double2(fma(w.y, xa.x, fma(-w.x, xa.y, xa.x)), fma(w.y, xa.y, fma(w.x, xa.x, xa.y)));
                    } else if constexpr (a_none) {
                        static_assert(b_all, "cut-offs");
                        const cplx xb = sf[kb];
                        // S = conj(xb), D = -conj(xb)
                        v[m] = make_double2(fma(-w.y, xb.x, fma(-w.x, xb.y, xb.x)), fma(w.y, xb.y, fma(-w.x, xb.x, -xb.y)));
                    } else {
                        cplx xa = make_double2(0.0, 0.0), xb = xa;
                        if (a_all || k < NKX) xa = sf[k];
                        if (b_all || kb < NKX) xb = sf[kb];
                        const double Sx = xa.x + xb.x, Sy = xa.y - xb.y, Dx = xa.x - xb.x, Dy = xa.y + xb.y;
                        v[m] = make_double2(fma(w.y, Dx, fma(-w.x, Dy, Sx)), fma(w.y, Dy, fma(w.x, Dx, Sy)));
                    }
                });
                RegFFT<R1, +1>::run(v);
                TwPow<R1> tp;
                tp.init(cmul(wj, wj));
                s[widx<LG>(jj, f)] = v[0];
                tp.each([&](int q, cplx wq) { s[widx<LG>(jj + S1 * q, f)] = cmultw<+1>(v[q], wq); });
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(bar_free);   // this field's staged row is consumed
            // ---- B: DIF pass R2, no twiddles (they are applied in the pointwise stage) ----
            {
                const int b = opaque(lane) & 31, row0 = (b >> 1) * LS + (b & 1);
                cplx v[R2];
#pragma unroll
                for (int m = 0; m < R2; ++m) v[m] = s[widx<LG>(row0 + 2 * m, f)];
                RegFFT<R2, +1>::run(v);
#pragma unroll
                for (int q = 0; q < R2; ++q) s[widx<LG>(row0 + 2 * q, f)] = v[q];
            }
        } else if (service) {
            if (lane == 0) {                        // all input warps are done with the stage: prefetch the next line
                mbar_wait(bar_free, parity);
                if (line + (int)gridDim.x < a.nlines) {
                    fence_proxy_async();
                    issue(line + gridDim.x);
                }
            }
        }
        parity ^= 1;
        __syncthreads();
        // ---- C: last DIF radix 2 (with the inner pass's twiddle), pointwise products, first DIT radix 2 ----
        {
            const int t = opaque(tid) & (NT - 1);
            static_assert(H / 2 == NT, "one row pair per thread");
            double p00[8], p01[8], p10[8], p11[8];
#pragma unroll
            for (int q = 0; q < NIN; ++q) {
                const cplx p = s[widx<LG>(2 * t, q)];
                cplx m = s[widx<LG>(2 * t + 1, q)];
                m = cmultw<+1>(m, wc);
                p00[q] = p.x + m.x; p01[q] = p.y + m.y;
                p10[q] = p.x - m.x; p11[q] = p.y - m.y;
            }
#pragma unroll
            for (int q = 0; q < NOUT; ++q) {
                double o00, o01, o10, o11;
                nl_quad<PHASE>(q, p00, p01, p10, p11, a.cs, o00, o01, o10, o11);
                s[widx<LG>(2 * t, q)] = make_double2(o00 + o10, o01 + o11);
                cplx m = make_double2(o00 - o10, o01 - o11);
                m = cmultw<-1>(m, wc);
                s[widx<LG>(2 * t + 1, q)] = m;
            }
        }
        __syncthreads();
        if constexpr (PHASE) {
            if (service && line + (int)gridDim.x < a.nlines) derive(parity);     // parity is already the next line's
        }
        if (f < NOUT) {
            // ---- D: DIT pass R2 (forward transform, sign -), no twiddles ----
            {
                const int b = opaque(lane) & 31, row0 = (b >> 1) * LS + (b & 1);
                cplx v[R2];
#pragma unroll
                for (int m = 0; m < R2; ++m) v[m] = s[widx<LG>(row0 + 2 * m, f)];
                RegFFT<R2, -1>::run(v);
#pragma unroll
                for (int q = 0; q < R2; ++q) s[widx<LG>(row0 + 2 * q, f)] = v[q];
            }
            __syncwarp();
            // ---- E: DIT pass R1; the results stay in registers ----
            cplx v[R1];
            {
                const int jj = opaque(j) & (S1 - 1);
                TwPow<R1> tp;
                tp.init(cmul(wj, wj));
                v[0] = s[widx<LG>(jj, f)];
                tp.each([&](int m, cplx wq) { v[m] = cmultw<-1>(s[widx<LG>(jj + S1 * m, f)], wq); });
                RegFFT<R1, -1>::run(v);
            }
            // ---- F: post-twiddle of row k = j + S1 q against its partner row H - k, truncated store.  The partner
            // is output R1 - 1 - q of butterfly S1 - j (output R1 - q of butterfly 0 for j = 0): a register of another
            // lane of THIS warp, fetched by shuffle - no shared-memory exchange and no barrier.
            {
                const int src = (S1 - j) & (S1 - 1);
                cplx *o = outf + base + j;
                static_for<0, R1>([&](auto Q) {
                    constexpr int q = decltype(Q)::value;
                    if constexpr (S1 * q < KXP) {
                        constexpr bool all = (S1 * q + S1 - 1 < NKX);
                        const cplx mine = (j == 0) ? v[(R1 - q) & (R1 - 1)] : v[R1 - 1 - q];
                        cplx zp;
                        zp.x = __shfl_sync(0xffffffffu, mine.x, src);
                        zp.y = __shfl_sync(0xffffffffu, mine.y, src);
                        const int k = j + S1 * q;
                        const cplx za = v[q];
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
            __syncwarp();     // this warp's F reads are done before its next stage A overwrites the field
        }
    }
}

// Multi-line generalisation for nx < 1024, where a pass has fewer than 32 butterflies per field: the 32 lanes of a
// field warp are LPI lines x S1 butterflies (LPI = 2 at nx = 512 and 256, 4 at 128, ..), the tile holds LPI lines.
// Kept as a second kernel: folded to LPI = 1 it is the kernel above instruction for instruction, yet measured 3 %
// slower at nx = 1024 (8.4 vs 8.16 ms), so nx = 1024 keeps the single-line form.
template <int L, bool PHASE>
__global__ void __launch_bounds__(XFW_THREADS, (L >= 1024 ? XF_MINB : (L >= 128 ? 2 : 3))) k_xfusedwm(const __grid_constant__ XFArgs a,
                                                                             const cplx *__restrict__ twx) {
    constexpr int H = L / 2;
    constexpr int R1 = XPlan<H>::R1, R2 = XPlan<H>::R2;
    constexpr int NT = XFW_THREADS;
    constexpr int S1 = H / R1;              // butterflies per field of pass R1 (<= 32)
    constexpr int LS = 2 * R2;              // sub-length of the inner pass
    constexpr int NB2 = H / R2;             // butterflies per field of the inner pass (<= 32)
    constexpr int LG = ilog2(LS) < 3 ? 3 : ilog2(LS);
    constexpr int NIN = PHASE ? 7 : 3, NOUT = PHASE ? 7 : 5;
    constexpr int NTMA = PHASE ? 6 : 3;
    constexpr int NST = xf_nstage<PHASE>();
    constexpr int LPI = xfw_lpi<L>();       // lines per iteration
    // compile-time cut-offs, as in k_xfusedw (the host checks a.nkx == NKX)
    constexpr int NKX = L / 3 + 1, KXP = (NKX + 7) & ~7;
    constexpr int SP = NKX | 1;
    static_assert(R1 * R2 * 2 == H && S1 * LPI == 32, "plan");
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cplx *s = reinterpret_cast<cplx *>(smem_raw);
    cplx *stage = s + LPI * H * TILE_LINES;         // [LPI][NST][spitch]
    constexpr int spitch = SP;
    unsigned long long *bar = reinterpret_cast<unsigned long long *>(stage + (size_t)LPI * NST * spitch);
    unsigned long long *bar_free = bar + 1;         // stage consumed by every input-field warp
    unsigned long long *bar_drv = bar + 2;          // i kx phi^ rows of the staged lines derived (service warp -> phx warp)
    const int tid = threadIdx.x, f = tid >> 5, lane = tid & 31;
    const bool service = (f == TILE_LINES - 1);     // eighth warp
    cplx *outf = a.out[f < NOUT ? f : 0];
    const double sc = 0.5 / L;
    constexpr unsigned row_bytes = (unsigned)(NKX * sizeof(cplx));
    const int ngroups = a.nlines / LPI;             // nlines = nz * ny is a multiple of LPI (ny >= 16, power of two)
    auto issue = [&](int grp) {
        mbar_expect_tx(bar, row_bytes * NTMA * LPI);
#pragma unroll
        for (int l = 0; l < LPI; ++l)
#pragma unroll
            for (int q = 0; q < NTMA; ++q)
                bulk_g2s(stage + (size_t)(l * NST + q) * spitch, a.in[q] + (size_t)(grp * LPI + l) * KXP, row_bytes, bar);
    };
    if (tid == 0) {
        mbar_init(bar, 1);
        mbar_init(bar_free, NIN);
        mbar_init(bar_drv, 1);
        if ((int)blockIdx.x < ngroups) issue(blockIdx.x);
    }
    __syncthreads();
    // row a1: phx^ = i kx phi^, formed in the stage by the service warp as soon as the rows have landed - for the first
    // group here, for every later group while the field warps run stages D-F of the group before
    auto derive = [&](unsigned par) {
        mbar_wait(bar, par);
#pragma unroll
        for (int l = 0; l < LPI; ++l)
            for (int k = lane; k < NKX; k += 32) {
                const cplx p = stage[(l * NST + 3) * spitch + k];
                const double kk = a.kxf * (double)k;
                stage[(l * NST + 6) * spitch + k] = make_double2(-kk * p.y, kk * p.x);
            }
        __syncwarp();
        if (lane == 0) mbar_arrive(bar_drv);
    };
    if constexpr (PHASE) {
        if (service && (int)blockIdx.x < ngroups) derive(0);
    }
    const int j = LPI == 1 ? lane : (lane & (S1 - 1)), ln = LPI == 1 ? 0 : lane / S1;   // butterfly of passes A, E, F; its line
    constexpr bool itemA = true;                    // S1 * LPI = 32: every lane owns a butterfly
    const int lrow = ln * H;                        // first tile row of that line
    cplx wj = twx[j];                               // w_L^j
    // pointwise-stage twiddle of this thread's row pair: w_LS^(t mod R2) = w_L^((t mod R2) L / LS)
    cplx wc = twx[(tid % R2) * (L / LS)];
    unsigned parity = 0;
    // field -> staged row: u v w phi phx phy phz  <-  0 1 2 3 6 4 5
    const int srow = !PHASE ? (f < NST ? f : 0) : (f < 4 ? f : (f == 4 ? 6 : (f < NIN ? f - 1 : 0)));
    const cplx *sf = stage + (size_t)(ln * NST + srow) * spitch;
    for (int grp = blockIdx.x; grp < ngroups; grp += gridDim.x) {
        const size_t base = (size_t)(grp * LPI + ln) * KXP;
        if (f < NIN) mbar_wait(bar, parity);
        if constexpr (PHASE) {
            if (srow == 6) mbar_wait(bar_drv, parity);
        }
        asm volatile("" : "+d"(wj.x), "+d"(wj.y), "+d"(wc.x), "+d"(wc.y));
        if (f < NIN) {
            // ---- A: pre-twiddle from the staged rows + DIF pass R1 (inverse transform, sign +) ----
            if (itemA) {
                const int jj = opaque(j) & (S1 - 1);
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
                        cplx xa = sf[k];
                        if (m == 0 && k == 0) xa.y = 0.0;           // reading S20
                        v[m] = make_double2(fma(w.y, xa.x, fma(-w.x, xa.y, xa.x)), fma(w.y, xa.y, fma(w.x, xa.x, xa.y)));
                    } else if constexpr (a_none) {
                        static_assert(b_all, "cut-offs");
                        const cplx xb = sf[kb];                     // S = conj(xb), D = -conj(xb)
                        v[m] = make_double2(fma(-w.y, xb.x, fma(-w.x, xb.y, xb.x)), fma(w.y, xb.y, fma(-w.x, xb.x, -xb.y)));
                    } else {
                        cplx xa = make_double2(0.0, 0.0), xb = xa;
                        if (a_all || k < NKX) xa = sf[k];
                        if (b_all || kb < NKX) xb = sf[kb];
                        if (m == 0 && k == 0) { xa.y = 0.0; xb.y = 0.0; }   // reading S20
                        const double Sx = xa.x + xb.x, Sy = xa.y - xb.y, Dx = xa.x - xb.x, Dy = xa.y + xb.y;
                        v[m] = make_double2(fma(w.y, Dx, fma(-w.x, Dy, Sx)), fma(w.y, Dy, fma(w.x, Dx, Sy)));
                    }
                });
                RegFFT<R1, +1>::run(v);
                TwPow<R1> tp;
                tp.init(cmul(wj, wj));
                s[widx<LG>(lrow + jj, f)] = v[0];
                tp.each([&](int q, cplx wq) { s[widx<LG>(lrow + jj + S1 * q, f)] = cmultw<+1>(v[q], wq); });
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(bar_free);   // this field's staged row is consumed
            // ---- B: DIF pass R2, no twiddles (they are applied in the pointwise stage) ----
            if constexpr (R2 > 1) {
#pragma unroll
                for (int it = 0; it < (LPI * NB2 + 31) / 32; ++it) {
                    const int b0 = opaque(lane) + 32 * it;
                    if (b0 < LPI * NB2) {
                        const int b = b0 % NB2, row0 = (b0 / NB2) * H + (b >> 1) * LS + (b & 1);
                        cplx v[R2];
#pragma unroll
                        for (int m = 0; m < R2; ++m) v[m] = s[widx<LG>(row0 + 2 * m, f)];
                        RegFFT<R2, +1>::run(v);
#pragma unroll
                        for (int q = 0; q < R2; ++q) s[widx<LG>(row0 + 2 * q, f)] = v[q];
                    }
                }
            }
        } else if (service) {
            if (lane == 0) {                        // all input warps are done with the stage: prefetch the next line
                mbar_wait(bar_free, parity);
                if (grp + (int)gridDim.x < ngroups) {
                    fence_proxy_async();
                    issue(grp + gridDim.x);
                }
            }
        }
        parity ^= 1;
        __syncthreads();
        // ---- C: last DIF radix 2 (with the inner pass's twiddle), pointwise products, first DIT radix 2 ----
        for (int t0 = opaque(tid); t0 < LPI * (H / 2); t0 += NT) {
            const int t = t0;                                // row pair (2t, 2t+1) of the LPI-line tile (line l starts at row l H)
            double p00[8], p01[8], p10[8], p11[8];
#pragma unroll
            for (int q = 0; q < NIN; ++q) {
                const cplx p = s[widx<LG>(2 * t, q)];
                cplx m = s[widx<LG>(2 * t + 1, q)];
                if (R2 > 1) m = cmultw<+1>(m, wc);
                p00[q] = p.x + m.x; p01[q] = p.y + m.y;
                p10[q] = p.x - m.x; p11[q] = p.y - m.y;
            }
#pragma unroll
            for (int q = 0; q < NOUT; ++q) {
                double o00, o01, o10, o11;
                nl_quad<PHASE>(q, p00, p01, p10, p11, a.cs, o00, o01, o10, o11);
                s[widx<LG>(2 * t, q)] = make_double2(o00 + o10, o01 + o11);
                cplx m = make_double2(o00 - o10, o01 - o11);
                if (R2 > 1) m = cmultw<-1>(m, wc);
                s[widx<LG>(2 * t + 1, q)] = m;
            }
        }
        __syncthreads();
        if constexpr (PHASE) {
            if (service && grp + (int)gridDim.x < ngroups) derive(parity);      // parity is already the next group's
        }
        if (f < NOUT) {
            // ---- D: DIT pass R2 (forward transform, sign -), no twiddles ----
            if constexpr (R2 > 1) {
#pragma unroll
                for (int it = 0; it < (LPI * NB2 + 31) / 32; ++it) {
                    const int b0 = opaque(lane) + 32 * it;
                    if (b0 < LPI * NB2) {
                        const int b = b0 % NB2, row0 = (b0 / NB2) * H + (b >> 1) * LS + (b & 1);
                        cplx v[R2];
#pragma unroll
                        for (int m = 0; m < R2; ++m) v[m] = s[widx<LG>(row0 + 2 * m, f)];
                        RegFFT<R2, -1>::run(v);
#pragma unroll
                        for (int q = 0; q < R2; ++q) s[widx<LG>(row0 + 2 * q, f)] = v[q];
                    }
                }
                __syncwarp();
            }
            // ---- E: DIT pass R1; the results stay in registers ----
            cplx v[R1];
            {
                const int jj = opaque(j) & (S1 - 1);
                TwPow<R1> tp;
                tp.init(cmul(wj, wj));
                v[0] = s[widx<LG>(lrow + jj, f)];
                tp.each([&](int m, cplx wq) { v[m] = cmultw<-1>(s[widx<LG>(lrow + jj + S1 * m, f)], wq); });
                RegFFT<R1, -1>::run(v);
            }
            // ---- F: post-twiddle of row k = j + S1 q against its partner row H - k, truncated store.  The partner
            // is output R1 - 1 - q of butterfly S1 - j (output R1 - q of butterfly 0 for j = 0): a register of another
            // lane of THIS warp, fetched by shuffle - no shared-memory exchange and no barrier.
            {
                const int src = ln * S1 + ((S1 - j) & (S1 - 1));
                cplx *o = outf + base + j;
                static_for<0, R1>([&](auto Q) {
                    constexpr int q = decltype(Q)::value;
                    if constexpr (S1 * q < KXP) {              // no row of this q is kept otherwise
                        constexpr bool all = (S1 * q + S1 - 1 < NKX);
                        const cplx mine = (j == 0) ? v[(R1 - q) & (R1 - 1)] : v[R1 - 1 - q];
                        cplx zp;
                        zp.x = __shfl_sync(0xffffffffu, mine.x, src);
                        zp.y = __shfl_sync(0xffffffffu, mine.y, src);
                        const int k = j + S1 * q;
                        const cplx za = v[q];
                        if (q == 0 && k == 0) zp = za;         // k = 0 is its own partner
                        const cplx w = q ? cmul(wj, make_double2(wc_re<2 * R1>(q), wc_im<2 * R1>(q))) : wj;
                        const double Sx = za.x + zp.x, Sy = za.y - zp.y, Dx = za.x - zp.x, Dy = za.y + zp.y;
                        // X_k = (S - i w D) / (2 L)
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
            __syncwarp();     // this warp's F reads are done before its next stage A overwrites the field
        }
    }
}

}  // namespace psdns
