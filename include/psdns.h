/*
 * libpsdns - B200-native (sm_100a, FP64) hot path of the pseudo-spectral multiphase channel
 * solver of arXiv 2406.01322: per time step, batched backward transforms
 * (Chebyshev in z, Fourier in y and x), pointwise non-linear terms in physical space,
 * forward transforms with 2/3 dealiasing, and the batched per-(kx,ky) Chebyshev-tau
 * Helmholtz / biharmonic solves of the IMEX scheme.
 *
 * Plain C ABI: opaque handle, POD structs, raw pointers, int status codes.  No exceptions,
 * no printing, no abort.  The library never allocates or frees device memory: every d_*
 * pointer and the workspace are DEVICE memory owned by the caller (e.g. torch tensors);
 * h_* pointers are HOST memory (pinned for asynchronous copies) owned by the caller.
 * All work is enqueued on the cudaStream_t given at init; calls return after enqueue and
 * the caller synchronises.  A handle is not thread-safe; distinct handles are independent.
 *
 * Layouts at the boundary (internal layouts are private):
 *   PSDNS_PHYSICAL : double  [nz][ny][nx]           x fastest; z index k <-> z_k = cos(pi k/(nz-1))
 *                                                   (k = 0 is the wall z = +1; Gauss-Lobatto, L134/L178)
 *   PSDNS_SPECTRAL : double  [nz][ny][nx/2+1][2]    interleaved complex; kx index i = 0..nx/2 fastest,
 *                                                   ky in FFT order (0..ny/2, -ny/2+1..-1), n = Chebyshev mode
 * Transform conventions (readings S1, S2 of DESIGN.md):
 *   forward : f^(i,j,n) = 1/(nx ny) sum_xy f e^{-i(kx x + ky y)}, then a_n = 2/(N c_n) sum_k f_k cos(pi n k/N)/c_k
 *   backward: f = sum f^ T_n(z_k) e^{+i(kx x + ky y)}, x real <-> half-complex (D2Z/Z2D, L176)
 */
#ifndef PSDNS_H
#define PSDNS_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct psdns_handle psdns_handle; /* opaque; host memory owned by the library */

/* Channel grid: nx, ny periodic equispaced points over lx, ly;
 * nz Chebyshev-Gauss-Lobatto points on z in [-1, 1].
 * Supported: nx, ny powers of two in [16, 1024]; nz - 1 a power of two in [8, 512]. */
typedef struct {
    int nx, ny, nz;
    double lx, ly;
} psdns_grid;

/* Dimensionless groups: Re (Eq. 9), Pe (Eq. 2), Ch (L70), We (Eq. 10); time step dt.
 * gradp_x   : constant mean forcing G added to S_x (reading S12; 2/Re keeps u = 1 - z^2 steady)
 * visc_ratio: lambda, viscosity ratio; 1.0 = matched; != 1 evaluates the
 *             explicit variable-viscosity stress pointwise (reading S14)
 * phase_field: 0 = single-phase Navier-Stokes only (the Fig. 3 workload, L231), 1 = + Cahn-Hilliard
 * wall_top, wall_bottom: velocity condition at z = +1 / z = -1.  Free-slip turns the condition on
 *             omega_z (and the mean flow) into d/dz = 0 and the second condition on w into d^2 w/dz^2 = 0 (continuity);
 *             phi keeps d phi/dz = d psi/dz = 0.  Zero-initialised structs give the no-slip channel.
 * convection_form: 1 evaluates the convective term as u x omega (vorticity of the truncated velocity formed in spectral
 *             space, three more backward fields); differs from form 0 by grad(|u|^2 / 2), see surface_tension_form.
 * surface_tension_form: 1 evaluates the surface tension as a force vector instead of a stress tensor.  The two differ by
 *             a gradient that Eqs. 14-15 annihilate, in the discrete problem only to truncation error, so it is a switch
 *             and not an optimisation; it costs one more backward field (lap phi) and three more forward fields, runs the
 *             three-kernel x path through physical-space arrays (part of its workspace) and is slower than form 0.
 * dealias   : must be 1 for psdns_step (2/3 rule in x, y, z; reading S3).  The round-trip
 *             call always runs with dealiasing off. */
typedef struct {
    double re, pe, ch, we, dt;
    double gradp_x;
    double visc_ratio;
    int phase_field;
    int dealias;
    int wall_top;    /* wall z = +1: 0 = no-slip (u = v = w = 0), 1 = free-slip (w = 0, du/dz = dv/dz = 0) - PAPER.md L52 */
    int wall_bottom; /* wall z = -1, same codes; "a combination of them" (L52) = different values at the two walls */
    int surface_tension_form; /* 0 = divergence of the Korteweg tensor, Eq. 8 as written (reading S5); 1 = the force
                               * -c_sigma lap(phi) grad(phi): needs phase_field = 1, visc_ratio = 1 */
    int convection_form;      /* 0 = divergence form -div(u u) (reading S4); 1 = rotational form u x omega;
                               * not together with visc_ratio != 1 */
} psdns_params;

enum { PSDNS_PHYSICAL = 0, PSDNS_SPECTRAL = 1 };

enum {
    PSDNS_OK = 0,
    PSDNS_EINVAL = -1, /* null pointer, unsupported size, non-positive dt/Re/..., bad enum */
    PSDNS_ENOMEM = -2, /* workspace too small or misaligned (256 B) */
    PSDNS_ESTATE = -3, /* step/get before set_state */
    PSDNS_ECUDA = -4   /* CUDA launch/runtime failure; text via psdns_last_error */
};

/* Bytes of device workspace psdns_init needs for this grid/params (0 on invalid input).
 * Holds twiddle tables, the retained-mode state (u^, v^, w^, phi^, theta^), the AB2 history,
 * per-wavenumber solver tables, transform scratch and host-staging buffers. */
size_t psdns_workspace_bytes(const psdns_grid *grid, const psdns_params *params);

/* Create a handle.  d_workspace: device memory, >= psdns_workspace_bytes, 256-byte aligned,
 * must outlive the handle.  cuda_stream: a cudaStream_t (NULL = default stream).  Builds the
 * twiddle tables and the per-(kx,ky) solver factorisations (enqueued on the stream). */
int psdns_init(const psdns_grid *grid, const psdns_params *params, void *d_workspace, size_t bytes,
               void *cuda_stream, psdns_handle **out);

/* Step i) of the time-step algorithm.  space = PSDNS_PHYSICAL: each field is
 * forward transformed (x, then y, then z; L154).  space = PSDNS_SPECTRAL: fields are taken as
 * given.  Only the retained (kx, ky) modes (i <= nx/3, |j'| <= ny/3) are kept; all nz Chebyshev
 * modes are kept.  Derives the hidden state theta^ = (D^2 - k^2) w^ and clears the
 * Adams-Bashforth history, so the next step is an explicit-Euler start (reading S7).
 * d_phi may be NULL iff phase_field == 0.  Inputs are not modified. */
int psdns_set_state(psdns_handle *h, int space, const void *d_u, const void *d_v, const void *d_w,
                    const void *d_phi);

/* Advance nsteps time steps (rows a1-a11 of DESIGN.md): non-linear terms by
 * backward transforms -> pointwise products -> forward transforms with dealiasing; AB2 for the
 * explicit terms; Crank-Nicolson Helmholtz solves for omega_z (Eq. 14) and the two-stage w problem
 * (Eq. 15) with u^, v^ from Eqs. 6 and 16; implicit-Euler two-stage solve for phi (Eq. 17).
 * Asynchronous on the stream. */
int psdns_step(psdns_handle *h, int nsteps);

/* Copy the state out in the requested space (outputs fully overwritten; non-retained modes are
 * zero in PSDNS_SPECTRAL).  d_phi may be NULL iff phase_field == 0. */
int psdns_get_state(psdns_handle *h, int space, void *d_u, void *d_v, void *d_w, void *d_phi);

/* Hidden state of the time integration, for an exact restart (SURVEY.md 8(b) "optional, for bit-exact restart";
 * the paper's demo run "starts ... in a flow field previously obtained" from another run):
 * theta^ = lap(w) carried from the last solve (reading S13), omega_z^, D phi^, the three Adams-Bashforth
 * history spectra (N_omega, N_w, S_phi of step n-1, reading S7) and the step counter, as ONE opaque blob in the
 * library's private layout.  Protocol: state = psdns_get_state(PSDNS_SPECTRAL), blob = psdns_get_history;
 * later, on a handle of the same grid and params: psdns_set_state(PSDNS_SPECTRAL, state) then
 * psdns_set_history(blob) - the following steps are bit-identical to the uninterrupted run.
 * d_blob: DEVICE memory of psdns_history_bytes(h) bytes (256-byte aligned), owned by the caller.
 * Between steps theta^ is held as the particular solution plus the coefficients of its influence-matrix correction
 * (option "lazy"); psdns_get_history first completes the array on the stream (one small kernel), which does not change
 * what the following steps compute.  Asynchronous on the stream.
 * PSDNS_ESTATE before the first set_state; PSDNS_EINVAL on a null pointer or a size mismatch. */
size_t psdns_history_bytes(const psdns_handle *h);
int psdns_get_history(psdns_handle *h, void *d_blob, size_t bytes);
int psdns_set_history(psdns_handle *h, const void *d_blob, size_t bytes);

/* One forward+backward 3-D transform of a single field with dealiasing OFF (full sizes).
 * start_space = PSDNS_PHYSICAL: d_in physical -> (d_mid spectral, nullable) -> d_out physical.
 * start_space = PSDNS_SPECTRAL: d_in spectral -> (d_mid physical, nullable) -> d_out spectral.
 * Does not touch the state. */
int psdns_transform_roundtrip(psdns_handle *h, int start_space, const void *d_in, void *d_out,
                              void *d_mid);

/* Host-buffer form of set_state -> step -> get_state, used for the end-to-end number.  The four fields are copied host ->
 * device on a side stream of the handle into one of two input staging sets, then set_state, nsteps steps and get_state
 * (into output staging buffers) run on the init stream, and the result is copied device -> host on a second side stream.
 * Consecutive calls on one handle therefore pipeline: the upload of call k + 1 and the copy-back of call k - 1 overlap the
 * compute of call k (PCIe is full duplex; the copies are 90 % of such a call).
 * h_in_* / h_out_* are HOST pointers (pinned, for the copies to be asynchronous) in the boundary layout of `space` (the
 * phi pair may be NULL iff phase_field == 0).  h_out_* are valid, and h_in_* may be modified again, after
 * psdns_run_host_wait(h) has returned - synchronising the init stream alone does NOT cover the side streams. */
int psdns_run_host(psdns_handle *h, int space, int nsteps, const void *h_in_u, const void *h_in_v,
                   const void *h_in_w, const void *h_in_phi, void *h_out_u, void *h_out_v,
                   void *h_out_w, void *h_out_phi);

/* Block the calling host thread until the device -> host copies of the last psdns_run_host have finished. */
int psdns_run_host_wait(psdns_handle *h);

/* Number of kernel launches the library has enqueued on this handle since init. */
long long psdns_launch_count(const psdns_handle *h);

/* Enable (1) / disable (0) CUDA-event timing of the kernel class `name` inside psdns_step
 * ("zbwd","ybwd","xbwd","pointwise","xfwd","yfwd","zfwd","rhs","solve", or "xfused").  When
 * enabled, psdns_step records events on the stream around every launch of that class;
 * psdns_kernel_time_ms returns the accumulated milliseconds and launch count after the caller
 * has synchronised.  Used by bench.py for the roofline of the dominant kernel. */
int psdns_kernel_timing(psdns_handle *h, const char *name, int enable);
int psdns_kernel_time_ms(psdns_handle *h, double *ms_total, long long *launches);

/* Diagnostics of the current state, computed on the device from the resident spectra (the fields a run
 * monitors) - no host round trip, asynchronous on the stream.  d_out: DEVICE memory, 8 doubles:
 *   [0] mean(phi)          volume average, 1/2 sum_{n even} phi^(0,0,n) 2/(1 - n^2)   (0 when phase_field == 0)
 *   [1] max |div u|        max over all retained coefficients of |i kx u^ + i ky v^ + D w^|  (Eq. 6)
 *   [2] kinetic energy     1/2 <u^2 + v^2 + w^2>: mean over x, y (Parseval over the retained modes), Clenshaw-Curtis
 *                          quadrature over the collocation points z_k, divided by the channel height 2
 *   [3] [4] wall shear     d u-bar/dz at z = +1 and at z = -1 (mean streamwise velocity, column (0,0))
 *   [5] bulk velocity      1/2 int u-bar dz
 *   [6] [7]                reserved, written as 0
 * Uses the transform scratch (not the state).  PSDNS_ESTATE before the first set_state. */
int psdns_diagnostics(psdns_handle *h, double *d_out);

/* psdns_diagnostics for callers that may not allocate device memory and have none to spare (code under CUDA graph
 * capture, tight serving loops, harnesses that forbid cudaMalloc): same inputs (the resident state), same 8 outputs in
 * DEVICE memory d_out, same kernels and launch shapes - the results are bit-identical to psdns_diagnostics - but the
 * per-block partials of the two reductions live in a file-scope `static __device__` array of
 * PSDNS_STATIC_SCRATCH_DOUBLES doubles (16 KiB, held by every GPU that loads the library until the process exits)
 * instead of the workspace's fourth Z array.  The call itself runs no cudaMalloc, cudaFree or allocating library routine.
 *   limit    ceil(ncols/256) + 8 * (number of SMs) <= PSDNS_STATIC_SCRATCH_DOUBLES, ncols = the retained (kx, ky) columns
 *            (1024 x 512 needs 459 + 1184 on a B200; 1024 x 1024 does not fit).  Beyond it: PSDNS_EINVAL, nothing launched,
 *            the text names the need and the limit.
 *   sharing  every handle and every call on one GPU shares the array.  Each call overwrites the slots it reads before it
 *            reads them, so the last call's contents never matter and nothing is cleared; but two calls that OVERLAP on
 *            the GPU (different streams or handles, no ordering between them) race on it - serialise them.
 *   errors   PSDNS_ESTATE before the first set_state or while psdns_kernel_timing is enabled (timing creates events);
 *            PSDNS_EINVAL on a null pointer, a device ordinal > 63 or a grid beyond the limit; PSDNS_ECUDA otherwise.
 * The device that owns the handle's workspace must be current, as for every other call. */
#define PSDNS_STATIC_SCRATCH_DOUBLES 2048
int psdns_diagnostics_static(psdns_handle *h, double *d_out);

/* Iso-surface ray-caster (Fig. 5: the drops are rendered as the iso-surface phi = 0).
 * Pure compute into headless DEVICE buffers, no graphics API.  One ray per pixel:
 *   camera : f = unit(target - eye), r = unit(f x up), v = r x f; pixel (px, py), py = 0 the top row:
 *            sx = (2 (px + 1/2)/width - 1) tan(fov_y/2) width/height, sy = (1 - 2 (py + 1/2)/height) tan(fov_y/2),
 *            direction = unit(f + sx r + sy v)
 *   box    : slab intersection with [0, lx] x [0, ly] x [-1, 1]; a miss gives intensity 0, depth -1
 *   field  : trilinear interpolation on the grid (periodic in x, y; z clamped to the Gauss-Lobatto points)
 *   march  : samples at t0 + i step (last one at the exit point); the first sign change of field - iso is refined by
 *            24 bisections; depth = ray parameter of the midpoint of the last bracket
 *   shade  : intensity = 0.2 + 0.8 |unit(grad) . unit(light)|, grad by central differences with steps (lx/nx, ly/ny, 1/N)
 * d_field: DEVICE double [nz][ny][nx] (PSDNS_PHYSICAL layout), or NULL = the current phase field phi of the state
 * (needs phase_field = 1 and a state).  d_intensity, d_depth: DEVICE double [height][width], fully overwritten. */
typedef struct {
    double eye[3], target[3], up[3];
    double fov_y_deg;
    int width, height;
    double step;
    double light[3];
} psdns_camera;
int psdns_render_isosurface(psdns_handle *h, const psdns_camera *cam, double iso, const void *d_field,
                            void *d_intensity, void *d_depth);

/* FP64 peak of this GPU as an FMA-chain microbenchmark measures it: 8 independent chains of dependent DFMAs
 * per thread, 8 CTAs of 256 threads per SM, best of three timed launches; *tflops in TFLOP/s (2 flops per FMA).
 * Synchronises the stream.  Used by bench.py as the denominator of the FP64 view of the fused x kernel's roofline. */
int psdns_measure_fp64_peak(psdns_handle *h, double *tflops);

/* Tuning and test switches.  None is needed for normal use; the defaults are the product path.  Changing an option
 * drops the captured CUDA graph of the step (it is re-captured by the next psdns_step).
 *   "graph"    1 (default) / 0 : replay one captured CUDA graph per step / launch the kernels directly
 *   "xfuse"    1 (default) / 0 : fused x kernel (rows a4-a6 in one kernel, physical space never in HBM) / the three-kernel
 *                                cross-check path x-backward -> pointwise -> x-forward through physical-space arrays;
 *                                0 needs a workspace of psdns_workspace_bytes_unfused() bytes at init, else PSDNS_ENOMEM
 *   "grid_cap" n >= 0          : upper bound on the grid of every persistent kernel (z, y, fused x passes); 0 = none.
 *                                Tests use a small cap so that each CTA walks many tiles / lines of a small grid.
 *   "ztma"     1 (default) / 0 : z passes fed by 2-D TMA tensor loads into a two-deep shared-memory stage (k_zpass_tma)
 *                                / by per-thread strided loads (k_zpass); same arithmetic at N < 512, radix plan differs
 *                                in the forward pass at N = 512
 *   "zgemm"    0 (default) / 1 : nz <= 65 only: Chebyshev transform as a dense FP64 matrix product on the tensor cores
 *                                (k_zgemm, DMMA) instead of the FFT path - kept for the measurement of SURVEY 8(f)-1
 *   "pf", "pf_rhs" n >= 0      : L2 prefetch distance, in rows, of the solver sweeps (defaults 2 and 4)
 *   "phi3"     1 (default) / 0 : phase field only: the second Helmholtz solve of the phi problem eliminated upwards inside
 *                                the up sweep that produces psi and back-substituted by the last (downward) sweep - three
 *                                sweeps over the phi column, psi never stored - / the five-sweep form; equal to rounding
 *   "w3"       1 (default) / 0 : the w problem likewise (its second solve eliminated upwards inside the up
 *                                sweep of the (omega_z, theta) pair, influence-matrix correction in the last sweep): the
 *                                solver stage is then three launches instead of five; needs "phi3" with a phase field
 *   "lazy"     1 (default) / 0 : with "w3": the influence-matrix correction of the hidden state theta^ is not written back
 *                                by the last sweep but applied by the next step's right-hand-side kernel where it reads
 *                                theta^ anyway (psdns_get_history and psdns_set_option materialise it first) / written back
 * PSDNS_EINVAL on an unknown name or a bad value. */
int psdns_set_option(psdns_handle *h, const char *name, double value);

/* Workspace size that also holds the physical-space arrays of the unfused cross-check path ("xfuse" 0). */
size_t psdns_workspace_bytes_unfused(const psdns_grid *grid, const psdns_params *params);

/* Introspection for tests and bench.py; -1 on an unknown name.  "<class>_grid" / "<class>_items": grid size and number
 * of work items (tiles or lines) of the last launch of the persistent kernel class <class> = zbwd | ybwd | xfused |
 * yfwd | zfwd; "n_sm"; "workspace_bytes"; "launches_per_step" (kernels in the captured graph of one step). */
double psdns_get_info(const psdns_handle *h, const char *name);

/* Release the handle (host memory only; the workspace stays the caller's). */
int psdns_destroy(psdns_handle *h);

/* Text of the last error on this handle ("" if none); valid until the next call. NULL-safe. */
const char *psdns_last_error(const psdns_handle *h);

#ifdef __cplusplus
}
#endif
#endif /* PSDNS_H */
