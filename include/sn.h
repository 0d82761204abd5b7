/*
 * sn.h -- C ABI of the B200-native split-step Schroedinger-Newton stepper (libsn.so).
 *
 * What the library computes.  The generalized Schroedinger-Newton system of PAPER.md:42-44
 * (section II, eq. (1),(2))
 *      i dpsi/dtau = A lap psi + B phi psi + G(|psi|^2) psi            (1)
 *      lap phi + C phi = D |psi|^2                                      (2)
 * on a periodic 2D/3D box, advanced with the "Symmetric Split-Step Fourier Method", eq. (2)
 * "also solved with spectral methods" (section III).  One step is
 *      K(dtau/2) N(dtau) K(dtau/2),
 *      K(s): psi^ *= exp(+i A k^2 s) in Fourier space,
 *      N(s): phi^ = D rho^/(C - k^2) (phi^(0) = 0 when C == 0), psi *= exp(-i s (B phi + G(rho))),
 * (readings Q1-Q10 of DESIGN.md).  All arithmetic is complex64/float32 on the GPU; every step
 * of the path runs in hand-written sm_100a kernels (no cuFFT, no CPU fallback).
 *
 * Conventions.
 *   - dims[0] is the slowest axis, dims[ndim-1] the contiguous one (C order).
 *   - psi is complex64, interleaved (re, im), ndim-dimensional, dense.
 *   - Pointers are tagged "host" or "device" below.  The library never allocates device
 *     memory: state, half-spectrum buffer and tables live in the caller's workspace
 *     (e.g. a torch uint8 tensor), which must stay alive until sn_destroy.
 *   - Every call returns 0 on success or a negative SN_ERR_* code; nothing throws, nothing
 *     calls exit.  Argument errors (every code except SN_ERR_CUDA) are detected before any
 *     device work is enqueued: outputs are untouched and the context is unchanged.  After
 *     SN_ERR_CUDA (a launch or copy failed part-way through a call) the state and the tables of
 *     the context are undefined: destroy it and create a new one.
 *   - A context is not thread-safe; different contexts are independent.
 *   - All device work is enqueued on the cudaStream_t given to sn_create, on the device that
 *     owns the workspace: every call switches to that device for its duration and restores the
 *     caller's current device on return.
 *   - The library reads no environment variables; every switch is an argument or sn_set_option.
 */
#ifndef SN_H
#define SN_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define SN_OK 0
#define SN_ERR_NULL -1      /* a required pointer is NULL */
#define SN_ERR_DIMS -2      /* ndim not 2/3, or an axis length that is not supported */
#define SN_ERR_PARAM -3     /* non-finite constant, L <= 0, n_g outside [0,4], nsteps < 0 */
#define SN_ERR_SINGULAR -4  /* C > 0 and C == k^2 for some grid mode: eq. (2) has no solution */
#define SN_ERR_WORKSPACE -5 /* workspace too small or not 256-byte aligned */
#define SN_ERR_STATE -6     /* step/get/diagnostics before sn_set_state */
#define SN_ERR_CUDA -7      /* a CUDA runtime call failed (sticky; text via sn_strerror) */
#define SN_ERR_NOMEM -8     /* host allocation failed */
#define SN_ERR_FEATURE -9   /* the call needs a workspace region that was not requested at create (sn_options.features) */
#define SN_ERR_TOO_LARGE -10 /* sn_norm_static: more cells than its fixed static scratch serves */

typedef struct sn_ctx sn_ctx; /* opaque host object, owned by the library */

/* Diagnostics (reading Q10 of DESIGN.md; the paper defines none):
 *   norm = sum |psi|^2 dV,
 *   H    = -A sum_k k^2 |psi^_k|^2 dV/prod N + (B/2) sum phi rho dV + sum F(rho) dV,
 *   F(rho) = sum_j g_j rho^(j+1)/(j+1). */
typedef struct {
    double norm, e_kin, e_nonlocal, e_local, e_total;
} sn_diag;

/* Optional workspace regions.  The stepper itself needs the state (8 B/cell), the half spectrum (~4 B/cell) and
 * the FFT tables: about 12 B/cell.  Everything else is requested at create time: */
#define SN_FEAT_STAGING 1u  /* 4 B/cell scratch: host destination of sn_debug_potential, host sources of sn_set_source_tables */
#define SN_FEAT_VEXT 2u     /* 4 B/cell: the external potential table of sn_set_external_potential */
#define SN_FEAT_SOURCE 4u   /* 8 B/cell: the interleaved (beta, gamma) tables of sn_set_source_tables */
#define SN_FEAT_ALL 7u

typedef struct {
    size_t struct_size;  /* sizeof(sn_options), filled in by the caller (a mismatch is SN_ERR_PARAM) */
    int64_t batch;       /* ensemble members, >= 1 (see sn_create_batch) */
    uint32_t features;   /* SN_FEAT_* bits */
    uint32_t dtype;      /* SN_DTYPE_C64 (default) or SN_DTYPE_C128 */
} sn_options;

/* Precision of the state and of all arithmetic.  SN_DTYPE_C64: complex64 / float32 (BASELINE.json's metric).
 * SN_DTYPE_C128: complex128 / float64, the precision the paper benchmarked: psi passed to
 * sn_set_state / sn_get_state is complex128 (16 B per cell), sn_debug_potential writes float64, the workspace is
 * about twice as large.  The complex128 path runs eq. (1),(2) with the polynomial G (Strang and order-4 steps,
 * ensembles, diagnostics, test hooks); the NEXT-1 terms (sn_set_local_terms, _external_potential, _source_tables,
 * _bohm) return SN_ERR_FEATURE there and features must be 0. */
#define SN_DTYPE_C64 0u
#define SN_DTYPE_C128 1u

/* Supported axis lengths: powers of two with 32 <= N <= 4096, and 3*2^a with 96 <= N <= 3072 (96, 192, 384, 768,
 * 1536, 3072: radix-4 stages, a leading radix-2 stage where needed, and one radix-6 stage; the grid-size sweep's 384^3).  Any other length: sn_workspace_bytes
 * returns 0 and sn_create returns SN_ERR_DIMS.  Bytes of device workspace needed. */
size_t sn_workspace_bytes(int ndim, const int64_t *dims /* host, ndim entries */);  /* = options {batch 1, features 0} */
size_t sn_workspace_bytes_opt(int ndim, const int64_t *dims /* host */, const sn_options *opt /* host */);

/* Create a context.
 *   out          host; receives the context
 *   dims, L      host; ndim axis lengths and box lengths (dims[0] slowest)
 *   A,B,C,D      constants of eq. (1),(2)
 *   g, n_g       host; G(rho) = sum_{j=1..n_g} g[j-1] rho^j, 0 <= n_g <= 4 (g may be NULL if n_g == 0)
 *   dtau         step; may be negative (time reversal) or zero
 *   d_workspace  DEVICE; >= sn_workspace_bytes(...) bytes, 256-byte aligned, caller-owned
 *   cuda_stream  cudaStream_t (0 = legacy default stream) */
int sn_create(sn_ctx **out, int ndim, const int64_t *dims, const double *L, double A, double B, double C,
              double D, const double *g, int n_g, double dtau, void *d_workspace, size_t workspace_bytes,
              void *cuda_stream);

/* Same with options (ensemble size, optional workspace regions).  sn_create = {batch 1, features 0};
 * sn_create_batch = {batch, features 0}. */
int sn_create_opt(sn_ctx **out, int ndim, const int64_t *dims, const double *L, double A, double B, double C,
                  double D, const double *g, int n_g, double dtau, void *d_workspace, size_t workspace_bytes,
                  void *cuda_stream, const sn_options *opt /* host */);

/* Ensemble of `batch` independent systems advanced together ("batched small-grid ensembles";
 * parameter scans such as PAPER.md:131 run many small meshes).  Same constants and dtau for every member.
 * ndim, dims, L: as for sn_create, describing ONE system.  Storage layout of every array of the context (state,
 * external potential, source tables): [dims[0]][batch][dims[1]]([dims[2]]), i.e. the member index sits right after
 * the slowest physical axis, so that the lines of every axis stay dense; member b of a (batch, dims...) array is at
 * [:, b, ...].  No pass runs along the member index.  sn_diagnostics returns the SUM over the ensemble.
 * 1 <= batch <= 2^20; batch = 1 is sn_create.  An ensemble whose line or column counts do not fit a 32-bit int
 * (more than 2^31-1 lines along any axis) is rejected with SN_ERR_DIMS. */
size_t sn_workspace_bytes_batch(int ndim, const int64_t *dims /* host, ndim */, int64_t batch);
int sn_create_batch(sn_ctx **out, int ndim, const int64_t *dims, int64_t batch, const double *L, double A, double B,
                    double C, double D, const double *g, int n_g, double dtau, void *d_workspace, size_t workspace_bytes,
                    void *cuda_stream);

/* Copy a complex64 state in.  psi: host (src_on_device == 0) or device pointer; prod(dims) complex64. */
int sn_set_state(sn_ctx *ctx, const void *psi, int src_on_device);

/* Advance nsteps Strang steps (tau += nsteps*dtau).  Enqueues kernels and returns without
 * synchronising.  Adjacent kinetic half steps are merged inside one call (mathematically identical). */
int sn_step(sn_ctx *ctx, int64_t nsteps);

/* Fourth-order variant (not in the paper, which uses the second-order symmetric scheme of
 * PAPER.md:113): one step is the Yoshida composition S2(w1 dtau) S2(w0 dtau) S2(w1 dtau) of three Strang steps,
 * w1 = 1/(2 - 2^(1/3)), w0 = 1 - 2 w1 (< 0), adjacent kinetic half steps merged.  Three N sub-steps per step. */
int sn_step_order4(sn_ctx *ctx, int64_t nsteps);

/* Copy the state out.  A host destination synchronises the stream. */
int sn_get_state(sn_ctx *ctx, void *psi_out, int dst_on_device);

/* Norm and energy of the current state (host struct).  Synchronises; the state is unchanged. */
int sn_diagnostics(sn_ctx *ctx, sn_diag *out);

/* Replace dtau (rebuilds the kinetic phase tables and the nonlinear coefficients; synchronises the stream). */
int sn_set_dtau(sn_ctx *ctx, double dtau);

/* ---- NEXT-1 terms of the local potential (eq. (15),(16)) ----
 * sn_set_local_terms: G(rho) += g_log ln(rho_f) + g_pow rho_f^p_pow, rho_f = max(rho, rho_floor) -- the pressure
 *   potential V_pressure = w ln(rho) (n = 1) or (n w/(n-1)) rho^(n-1) of eq. (16).  rho_floor > 0 (reading Q15:
 *   the paper does not say how ln(0) is avoided), p_pow != -1.  g_log = g_pow = 0 switches the terms off.
 * sn_set_external_potential: a fixed real potential V(x) (float32, prod(dims) values, layout of psi; host or
 *   device pointer, copied into the workspace; needs SN_FEAT_VEXT) enters the N sub-step as exp(-i s (B phi + G(rho) + V)) -- phi_C
 *   of eq. (11),(15).  NULL removes it.  exp(-i s V) commutes with the rest of the N phase, so it is applied by the
 *   contiguous-axis kinetic pass that precedes each N sub-step (by the axis-0 pass when that one is first-path).
 * Both rebuild the nonlinear-phase coefficients; e_local of sn_diagnostics then includes sum (F(rho) + V rho) dV. */
/* sn_set_source_tables: eq. (12), PAPER.md:92 -- lap phi + C phi = D (gamma(x) rho + beta(x) lap rho) instead of
 *   eq. (2).  beta, gamma: float32, prod(dims) values each, layout of psi, host or device (copied into the
 *   workspace; needs SN_FEAT_SOURCE, host sources also SN_FEAT_STAGING); two NULLs restore eq. (2) (= gamma 1, beta 0).  Costs one more half-spectrum chain and one more
 *   axis-0 pass per step.  e_nonlocal of sn_diagnostics stays (B/2) sum phi rho dV (no longer a conserved energy
 *   when beta, gamma vary in space: the kernel of phi[rho] is not symmetric). */
/* sn_set_bohm: the Bohm quantum potential of eq. (15), PAPER.md:102 -- the N sub-step phase gains the factor
 *   exp(-i s c_bohm V_B), V_B = lap sqrt(rho) / (2 max(sqrt(rho), sqrt_floor)) (c_bohm = nu^2 in eq. (15); with
 *   c_bohm = -2A it cancels the quantum pressure of the kinetic operator and real states become stationary).
 *   sqrt_floor > 0 is reading Q17 (the paper does not regularise 1/sqrt(rho)).  Costs one more r2c + half-spectrum
 *   chain + axis-0 pass per N sub-step.  c_bohm = 0 switches it off.  Not included in sn_diagnostics' energies. */
int sn_set_bohm(sn_ctx *ctx, double c_bohm, double sqrt_floor);
int sn_set_local_terms(sn_ctx *ctx, double g_log, double rho_floor, double g_pow, double p_pow);
int sn_set_source_tables(sn_ctx *ctx, const float *beta, const float *gamma, int src_on_device);
int sn_set_external_potential(sn_ctx *ctx, const float *v, int src_on_device);

/* ---- NEXT-4b: coupled wave functions ("Equations (1) and (2) can be further generalized if one considers
 * multiple wave functions coupled through the different nonlinearities of the system"; the paper does not write the
 * system down -- reading Q18 of DESIGN.md) ----
 *      i dpsi_c/dtau = A_c lap psi_c + B_c phi psi_c + (sum_c' g_cc' |psi_c'|^2) psi_c,   c = 0..n_comp-1
 *      lap phi + C phi = D sum_c w_c |psi_c|^2
 * advanced by the same Strang step: K(s) acts on every component with its own A_c; N(s) is exact for its sub-flow
 * (every |psi_c|^2 is invariant under it).  1 <= n_comp <= 4; A, B, w: n_comp values; g: n_comp x n_comp, row-major
 * (g[c * n_comp + c'] multiplies |psi_c'|^2 in the equation of component c); all host pointers.  complex64.
 * State layout for sn_set_state / sn_get_state: [n_comp][dims...] (component-major).  Calls that work on such a
 * context: sn_set_state, sn_step, sn_get_state, sn_set_dtau, sn_mc_norms, sn_set_option, sn_profile*, sn_destroy;
 * the others return SN_ERR_FEATURE.  sn_mc_norms: norms[c] = sum |psi_c|^2 dV (each conserved); host, n_comp doubles. */
size_t sn_workspace_bytes_mc(int ndim, const int64_t *dims /* host */, int n_comp);
int sn_create_mc(sn_ctx **out, int ndim, const int64_t *dims, const double *L, int n_comp, const double *A,
                 const double *B, double C, double D, const double *w, const double *g, double dtau,
                 void *d_workspace, size_t workspace_bytes, void *cuda_stream);
int sn_mc_norms(sn_ctx *ctx, double *norms);

/* ---- NEXT-2: slab-decomposed step for R ranks (the paper's solver is single-device,
 * PAPER.md:113) ----
 * 3D, complex64, eq. (1),(2) with the polynomial G.  The grid dims[0] x dims[1] x dims[2] is split over nranks
 * ranks; rank r owns the z-slab rows [r dims[0]/R, (r+1) dims[0]/R) of axis 0 ("view A", [dims[0]/R][dims[1]][dims[2]]:
 * the layout of sn_set_state / sn_get_state on such a context).  Lines along axes 1 and 2 are whole in view A; for
 * the passes along axis 0 the data is moved to the y-slab view B = [dims[0]][dims[1]/R][dims[2]] by an all-to-all,
 * and back: 4 exchanges per step (psi twice, 8 B/cell; the half spectrum twice, 4 B/cell).  The library runs the LOCAL
 * passes (sn_slab_stage) and the pack/unpack copies; the exchange itself belongs to the caller: sn_slab_exchange_local
 * for R contexts on ONE device and stream (virtual ranks: how the path is validated on one GPU), or, one process per
 * GPU, any all-to-all over the buffers of sn_slab_buffer (paper_1909_08354_b200/slab.py uses torch.distributed, i.e.
 * NCCL over NVLink; not measured on hardware in this build).  Requirements: dims[0], dims[1] and dims[0]/2 divisible
 * by nranks; (dims[1]/nranks) * dims[2] a multiple of 32.  The half-spectrum rows 0..dims[0]/2 are dealt out
 * (dims[0]/2)/nranks per rank, the Nyquist row to the last rank.
 * One call of n steps, psi starting and ending in view A (half_phase = 1 on the first and last kinetic sweep):
 *   KIN_A(half) | psi A->B | KIN0_B(half)
 *   n times: R2C_B | hs B->A | CHAIN_A | hs A->B | NLKIN_B(half on the last step) | psi B->A | KIN_A(same) | psi A->B
 *   (the last psi A->B is dropped)
 * Exchange buffers: view-B buffers hold the block for / from rank r contiguously (rows r dims[0]/R ... of psi_B, rows
 * h_lo(r) ... of hs_B); sn_slab_pack gathers the blocks of a view-A buffer into the staging buffer in rank order
 * (unpack = 0) or scatters them back (unpack = 1).  sn_step and the other whole-grid calls return SN_ERR_FEATURE on a
 * slab context; sn_set_state, sn_get_state, sn_set_dtau, sn_destroy, sn_profile*, sn_launch_count work. */
#define SN_SLAB_KIN_A 0    /* stages of sn_slab_stage */
#define SN_SLAB_KIN0_B 1
#define SN_SLAB_R2C_B 2
#define SN_SLAB_CHAIN_A 3
#define SN_SLAB_NLKIN_B 4
#define SN_SLAB_PSI_A 0    /* buffers of sn_slab_buffer; PSI_A / HS_A also name WHAT an exchange or a pack moves */
#define SN_SLAB_PSI_B 1
#define SN_SLAB_HS_A 2
#define SN_SLAB_HS_B 3
#define SN_SLAB_STAGING 4
size_t sn_slab_workspace_bytes(const int64_t *dims /* host, 3 */, int nranks, int rank);
int sn_slab_create(sn_ctx **out, const int64_t *dims, const double *L, double A, double B, double C, double D,
                   const double *g, int n_g, double dtau, int nranks, int rank, void *d_workspace,
                   size_t workspace_bytes, void *cuda_stream);
int sn_slab_stage(sn_ctx *ctx, int stage, int half_phase);
int sn_slab_buffer(sn_ctx *ctx, int which, void **ptr /* host; receives a DEVICE pointer */, int64_t *elems /* complex64 */);
int sn_slab_pack(sn_ctx *ctx, int what /* SN_SLAB_PSI_A or SN_SLAB_HS_A */, int unpack);
int sn_slab_exchange_local(sn_ctx **ctxs /* host, nranks contexts in rank order */, int nranks, int what, int to_a);
int sn_slab_local_norm(sn_ctx *ctx, double *sum_abs2_dv /* host: this rank's part of the norm */);

/* ---- allocation-free entry point (no context, no workspace) ----
 * For callers that cannot allocate device memory at the call site (code under CUDA graph capture, tight serving loops,
 * harnesses that forbid cudaMalloc): norm = dv * sum_{i < n_cells} |psi_i|^2 of a complex64 DEVICE array (the norm of the
 * diagnostics, S12: fp32 data, fp64 accumulation), written to the DEVICE double *norm_out.  Enqueued on cuda_stream
 * (two kernel launches), returns without synchronising; runs on the device that owns psi and restores the caller's
 * current device.  Calls no cudaMalloc / cudaFree / allocating routine: its scratch (one partial sum per 8192 cells) is a
 * file-scope __device__ array of SN_STATIC_NORM_SCRATCH_DOUBLES doubles = 256 KiB that every GPU which loads the library
 * holds until the process exits.  Hence the limit: n_cells <= SN_STATIC_NORM_MAX_CELLS = 2^28 (a 2 GiB state; 512^3 is
 * 2^27), beyond it SN_ERR_TOO_LARGE and nothing is launched.  n_cells = 0 gives 0.  The sum is taken in a fixed order:
 * bitwise reproducible.  ALL calls on a device share the scratch array: each call overwrites the slots it reads (nothing
 * needs clearing between calls), but two calls that OVERLAP on the GPU -- different streams, concurrently replayed
 * graphs -- race on it and give wrong sums: keep calls on one stream or order them with events. */
#define SN_STATIC_NORM_SCRATCH_DOUBLES 32768
#define SN_STATIC_NORM_MAX_CELLS ((int64_t)1 << 28)
int sn_norm_static(const void *psi /* DEVICE, n_cells complex64 */, int64_t n_cells, double dv,
                   double *norm_out /* DEVICE, 1 double */, void *cuda_stream);

int sn_destroy(sn_ctx *ctx);

/* Text for an error code; for SN_ERR_CUDA the last CUDA error string seen by this thread. */
const char *sn_strerror(int code);

/* Number of kernels this context has launched since creation (for bench.py's gpu_launches). */
int64_t sn_launch_count(const sn_ctx *ctx);

/* ---- per-launch timing (bench.py's roofline) ----
 * With profiling enabled every kernel launch is bracketed by a cudaEvent pair on the context's
 * stream; sn_profile_read synchronises and returns, per pass kind, the summed device time in
 * milliseconds and the number of launches since the last reset.  Pass kinds (index):
 *   0 S_FFT  strided-axis plain transform          1 S_KIN  strided-axis forward-phase-inverse
 *   2 S_KDIAG strided-axis kinetic-energy sum      3 H_NLKIN axis-0 c2r + nonlinear phase + kinetic
 *   4 H_R2C  axis-0 density + packed r2c           5 H_POT  axis-0 c2r -> phi (test hook)
 *   6 H_DIAG axis-0 c2r + energy sums              7 X_FFT  contiguous-axis plain transform
 *   8 X_KIN  contiguous-axis forward-phase-inverse 9 X_POISSON contiguous-axis forward-D/(C-k^2)-inverse
 *  10 X_KDIAG contiguous-axis kinetic-energy sum  11 H_SRC axis-0 source gamma rho + beta lap rho (eq. (12))
 *  12 H_BOHM axis-0 Bohm phase (eq. (15))       13 H_R2C_MC weighted density of coupled components + packed r2c
 *  14 H_NL_MC axis-0 c2r + nonlinear phases of coupled components
 *  15 R_STEPS the cluster-resident kernel: one launch = ALL steps of an sn_step call (small square 2D grids) */
#define SN_NUM_PASS_KINDS 16
int sn_profile(sn_ctx *ctx, int enable);
int sn_profile_read(sn_ctx *ctx, double *ms_by_kind /* host, 16 */, int64_t *launches_by_kind /* host, 16 */,
                    int reset);

/* ---- test hooks (used by the acceptance tests, not by users) ---- */

/* Switches for A/B runs and tests (none changes results beyond rounding).  Takes effect from the next call;
 * synchronises the stream.
 *   SN_OPT_GRAPH    1 (default): sn_step(n >= 4) on grids of <= 2^24 cells replays a captured CUDA graph of the
 *                   interior step; 0: plain stream launches.
 *   SN_OPT_DISPATCH 0 (default): each pass runs the kernel measured fastest for its line length; 1: first-path
 *                   kernels (sn_kernels.cu) everywhere; 2: TMA-pipelined kernels (sn_pipe.cu) wherever instantiated. */
#define SN_OPT_GRAPH 1
#define SN_OPT_DISPATCH 2
#define SN_OPT_GRAPH_STEPS 3 /* interior steps captured per replayed graph, 1 ... 64 (launch-bound grids; default 8; the interior
                              * steps a call leaves over replay a one-step graph, the closing step runs as plain launches) */
/*   SN_OPT_RESIDENT 1 (default): sn_step / sn_step_order4 on a complex64 2D grid with n0 == n1 in {64, 128}, local
 *                   nonlinearities and / or an external potential (no sn_set_bohm / _source_tables in effect), the default
 *                   SN_OPT_DISPATCH and at most 32 (128^2) / 256 (64^2) ensemble members runs as ONE launch of the
 *                   cluster-resident kernel:
 *                   the state stays in the distributed shared memory of a cluster of 8 CTAs for all n steps of the
 *                   call (one cluster per member); 0: the pass kernels.  sn_create checks once that the device can hold
 *                   such a cluster (cudaOccupancyMaxActiveClusters); where it cannot, the option stays 0 and the pass
 *                   kernels serve the context.  Same schedule and arithmetic; the density is
 *                   transformed as a complex field there, so the two paths agree to rounding, not bit for bit. */
#define SN_OPT_RESIDENT 4
int sn_set_option(sn_ctx *ctx, int option, int value);

/* In-place d-dimensional FFT of the internal state: direction +1 forward (e^{-i k x}, unscaled),
 * -1 inverse (scaled by 1/prod N).  Uses the same line-FFT engine as sn_step. */
int sn_debug_fft(sn_ctx *ctx, int direction);

/* phi (float32, prod(dims) values, same layout as psi) solving eq. (2) for the current state.  A host destination
 * needs SN_FEAT_STAGING. */
int sn_debug_potential(sn_ctx *ctx, float *phi_out, int dst_on_device);

#ifdef __cplusplus
}
#endif
#endif /* SN_H */
