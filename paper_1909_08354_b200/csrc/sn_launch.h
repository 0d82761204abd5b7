// sn_launch.h -- internal interface between the scheduler (sn_api.cu) and the per-length kernel
// translation units (sn_kernels.cu compiled once per line length with -DSN_LEN=N).
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>

namespace snk {

enum PassKind {
    P_S_FFT = 0,   // strided axis: plain c2c transform (dir, hilo, scale)
    P_S_KIN,       // strided axis: forward -> kinetic phase -> inverse            (S1-S3 per axis)
    P_S_KDIAG,     // strided axis: forward, accumulate sum k_a^2 |psi^|^2         (S12)
    P_H_NLKIN,     // axis 0: c2r of phi^ -> nonlinear phase -> fwd -> phase -> inv (S7,S8,S1-S3)
    P_H_R2C,       // axis 0: rho = |psi|^2 -> packed r2c -> half spectrum          (S4,S5)
    P_H_POT,       // axis 0: c2r of phi^ -> phi (float) out                        (test hook)
    P_H_DIAG,      // axis 0: c2r of phi^ -> sums of rho, phi rho, F(rho)           (S12)
    P_X_FFT,       // contiguous axis: plain c2c transform
    P_X_KIN,       // contiguous axis: forward -> kinetic phase -> inverse
    P_X_POISSON,   // contiguous axis of the half spectrum: forward -> D/(C-k^2) -> inverse (S5-S7)
    P_X_KDIAG,     // contiguous axis: forward, accumulate sum k_x^2 |psi^|^2
    P_H_SRC,       // axis 0: c2r of F[lap rho] -> s = gamma rho + beta lap rho -> packed r2c   (eq. (12), NEXT-1)
    P_H_BOHM,      // axis 0: c2r of F[lap sqrt(rho)] -> psi *= exp(-i s c_B lap sqrt(rho)/(2 sqrt(rho)))  (eq. (15))
    P_H_R2C_MC,    // axis 0, coupled components: rho = sum_c w_c |psi_c|^2 -> packed r2c
    P_H_NL_MC,     // axis 0, coupled components: c2r of phi^ -> psi_c *= exp(-i s (B_c phi + sum_c' g_cc' rho_c')) for every c
    P_R_STEPS      // cluster-resident kernel: ALL steps of an sn_step(n) call on a small 2D grid in one launch (sn_resident.cu)
};

// Coupled wave functions (NEXT-4b; reading Q18 of DESIGN.md): up to 4 components, stored one after the other
// (component c at data + c * comp_stride); half-angle coefficients like NLParams.
struct MCParams {
    int ncomp;
    long long comp_stride; // complex elements between components
    float w[4];            // source weights of eq. (2')
    float hb[4];           // -s/2 * B_c
    float hg[4][4];        // -s/2 * g_cc'
};

// Nonlinear phase psi *= exp(-i dtau (B phi + sum_j g_j rho^j)), stored as HALF-angle
// coefficients: theta/2 = hb * phi + rho (hg[0] + rho (hg[1] + rho (hg[2] + rho hg[3]))).
struct NLParams {
    float hb;
    float hg[4];
    float fg[4]; // F(rho) = rho^2 (fg[0] + rho (fg[1] + ...)), fg[j] = g_j/(j+2)   (diagnostics)
    // NEXT-1 terms (eq. (15),(16) PAPER.md:102-107), all zero / off by default (flags == 0):
    int flags;        // bit 0: logarithmic / power-law terms present; bit 1: external potential present
    float hlog, hpow; // half-angle coefficients -dtau/2 * g_log, -dtau/2 * g_pow
    float floor_, ppow; // rho_f = max(rho, floor_); rho_f^ppow
    float hv;         // -dtau/2 (multiplies the external potential)
    float flog, fpow; // diagnostics: g_log, g_pow/(ppow+1)
};

struct PassArgs {
    int kind;
    int dir;  // +1 forward, -1 inverse (P_S_FFT / P_X_FFT)
    int hilo; // 1: hi/lo twiddles (psi transforms); 0: plain (density / potential transforms)
    float2 *data;      // DEVICE: array transformed in place (psi, or the half spectrum)
    float2 *hs;        // DEVICE: half-spectrum buffer (P_H_* kinds)
    long long row_stride;   // elements between consecutive points of a line (strided kinds)
    long long outer_stride; // elements between outer blocks
    int ncols;              // contiguous columns per outer block
    int n_outer;
    int axis;               // strided kinds: 0 or 1 (which view of the array the lines run along)
    int nlines;             // contiguous kinds: number of lines (even)
    const float4 *tw;       // DEVICE: twiddle table for this length
    const float4 *phase;    // DEVICE: kinetic phase table (hi/lo, includes 1/N)
    const float *ksq;       // DEVICE: k_a^2 per index of this axis
    const float2 *ksq2;     // DEVICE: P_X_POISSON: k_x^2 per index of the contiguous axis as hi + lo
    const float2 *dko;      // DEVICE: P_X_POISSON: per line, C - (other axes' k^2) (lap: -(other axes' k^2)) as hi + lo
    float scale;            // P_*_FFT: output scale (1/N on inverse)
    float pscale;           // P_X_POISSON: D * 0.5 / prod(N)   (0.5 from the packed r2c)
    NLParams nl;
    float *phi_out;         // DEVICE: P_H_POT
    const float *vext;      // DEVICE: external potential (same layout as psi, float) or nullptr
    const float2 *bg;       // DEVICE: P_H_SRC source tables of eq. (12), interleaved (beta, gamma) per cell, layout of psi
    int lap;                // P_X_POISSON: multiply by d * pscale instead of pscale/d, d = (dko - ksq2) = -k^2
    int sqrt_rho;           // P_H_R2C: transform sqrt(rho) instead of rho (Bohm term)
    float hbohm, sfloor;    // P_H_BOHM: half angle = hbohm * W / max(sqrt(rho), sfloor), hbohm = -s c_B/4; floor of sqrt(rho)
    double *diag;           // DEVICE: accumulators
    int nl_slot;            // which nonlinear sub-step the coefficients in `nl` belong to (scheduler bookkeeping)
    MCParams mc;            // P_H_R2C_MC / P_H_NL_MC
    cudaStream_t stream;
};

// cudaFuncSetAttribute(MaxDynamicSharedMemorySize) is needed once per kernel and device, not per launch
// (it costs ~1 us of host time per call); the set of kernels already configured lives in sn_api.cu.
bool smem_attr_done(const void *kernel);
void smem_attr_mark(const void *kernel);

// Returns cudaError_t as int.  Explicitly instantiated for N in {64,...,4096}.
template <int N>
int launch_pass(const PassArgs &a);

// ---- pipelined (persistent, TMA-fed) variants of the hot passes: sn_pipe.cu ----
// One CTA per SM (512 threads, 64 KB tiles for N = 2^n; 256 threads, 48 KB tiles for N = 3*2^a) walks over the
// tiles of a pass; tiles are moved by the TMA unit between HBM and a ring of shared-memory stages, so loads and
// stores of neighbouring tiles overlap the butterflies of the current one.  Kinds served: P_S_FFT, P_S_KIN,
// P_H_NLKIN, P_H_R2C, P_X_KIN, P_X_POISSON.  Tensor maps view an array as [outer][row][2*cols floats]; a box is
// 2*CPW complex wide (CPW = pipe_cpw(N) column pairs: 128, 64, 32 or 16 bytes) and swizzled over exactly that width.
struct PipeArgs {
    CUtensorMap m_data;   // psi (or the half spectrum for P_S_FFT): box {4*CPW floats, pipe_box_rows(N) rows, 1}
    CUtensorMap m_hs;     // P_H_*: half spectrum [N/2+1 rows][2*cols floats]: box {4*CPW, pipe_box_rows(N/2) rows, 1}
    CUtensorMap m_hs_row; // P_H_*: same tensor, box {4*CPW, 1, 1} (the row N/2)
    CUtensorMap m_bg;     // P_H_SRC: the interleaved (beta, gamma) table, same geometry as m_data
    PassArgs a;
    int n_tiles;          // tiles of this pass
    int tiles_per_outer;  // strided kinds: column blocks per outer index
    int grid;             // CTAs to launch (<= number of SMs)
    int *sched;           // device: {next tile, CTAs finished} of the dynamically scheduled kernels (k_pipe_haxis); both 0 between launches
};

// geometry of the pipelined kernels, shared by the scheduler (tensor maps, tile counts) and sn_pipe.cu:
// 8 points per thread and 512 threads for N = 2^n; 12 points per thread and 256 threads for N = 3*2^a
__host__ __device__ constexpr int pipe_ppt(int N) { return N % 3 == 0 ? 12 : 8; }
// N = 384 (BASELINE.json's sweep size): 12 warps of 168 registers (12 line pairs, 72 KB tiles, 64-byte rows) instead of 8
// warps of ~195: H_NLKIN 0.613 -> 0.460 ms.  Measured for the other 3*2^a lengths and not taken: 192^3 0.236 -> 0.221
// ms/step, 768^3 16.8 -> 18.2 (6 groups: 32-byte rows instead of 64), N = 96 does not fit (48 groups: 2 x 114 KB stages).
#ifndef SN_PIPE_THREADS_384
#define SN_PIPE_THREADS_384 384 // 256 = the round-1 geometry (A/B builds)
#endif
__host__ __device__ constexpr int pipe_threads(int N) { return N == 384 ? SN_PIPE_THREADS_384 : N % 3 == 0 ? 256 : 512; }
__host__ __device__ constexpr int pipe_groups(int N) { return pipe_threads(N) / (N / pipe_ppt(N)); } // line pairs per tile
__host__ __device__ constexpr int pipe_cpw(int N) // largest power of two <= 8 that divides the group count
{
    int c = 8;
    while (pipe_groups(N) % c) c /= 2;
    return c;
}
__host__ __device__ constexpr int pipe_box_rows(int rows) // largest divisor of `rows` that is <= 256 (rows = 2^a 3^b)
{
    int r = rows;
    while (r > 256) r = (r % 2 == 0) ? r / 2 : r / 3;
    return r;
}

// true when launch_pipe<N> can serve this kind/geometry (whether it is also the faster choice is decided per line
// length in sn_api.cu); otherwise launch_pass<N>
inline bool pipe_supported(int N, int kind, long long ncols, long long nlines)
{
    // 3*2^a lengths: measured at 384^3, the pipelined CTA (12 points per thread: 12 warps of 168 registers at N = 384, 8
    // warps of ~195 elsewhere) only beats the first-path kernels (2-3 CTAs per SM) for the axis-0 passes -- H_NLKIN 0.46
    // vs 1.24 ms, H_R2C 0.199 vs 0.222 (N = 384) -- and loses for the others (S_KIN 0.49 vs 0.31, X_KIN 0.44 vs 0.28,
    // X_POISSON 0.21 vs 0.15, S_FFT 0.11 vs 0.09 ms): those stay first-path even under SN_OPT_DISPATCH = 2
    if (N % 3 == 0 && kind != P_H_NLKIN && !(N == 384 && kind == P_H_R2C)) return false;
    if (N < 64) return false; // 32-point lines: first-path kernels only (no pipelined instantiation)
    switch (kind) {
    case P_S_FFT:
    case P_S_KIN:
    case P_H_NLKIN:
    case P_H_R2C:
    case P_H_SRC:
    case P_H_BOHM:
        return ncols % (2 * pipe_groups(N)) == 0; // a tile is 2 G columns wide
    case P_X_KIN:
    case P_X_POISSON:
        return nlines % 2 == 0;
    default:
        return false;
    }
}

template <int N>
int launch_pipe(const PipeArgs &a);

// ---- complex128 path (sn_kernels_f64.cu; the precision the paper benchmarked) ----
// Same pass kinds and geometry fields as PassArgs; a double2 point is one complex128 value.
struct NLParamsD {
    double hb;     // -s B: theta = hb phi + rho (hg[0] + rho (hg[1] + ...)), psi *= exp(i theta)
    double hg[4];  // -s g_j
    double fg[4];  // g_j/(j+2)   (diagnostics: F(rho) = rho^2 (fg[0] + rho (fg[1] + ...)))
};
struct PassArgsD {
    int kind, dir;
    double2 *data;          // DEVICE: array transformed in place (psi, or the half spectrum)
    double2 *hs;            // DEVICE: half-spectrum buffer (P_H_* kinds)
    long long row_stride, outer_stride;
    int ncols, n_outer, axis, nlines;
    const double2 *tw;      // DEVICE: twiddles exp(-2 pi i r kp/(NS R)), table layout of the complex64 engine
    const double2 *phase;   // DEVICE: kinetic phase exp(i A k^2 s)/N per index of this axis
    const double *ksq;      // DEVICE: k_a^2 per index of this axis
    const double *dko;      // DEVICE: P_X_POISSON: per line, C - (other axes' k^2) (lap: -(other axes' k^2))
    double scale;           // P_*_FFT: output scale (1/N on inverse)
    double pscale;          // P_X_POISSON: D * 0.5 / prod(N)
    int lap;
    NLParamsD nl;
    double *phi_out;        // DEVICE: P_H_POT
    double *diag;           // DEVICE: accumulators
    cudaStream_t stream;
};
template <int N>
int launch_pass_d(const PassArgsD &a);

// ---- cluster-resident step (sn_resident.cu): small square 2D grids, complex64, hot-path terms only ----
// The state lives in the distributed shared memory of a cluster of RES_CLUSTER CTAs for a whole sn_step(n) call.
constexpr int RES_CLUSTER = 8;
constexpr int RES_PH_SLOTS = 4; // kinetic phase tables a call can use
struct ResidentArgs {
    float2 *psi;              // DEVICE: state, storage [n0][batch][n1]
    long long row_stride;     // elements between consecutive rows of one member (batch * n1)
    int batch;                // ensemble members: one cluster each
    // The call as a program: K(ph_open) then nsub sub-steps [N(nl[nl_of[i % period]]) K(ph_of[i % period])], the last K
    // with ph_last instead.  Strang (sn_step): period 1, K(dtau/2) [N(dtau) K(dtau)]^(n-1) N(dtau) K(dtau/2); the
    // fourth-order composition (sn_step_order4): period 3.
    long long nsub;           // sub-steps of this call (>= 1)
    int period;               // 1 or 3
    int nl_of[3], ph_of[3];   // per position in the period: index into nl[] / into ph[] (the K after that N)
    int ph_open, ph_last;     // phase slots of the opening and of the closing kinetic sweep
    const float4 *tw;         // DEVICE: twiddle table of the (common) line length
    const float4 *ph[RES_PH_SLOTS][2]; // DEVICE: kinetic phase tables [slot][axis] (unused slots: nullptr)
    const float2 *ksq2_1;     // DEVICE: k_1^2 per index of axis 1 as hi + lo
    const float2 *dk0;        // DEVICE: C - k_0^2 as hi + lo per half-spectrum row and member ([n0/2+1][batch])
    float pscale;             // D / (n0 n1)
    const float *vext;        // DEVICE: external potential V(x) (layout of psi, float) or nullptr  (phi_C of eq. (15))
    NLParams nl[3];
    cudaStream_t stream;
};
inline bool resident_supported(int n0, int n1) { return n0 == n1 && (n0 == 64 || n0 == 128); }
template <int N>
int launch_resident(const ResidentArgs &a);
template <int N>
int resident_max_clusters(); // clusters the device can hold at once; <= 0: the kernel cannot run here

// sum |psi|^2 over n complex64 values, accumulated in double into *out (sn_mc_norms)
int launch_norm(const float2 *psi, long long n, double *out, cudaStream_t stream);

// setup helper (not part of a step): bg[i] = (beta[i], gamma[i])
int launch_interleave(const float *beta, const float *gamma, float2 *bg, long long n, cudaStream_t stream);

} // namespace snk
