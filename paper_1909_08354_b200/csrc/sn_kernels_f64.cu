// sn_kernels_f64.cu -- the pass kernels of the split-step path in complex128, compiled once per line length
// (-DSN_LEN=N).  SURVEY.md 8(f) item 3: the paper benchmarked its solver in double precision ("number
// representation of 64 bits"); this is that precision on the same pass structure as the complex64
// path: one pass per axis, each forward -> pointwise -> inverse along that axis alone; packed
// real-to-complex transform of the density along axis 0; eq. (2) solved in a fused pass along the
// contiguous axis of the half spectrum.  Every kernel is "load a tile of lines -> transform in registers / shared
// memory with the pointwise work fused at both ends -> store".
#include "sn_fft_core_f64.cuh"
#include "sn_launch.h"

#ifndef SN_LEN
#error "compile with -DSN_LEN=<line length>"
#endif

namespace snd {

using namespace snk; // pass kinds, PassArgsD

__device__ __forceinline__ double abs2(cd v) { return fma(v.x, v.x, v.y * v.y); }

// psi *= exp(i theta), theta = hb phi + rho poly(rho)   (S8; eq. (1), reading Q3)
// |theta| <= pi/4 (every cell of every config: theta = dtau * O(potential)): the double-precision minimax kernels of the
// Cephes library on [-pi/4, pi/4] (sin x = x + x z S(z), cos x = 1 - z/2 + z^2 C(z), z = x^2; < 1 ulp), no range
// reduction -- a third of the cost of sincos(); otherwise sincos().
__device__ __forceinline__ cd nl_phase(cd psi, double phi, const NLParamsD &nl)
{
    const double rho = abs2(psi);
    const double th = fma(nl.hb, phi, rho * fma(rho, fma(rho, fma(rho, nl.hg[3], nl.hg[2]), nl.hg[1]), nl.hg[0]));
    double s, c;
    if (fabs(th) <= 0.78539816339744830962) {
        const double z = th * th;
        double ps = 1.58962301576546568060e-10;
        ps = fma(ps, z, -2.50507477628578072866e-8);
        ps = fma(ps, z, 2.75573136213857245213e-6);
        ps = fma(ps, z, -1.98412698295895385996e-4);
        ps = fma(ps, z, 8.33333333332211858878e-3);
        ps = fma(ps, z, -1.66666666666666307295e-1);
        double pc = -1.13585365213876817300e-11;
        pc = fma(pc, z, 2.08757008419747316778e-9);
        pc = fma(pc, z, -2.75573141792967388112e-7);
        pc = fma(pc, z, 2.48015872888517045348e-5);
        pc = fma(pc, z, -1.38888888888730564116e-3);
        pc = fma(pc, z, 4.16666666666665929218e-2);
        s = fma(th * z, ps, th);
        c = fma(z * z, pc, fma(-0.5, z, 1.0));
    } else {
        sincos(th, &s, &c);
    }
    return make_double2(fma(psi.x, c, -psi.y * s), fma(psi.x, s, psi.y * c));
}

// block-wide sum of NV doubles, one atomicAdd per block and value
template <int NV>
__device__ __forceinline__ void block_accumulate(double (&v)[NV], double *out)
{
    __shared__ double red[NV][32];
#pragma unroll
    for (int i = 0; i < NV; i++)
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v[i] += __shfl_xor_sync(0xffffffffu, v[i], o);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
    if (lane == 0)
        for (int i = 0; i < NV; i++) red[i][warp] = v[i];
    __syncthreads();
    if (warp == 0) {
#pragma unroll
        for (int i = 0; i < NV; i++) {
            double s = lane < nw ? red[i][lane] : 0.0;
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
            if (lane == 0) atomicAdd(out + i, s);
        }
    }
}

// columns per CTA tile of the strided kernels: 256-thread CTAs (two or three resident per SM: the loads of one overlap
// the butterflies of another -- with one 512-thread CTA per SM the 512^3 passes ran at 22-34 % of DRAM throughput,
// profiles/r02g) with rows of 128 bytes up to N = 256, 64 bytes at 512, 32 bytes (one sector) at 1024 and 2048
#ifndef SN_F64_CP512
#define SN_F64_CP512 4
#endif
__host__ __device__ constexpr int cpd_for(int N)
{
    return N <= 384 ? 8 : (N <= 768 ? SN_F64_CP512 : (N <= 2048 ? 2 : 1));
}
__host__ __device__ constexpr int sthreads(int N) { return cpd_for(N) * (N / ppt_for(N)); }
__host__ __device__ constexpr int sblocks(int N) { return sthreads(N) <= 256 ? 2 : 1; }
// axis-0 kernel: the modes without a psi transform (r2c, potential, diagnostics) fit 85 registers and run three CTAs per
// SM; the nonlinear mode needs its 128 (at 85 it spills 420 bytes, also with phi parked in shared memory: measured with
// -Xptxas -v), and the 12-point engine of the 3*2^a lengths one CTA per SM (240 bytes of spills at 128 registers)
__host__ __device__ constexpr int hblocks(int N, int mode)
{
    return sthreads(N) <= 256 ? (mode == P_H_NLKIN ? (N % 3 == 0 ? 1 : 2) : 3) : 1;
}

// ---------------------------------------------------------------------------- strided axis
// Tile: N rows (points of the line, row_stride elements apart) x CP adjacent columns; thread (t, j): column t,
// points j + T*m.  8 adjacent lanes read/write one 128-byte row segment.
template <int N, int CP, int MODE, int DIR>
__global__ void __launch_bounds__(sthreads(N), sblocks(N)) kd_strided(const PassArgsD p)
{
    extern __shared__ double2 smem_d[];
    constexpr int P = ppt_for(N), T = N / P;
    const int t = threadIdx.x % CP, j = threadIdx.x / CP;
    const int tiles_per_outer = p.ncols / CP;
    const int outer = blockIdx.x / tiles_per_outer, tile = blockIdx.x % tiles_per_outer;
    cd *g = p.data + (long long)outer * p.outer_stride + (long long)tile * CP + t;
    SmemTileD<CP> sm{smem_d, t};

    cd x[P];
#pragma unroll
    for (int m = 0; m < P; m++) x[m] = g[(long long)(j + T * m) * p.row_stride];
    if (MODE == P_S_FFT) {
        fft_line<N, DIR>(x, j, p.tw, sm);
#pragma unroll
        for (int m = 0; m < P; m++) {
            if (DIR < 0) x[m] = make_double2(x[m].x * p.scale, x[m].y * p.scale);
            g[(long long)(j + T * m) * p.row_stride] = x[m];
        }
    } else if (MODE == P_S_KIN) {
        fft_line<N, +1>(x, j, p.tw, sm);
#pragma unroll
        for (int m = 0; m < P; m++) x[m] = cmul<+1>(x[m], __ldg(p.phase + j + T * m));
        fft_line<N, -1>(x, j, p.tw, sm);
#pragma unroll
        for (int m = 0; m < P; m++) g[(long long)(j + T * m) * p.row_stride] = x[m];
    } else { // P_S_KDIAG
        fft_line<N, +1>(x, j, p.tw, sm);
        double v[1] = {0.0};
#pragma unroll
        for (int m = 0; m < P; m++) v[0] = fma(__ldg(p.ksq + j + T * m), abs2(x[m]), v[0]);
        block_accumulate<1>(v, p.diag);
    }
}

// ---------------------------------------------------------------------------- axis 0 ("h") kernels
// Tile: N rows x 2*CP columns; thread (t, j) owns two columns of the tile, S apart.  The two REAL columns of rho / phi
// travel as one complex line z = x + i y (two-for-one trick).  Which two columns are paired is free per kernel -- once
// untangled, column c of the half spectrum holds the spectrum of real column c -- so each mode picks the pairing that
// gives whole 32-byte sectors: the modes that read both psi columns at once (R2C, DIAG, POT) pair 2t with 2t+1 (S = 1,
// 32 contiguous bytes per thread); NLKIN, which transforms one psi column after the other, pairs t with CP + t (S = CP:
// the CP lanes of a row read CP adjacent 16-byte values in each column pass).  Measured at 512^3: NLKIN 2.68 -> 2.49 ms
// with S = CP, R2C 0.73 -> 1.02 ms if it used S = CP too.
//   X[k] = (Z[k] + conj Z[N-k])/2,  Y[k] = (Z[k] - conj Z[N-k])/(2i),  k = 0..N/2;
//   inverse: Z[k] = X[k] + i Y[k] (k <= N/2), Z[N-k] = conj X[k] + i conj Y[k];
// the factor 1/2 is folded into the Poisson multiplier (PassArgsD::pscale).  The half spectrum stores X[k] in column
// of the first and Y[k] in the column of the second real column, row k.
template <int N, int CP, int MODE>
__global__ void __launch_bounds__(sthreads(N), hblocks(N, MODE)) kd_haxis(const PassArgsD p)
{
    extern __shared__ double2 smem_d[];
    constexpr int P = ppt_for(N), T = N / P;
    const int t = threadIdx.x % CP, j = threadIdx.x / CP;
    const long long rs = p.row_stride;
    constexpr int S = MODE == P_H_NLKIN ? CP : 1;              // distance between the thread's two columns
    const long long col = (long long)blockIdx.x * 2 * CP + (S == 1 ? 2 * t : t);
    cd *psi = p.data + col;
    cd *hs = p.hs + col;
    SmemTileD<CP> sm{smem_d, t};

    cd z[P];
    if (MODE == P_H_R2C) {
#pragma unroll
        for (int m = 0; m < P; m++) {
            const long long row = (long long)(j + T * m) * rs;
            z[m] = make_double2(abs2(psi[row]), abs2(psi[row + S]));
        }
        fft_line<N, +1>(z, j, p.tw, sm);
        sm.sync();
#pragma unroll
        for (int m = 0; m < P; m++) sm.st(j + T * m, z[m]);
        sm.sync();
#pragma unroll
        for (int m = 0; m <= P / 2; m++) {
            if (m < P / 2 || j == 0) {
                const int k = j + T * m;
                const cd y = sm.ld((N - k) % N);
                hs[(long long)k * rs] = make_double2(z[m].x + y.x, z[m].y - y.y);
                hs[(long long)k * rs + S] = make_double2(z[m].y + y.y, y.x - z[m].x);
            }
        }
        return;
    }

    // c2r of phi^ (S7): z[m] = (phi[col 2t], phi[col 2t+1]) at row j + T m
#pragma unroll
    for (int m = 0; m < P; m++) {
        const int km = j + T * m;
        const int src = m < P / 2 ? km : N - km; // m >= P/2: km >= N/2, mirrored row in [0, N/2]
        const cd u = hs[(long long)src * rs], v = hs[(long long)src * rs + S];
        z[m] = m < P / 2 ? make_double2(u.x - v.y, u.y + v.x) : make_double2(u.x + v.y, v.x - u.y);
    }
    fft_line<N, -1>(z, j, p.tw, sm);

    if (MODE == P_H_POT) {
        double *out = p.phi_out + col;
#pragma unroll
        for (int m = 0; m < P; m++) {
            out[(long long)(j + T * m) * rs] = z[m].x;
            out[(long long)(j + T * m) * rs + S] = z[m].y;
        }
        return;
    }
    if (MODE == P_H_DIAG) {
        double v[3] = {0.0, 0.0, 0.0};
#pragma unroll
        for (int m = 0; m < P; m++) {
            const long long row = (long long)(j + T * m) * rs;
            const double r[2] = {abs2(psi[row]), abs2(psi[row + S])};
            const double ph[2] = {z[m].x, z[m].y};
#pragma unroll
            for (int c = 0; c < 2; c++) {
                v[0] += r[c];
                v[1] = fma(ph[c], r[c], v[1]);
                const double f = fma(r[c], fma(r[c], fma(r[c], p.nl.fg[3], p.nl.fg[2]), p.nl.fg[1]), p.nl.fg[0]);
                v[2] = fma(r[c] * r[c], f, v[2]);
            }
        }
        block_accumulate<3>(v, p.diag);
        return;
    }

    // P_H_NLKIN (S8, S1-S3 along axis 0): nonlinear phase with phi, then forward -> kinetic phase -> inverse,
    // one column after the other (a column is one complex128 line)
#pragma unroll
    for (int c = 0; c < 2; c++) {
        cd x[P];
#pragma unroll
        for (int m = 0; m < P; m++)
            x[m] = nl_phase(psi[(long long)(j + T * m) * rs + c * S], c == 0 ? z[m].x : z[m].y, p.nl);
        fft_line<N, +1>(x, j, p.tw, sm);
#pragma unroll
        for (int m = 0; m < P; m++) x[m] = cmul<+1>(x[m], __ldg(p.phase + j + T * m));
        fft_line<N, -1>(x, j, p.tw, sm);
#pragma unroll
        for (int m = 0; m < P; m++) psi[(long long)(j + T * m) * rs + c * S] = x[m];
    }
}

// ---------------------------------------------------------------------------- contiguous axis
// A group of T = N/P threads owns one line; lanes are consecutive j, so a warp's access is one contiguous
// 512-byte run of the line.
__host__ __device__ constexpr int xthreads(int N) { return N / ppt_for(N) >= 256 ? N / ppt_for(N) : 256; }

template <int N, int MODE, int DIR>
__global__ void __launch_bounds__(xthreads(N)) kd_contig(const PassArgsD p)
{
    extern __shared__ double2 smem_d[];
    constexpr int P = ppt_for(N), T = N / P, G = xthreads(N) / T;
    const int j = threadIdx.x % T, grp = threadIdx.x / T;
    const long long line = (long long)blockIdx.x * G + grp;
    const bool active = line < p.nlines;
    if (MODE != P_X_KDIAG && !active) return;
    cd *l = p.data + (active ? line : 0) * N;
    SmemLineD<T> sm{smem_d + grp * N, 1 + grp, G == 1};

    cd x[P];
#pragma unroll
    for (int m = 0; m < P; m++) x[m] = l[j + T * m];
    if (MODE == P_X_FFT) {
        fft_line<N, DIR>(x, j, p.tw, sm);
#pragma unroll
        for (int m = 0; m < P; m++) {
            if (DIR < 0) x[m] = make_double2(x[m].x * p.scale, x[m].y * p.scale);
            l[j + T * m] = x[m];
        }
    } else if (MODE == P_X_KIN) {
        fft_line<N, +1>(x, j, p.tw, sm);
#pragma unroll
        for (int m = 0; m < P; m++) x[m] = cmul<+1>(x[m], __ldg(p.phase + j + T * m));
        fft_line<N, -1>(x, j, p.tw, sm);
#pragma unroll
        for (int m = 0; m < P; m++) l[j + T * m] = x[m];
    } else if (MODE == P_X_POISSON) {
        // eq. (2) in Fourier space: phi^ = D rho^/(C - k^2); C == 0: phi^(k=0) = 0; lap: -k^2 rho^
        fft_line<N, +1>(x, j, p.tw, sm);
        const double dk = __ldg(p.dko + line);
#pragma unroll
        for (int m = 0; m < P; m++) {
            const double d = dk - __ldg(p.ksq + j + T * m);
            const double gm = p.lap ? d * p.pscale : (d == 0.0 ? 0.0 : p.pscale / d);
            x[m] = make_double2(x[m].x * gm, x[m].y * gm);
        }
        fft_line<N, -1>(x, j, p.tw, sm);
#pragma unroll
        for (int m = 0; m < P; m++) l[j + T * m] = x[m];
    } else { // P_X_KDIAG
        fft_line<N, +1>(x, j, p.tw, sm);
        double v[1] = {0.0};
#pragma unroll
        for (int m = 0; m < P; m++) v[0] = fma(__ldg(p.ksq + j + T * m), abs2(x[m]), v[0]);
        if (!active) v[0] = 0.0;
        block_accumulate<1>(v, p.diag);
    }
}

// ---------------------------------------------------------------------------- launchers

template <class K>
static int launch_kernel(K kern, unsigned grid, int threads, size_t smem_bytes, const PassArgsD &a)
{
    if (smem_bytes > 40 * 1024 && !smem_attr_done(reinterpret_cast<const void *>(kern))) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_bytes);
        if (e != cudaSuccess) return (int)e;
        smem_attr_mark(reinterpret_cast<const void *>(kern));
    }
    kern<<<grid, threads, smem_bytes, a.stream>>>(a);
    return (int)cudaGetLastError();
}

} // namespace snd

namespace snk {

template <int N>
int launch_pass_d(const PassArgsD &a)
{
    using namespace snd;
    constexpr int CP = cpd_for(N), T = N / ppt_for(N);
    constexpr int ST = CP * T;
    constexpr size_t SSMEM = (size_t)N * CP * 16; // one double2 per point and column
    constexpr int XT = xthreads(N), G = XT / T;
    constexpr size_t XSMEM = (size_t)N * G * 16;
    switch (a.kind) {
    case P_S_FFT:
    case P_S_KIN:
    case P_S_KDIAG: {
        const unsigned grid = (unsigned)((long long)a.n_outer * (a.ncols / CP));
        if (a.kind == P_S_KIN) return launch_kernel(kd_strided<N, CP, P_S_KIN, +1>, grid, ST, SSMEM, a);
        if (a.kind == P_S_KDIAG) return launch_kernel(kd_strided<N, CP, P_S_KDIAG, +1>, grid, ST, SSMEM, a);
        return a.dir > 0 ? launch_kernel(kd_strided<N, CP, P_S_FFT, +1>, grid, ST, SSMEM, a)
                         : launch_kernel(kd_strided<N, CP, P_S_FFT, -1>, grid, ST, SSMEM, a);
    }
    case P_H_NLKIN:
    case P_H_R2C:
    case P_H_POT:
    case P_H_DIAG: {
        const unsigned grid = (unsigned)(a.ncols / (2 * CP));
        if (a.kind == P_H_NLKIN) return launch_kernel(kd_haxis<N, CP, P_H_NLKIN>, grid, ST, SSMEM, a);
        if (a.kind == P_H_R2C) return launch_kernel(kd_haxis<N, CP, P_H_R2C>, grid, ST, SSMEM, a);
        if (a.kind == P_H_POT) return launch_kernel(kd_haxis<N, CP, P_H_POT>, grid, ST, SSMEM, a);
        return launch_kernel(kd_haxis<N, CP, P_H_DIAG>, grid, ST, SSMEM, a);
    }
    case P_X_FFT:
    case P_X_KIN:
    case P_X_POISSON:
    case P_X_KDIAG: {
        const unsigned grid = (unsigned)((a.nlines + G - 1) / G);
        if (a.kind == P_X_KIN) return launch_kernel(kd_contig<N, P_X_KIN, +1>, grid, XT, XSMEM, a);
        if (a.kind == P_X_POISSON) return launch_kernel(kd_contig<N, P_X_POISSON, +1>, grid, XT, XSMEM, a);
        if (a.kind == P_X_KDIAG) return launch_kernel(kd_contig<N, P_X_KDIAG, +1>, grid, XT, XSMEM, a);
        return a.dir > 0 ? launch_kernel(kd_contig<N, P_X_FFT, +1>, grid, XT, XSMEM, a)
                         : launch_kernel(kd_contig<N, P_X_FFT, -1>, grid, XT, XSMEM, a);
    }
    default:
        return (int)cudaErrorInvalidValue;
    }
}

template int launch_pass_d<SN_LEN>(const PassArgsD &a);

} // namespace snk
