// sn_kernels.cu -- the pass kernels of the split-step path, compiled once per line length
// (-DSN_LEN=N).  Every kernel is "load a tile of lines -> transform in registers/shared memory
// with pointwise work fused at both ends -> store"; no standalone elementwise kernel exists.
//
// Pass structure of one Strang step (operations S1-S12 of SURVEY.md 8(a)):
//   the kinetic operator exp(i A k^2 s) = prod_a exp(i A k_a^2 s) is separable, so it is applied
//   as ONE pass per axis, each doing forward FFT -> phase -> inverse FFT along that axis alone.
//   The density transform is a packed real-to-complex transform along axis 0 (two real lines
//   in one complex line); eq. (2) is solved in a fused forward -> D/(C-k^2) -> inverse pass
//   along the contiguous axis of the half spectrum.
#include "sn_fft_core.cuh"
#include "sn_launch.h"
#include "sn_pointwise.cuh"

#ifndef SN_LEN
#error "compile with -DSN_LEN=<line length>"
#endif

namespace snk {

// block-wide sum of up to 3 doubles, one atomicAdd per block and value
template <int NV>
__device__ __forceinline__ void block_accumulate(double (&v)[NV], double *out)
{
    __shared__ double red[NV][32];
#pragma unroll
    for (int i = 0; i < NV; i++) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v[i] += __shfl_xor_sync(0xffffffffu, v[i], o);
    }
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

// column pairs per CTA tile: 512-point lines run as two 256-thread CTAs per SM (measured 15-30 % faster
// than one 512-thread CTA: the second CTA's loads overlap the first one's butterflies); 384-point lines with
// 128-byte rows (CP = 8; 384^3 step 2.075 -> 2.036 ms against CP = 4)
__host__ __device__ constexpr int cp_for(int N) { return N <= 384 ? 8 : (N <= 1024 ? 4 : (N <= 2048 ? 2 : 1)); }
__host__ __device__ constexpr int sthreads(int N) { return cp_for(N) * (N / ppt_for(N)); }
// resident CTAs per SM asked of the compiler: 128-thread CTAs (N = 384 and N <= 128) run three (measured at 384^3:
// S_KIN 0.358 -> 0.329 ms against two), 256-thread CTAs two, 512-thread CTAs one
__host__ __device__ constexpr int sblocks(int N) { return sthreads(N) <= 128 ? 3 : (sthreads(N) <= 256 ? 2 : 1); }

// ---------------------------------------------------------------------------- strided axis
// Tile: N rows (points of the line, `row_stride` elements apart) x 2*CP adjacent columns.
// Thread (t, j): column pair t, points j + T*m.  All global accesses are 128-bit; 8 adjacent
// lanes read/write one 128-byte row segment.

template <int N, int CP, int MODE, int DIR, bool HILO>
__global__ void __launch_bounds__(sthreads(N), sblocks(N)) k_strided(const PassArgs p)
{
    extern __shared__ float4 smem[];
    constexpr int P = ppt_for(N), T = N / P;
    const int t = threadIdx.x % CP, j = threadIdx.x / CP;
    const int tiles_per_outer = p.ncols / (2 * CP);
    const int outer = blockIdx.x / tiles_per_outer, tile = blockIdx.x % tiles_per_outer;
    float4 *g4 = reinterpret_cast<float4 *>(p.data + (long long)outer * p.outer_stride + (long long)tile * 2 * CP) + t;
    const long long rs4 = p.row_stride / 2;
    SmemTile<CP> sm{smem, t};

    float2 a[P], b[P];
#pragma unroll
    for (int m = 0; m < P; m++) {
        const float4 v = g4[(long long)(j + T * m) * rs4];
        a[m] = lo2(v);
        b[m] = hi2(v);
    }
    if (MODE == P_S_FFT) {
        fft_pair<N, DIR, HILO>(a, b, j, p.tw, sm);
        const float s = p.scale;
#pragma unroll
        for (int m = 0; m < P; m++) {
            if (DIR < 0) {
                a[m].x *= s; a[m].y *= s; b[m].x *= s; b[m].y *= s;
            }
            g4[(long long)(j + T * m) * rs4] = pack4(a[m], b[m]);
        }
    } else if (MODE == P_S_KIN) {
        fft_pair<N, +1, true>(a, b, j, p.tw, sm);
#pragma unroll
        for (int m = 0; m < P; m++) {
            const float4 ph = __ldg(p.phase + j + T * m);
            a[m] = twmul<+1, true>(a[m], ph);
            b[m] = twmul<+1, true>(b[m], ph);
        }
        fft_pair<N, -1, true>(a, b, j, p.tw, sm);
#pragma unroll
        for (int m = 0; m < P; m++) g4[(long long)(j + T * m) * rs4] = pack4(a[m], b[m]);
    } else { // P_S_KDIAG
        fft_pair<N, +1, true>(a, b, j, p.tw, sm);
        double v[1] = {0.0}; // fp32 data, fp64 accumulation from the first addition on (S12)
#pragma unroll
        for (int m = 0; m < P; m++) v[0] += (double)__ldg(p.ksq + j + T * m) * ((double)abs2(a[m]) + (double)abs2(b[m]));
        block_accumulate<1>(v, p.diag);
    }
}

// ---------------------------------------------------------------------------- axis 0 ("h") kernels
// Tile: N rows x 4*CP columns = two half-tiles of CP column pairs.  Thread (t, j) owns column
// pairs t (columns 2t, 2t+1) and CP + t of the tile.  Two REAL columns 2t, 2t+1 travel as one
// complex line re + i im, so the four real columns of a thread are one fft_pair.
//
// Packed real transforms (two-for-one trick): Z = FFT(x + i y), x, y real =>
//   X[k] = (Z[k] + conj Z[N-k])/2,  Y[k] = (Z[k] - conj Z[N-k])/(2i),  k = 0..N/2;
// inverse: Z[k] = X[k] + i Y[k] (k <= N/2), Z[N-k] = conj X[k] + i conj Y[k].
// The factor 1/2 is folded into the Poisson multiplier (PassArgs::pscale).

template <int N, int CP, class SM>
__device__ __forceinline__ void c2r_potential(const PassArgs &p, const float4 *hs4, long long rs4, int t, int j,
                                              float2 (&fa)[ppt_for(N)], float2 (&fb)[ppt_for(N)], SM &sm)
{
    constexpr int P = ppt_for(N), T = N / P;
#pragma unroll
    for (int m = 0; m < P; m++) {
        const int km = j + T * m;
        const int src = m < P / 2 ? km : N - km; // m >= P/2: km >= N/2, mirrored row in [0, N/2]
        const float4 u = hs4[(long long)src * rs4 + t];
        const float4 v = hs4[(long long)src * rs4 + CP + t];
        if (m < P / 2) {
            fa[m] = make_float2(u.x - u.w, u.y + u.z);
            fb[m] = make_float2(v.x - v.w, v.y + v.z);
        } else {
            fa[m] = make_float2(u.x + u.w, u.z - u.y);
            fb[m] = make_float2(v.x + v.w, v.z - v.y);
        }
    }
    fft_pair<N, -1, false>(fa, fb, j, p.tw, sm);
    // now fa[m] = (phi[col 2t], phi[col 2t+1]), fb[m] = same for column pair CP+t, at row j+T*m
}

template <int N, int CP, int MODE>
__global__ void __launch_bounds__(sthreads(N), sblocks(N)) k_haxis(const PassArgs p)
{
    extern __shared__ float4 smem[];
    constexpr int P = ppt_for(N), T = N / P;
    const int t = threadIdx.x % CP, j = threadIdx.x / CP;
    const long long rs4 = p.row_stride / 2;
    const long long col4 = (long long)blockIdx.x * 2 * CP; // first column pair of the tile
    float4 *psi4 = reinterpret_cast<float4 *>(p.data) + col4;
    float4 *hs4 = reinterpret_cast<float4 *>(p.hs) + col4;
    SmemTile<CP> sm{smem, t};

    if (MODE == P_H_R2C || MODE == P_H_SRC) {
        float2 a[P], b[P];
        if (MODE == P_H_SRC) {
            // eq. (12): the half spectrum holds F[lap rho]; bring it back along axis 0 and form the source
            // s = gamma(x) rho + beta(x) lap rho for the thread's four real columns, then transform s like rho
            c2r_potential<N, CP>(p, hs4, rs4, t, j, a, b, sm);
            const float4 *bg4 = reinterpret_cast<const float4 *>(p.bg) + col4; // (beta, gamma) of two adjacent columns
#pragma unroll
            for (int m = 0; m < P; m++) {
                const long long row = (long long)(j + T * m) * rs4;
                const float4 u = psi4[row + t], v = psi4[row + CP + t];
                const float4 q0 = __ldg(bg4 + row + t), q1 = __ldg(bg4 + row + CP + t);
                a[m] = make_float2(fmaf(q0.y, abs2(lo2(u)), q0.x * a[m].x), fmaf(q0.w, abs2(hi2(u)), q0.z * a[m].y));
                b[m] = make_float2(fmaf(q1.y, abs2(lo2(v)), q1.x * b[m].x), fmaf(q1.w, abs2(hi2(v)), q1.z * b[m].y));
            }
        } else {
#pragma unroll
            for (int m = 0; m < P; m++) {
                const float4 u = psi4[(long long)(j + T * m) * rs4 + t];
                const float4 v = psi4[(long long)(j + T * m) * rs4 + CP + t];
                a[m] = make_float2(abs2(lo2(u)), abs2(hi2(u)));
                b[m] = make_float2(abs2(lo2(v)), abs2(hi2(v)));
                if (p.sqrt_rho) { // Bohm term: the transform of sqrt(rho)
                    a[m] = make_float2(sqrtf(a[m].x), sqrtf(a[m].y));
                    b[m] = make_float2(sqrtf(b[m].x), sqrtf(b[m].y));
                }
            }
        }
        fft_pair<N, +1, false>(a, b, j, p.tw, sm);
        sm.sync();
#pragma unroll
        for (int m = 0; m < P; m++) sm.st(j + T * m, a[m], b[m]);
        sm.sync();
#pragma unroll
        for (int m = 0; m <= P / 2; m++) {
            if (m < P / 2 || j == 0) {
                const int k = j + T * m;
                float2 ya, yb;
                sm.ld((N - k) % N, ya, yb);
                hs4[(long long)k * rs4 + t] = make_float4(a[m].x + ya.x, a[m].y - ya.y, a[m].y + ya.y, ya.x - a[m].x);
                hs4[(long long)k * rs4 + CP + t] =
                    make_float4(b[m].x + yb.x, b[m].y - yb.y, b[m].y + yb.y, yb.x - b[m].x);
            }
        }
        return;
    }

    if (MODE == P_H_R2C_MC) {
        // coupled components (reading Q18): the source of eq. (2') is sum_c w_c |psi_c|^2
        float2 a[P], b[P];
        const long long cs4 = p.mc.comp_stride / 2;
#pragma unroll
        for (int m = 0; m < P; m++) {
            a[m] = make_float2(0.f, 0.f);
            b[m] = make_float2(0.f, 0.f);
            for (int c = 0; c < p.mc.ncomp; c++) {
                const float4 u = psi4[c * cs4 + (long long)(j + T * m) * rs4 + t];
                const float4 v = psi4[c * cs4 + (long long)(j + T * m) * rs4 + CP + t];
                const float w = p.mc.w[c];
                a[m] = make_float2(fmaf(w, abs2(lo2(u)), a[m].x), fmaf(w, abs2(hi2(u)), a[m].y));
                b[m] = make_float2(fmaf(w, abs2(lo2(v)), b[m].x), fmaf(w, abs2(hi2(v)), b[m].y));
            }
        }
        fft_pair<N, +1, false>(a, b, j, p.tw, sm);
        sm.sync();
#pragma unroll
        for (int m = 0; m < P; m++) sm.st(j + T * m, a[m], b[m]);
        sm.sync();
#pragma unroll
        for (int m = 0; m <= P / 2; m++) {
            if (m < P / 2 || j == 0) {
                const int k = j + T * m;
                float2 ya, yb;
                sm.ld((N - k) % N, ya, yb);
                hs4[(long long)k * rs4 + t] = make_float4(a[m].x + ya.x, a[m].y - ya.y, a[m].y + ya.y, ya.x - a[m].x);
                hs4[(long long)k * rs4 + CP + t] =
                    make_float4(b[m].x + yb.x, b[m].y - yb.y, b[m].y + yb.y, yb.x - b[m].x);
            }
        }
        return;
    }

    float2 fa[P], fb[P];
    c2r_potential<N, CP>(p, hs4, rs4, t, j, fa, fb, sm);

    if (MODE == P_H_NL_MC) {
        // psi_c *= exp(-i s (B_c phi + sum_c' g_cc' rho_c')): every rho_c is read before any component is rewritten
        const long long cs4 = p.mc.comp_stride / 2;
        const int M = p.mc.ncomp;
#pragma unroll
        for (int half = 0; half < 2; half++) {
#pragma unroll
            for (int m = 0; m < P; m++) {
                float4 *g4 = psi4 + half * CP + t + (long long)(j + T * m) * rs4;
                const float2 ph = half == 0 ? fa[m] : fb[m];
                float4 v[4];
                float2 rho[4];
#pragma unroll
                for (int c = 0; c < 4; c++)
                    if (c < M) {
                        v[c] = g4[c * cs4];
                        rho[c] = make_float2(abs2(lo2(v[c])), abs2(hi2(v[c])));
                    }
#pragma unroll
                for (int c = 0; c < 4; c++)
                    if (c < M) {
                        float tx = p.mc.hb[c] * ph.x, ty = p.mc.hb[c] * ph.y;
#pragma unroll
                        for (int d = 0; d < 4; d++)
                            if (d < M) {
                                tx = fmaf(p.mc.hg[c][d], rho[d].x, tx);
                                ty = fmaf(p.mc.hg[c][d], rho[d].y, ty);
                            }
                        g4[c * cs4] = pack4(rotate_half_angle(lo2(v[c]), tx), rotate_half_angle(hi2(v[c]), ty));
                    }
            }
        }
        return;
    }

    if (MODE == P_H_POT) {
        float2 *out = reinterpret_cast<float2 *>(p.phi_out) + col4;
#pragma unroll
        for (int m = 0; m < P; m++) {
            out[(long long)(j + T * m) * rs4 + t] = fa[m];
            out[(long long)(j + T * m) * rs4 + CP + t] = fb[m];
        }
        return;
    }
    if (MODE == P_H_DIAG) {
        double s_rho = 0.0, s_pr = 0.0, s_f = 0.0; // fp32 data, fp64 accumulation from the first addition on (S12)
#pragma unroll
        for (int m = 0; m < P; m++) {
            const float4 u = psi4[(long long)(j + T * m) * rs4 + t];
            const float4 v = psi4[(long long)(j + T * m) * rs4 + CP + t];
            const float r[4] = {abs2(lo2(u)), abs2(hi2(u)), abs2(lo2(v)), abs2(hi2(v))};
            const float ph[4] = {fa[m].x, fa[m].y, fb[m].x, fb[m].y};
            float ve[4] = {0.f, 0.f, 0.f, 0.f};
            if (p.nl.flags & 2) {
                const float2 *v2 = reinterpret_cast<const float2 *>(p.vext) + col4 + (long long)(j + T * m) * rs4;
                const float2 e0 = __ldg(v2 + t), e1 = __ldg(v2 + CP + t);
                ve[0] = e0.x; ve[1] = e0.y; ve[2] = e1.x; ve[3] = e1.y;
            }
#pragma unroll
            for (int c = 0; c < 4; c++) {
                s_rho += (double)r[c];
                s_pr += (double)ph[c] * (double)r[c];
                const float f = fmaf(r[c], fmaf(r[c], fmaf(r[c], p.nl.fg[3], p.nl.fg[2]), p.nl.fg[1]), p.nl.fg[0]);
                s_f += (double)(r[c] * r[c]) * (double)f;
                if (p.nl.flags) { // F_log = g_log (rho ln rho_f - rho), F_pow = g_pow rho rho_f^p/(p+1), V rho
                    const float rf = fmaxf(r[c], p.nl.floor_);
                    float e = ve[c];
                    if (p.nl.flog != 0.f) e += p.nl.flog * (logf(rf) - 1.f);
                    if (p.nl.fpow != 0.f) e = fmaf(p.nl.fpow, powf(rf, p.nl.ppow), e);
                    s_f += (double)r[c] * (double)e;
                }
            }
        }
        double v[3] = {s_rho, s_pr, s_f};
        block_accumulate<3>(v, p.diag);
        return;
    }

    if (MODE == P_H_BOHM) { // fa, fb hold W = lap sqrt(rho): rotate psi by -s c_B W/(2 max(sqrt(rho), floor))
#pragma unroll
        for (int half = 0; half < 2; half++) {
            float4 *g4 = psi4 + half * CP + t;
#pragma unroll
            for (int m = 0; m < P; m++) {
                const float4 v = g4[(long long)(j + T * m) * rs4];
                const float2 w = half == 0 ? fa[m] : fb[m];
                const float2 x0 = rotate_half_angle(lo2(v), p.hbohm * w.x / fmaxf(sqrtf(abs2(lo2(v))), p.sfloor));
                const float2 x1 = rotate_half_angle(hi2(v), p.hbohm * w.y / fmaxf(sqrtf(abs2(hi2(v))), p.sfloor));
                g4[(long long)(j + T * m) * rs4] = pack4(x0, x1);
            }
        }
        return;
    }

    // P_H_NLKIN: nonlinear phase with phi, then the axis-0 kinetic pass, half-tile by half-tile
#pragma unroll
    for (int half = 0; half < 2; half++) {
        float4 *g4 = psi4 + half * CP + t;
        float2 a[P], b[P];
#pragma unroll
        for (int m = 0; m < P; m++) {
            const float4 v = g4[(long long)(j + T * m) * rs4];
            const float2 ph = half == 0 ? fa[m] : fb[m];
            float2 ve = make_float2(0.f, 0.f);
            if (p.nl.flags & 2)
                ve = __ldg(reinterpret_cast<const float2 *>(p.vext) + col4 + half * CP + t + (long long)(j + T * m) * rs4);
            a[m] = nl_phase(lo2(v), ph.x, p.nl, ve.x);
            b[m] = nl_phase(hi2(v), ph.y, p.nl, ve.y);
        }
        fft_pair<N, +1, true>(a, b, j, p.tw, sm);
#pragma unroll
        for (int m = 0; m < P; m++) {
            const float4 ph = __ldg(p.phase + j + T * m);
            a[m] = twmul<+1, true>(a[m], ph);
            b[m] = twmul<+1, true>(b[m], ph);
        }
        fft_pair<N, -1, true>(a, b, j, p.tw, sm);
#pragma unroll
        for (int m = 0; m < P; m++) g4[(long long)(j + T * m) * rs4] = pack4(a[m], b[m]);
    }
}

// ---------------------------------------------------------------------------- contiguous axis
// A group of T = N/8 threads owns two adjacent lines; lanes are consecutive j, so every global
// access of a warp is one contiguous 256-byte run of a line.

__host__ __device__ constexpr int xthreads(int N) { return N / ppt_for(N) >= 256 ? N / ppt_for(N) : 256; }

template <int N, int MODE, int DIR, bool HILO>
__global__ void __launch_bounds__(xthreads(N), xthreads(N) <= 256 ? 2 : 1) k_contig(const PassArgs p)
{
    extern __shared__ float4 smem[];
    constexpr int P = ppt_for(N), T = N / P, G = xthreads(N) / T;
    const int j = threadIdx.x % T, grp = threadIdx.x / T;
    const long long pair = (long long)blockIdx.x * G + grp;
    const bool active = 2 * pair < p.nlines;
    if (MODE != P_X_KDIAG && !active) return;
    float2 *la = p.data + (active ? 2 * pair : 0) * N;
    float2 *lb = la + N;
    SmemLine<T> sm{smem + grp * N, 1 + grp, G == 1};

    float2 a[P], b[P];
#pragma unroll
    for (int m = 0; m < P; m++) {
        a[m] = la[j + T * m];
        b[m] = lb[j + T * m];
    }
    if (MODE == P_X_FFT) {
        fft_pair<N, DIR, HILO>(a, b, j, p.tw, sm);
        const float s = p.scale;
#pragma unroll
        for (int m = 0; m < P; m++) {
            if (DIR < 0) {
                a[m].x *= s; a[m].y *= s; b[m].x *= s; b[m].y *= s;
            }
            la[j + T * m] = a[m];
            lb[j + T * m] = b[m];
        }
    } else if (MODE == P_X_KIN) {
        fft_pair<N, +1, true>(a, b, j, p.tw, sm);
#pragma unroll
        for (int m = 0; m < P; m++) {
            const float4 ph = __ldg(p.phase + j + T * m);
            a[m] = twmul<+1, true>(a[m], ph);
            b[m] = twmul<+1, true>(b[m], ph);
        }
        fft_pair<N, -1, true>(a, b, j, p.tw, sm);
#pragma unroll
        for (int m = 0; m < P; m++) {
            la[j + T * m] = a[m];
            lb[j + T * m] = b[m];
        }
    } else if (MODE == P_X_POISSON) {
        // eq. (2) in Fourier space: phi^ = D rho^/(C - k^2); C == 0: phi^(k=0) = 0
        fft_pair<N, +1, false>(a, b, j, p.tw, sm);
        const float2 ka = __ldg(p.dko + 2 * pair), kb = __ldg(p.dko + 2 * pair + 1);
#pragma unroll
        for (int m = 0; m < P; m++) {
            const float2 kx = __ldg(p.ksq2 + j + T * m);
            const float ga = helmholtz_mult(ka, kx, p.pscale, p.lap), gb = helmholtz_mult(kb, kx, p.pscale, p.lap);
            a[m].x *= ga; a[m].y *= ga; b[m].x *= gb; b[m].y *= gb;
        }
        fft_pair<N, -1, false>(a, b, j, p.tw, sm);
#pragma unroll
        for (int m = 0; m < P; m++) {
            la[j + T * m] = a[m];
            lb[j + T * m] = b[m];
        }
    } else { // P_X_KDIAG
        fft_pair<N, +1, true>(a, b, j, p.tw, sm);
        double v[1] = {0.0};
#pragma unroll
        for (int m = 0; m < P; m++) v[0] += (double)__ldg(p.ksq + j + T * m) * ((double)abs2(a[m]) + (double)abs2(b[m]));
        if (!active) v[0] = 0.0;
        block_accumulate<1>(v, p.diag);
    }
}

// ---------------------------------------------------------------------------- launchers

template <class K>
static int launch_kernel(K kern, unsigned grid, int threads, size_t smem_bytes, const PassArgs &a)
{
    // static shared memory (block_accumulate) counts against the 48 KB default too
    if (smem_bytes > 40 * 1024 && !smem_attr_done(reinterpret_cast<const void *>(kern))) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_bytes);
        if (e != cudaSuccess) return (int)e;
        smem_attr_mark(reinterpret_cast<const void *>(kern));
    }
    kern<<<grid, threads, smem_bytes, a.stream>>>(a);
    return (int)cudaGetLastError();
}

template <int N>
int launch_pass(const PassArgs &a)
{
    constexpr int CP = cp_for(N), T = N / ppt_for(N);
    constexpr int ST = CP * T;                       // threads of a strided-axis CTA
    constexpr size_t SSMEM = (size_t)N * CP * 16;    // one float4 per point and column pair
    constexpr int XT = xthreads(N), G = XT / T;
    constexpr size_t XSMEM = (size_t)N * G * 16;
    switch (a.kind) {
    case P_S_FFT:
    case P_S_KIN:
    case P_S_KDIAG: {
        const unsigned grid = (unsigned)((long long)a.n_outer * (a.ncols / (2 * CP)));
        if (a.kind == P_S_KIN) return launch_kernel(k_strided<N, CP, P_S_KIN, +1, true>, grid, ST, SSMEM, a);
        if (a.kind == P_S_KDIAG) return launch_kernel(k_strided<N, CP, P_S_KDIAG, +1, true>, grid, ST, SSMEM, a);
        if (a.dir > 0)
            return a.hilo ? launch_kernel(k_strided<N, CP, P_S_FFT, +1, true>, grid, ST, SSMEM, a)
                          : launch_kernel(k_strided<N, CP, P_S_FFT, +1, false>, grid, ST, SSMEM, a);
        return a.hilo ? launch_kernel(k_strided<N, CP, P_S_FFT, -1, true>, grid, ST, SSMEM, a)
                      : launch_kernel(k_strided<N, CP, P_S_FFT, -1, false>, grid, ST, SSMEM, a);
    }
    case P_H_NLKIN:
    case P_H_R2C:
    case P_H_POT:
    case P_H_SRC:
    case P_H_BOHM:
    case P_H_R2C_MC:
    case P_H_NL_MC:
    case P_H_DIAG: {
        const unsigned grid = (unsigned)(a.ncols / (4 * CP));
        if (a.kind == P_H_R2C_MC) return launch_kernel(k_haxis<N, CP, P_H_R2C_MC>, grid, ST, SSMEM, a);
        if (a.kind == P_H_NL_MC) return launch_kernel(k_haxis<N, CP, P_H_NL_MC>, grid, ST, SSMEM, a);
        if (a.kind == P_H_NLKIN) return launch_kernel(k_haxis<N, CP, P_H_NLKIN>, grid, ST, SSMEM, a);
        if (a.kind == P_H_R2C) return launch_kernel(k_haxis<N, CP, P_H_R2C>, grid, ST, SSMEM, a);
        if (a.kind == P_H_POT) return launch_kernel(k_haxis<N, CP, P_H_POT>, grid, ST, SSMEM, a);
        if (a.kind == P_H_SRC) return launch_kernel(k_haxis<N, CP, P_H_SRC>, grid, ST, SSMEM, a);
        if (a.kind == P_H_BOHM) return launch_kernel(k_haxis<N, CP, P_H_BOHM>, grid, ST, SSMEM, a);
        return launch_kernel(k_haxis<N, CP, P_H_DIAG>, grid, ST, SSMEM, a);
    }
    case P_X_FFT:
    case P_X_KIN:
    case P_X_POISSON:
    case P_X_KDIAG: {
        const long long pairs = a.nlines / 2;
        const unsigned grid = (unsigned)((pairs + G - 1) / G);
        if (a.kind == P_X_KIN) return launch_kernel(k_contig<N, P_X_KIN, +1, true>, grid, XT, XSMEM, a);
        if (a.kind == P_X_POISSON) return launch_kernel(k_contig<N, P_X_POISSON, +1, false>, grid, XT, XSMEM, a);
        if (a.kind == P_X_KDIAG) return launch_kernel(k_contig<N, P_X_KDIAG, +1, true>, grid, XT, XSMEM, a);
        return a.dir > 0 ? launch_kernel(k_contig<N, P_X_FFT, +1, true>, grid, XT, XSMEM, a)
                         : launch_kernel(k_contig<N, P_X_FFT, -1, true>, grid, XT, XSMEM, a);
    }
    default:
        return (int)cudaErrorInvalidValue;
    }
}

template int launch_pass<SN_LEN>(const PassArgs &a);

#if SN_LEN == 64
// setup only (sn_set_source_tables), never inside a step: interleave the two source tables of eq. (12)
__global__ void k_interleave(const float *__restrict__ beta, const float *__restrict__ gamma, float2 *__restrict__ bg, long long n)
{
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x)
        bg[i] = make_float2(beta[i], gamma[i]);
}
int launch_interleave(const float *beta, const float *gamma, float2 *bg, long long n, cudaStream_t stream)
{
    k_interleave<<<1184, 256, 0, stream>>>(beta, gamma, bg, n);
    return (int)cudaGetLastError();
}

// per-component norms of the coupled-field path (sn_mc_norms): fp32 squares, fp64 accumulation
__global__ void k_norm(const float2 *__restrict__ psi, long long n, double *out)
{
    double v[1] = {0.0};
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x)
        v[0] += (double)abs2(psi[i]);
    block_accumulate<1>(v, out);
}
int launch_norm(const float2 *psi, long long n, double *out, cudaStream_t stream)
{
    k_norm<<<1184, 256, 0, stream>>>(psi, n, out);
    return (int)cudaGetLastError();
}
#endif

} // namespace snk
