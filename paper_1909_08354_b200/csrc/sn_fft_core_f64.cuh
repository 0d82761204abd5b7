// sn_fft_core_f64.cuh -- complex128 line-FFT engine (sm_100a): the precision the paper benchmarked
// ("number representation of 64 bits", section III).
//
// Same Stockham structure as the complex64 engine (sn_fft_core.cuh): one line of N points is held by
// T = N/P threads, P = 8 points per thread (12 for N = 3*2^a), radix-8 stages with a trailing radix-4/2
// (radix-4 stages and a final radix-6 for 3*2^a), exchanges through shared memory in autosort order, so the
// forward transform leaves thread j with outputs j + T*m -- the operands of the first inverse stage.
// Differences: a thread carries ONE line (a double2 point is 16 bytes, what the complex64 engine moves for a
// line PAIR, so the exchange layouts and their XOR-linear addressing carry over unchanged with "column pair"
// read as "column"); twiddles are plain double2 (no hi/lo split: a correctly rounded double twiddle is off the
// unit circle by 1e-16, far below anything 10^3 steps can accumulate).
#pragma once
#include "sn_fft_core.cuh"

namespace snd {

using snk::comb;
using snk::ppt_for;
using snk::radix_for;
using snk::twiddle_entries;

typedef double2 cd;

constexpr double SQRT_HALF = 0.70710678118654752440084436210485;
constexpr double SIN60 = 0.86602540378443864676372317075294;

__device__ __forceinline__ cd cadd(cd a, cd b) { return make_double2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ cd csub(cd a, cd b) { return make_double2(a.x - b.x, a.y - b.y); }
// v * w, w the FORWARD twiddle e^{-i theta}; DIR < 0: v * conj(w)
template <int DIR>
__device__ __forceinline__ cd cmul(cd v, cd w)
{
    const double wi = DIR > 0 ? w.y : -w.y;
    return make_double2(fma(v.x, w.x, -v.y * wi), fma(v.x, wi, v.y * w.x));
}
template <int DIR>
__device__ __forceinline__ cd mul_w8_1(cd v)
{
    return DIR > 0 ? make_double2(SQRT_HALF * (v.x + v.y), SQRT_HALF * (v.y - v.x))
                   : make_double2(SQRT_HALF * (v.x - v.y), SQRT_HALF * (v.x + v.y));
}
template <int DIR>
__device__ __forceinline__ cd mul_w8_3(cd v)
{
    return DIR > 0 ? make_double2(SQRT_HALF * (v.y - v.x), -SQRT_HALF * (v.x + v.y))
                   : make_double2(-SQRT_HALF * (v.x + v.y), SQRT_HALF * (v.x - v.y));
}
template <int DIR>
__device__ __forceinline__ cd mul_w4_1(cd v)
{
    return DIR > 0 ? make_double2(v.y, -v.x) : make_double2(-v.y, v.x);
}

template <int DIR>
__device__ __forceinline__ void bf2(cd &x0, cd &x1)
{
    const cd t = x0;
    x0 = cadd(t, x1);
    x1 = csub(t, x1);
}
template <int DIR>
__device__ __forceinline__ void bf4(cd &x0, cd &x1, cd &x2, cd &x3)
{
    const cd c0 = cadd(x0, x2), d0 = csub(x0, x2);
    const cd c1 = cadd(x1, x3), d1 = mul_w4_1<DIR>(csub(x1, x3));
    x0 = cadd(c0, c1);
    x2 = csub(c0, c1);
    x1 = cadd(d0, d1);
    x3 = csub(d0, d1);
}
template <int DIR>
__device__ __forceinline__ void bf8(cd &x0, cd &x1, cd &x2, cd &x3, cd &x4, cd &x5, cd &x6, cd &x7)
{
    cd a0 = cadd(x0, x4), b0 = csub(x0, x4);
    cd a1 = cadd(x1, x5), b1 = mul_w8_1<DIR>(csub(x1, x5));
    cd a2 = cadd(x2, x6), b2 = mul_w4_1<DIR>(csub(x2, x6));
    cd a3 = cadd(x3, x7), b3 = mul_w8_3<DIR>(csub(x3, x7));
    bf4<DIR>(a0, a1, a2, a3);
    bf4<DIR>(b0, b1, b2, b3);
    x0 = a0; x1 = b0; x2 = a1; x3 = b1; x4 = a2; x5 = b2; x6 = a3; x7 = b3;
}
template <int DIR>
__device__ __forceinline__ void bf3(cd &x0, cd &x1, cd &x2)
{
    const cd t = cadd(x1, x2), u = csub(x1, x2);
    const cd m = make_double2(fma(-0.5, t.x, x0.x), fma(-0.5, t.y, x0.y));
    const double vx = u.x * SIN60, vy = u.y * SIN60;
    const cd iv = DIR > 0 ? make_double2(vy, -vx) : make_double2(-vy, vx);
    x0 = cadd(x0, t);
    x1 = cadd(m, iv);
    x2 = csub(m, iv);
}
// 6-point DFT as 2 x 3 with the prime-factor index maps (no twiddles between the factors)
template <int DIR>
__device__ __forceinline__ void bf6(cd &x0, cd &x1, cd &x2, cd &x3, cd &x4, cd &x5)
{
    cd s0 = cadd(x0, x3), d0 = csub(x0, x3);
    cd s1 = cadd(x2, x5), d1 = csub(x2, x5);
    cd s2 = cadd(x4, x1), d2 = csub(x4, x1);
    bf3<DIR>(s0, s1, s2);
    bf3<DIR>(d0, d1, d2);
    x0 = s0; x4 = s1; x2 = s2; x3 = d0; x1 = d1; x5 = d2;
}
template <int R, int NB, int DIR, int P>
__device__ __forceinline__ void butterfly(cd (&x)[P], int q)
{
    if constexpr (R == 8) {
        bf8<DIR>(x[q], x[q + NB], x[q + 2 * NB], x[q + 3 * NB], x[q + 4 * NB], x[q + 5 * NB], x[q + 6 * NB], x[q + 7 * NB]);
    } else if constexpr (R == 6) {
        bf6<DIR>(x[q], x[q + NB], x[q + 2 * NB], x[q + 3 * NB], x[q + 4 * NB], x[q + 5 * NB]);
    } else if constexpr (R == 4) {
        bf4<DIR>(x[q], x[q + NB], x[q + 2 * NB], x[q + 3 * NB]);
    } else {
        bf2<DIR>(x[q], x[q + NB]);
    }
}

// One Stockham stage (NS, R): twiddle exp(-/+ 2 pi i r (bq % NS)/(NS R)) at tw[OFF + (r-1) NS + bq % NS] (the
// table layout of the complex64 engine), then the radix-R butterflies.
template <int N, int R, int NS, int OFF, int DIR, int P>
__device__ __forceinline__ void stage(cd (&x)[P], int j, const cd *__restrict__ tw)
{
    constexpr int T = N / P, NB = P / R;
#pragma unroll
    for (int q = 0; q < NB; q++) {
        if constexpr (NS > 1) {
            const int kp = (j + T * q) & (NS - 1);
#pragma unroll
            for (int r = 1; r < R; r++) x[q + r * NB] = cmul<DIR>(x[q + r * NB], __ldg(tw + OFF + (r - 1) * NS + kp));
        }
        butterfly<R, NB, DIR>(x, q);
    }
}

template <int N, int R, int NS, class SM, int P>
__device__ __forceinline__ void exchange(cd (&x)[P], int j, SM &sm)
{
    constexpr int T = N / P, NB = P / R;
    constexpr int WPM = ((T - 1) & ~(NS - 1)) * R | ((T - 1) & (NS - 1));
    sm.sync(); // previous readers of the buffer are done
    const int tbw = sm.idx((j & ~(NS - 1)) * R + (j & (NS - 1)));
#pragma unroll
    for (int q = 0; q < NB; q++) {
        const int kq = ((T * q) & ~(NS - 1)) * R + ((T * q) & (NS - 1));
#pragma unroll
        for (int r = 0; r < R; r++) sm.st_i(comb<SM>(tbw, kq + r * NS, WPM), x[q + r * NB]);
    }
    sm.sync();
    const int tbr = sm.idx(j);
#pragma unroll
    for (int m = 0; m < P; m++) x[m] = sm.ld_i(comb<SM>(tbr, T * m, T - 1));
}

template <int N, int NSP, int RP, int OFF, int DIR, class SM, int P>
__device__ __forceinline__ void fft_next(cd (&x)[P], int j, const cd *__restrict__ tw, SM &sm)
{
    constexpr int NS = NSP * RP, R = radix_for(N, NS);
    exchange<N, RP, NSP>(x, j, sm);
    stage<N, R, NS, OFF, DIR>(x, j, tw);
    if constexpr (NS * R < N) fft_next<N, NS, R, OFF + NS * (R - 1), DIR, SM>(x, j, tw, sm);
}

// Unscaled DFT of one line.  In: thread j holds points j + T*m (T = N/P); out: outputs j + T*m.
// DIR = +1: sum x e^{-2 pi i jk/N}; DIR = -1: e^{+...}.
template <int N, int DIR, class SM, int P>
__device__ __forceinline__ void fft_line(cd (&x)[P], int j, const cd *__restrict__ tw, SM &sm)
{
    static_assert(P == ppt_for(N), "points per thread");
    constexpr int R = radix_for(N, 1);
    stage<N, R, 1, 0, DIR>(x, j, tw);
    if constexpr (R < N) fft_next<N, 1, R, 0, DIR, SM>(x, j, tw, sm);
}

// ---- shared-memory accessors (one double2 per position; index maps of snk::SmemTile / snk::SmemLine) ----
template <int CP>
struct SmemTileD {
    cd *base;
    int t;
    static constexpr int TMASK = CP - 1;
    __host__ __device__ static constexpr int lin(int pos) { return snk::SmemTile<CP>::lin(pos); }
    __device__ __forceinline__ int idx(int pos) const { return lin(pos) ^ t; }
    __device__ __forceinline__ void st_i(int i, cd v) const { base[i] = v; }
    __device__ __forceinline__ cd ld_i(int i) const { return base[i]; }
    __device__ __forceinline__ void st(int pos, cd v) const { st_i(idx(pos), v); }
    __device__ __forceinline__ cd ld(int pos) const { return ld_i(idx(pos)); }
    __device__ __forceinline__ void sync() const { __syncthreads(); }
};

template <int T>
struct SmemLineD {
    cd *base;
    int bar_id;
    bool whole_cta;
    static constexpr int TMASK = 0;
    __host__ __device__ static constexpr int lin(int pos) { return pos ^ ((pos >> 3) & 7); }
    __device__ __forceinline__ int idx(int pos) const { return lin(pos); }
    __device__ __forceinline__ void st_i(int i, cd v) const { base[i] = v; }
    __device__ __forceinline__ cd ld_i(int i) const { return base[i]; }
    __device__ __forceinline__ void sync() const
    {
        if (T <= 32) {
            __syncwarp();
        } else if (whole_cta) {
            __syncthreads();
        } else {
            asm volatile("bar.sync %0, %1;" ::"r"(bar_id), "r"(T) : "memory");
        }
    }
};

} // namespace snd
