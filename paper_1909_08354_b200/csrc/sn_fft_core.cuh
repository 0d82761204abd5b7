// sn_fft_core.cuh -- register/shared-memory Stockham line FFT engine (sm_100a).
//
// The "Fourier methods" of PAPER.md:113 (section III) are hand-written here: one line of
// N = 2^n complex64 points is held by T = N/8 threads, 8 points per thread in registers
// (N = 3*2^a: T = N/12 threads, 12 points per thread, radix-4 stages and a final radix-6 stage
// done as 2 x 3 with prime-factor index maps).
// Every thread carries TWO independent lines (a[], b[]) so that each twiddle load, each
// shared-memory instruction (128-bit: one point of each line) and each index computation is
// amortised over two transforms.  Stages are radix-8 (a trailing radix-2/4 stage when n is
// not a multiple of 3); between stages the lines are exchanged through shared memory in
// Stockham (autosort) order, so forward output is in natural order, thread j holding points
// j + T*m (m = 0..7) -- exactly the operands its first inverse stage needs.  A fused
// forward -> pointwise -> inverse pass therefore needs no exchange at the junction.
//
// Twiddles are stored as hi+lo float pairs (float4 = wr_hi, wi_hi, wr_lo, wi_lo) built in
// float64 on the host and applied with an FMA chain.  A plain fp32 twiddle has |w| != 1 by a
// FIXED ~1e-8 relative amount; used by a fixed fraction of the butterflies this gives a
// systematic, non-averaging gain per transform that breaks norm conservation at the 1e-5
// level over 10^3 steps.  The lo part enters the FMA chain
// before the final rounding, which removes the bias.  HILO=false (plain float2 twiddles) is
// used for the density/potential transforms, where a 1e-7 gain is harmless.
#pragma once
#include <cuda_runtime.h>

namespace snk {

constexpr double SQRT_HALF_D = 0.70710678118654752440084436210485;
constexpr float C8_HI = (float)SQRT_HALF_D;
constexpr float C8_LO = (float)(SQRT_HALF_D - (double)C8_HI);
constexpr double SIN60_D = 0.86602540378443864676372317075294;
constexpr float S3_HI = (float)SIN60_D;
constexpr float S3_LO = (float)(SIN60_D - (double)S3_HI);

__device__ __forceinline__ float2 cadd(float2 a, float2 b) { return make_float2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ float2 csub(float2 a, float2 b) { return make_float2(a.x - b.x, a.y - b.y); }

// v * w, w the FORWARD twiddle (e^{-i theta}) as hi/lo; DIR < 0 multiplies by conj(w).
template <int DIR, bool HILO>
__device__ __forceinline__ float2 twmul(float2 v, float4 w)
{
    const float wi = DIR > 0 ? w.y : -w.y;
    float2 o;
    if (HILO) {
        const float li = DIR > 0 ? w.w : -w.w;
        o.x = fmaf(v.x, w.x, fmaf(-v.y, wi, fmaf(v.x, w.z, -v.y * li)));
        o.y = fmaf(v.x, wi, fmaf(v.y, w.x, fmaf(v.x, li, v.y * w.z)));
    } else {
        o.x = fmaf(v.x, w.x, -v.y * wi);
        o.y = fmaf(v.x, wi, v.y * w.x);
    }
    return o;
}

template <bool HILO>
__device__ __forceinline__ float scale8(float s)
{
    return HILO ? fmaf(s, C8_HI, s * C8_LO) : s * C8_HI;
}

// x *= W8^1 (forward: e^{-i pi/4}; DIR < 0: conjugate)
template <int DIR, bool HILO>
__device__ __forceinline__ float2 mul_w8_1(float2 v)
{
    return DIR > 0 ? make_float2(scale8<HILO>(v.x + v.y), scale8<HILO>(v.y - v.x))
                   : make_float2(scale8<HILO>(v.x - v.y), scale8<HILO>(v.x + v.y));
}
// x *= W8^3
template <int DIR, bool HILO>
__device__ __forceinline__ float2 mul_w8_3(float2 v)
{
    return DIR > 0 ? make_float2(scale8<HILO>(v.y - v.x), scale8<HILO>(-v.x - v.y))
                   : make_float2(scale8<HILO>(-v.x - v.y), scale8<HILO>(v.x - v.y));
}
// x *= W4^1 = -i (forward) / +i (inverse)
template <int DIR>
__device__ __forceinline__ float2 mul_w4_1(float2 v)
{
    return DIR > 0 ? make_float2(v.y, -v.x) : make_float2(-v.y, v.x);
}

template <int DIR>
__device__ __forceinline__ void bf2(float2 &x0, float2 &x1)
{
    const float2 t = x0;
    x0 = cadd(t, x1);
    x1 = csub(t, x1);
}

// 4-point DFT, natural order in and out
template <int DIR>
__device__ __forceinline__ void bf4(float2 &x0, float2 &x1, float2 &x2, float2 &x3)
{
    const float2 c0 = cadd(x0, x2), d0 = csub(x0, x2);
    const float2 c1 = cadd(x1, x3), d1 = mul_w4_1<DIR>(csub(x1, x3));
    x0 = cadd(c0, c1);
    x2 = csub(c0, c1);
    x1 = cadd(d0, d1);
    x3 = csub(d0, d1);
}

// 8-point DFT, natural order in and out
template <int DIR, bool HILO>
__device__ __forceinline__ void bf8(float2 &x0, float2 &x1, float2 &x2, float2 &x3, float2 &x4, float2 &x5,
                                    float2 &x6, float2 &x7)
{
    float2 a0 = cadd(x0, x4), b0 = csub(x0, x4);
    float2 a1 = cadd(x1, x5), b1 = mul_w8_1<DIR, HILO>(csub(x1, x5));
    float2 a2 = cadd(x2, x6), b2 = mul_w4_1<DIR>(csub(x2, x6));
    float2 a3 = cadd(x3, x7), b3 = mul_w8_3<DIR, HILO>(csub(x3, x7));
    bf4<DIR>(a0, a1, a2, a3); // X0 X2 X4 X6
    bf4<DIR>(b0, b1, b2, b3); // X1 X3 X5 X7
    x0 = a0; x1 = b0; x2 = a1; x3 = b1; x4 = a2; x5 = b2; x6 = a3; x7 = b3;
}

// 3-point DFT in place; W3 = -1/2 -+ i sqrt(3)/2 (sqrt(3)/2 as hi/lo like the twiddles)
template <int DIR, bool HILO>
__device__ __forceinline__ void bf3(float2 &x0, float2 &x1, float2 &x2)
{
    const float2 t = cadd(x1, x2), u = csub(x1, x2);
    const float2 m = make_float2(fmaf(-0.5f, t.x, x0.x), fmaf(-0.5f, t.y, x0.y));
    const float vx = HILO ? fmaf(u.x, S3_HI, u.x * S3_LO) : u.x * S3_HI;
    const float vy = HILO ? fmaf(u.y, S3_HI, u.y * S3_LO) : u.y * S3_HI;
    // forward: X1 = m - i v, X2 = m + i v; inverse: swapped
    const float2 iv = DIR > 0 ? make_float2(vy, -vx) : make_float2(-vy, vx);
    x0 = cadd(x0, t);
    x1 = cadd(m, iv);
    x2 = csub(m, iv);
}

// 6-point DFT, natural order in and out, as 2 x 3 with the prime-factor index maps
// n = (3 n1 + 2 n2) mod 6, k = (3 k1 + 4 k2) mod 6 (no twiddles between the factors).
template <int DIR, bool HILO>
__device__ __forceinline__ void bf6(float2 &x0, float2 &x1, float2 &x2, float2 &x3, float2 &x4, float2 &x5)
{
    float2 s0 = cadd(x0, x3), d0 = csub(x0, x3); // n2 = 0: x[0], x[3]
    float2 s1 = cadd(x2, x5), d1 = csub(x2, x5); // n2 = 1: x[2], x[5]
    float2 s2 = cadd(x4, x1), d2 = csub(x4, x1); // n2 = 2: x[4], x[1]
    bf3<DIR, HILO>(s0, s1, s2);                  // k1 = 0: X[0], X[4], X[2]
    bf3<DIR, HILO>(d0, d1, d2);                  // k1 = 1: X[3], X[1], X[5]
    x0 = s0; x4 = s1; x2 = s2; x3 = d0; x1 = d1; x5 = d2;
}

// radix-R butterfly on x[q + r*NB], r = 0..R-1
template <int R, int NB, int DIR, bool HILO, int P>
__device__ __forceinline__ void butterfly(float2 (&x)[P], int q)
{
    if constexpr (R == 8) {
        bf8<DIR, HILO>(x[q], x[q + NB], x[q + 2 * NB], x[q + 3 * NB], x[q + 4 * NB], x[q + 5 * NB], x[q + 6 * NB],
                       x[q + 7 * NB]);
    } else if constexpr (R == 6) {
        bf6<DIR, HILO>(x[q], x[q + NB], x[q + 2 * NB], x[q + 3 * NB], x[q + 4 * NB], x[q + 5 * NB]);
    } else if constexpr (R == 4) {
        bf4<DIR>(x[q], x[q + NB], x[q + 2 * NB], x[q + 3 * NB]);
    } else {
        bf2<DIR>(x[q], x[q + NB]);
    }
}

// Engine shape per length.  N = 2^n: 8 points per thread and line, radix-8 stages with a trailing
// radix-4/2.  N = 3 * 2^a (96 ... 3072): 12 points per thread, radix-4 stages (after one leading radix-2 stage
// when N/6 is not a power of 4) and a final radix-6.
__host__ __device__ constexpr int ppt_for(int N) { return N % 3 == 0 ? 12 : 8; }
__host__ __device__ constexpr int radix_for(int N, int NS)
{
    const int rem = N / NS;
    if (N % 3 == 0) {
        if (rem == 6) return 6;
        // N/6 = 2 * 4^a (192, 768, 3072): one leading radix-2 stage (untwiddled), then radix 4
        int m = N / 6;
        while (m % 4 == 0) m /= 4;
        return (NS == 1 && m == 2) ? 2 : 4;
    }
    return rem >= 8 ? 8 : rem;
}

// Number of float4 twiddle entries of the table for length N (all stages with NS > 1).
__host__ __device__ constexpr int twiddle_entries(int N)
{
    int total = 0, ns = 1;
    while (ns < N) {
        const int r = radix_for(N, ns);
        if (ns > 1) total += ns * (r - 1);
        ns *= r;
    }
    return total;
}

// One Stockham stage on both lines: twiddle (if NS > 1) then radix-R butterflies.
// Butterfly q of thread j is butterfly number bq = j + T*q of the stage; its inputs are the
// thread's own points j + T*(q + r*NB) = bq + r*N/R; twiddle exp(-/+ 2 pi i r (bq % NS)/(NS R)),
// stored at tw[(r-1)*NS + (bq % NS)] so that lanes with consecutive j read consecutive entries.
// ONE = true: only line a is transformed (b is never touched).
#ifndef SN_TW_PREFETCH
#define SN_TW_PREFETCH 1 // load a stage's twiddles between the exchange's stores and loads (data registers are dead there)
#endif

// Table of length N: twiddle_entries(N) float4 (hi + lo) followed by the same entries as plain float2 (hi only).
// A stage whose twiddles are applied plainly reads the compact float2 copy: 256 B instead of 512 B per warp-wide
// load, i.e. 2 instead of 4 L1 wavefronts -- the pass kernels are bound by L1/shared-memory wavefronts
// (profiles/r02c).  OFF = entries of the earlier stages.
#ifndef SN_HILO_MAX_NS
#define SN_HILO_MAX_NS (1 << 30) // hi/lo twiddles on stages with NS <= this (psi transforms); larger NS: plain
#endif
template <bool HILO, int NS>
__host__ __device__ constexpr bool stage_hilo() { return HILO && NS <= SN_HILO_MAX_NS; }

// The pass kernels read the tables from global memory through the read-only path; a kernel that keeps its tables in
// shared memory (sn_resident.cu) defines SN_TW_LOAD as a plain load before including this header.
#ifndef SN_TW_LOAD
#define SN_TW_LOAD(p) __ldg(p)
#endif
template <int N, int R, int NS, int OFF, bool HILO, int P>
__device__ __forceinline__ void load_twiddles(float4 (&w)[(P / R) * (R - 1)], int j, const float4 *__restrict__ tw)
{
    constexpr int T = N / P, NB = P / R;
    const float2 *__restrict__ tw2 = reinterpret_cast<const float2 *>(tw + twiddle_entries(N));
#pragma unroll
    for (int q = 0; q < NB; q++) {
        const int kp = (j + T * q) & (NS - 1);
#pragma unroll
        for (int r = 1; r < R; r++) {
            if (HILO) {
                w[q * (R - 1) + r - 1] = SN_TW_LOAD(tw + OFF + kp + (r - 1) * NS);
            } else {
                const float2 h = SN_TW_LOAD(tw2 + OFF + kp + (r - 1) * NS);
                w[q * (R - 1) + r - 1] = make_float4(h.x, h.y, 0.f, 0.f);
            }
        }
    }
}

template <int N, int R, int NS, int DIR, bool HILO, bool ONE, int P>
__device__ __forceinline__ void stage_compute(float2 (&a)[P], float2 (&b)[P], const float4 (&w)[(P / R) * (R - 1)])
{
    constexpr int NB = P / R;
#pragma unroll
    for (int q = 0; q < NB; q++) {
        if constexpr (NS > 1) {
#pragma unroll
            for (int r = 1; r < R; r++) {
                const float4 ww = w[q * (R - 1) + r - 1];
                a[q + r * NB] = twmul<DIR, HILO>(a[q + r * NB], ww);
                if (!ONE) b[q + r * NB] = twmul<DIR, HILO>(b[q + r * NB], ww);
            }
        }
        butterfly<R, NB, DIR, HILO>(a, q);
        if (!ONE) butterfly<R, NB, DIR, HILO>(b, q);
    }
}

// ---- XOR-linear shared-memory addressing --------------------------------------------------
// Every exchange layout below is a GF(2)-linear map of the position bits (shifts, masks, XOR
// swizzles) XORed with a per-group constant.  An exchange position is (thread part) ^ (compile-
// time part) with disjoint bits, so   idx(pos) = idx(thread part) ^ lin(compile-time part):
// ONE runtime index per stage and thread, and per access an XOR with an immediate (bits that the
// thread part can also set) plus an immediate offset (bits it cannot).  Without this the compiler
// precomputes ~20 addresses per thread, keeps them across tiles and spills them.
template <class SM>
__host__ __device__ constexpr int lin_mask(int posmask)
{
    int m = 0;
    for (int bit = 0; bit < 16; bit++)
        if (posmask >> bit & 1) m |= SM::lin(1 << bit);
    return m;
}
// index of position (thread part ^ K) given tb = idx(thread part); PM = bits the thread part may set
template <class SM>
__device__ __forceinline__ int comb(int tb, int K, int PM)
{
    const int TM = lin_mask<SM>(PM) | SM::TMASK;
    const int L = SM::lin(K);
    const int X = L & TM, A = L & ~TM;
    return (tb ^ X) + A;
}

// Stockham exchange after a stage (NS, R): output r of butterfly bq goes to position
// (bq / NS) * NS * R + (bq % NS) + r * NS; afterwards thread j re-reads points j + T*m.
template <int N, int R, int NS, class SM, int P>
__device__ __forceinline__ void exchange_store(float2 (&a)[P], float2 (&b)[P], int j, SM &sm)
{
    constexpr int T = N / P, NB = P / R;
    constexpr int WPM = ((T - 1) & ~(NS - 1)) * R | ((T - 1) & (NS - 1)); // position bits of butterfly j's base
    sm.sync(); // previous readers of the buffer are done
    const int tbw = sm.idx((j & ~(NS - 1)) * R + (j & (NS - 1)));
#pragma unroll
    for (int q = 0; q < NB; q++) {
        const int kq = ((T * q) & ~(NS - 1)) * R + ((T * q) & (NS - 1)); // base of butterfly T*q (compile time)
#pragma unroll
        for (int r = 0; r < R; r++) sm.st_i(comb<SM>(tbw, kq + r * NS, WPM), a[q + r * NB], b[q + r * NB]);
    }
}
template <int N, class SM, int P>
__device__ __forceinline__ void exchange_load(float2 (&a)[P], float2 (&b)[P], int j, SM &sm)
{
    constexpr int T = N / P;
    sm.sync();
    const int tbr = sm.idx(j);
#pragma unroll
    for (int m = 0; m < P; m++) sm.ld_i(comb<SM>(tbr, T * m, T - 1), a[m], b[m]);
}

// exchange after stage (NSP, RP), then stage NS = NSP * RP and everything after it (OFF: table entries before it)
template <int N, int NSP, int RP, int OFF, int DIR, bool HILO, bool ONE, class SM, int P>
__device__ __forceinline__ void fft_next(float2 (&a)[P], float2 (&b)[P], int j, const float4 *__restrict__ tw, SM &sm)
{
    constexpr int NS = NSP * RP, R = radix_for(N, NS);
    constexpr bool H = stage_hilo<HILO, NS>();
    float4 w[(P / R) * (R - 1)];
    exchange_store<N, RP, NSP>(a, b, j, sm);
    if (SN_TW_PREFETCH) load_twiddles<N, R, NS, OFF, H, P>(w, j, tw);
    exchange_load<N>(a, b, j, sm);
    if (!SN_TW_PREFETCH) load_twiddles<N, R, NS, OFF, H, P>(w, j, tw);
    stage_compute<N, R, NS, DIR, H, ONE>(a, b, w);
    if constexpr (NS * R < N) fft_next<N, NS, R, OFF + NS * (R - 1), DIR, HILO, ONE, SM>(a, b, j, tw, sm);
}

template <int N, int NS, int DIR, bool HILO, bool ONE, class SM, int P>
__device__ __forceinline__ void fft_stages(float2 (&a)[P], float2 (&b)[P], int j, const float4 *__restrict__ tw,
                                           SM &sm)
{
    static_assert(P == ppt_for(N), "points per thread");
    static_assert(NS == 1, "entry point is the first (untwiddled) stage");
    constexpr int R = radix_for(N, 1);
    const float4 none[(P / R) * (R - 1)] = {};
    stage_compute<N, R, 1, DIR, HILO, ONE>(a, b, none);
    if constexpr (R < N) fft_next<N, 1, R, 0, DIR, HILO, ONE, SM>(a, b, j, tw, sm);
}

// Unscaled DFT of two lines.  In: thread j holds points j + T*m of each line (T = N/P, P = ppt_for(N)).
// Out: thread j holds outputs j + T*m.  DIR = +1: sum x e^{-2 pi i jk/N}; DIR = -1: e^{+...}.
template <int N, int DIR, bool HILO, class SM, int P>
__device__ __forceinline__ void fft_pair_scalar(float2 (&a)[P], float2 (&b)[P], int j, const float4 *__restrict__ tw, SM &sm)
{
    fft_stages<N, 1, DIR, HILO, false, SM>(a, b, j, tw, sm);
}

// Same for ONE line (a); the accessor SM stores/loads only a.
template <int N, int DIR, bool HILO, class SM, int P>
__device__ __forceinline__ void fft_single(float2 (&a)[P], int j, const float4 *__restrict__ tw, SM &sm)
{
    float2 dummy[P];
    fft_stages<N, 1, DIR, HILO, true, SM>(a, dummy, j, tw, sm);
}

// ---- packed (fp32x2) line-pair engine ------------------------------------------------------
// The two lines of a pair see the same twiddles and the same butterfly structure, so point m of the pair is held
// as two register pairs  r = (a.re, b.re), i = (a.im, b.im)  and every operation is one sm_100 packed instruction
// (FADD2 / FMUL2 / FFMA2: two fp32 lanes per thread, a twiddle enters as a broadcast scalar operand) instead of two
// scalar ones.  The fp32 pipe does the same lane-work either way; what halves is the number of ISSUED floating-point
// instructions, and the pass kernels are issue-bound (profiles/r01g: issue slots 65 % busy, fp32 pipe ~50 %).
// Multiplications by -i / +i are register renames plus sign flips that fold into operand modifiers.
// Rounding is identical to the scalar engine (same operations in the same order, lane by lane).
#ifndef SN_PACKED
#define SN_PACKED 1 // 0: scalar engine everywhere (A/B builds)
#endif
#ifndef SN_PACKED_3
// packed engine for the 3*2^a lengths too?  No: measured at 384^3 (12 points per thread, radix-4/6 stages, ~195
// registers) the packed form is SLOWER -- pipelined H_NLKIN 0.611 -> 0.877 ms, first-path S_KIN 0.314 -> 0.345 ms
// (the 64-bit register pairs cost that kernel the freedom it needs at its register budget); profiles/r02o.
#define SN_PACKED_3 0
#endif
__host__ __device__ constexpr bool packed_for(int N) { return SN_PACKED && (N % 3 != 0 || SN_PACKED_3); }

struct cp2 {
    float2 r, i;
};

__device__ __forceinline__ float2 neg2(float2 v) { return make_float2(-v.x, -v.y); }
__device__ __forceinline__ float2 add2(float2 a, float2 b) { return __fadd2_rn(a, b); }
__device__ __forceinline__ float2 sub2(float2 a, float2 b) { return __fadd2_rn(a, neg2(b)); }
__device__ __forceinline__ float2 mul2s(float2 a, float s) { return __fmul2_rn(a, make_float2(s, s)); }
__device__ __forceinline__ float2 fma2s(float2 a, float s, float2 c) { return __ffma2_rn(a, make_float2(s, s), c); }

__device__ __forceinline__ cp2 cadd(cp2 a, cp2 b) { return cp2{add2(a.r, b.r), add2(a.i, b.i)}; }
__device__ __forceinline__ cp2 csub(cp2 a, cp2 b) { return cp2{sub2(a.r, b.r), sub2(a.i, b.i)}; }

__device__ __forceinline__ cp2 pack_pair(float2 a, float2 b) { return cp2{make_float2(a.x, b.x), make_float2(a.y, b.y)}; }
__device__ __forceinline__ float2 line_a(cp2 v) { return make_float2(v.r.x, v.i.x); }
__device__ __forceinline__ float2 line_b(cp2 v) { return make_float2(v.r.y, v.i.y); }

// tile slot (a.re, a.im, b.re, b.im) <-> packed pair
__device__ __forceinline__ cp2 unpack4(float4 v) { return cp2{make_float2(v.x, v.z), make_float2(v.y, v.w)}; }
__device__ __forceinline__ float4 pack4(cp2 v) { return make_float4(v.r.x, v.i.x, v.r.y, v.i.y); }
// both lines times a real scalar / times one real factor per line (ga for line a, gb for line b)
__device__ __forceinline__ cp2 cscale(cp2 v, float s) { return cp2{mul2s(v.r, s), mul2s(v.i, s)}; }
__device__ __forceinline__ cp2 cscale(cp2 v, float ga, float gb)
{
    const float2 g = make_float2(ga, gb);
    return cp2{__fmul2_rn(v.r, g), __fmul2_rn(v.i, g)};
}

// v * w for both lines (w as in twmul)
template <int DIR, bool HILO>
__device__ __forceinline__ cp2 twmul(cp2 v, float4 w)
{
    const float wi = DIR > 0 ? w.y : -w.y;
    const float2 ni = neg2(v.i);
    cp2 o;
    if (HILO) {
        const float li = DIR > 0 ? w.w : -w.w;
        o.r = fma2s(v.r, w.x, fma2s(ni, wi, fma2s(v.r, w.z, mul2s(ni, li))));
        o.i = fma2s(v.r, wi, fma2s(v.i, w.x, fma2s(v.r, li, mul2s(v.i, w.z))));
    } else {
        o.r = fma2s(v.r, w.x, mul2s(ni, wi));
        o.i = fma2s(v.r, wi, mul2s(v.i, w.x));
    }
    return o;
}

template <bool HILO>
__device__ __forceinline__ float2 scale8(float2 s)
{
    return HILO ? fma2s(s, C8_HI, mul2s(s, C8_LO)) : mul2s(s, C8_HI);
}
template <int DIR, bool HILO>
__device__ __forceinline__ cp2 mul_w8_1(cp2 v)
{
    return DIR > 0 ? cp2{scale8<HILO>(add2(v.r, v.i)), scale8<HILO>(sub2(v.i, v.r))}
                   : cp2{scale8<HILO>(sub2(v.r, v.i)), scale8<HILO>(add2(v.r, v.i))};
}
template <int DIR, bool HILO>
__device__ __forceinline__ cp2 mul_w8_3(cp2 v)
{
    return DIR > 0 ? cp2{scale8<HILO>(sub2(v.i, v.r)), scale8<HILO>(neg2(add2(v.r, v.i)))}
                   : cp2{scale8<HILO>(neg2(add2(v.r, v.i))), scale8<HILO>(sub2(v.r, v.i))};
}
template <int DIR>
__device__ __forceinline__ cp2 mul_w4_1(cp2 v)
{
    return DIR > 0 ? cp2{v.i, neg2(v.r)} : cp2{neg2(v.i), v.r};
}

template <int DIR>
__device__ __forceinline__ void bf2(cp2 &x0, cp2 &x1)
{
    const cp2 t = x0;
    x0 = cadd(t, x1);
    x1 = csub(t, x1);
}
template <int DIR>
__device__ __forceinline__ void bf4(cp2 &x0, cp2 &x1, cp2 &x2, cp2 &x3)
{
    const cp2 c0 = cadd(x0, x2), d0 = csub(x0, x2);
    const cp2 c1 = cadd(x1, x3), d1 = mul_w4_1<DIR>(csub(x1, x3));
    x0 = cadd(c0, c1);
    x2 = csub(c0, c1);
    x1 = cadd(d0, d1);
    x3 = csub(d0, d1);
}
template <int DIR, bool HILO>
__device__ __forceinline__ void bf8(cp2 &x0, cp2 &x1, cp2 &x2, cp2 &x3, cp2 &x4, cp2 &x5, cp2 &x6, cp2 &x7)
{
    cp2 a0 = cadd(x0, x4), b0 = csub(x0, x4);
    cp2 a1 = cadd(x1, x5), b1 = mul_w8_1<DIR, HILO>(csub(x1, x5));
    cp2 a2 = cadd(x2, x6), b2 = mul_w4_1<DIR>(csub(x2, x6));
    cp2 a3 = cadd(x3, x7), b3 = mul_w8_3<DIR, HILO>(csub(x3, x7));
    bf4<DIR>(a0, a1, a2, a3);
    bf4<DIR>(b0, b1, b2, b3);
    x0 = a0; x1 = b0; x2 = a1; x3 = b1; x4 = a2; x5 = b2; x6 = a3; x7 = b3;
}
template <int DIR, bool HILO>
__device__ __forceinline__ void bf3(cp2 &x0, cp2 &x1, cp2 &x2)
{
    const cp2 t = cadd(x1, x2), u = csub(x1, x2);
    const cp2 m{fma2s(t.r, -0.5f, x0.r), fma2s(t.i, -0.5f, x0.i)};
    const float2 vx = HILO ? fma2s(u.r, S3_HI, mul2s(u.r, S3_LO)) : mul2s(u.r, S3_HI);
    const float2 vy = HILO ? fma2s(u.i, S3_HI, mul2s(u.i, S3_LO)) : mul2s(u.i, S3_HI);
    const cp2 iv = DIR > 0 ? cp2{vy, neg2(vx)} : cp2{neg2(vy), vx};
    x0 = cadd(x0, t);
    x1 = cadd(m, iv);
    x2 = csub(m, iv);
}
template <int DIR, bool HILO>
__device__ __forceinline__ void bf6(cp2 &x0, cp2 &x1, cp2 &x2, cp2 &x3, cp2 &x4, cp2 &x5)
{
    cp2 s0 = cadd(x0, x3), d0 = csub(x0, x3);
    cp2 s1 = cadd(x2, x5), d1 = csub(x2, x5);
    cp2 s2 = cadd(x4, x1), d2 = csub(x4, x1);
    bf3<DIR, HILO>(s0, s1, s2);
    bf3<DIR, HILO>(d0, d1, d2);
    x0 = s0; x4 = s1; x2 = s2; x3 = d0; x1 = d1; x5 = d2;
}
template <int R, int NB, int DIR, bool HILO, int P>
__device__ __forceinline__ void butterfly(cp2 (&x)[P], int q)
{
    if constexpr (R == 8) {
        bf8<DIR, HILO>(x[q], x[q + NB], x[q + 2 * NB], x[q + 3 * NB], x[q + 4 * NB], x[q + 5 * NB], x[q + 6 * NB],
                       x[q + 7 * NB]);
    } else if constexpr (R == 6) {
        bf6<DIR, HILO>(x[q], x[q + NB], x[q + 2 * NB], x[q + 3 * NB], x[q + 4 * NB], x[q + 5 * NB]);
    } else if constexpr (R == 4) {
        bf4<DIR>(x[q], x[q + NB], x[q + 2 * NB], x[q + 3 * NB]);
    } else {
        bf2<DIR>(x[q], x[q + NB]);
    }
}

template <int N, int R, int NS, int DIR, bool HILO, int P>
__device__ __forceinline__ void stage_compute(cp2 (&x)[P], const float4 (&w)[(P / R) * (R - 1)])
{
    constexpr int NB = P / R;
#pragma unroll
    for (int q = 0; q < NB; q++) {
        if constexpr (NS > 1) {
#pragma unroll
            for (int r = 1; r < R; r++) x[q + r * NB] = twmul<DIR, HILO>(x[q + r * NB], w[q * (R - 1) + r - 1]);
        }
        butterfly<R, NB, DIR, HILO>(x, q);
    }
}

// the exchange stores one float4 per position: (r.x, r.y, i.x, i.y) = (a.re, b.re, a.im, b.im)
template <int N, int R, int NS, class SM, int P>
__device__ __forceinline__ void exchange_store(cp2 (&x)[P], int j, SM &sm)
{
    constexpr int T = N / P, NB = P / R;
    constexpr int WPM = ((T - 1) & ~(NS - 1)) * R | ((T - 1) & (NS - 1));
    sm.sync();
    const int tbw = sm.idx((j & ~(NS - 1)) * R + (j & (NS - 1)));
#pragma unroll
    for (int q = 0; q < NB; q++) {
        const int kq = ((T * q) & ~(NS - 1)) * R + ((T * q) & (NS - 1));
#pragma unroll
        for (int r = 0; r < R; r++) sm.st_i(comb<SM>(tbw, kq + r * NS, WPM), x[q + r * NB].r, x[q + r * NB].i);
    }
}
template <int N, class SM, int P>
__device__ __forceinline__ void exchange_load(cp2 (&x)[P], int j, SM &sm)
{
    constexpr int T = N / P;
    sm.sync();
    const int tbr = sm.idx(j);
#pragma unroll
    for (int m = 0; m < P; m++) sm.ld_i(comb<SM>(tbr, T * m, T - 1), x[m].r, x[m].i);
}

// ---- resident last-stage twiddles ----
// The twiddles of the LAST stage depend on the thread (kp = (j + T q) mod NS) but not on the tile, and the forward and
// the inverse transform use the same values (conjugated).  A persistent pass kernel can load them once per CTA
// lifetime and keep them in registers (7 float4 at N = 512): per 64 KB tile and warp that removes 2 x 7 warp-wide
// 128-bit loads = 56 of the ~420 L1 wavefronts of a kinetic pass -- and L1/shared-memory wavefronts are what bounds
// these kernels.
__host__ __device__ constexpr int last_stage_ns(int N)
{
    int ns = 1;
    while (ns * radix_for(N, ns) < N) ns *= radix_for(N, ns);
    return ns;
}
__host__ __device__ constexpr int last_stage_off(int N)
{
    int ns = 1, off = 0;
    while (ns * radix_for(N, ns) < N) {
        if (ns > 1) off += ns * (radix_for(N, ns) - 1);
        ns *= radix_for(N, ns);
    }
    return off;
}
template <int N>
struct LastTw {
    static constexpr int P = ppt_for(N), NS = last_stage_ns(N), R = radix_for(N, NS), OFF = last_stage_off(N);
    static constexpr int COUNT = (P / R) * (R - 1);
    float4 w[COUNT];
    template <bool HILO>
    __device__ __forceinline__ void load(int j, const float4 *__restrict__ tw)
    {
        load_twiddles<N, R, NS, OFF, HILO, P>(w, j, tw);
    }
};

template <int N, int NSP, int RP, int OFF, int DIR, bool HILO, class SM, int P>
__device__ __forceinline__ void fft_next(cp2 (&x)[P], int j, const float4 *__restrict__ tw, SM &sm,
                                         const LastTw<N> *res = nullptr)
{
    constexpr int NS = NSP * RP, R = radix_for(N, NS);
    constexpr bool H = stage_hilo<HILO, NS>();
    if constexpr (NS * R == N) {
        if (res != nullptr) { // last stage with resident twiddles (res is a compile-time-known pointer after inlining)
            exchange_store<N, RP, NSP>(x, j, sm);
            exchange_load<N>(x, j, sm);
            stage_compute<N, R, NS, DIR, H>(x, res->w);
            return;
        }
    }
    float4 w[(P / R) * (R - 1)];
    exchange_store<N, RP, NSP>(x, j, sm);
    if (SN_TW_PREFETCH) load_twiddles<N, R, NS, OFF, H, P>(w, j, tw);
    exchange_load<N>(x, j, sm);
    if (!SN_TW_PREFETCH) load_twiddles<N, R, NS, OFF, H, P>(w, j, tw);
    stage_compute<N, R, NS, DIR, H>(x, w);
    if constexpr (NS * R < N) fft_next<N, NS, R, OFF + NS * (R - 1), DIR, HILO, SM>(x, j, tw, sm, res);
}

// Unscaled DFT of a packed line pair; same contract as fft_pair.
template <int N, int DIR, bool HILO, class SM, int P>
__device__ __forceinline__ void fft_pair(cp2 (&x)[P], int j, const float4 *__restrict__ tw, SM &sm,
                                         const LastTw<N> *res = nullptr)
{
    static_assert(P == ppt_for(N), "points per thread");
    if constexpr (packed_for(N)) {
        constexpr int R = radix_for(N, 1);
        const float4 none[(P / R) * (R - 1)] = {};
        stage_compute<N, R, 1, DIR, HILO>(x, none);
        if constexpr (R < N) fft_next<N, 1, R, 0, DIR, HILO, SM>(x, j, tw, sm, res);
    } else { // scalar engine on the same registers (the repacking is register naming)
        float2 a[P], b[P];
#pragma unroll
        for (int m = 0; m < P; m++) {
            a[m] = line_a(x[m]);
            b[m] = line_b(x[m]);
        }
        fft_pair_scalar<N, DIR, HILO>(a, b, j, tw, sm);
#pragma unroll
        for (int m = 0; m < P; m++) x[m] = pack_pair(a[m], b[m]);
    }
}

// Line pair given as two complex arrays: through the packed engine (the repacking is register naming).
template <int N, int DIR, bool HILO, class SM, int P>
__device__ __forceinline__ void fft_pair(float2 (&a)[P], float2 (&b)[P], int j, const float4 *__restrict__ tw, SM &sm)
{
    if constexpr (packed_for(N)) {
        cp2 x[P];
#pragma unroll
        for (int m = 0; m < P; m++) x[m] = pack_pair(a[m], b[m]);
        fft_pair<N, DIR, HILO>(x, j, tw, sm);
#pragma unroll
        for (int m = 0; m < P; m++) {
            a[m] = line_a(x[m]);
            b[m] = line_b(x[m]);
        }
    } else {
        fft_pair_scalar<N, DIR, HILO>(a, b, j, tw, sm);
    }
}

// ---- shared-memory accessors -------------------------------------------------------------
// One exchange position = one float4 (two register pairs of the packed engine: r = (a.re, b.re), i = (a.im, b.im); or the
// two complex values of the scalar engine).  Written as `*p = make_float4(...)`, ptxas builds the four CONSECUTIVE
// registers of the STS.128 with four MOVs per store (S_KIN at N = 512: 160 of 1150 instructions; the cluster-resident
// kernel: 14 % of its instruction stream).  Written as two 64-bit stores in inline PTX it allocates the two pairs
// adjacently and still fuses them into one STS.128 (SASS checked: same STS.128 count, MOVs gone).
#ifndef SN_XCH_PTX_STORES
#define SN_XCH_PTX_STORES 1 // 0: plain C++ store (A/B builds)
#endif
__device__ __forceinline__ void xch_store(float4 *p, float2 a, float2 b)
{
#if SN_XCH_PTX_STORES
    const unsigned addr = (unsigned)__cvta_generic_to_shared(p);
    asm volatile("st.shared.v2.f32 [%0], {%1, %2};" ::"r"(addr), "f"(a.x), "f"(a.y) : "memory");
    asm volatile("st.shared.v2.f32 [%0+8], {%1, %2};" ::"r"(addr), "f"(b.x), "f"(b.y) : "memory");
#else
    *p = make_float4(a.x, a.y, b.x, b.y);
#endif
}

// One float4 per point position: (a.re, a.im, b.re, b.im).  Interface: lin(pos) = linear index of a
// position (group constant excluded), TMASK = index bits the group constant occupies,
// idx(pos) = lin(pos) ^ group constant, st_i / ld_i = access by index.

// Tile of CP column pairs per row (strided-axis kernels); thread t owns column pair t.  With
// CP = 8 a row is 128 B = all 32 banks and 8 adjacent lanes cover it, so every 128-bit access
// phase is conflict-free for any row pattern.  Narrower tiles (long lines) XOR the chunk index
// with row bits 3.. so that the stride-8 rows written after the first stage spread over banks.
template <int CP>
struct SmemTile {
    float4 *base;
    int t;
    static constexpr int TMASK = CP - 1;
    __host__ __device__ static constexpr int lin(int pos)
    {
        if (CP == 8) return pos * 8;
        if (CP == 4) return (pos * 4) ^ (((pos >> 3) & 1) << 2);
        if (CP == 2) return (pos * 2) ^ (((pos >> 3) & 3) << 1);
        return pos ^ ((pos >> 3) & 7);
    }
    __device__ __forceinline__ int idx(int pos) const { return lin(pos) ^ t; }
    __device__ __forceinline__ void st_i(int i, float2 a, float2 b) const { xch_store(base + i, a, b); }
    __device__ __forceinline__ void ld_i(int i, float2 &a, float2 &b) const
    {
        const float4 v = base[i];
        a = make_float2(v.x, v.y);
        b = make_float2(v.z, v.w);
    }
    __device__ __forceinline__ void st(int pos, float2 a, float2 b) const { st_i(idx(pos), a, b); }
    __device__ __forceinline__ void ld(int pos, float2 &a, float2 &b) const { ld_i(idx(pos), a, b); }
    __device__ __forceinline__ void sync() const { __syncthreads(); }
};

// One line pair per T-thread group, lanes = consecutive j (contiguous-axis kernel).  XOR
// swizzle of the low 3 position bits with bits 3..5 makes the stride-8 writes of the first
// stage conflict-free and keeps unit-stride accesses conflict-free.
template <int T>
struct SmemLine {
    float4 *base;
    int bar_id; // named barrier for this group when T > 32 and the CTA holds several groups
    bool whole_cta;
    static constexpr int TMASK = 0;
    __host__ __device__ static constexpr int lin(int pos) { return pos ^ ((pos >> 3) & 7); }
    __device__ __forceinline__ int idx(int pos) const { return lin(pos); }
    __device__ __forceinline__ void st_i(int i, float2 a, float2 b) const { xch_store(base + i, a, b); }
    __device__ __forceinline__ void ld_i(int i, float2 &a, float2 &b) const
    {
        const float4 v = base[i];
        a = make_float2(v.x, v.y);
        b = make_float2(v.z, v.w);
    }
    __device__ __forceinline__ void st(int pos, float2 a, float2 b) const { st_i(idx(pos), a, b); }
    __device__ __forceinline__ void ld(int pos, float2 &a, float2 &b) const { ld_i(idx(pos), a, b); }
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

} // namespace snk
