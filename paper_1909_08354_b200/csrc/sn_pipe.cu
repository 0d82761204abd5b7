// sn_pipe.cu -- pipelined, persistent, TMA-fed versions of the hot pass kernels (sm_100a),
// compiled once per line length (-DSN_LEN=N).
//
// Why: the first-path kernels (sn_kernels.cu) are "load tile -> FFT -> store" with the three
// phases serialised inside a CTA whose 128 registers/thread allow one 512-thread CTA per SM:
// ncu showed DRAM 20-58 % busy, issue slots 25-57 % busy, the dominant stall the global loads
// (profiles/r01a_first_path_C5_512.md).  Here one 512-thread CTA per SM loops over tiles; the
// TMA unit moves 64 KB tiles between HBM and a ring of shared-memory stages
// (cp.async.bulk.tensor with 128-byte swizzle for strided lines, cp.async.bulk for contiguous
// lines), completion is tracked with mbarriers, and the butterflies of tile k run while tile
// k+1/k+2 are landing and tile k-1 is draining.  No register is spent on global addresses.
//
// Tile geometry (strided kinds): T = N/P threads carry one PAIR of adjacent columns (a "line pair", one float4 =
// 2 complex per row; P = 8 points per thread, 12 for N = 3*2^a); G = threads/T groups per CTA; a tile is N rows x
// 2G columns, stored as sub-tiles of [N rows][16*CPW bytes], CPW = min(G, 8) column pairs per row.  The TMA
// swizzle of that width (128B / 64B / 32B / none) puts the 16-byte chunk c of row r at chunk c ^ swz(r), and in
// every case the bank unit is a bijection of (r & 7): the 8 lanes of a quarter-warp (consecutive rows, same
// column pair) hit 8 different bank groups, so every 128-bit access is conflict-free.  A group only ever touches
// its own N slots (one per row), so the Stockham exchanges of its FFT run IN PLACE in the tile, position pos
// living in the slot of row pos ^ ((pos >> 3) & 7).
//
// Which passes actually run these kernels is decided per line length in sn_api.cu (run_pass_raw): measured, the
// axis-0 nonlinear pass always, the other kinds at N = 512 and N >= 2048.
#include "sn_fft_core.cuh"
#include "sn_launch.h"
#include "sn_pointwise.cuh"
#include "sn_tma.cuh"

#ifndef SN_LEN
#error "compile with -DSN_LEN=<line length>"
#endif

namespace snk {

// keep the last stage's hi/lo twiddles of the psi transforms in registers across tiles (sn_fft_core.cuh, LastTw)?
#ifndef SN_RES_TW
#define SN_RES_TW 1
#endif
#ifndef SN_RES_TW_ALL
#define SN_RES_TW_ALL 0
#endif
// (N <= 512: at 1024 and above the extra live registers spill, measured with -Xptxas -v)
__host__ __device__ constexpr bool res_tw_for(int N) { return SN_RES_TW && packed_for(N) && (N <= 512 || SN_RES_TW_ALL); }

template <int N>
struct Geo {
    static constexpr int P = pipe_ppt(N);                 // points per thread and line
    static constexpr int NTHR = pipe_threads(N);          // threads per CTA
    static constexpr int NWARP = NTHR / 32;
    static constexpr int T = N / P;                       // threads per line pair
    static constexpr int G = NTHR / T;                    // line pairs (groups) per tile
    static constexpr int TILE_BYTES = N * 2 * G * 8;      // 64 KB (N = 2^n) or 48 KB (N = 3*2^a)
    static constexpr int CPW = pipe_cpw(N);               // column pairs per sub-tile row (8 for N <= 512, then 4, 2, 1; 4 at N = 384)
    static constexpr int RBY = 16 * CPW;                  // bytes of a sub-tile row: 128, 64, 32, 16
    static constexpr int SUB = G / CPW;                   // sub-tiles per tile
    static constexpr int RB = pipe_box_rows(N);           // rows per TMA box
    static constexpr int NBOX = N / RB;
    static constexpr int SUB_F4 = N * CPW;                // float4 slots of a psi sub-tile
    static constexpr int SUB_BYTES = N * RBY;
    static constexpr int HROWS = N / 2 + 1;               // rows of the half spectrum
    static constexpr int HB = pipe_box_rows(N / 2);       // rows per TMA box of the half spectrum (rows 0..N/2-1)
    static constexpr int NHBOX = (N / 2) / HB;
    static constexpr int HS_SUB_BYTES = (HROWS * RBY + 1023) / 1024 * 1024;
    static constexpr int HS_SUB_F4 = HS_SUB_BYTES / 16;
    static constexpr int HS_TX = SUB * HROWS * RBY;       // bytes one hs tile load delivers
    static_assert(T % 8 == 0 && G * T == NTHR && SUB * CPW == G && NBOX * RB == N && NHBOX * HB == N / 2, "geometry");
};

// Slot (float4 index inside a sub-tile) of row r for column pair t < CPW: the layout the TMA swizzle of a
// RBY-byte-wide box produces (SWIZZLE_128B / 64B / 32B / none): chunk t of row r sits at chunk t ^ swz(r).
// In every case the 16-byte bank unit (slot mod 8) is a bijection of (r & 7) for fixed t, so 8 lanes on 8
// consecutive rows never conflict.
template <int CPW>
__host__ __device__ constexpr int swz(int r)
{
    return CPW == 8 ? (r & 7) : CPW == 4 ? ((r >> 1) & 3) : CPW == 2 ? ((r >> 2) & 1) : 0;
}
template <int CPW>
__device__ __forceinline__ int nat_slot(int r, int t) { return r * CPW + (t ^ swz<CPW>(r)); }

// Exchange accessor for a line PAIR living in its own slots of a swizzled sub-tile: position pos
// lives in the slot of row pos ^ ((pos >> 3) & 7).
template <int T, int CPW>
struct SmemSub {
    float4 *sub;
    int t, bar_id;
    static constexpr int TMASK = CPW - 1;
    __host__ __device__ static constexpr int lin(int pos)
    {
        const int r = pos ^ ((pos >> 3) & 7);
        return (r * CPW) | swz<CPW>(r);
    }
    __device__ __forceinline__ int idx(int pos) const { return lin(pos) ^ t; }
    __device__ __forceinline__ void st_i(int i, float2 a, float2 b) const { xch_store(sub + i, a, b); }
    __device__ __forceinline__ void ld_i(int i, float2 &a, float2 &b) const
    {
        const float4 v = sub[i];
        a = lo2(v);
        b = hi2(v);
    }
    __device__ __forceinline__ void sync() const
    {
        if (T <= 32) __syncwarp();
        else named_bar_sync(bar_id, T);
    }
};

// Exchange accessor for ONE line (float2 per position) living in the first N/2 slots of a group's
// column pair: position pos -> row q ^ ((q >> 2) & 7) ^ (4 if q bit 5), q = pos >> 1, half (pos ^ (pos >> 6)) & 1.
// A 64-bit access is served per half-warp, so 16 lanes must land on 16 different 8-byte bank pairs: position bit 6
// (lane bit 3 in the stores after the NS = 8 stage) has to reach the row bits as well as the half bit -- without the
// "^ 4" term those stores were 2-way conflicted (ncu source page, profiles/r02g: 8 STS.64 per transform at twice
// their ideal wavefronts, 10 % of the r2c kernel's shared-memory wavefronts).
template <int T, int CPW>
struct SmemSubOne {
    float2 *sub2; // the sub-tile as float2
    int t, bar_id;
    static constexpr int TMASK = (CPW - 1) << 1;
    __host__ __device__ static constexpr int lin(int pos)
    {
#ifndef SN_SUBONE_BIT6
#define SN_SUBONE_BIT6 1
#endif
        const int q = pos >> 1, r = q ^ ((q >> 2) & 7) ^ (SN_SUBONE_BIT6 ? ((q >> 5) & 1) << 2 : 0);
        return (((r * CPW) | swz<CPW>(r)) << 1) | ((pos ^ (pos >> 6)) & 1);
    }
    __device__ __forceinline__ int idx(int pos) const { return lin(pos) ^ (t << 1); }
    __device__ __forceinline__ void st_i(int i, float2 a, float2) const { sub2[i] = a; }
    __device__ __forceinline__ void ld_i(int i, float2 &a, float2 &) const { a = sub2[i]; }
    __device__ __forceinline__ void st(int pos, float2 a, float2 b) const { st_i(idx(pos), a, b); }
    __device__ __forceinline__ void ld(int pos, float2 &a, float2 &b) const { ld_i(idx(pos), a, b); }
    __device__ __forceinline__ void sync() const
    {
        if (T <= 32) __syncwarp();
        else named_bar_sync(bar_id, T);
    }
};

// a value the compiler cannot hoist out of the tile loop or merge with another copy (keeps it from
// precomputing per-thread address tables / re-using twiddles across transforms through local memory)
__device__ __forceinline__ int opaque(int v)
{
    asm volatile("" : "+r"(v));
    return v;
}

__device__ __forceinline__ uint8_t *align_1024(uint8_t *p)
{
    return p + ((1024u - (smem_u32(p) & 1023u)) & 1023u);
}

// all warps: "this warp is done with the stage" (generic writes fenced for the TMA store)
__device__ __forceinline__ void warp_arrive_done(uint64_t *bar)
{
    fence_proxy_async();
    __syncwarp();
    if ((threadIdx.x & 31) == 0) mbar_arrive(bar);
}

// kinetic phase on a line pair: a, b *= phase[j + T m]   (S2 of SURVEY.md 8(a), separable per axis)
template <int T, int P>
__device__ __forceinline__ void apply_phase(cp2 (&x)[P], int j, const float4 *__restrict__ phase)
{
#pragma unroll
    for (int m = 0; m < P; m++) x[m] = twmul<+1, true>(x[m], __ldg(phase + j + T * m));
}

// ---------------------------------------------------------------------------- strided axis
// P_S_KIN: forward -> kinetic phase -> inverse along a strided axis; P_S_FFT: plain transform.
// 3-stage ring.  Thread 0 is the issuer: at the end of tile k it waits until every warp has
// released the stage, stores it, and reloads the stage that tile k-1 was stored from with tile k+2.

template <int N, int MODE, int DIR, bool HILO>
__global__ void __launch_bounds__(pipe_threads(N), 1) k_pipe_strided(const __grid_constant__ PipeArgs p)
{
    using g_ = Geo<N>;
    constexpr int P = g_::P, TILE_BYTES = g_::TILE_BYTES, PIPE_WARPS = g_::NWARP, T = g_::T, G = g_::G, CPW = g_::CPW, RBY = g_::RBY, SUB = g_::SUB, RB = g_::RB, NBOX = g_::NBOX, NST = 3;
    extern __shared__ uint8_t smem_raw[];
    uint8_t *base = align_1024(smem_raw);
    uint64_t *full = reinterpret_cast<uint64_t *>(base + NST * TILE_BYTES), *done = full + NST;
    const int tid = threadIdx.x, g = tid / T, j = tid % T, s = g / CPW, t = g % CPW;

    if (tid == 0) {
        for (int i = 0; i < NST; i++) {
            mbar_init(full + i, 1);
            mbar_init(done + i, PIPE_WARPS);
        }
        mbar_fence_init();
    }
    __syncthreads();

    const int nk = (p.n_tiles - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x;
    auto tile_coords = [&](int k, int &outer, int &col0) {
        const int tile = blockIdx.x + k * gridDim.x;
        outer = tile / p.tiles_per_outer;
        col0 = (tile % p.tiles_per_outer) * 2 * G;
    };
    auto issue_load = [&](int k) {
        int outer, col0;
        tile_coords(k, outer, col0);
        const int b = k % NST;
        mbar_arrive_expect_tx(full + b, TILE_BYTES);
#pragma unroll
        for (int ss = 0; ss < SUB; ss++)
#pragma unroll
            for (int bx = 0; bx < NBOX; bx++)
                tma_load_3d(base + b * TILE_BYTES + ss * g_::SUB_BYTES + bx * RB * RBY, &p.m_data, full + b,
                            2 * (col0 + 2 * CPW * ss), bx * RB, outer);
    };
    if (tid == 0) {
        if (nk > 0) issue_load(0);
        if (nk > 1) issue_load(1);
    }
    LastTw<N> wres;
    constexpr bool RES = res_tw_for(N);
    if (RES) wres.template load<MODE == P_S_KIN || HILO>(j, p.a.tw);
    const LastTw<N> *res = RES ? &wres : nullptr;

    for (int k = 0; k < nk; k++) {
        const int b = k % NST;
        const uint32_t par = (k / NST) & 1;
        float4 *sub = reinterpret_cast<float4 *>(base + b * TILE_BYTES) + s * g_::SUB_F4;
        SmemSub<T, CPW> sm{sub, t, 1 + g};
        mbar_wait(full + b, par);

        const int jf = opaque(j), ji = opaque(j); // per-tile copies: see opaque()
        float4 *mine = sub + nat_slot<CPW>(jf, t);     // row jf; rows jf + T m are CPW T m slots further (T % 8 == 0)
        cp2 x[P]; // the column pair, packed (sn_fft_core.cuh)
#pragma unroll
        for (int m = 0; m < P; m++) x[m] = unpack4(mine[CPW * T * m]);
        if (MODE == P_S_FFT) {
            fft_pair<N, DIR, HILO>(x, jf, p.a.tw, sm, res);
            if (DIR < 0) {
                const float sc = p.a.scale;
#pragma unroll
                for (int m = 0; m < P; m++) x[m] = cscale(x[m], sc);
            }
        } else { // P_S_KIN
            fft_pair<N, +1, true>(x, jf, p.a.tw, sm, res);
            apply_phase<T, P>(x, jf, p.a.phase);
            fft_pair<N, -1, true>(x, ji, p.a.tw, sm, res);
        }
        // the last exchange's reads and these writes can only collide inside an aligned group of 8 lanes
        __syncwarp();
#pragma unroll
        for (int m = 0; m < P; m++) mine[CPW * T * m] = pack4(x[m]);
        warp_arrive_done(done + b);

        if (tid == 0) {
            mbar_wait(done + b, par);
            int outer, col0;
            tile_coords(k, outer, col0);
#pragma unroll
            for (int ss = 0; ss < SUB; ss++)
#pragma unroll
                for (int bx = 0; bx < NBOX; bx++)
                    tma_store_3d(&p.m_data, base + b * TILE_BYTES + ss * g_::SUB_BYTES + bx * RB * RBY, 2 * (col0 + 2 * CPW * ss),
                                 bx * RB, outer);
            bulk_commit();
            if (k + 2 < nk) {
                bulk_wait_read<1>(); // the store of tile k-1 has left its stage
                issue_load(k + 2);
            }
        }
    }
    if (tid == 0) bulk_wait<0>();
}

// ---------------------------------------------------------------------------- axis 0 ("h") kernels
// P_H_NLKIN (S7, S8, S1-S3 of SURVEY.md 8(a)): c2r of phi^ along axis 0 -> nonlinear phase on psi ->
// forward -> kinetic phase -> inverse along axis 0.  P_H_R2C (S4, S5): rho = |psi|^2 -> packed r2c.
// A group's two psi columns 2t, 2t+1 carry two REAL columns of rho / phi as ONE complex line
// z = x + i y (two-for-one trick):
//   X[k] = (Z[k] + conj Z[N-k])/2,  Y[k] = (Z[k] - conj Z[N-k])/(2i),  k = 0..N/2;
//   inverse: Z[k] = X[k] + i Y[k] (k <= N/2), Z[N-k] = conj X[k] + i conj Y[k];
// the factor 1/2 is folded into the Poisson multiplier (PassArgs::pscale).
// Stage = psi tile (64 KB) + half-spectrum tile ((N/2+1) rows, <= 33 KB); 2-stage ring.  The stage
// that tile k was stored from is reloaded with tile k+2 from a point INSIDE tile k+1's compute, so
// the issuer never waits for its own store to drain.

template <int N, int MODE, bool EXTRA>
__global__ void __launch_bounds__(pipe_threads(N), 1) k_pipe_haxis(const __grid_constant__ PipeArgs p)
{
    using g_ = Geo<N>;
    constexpr int P = g_::P, TILE_BYTES = g_::TILE_BYTES, PIPE_WARPS = g_::NWARP, T = g_::T, G = g_::G, CPW = g_::CPW, RBY = g_::RBY, SUB = g_::SUB, RB = g_::RB, NBOX = g_::NBOX, NST = 2;
    constexpr int STAGE_BYTES = TILE_BYTES + SUB * g_::HS_SUB_BYTES;
    constexpr bool LOAD_HS = true;
    static_assert(MODE == P_H_NLKIN || MODE == P_H_BOHM, "k_pipe_haxis serves P_H_NLKIN and P_H_BOHM");
    extern __shared__ uint8_t smem_raw[];
    uint8_t *base = align_1024(smem_raw);
    uint64_t *full = reinterpret_cast<uint64_t *>(base + NST * STAGE_BYTES), *done = full + NST;
    // tiles are handed out by a device-wide counter (p.sched[0]), not round-robin: measured at 384^3 and 256^3 a
    // few CTAs of the static schedule ran up to twice as long as the rest (sm__cycles_active min/avg/max
    // 0.93/1.2/1.9 Mcycles, profiles/r01i).  tile_of[stage] = tile in that stage, -1 = no tile left.
    volatile int *tile_of = reinterpret_cast<volatile int *>(done + NST);
    const int tid = threadIdx.x, g = tid / T, j = tid % T, s = g / CPW, t = g % CPW;

    if (tid == 0) {
        for (int i = 0; i < NST; i++) {
            mbar_init(full + i, 1);
            mbar_init(done + i, PIPE_WARPS);
        }
        mbar_fence_init();
    }
    __syncthreads();

    bool more = true; // issuer only: the counter has not run out yet
    // launch-bound grids (a tile or two per CTA) keep the round-robin order: there the atomics' latency is not hidden
    // (C2 37 -> 41 us/step, 64^3 29 -> 32 with the counter)
    const bool dyn = p.n_tiles > 2 * (int)gridDim.x;
    auto issue_load = [&](int k) {
        const int b = k % NST;
        const int tile = dyn ? atomicAdd(p.sched, 1) : (int)(blockIdx.x + k * gridDim.x);
        if (tile >= p.n_tiles) {
            more = false;
            tile_of[b] = -1;
            mbar_arrive(full + b); // completes the phase with no bytes: every warp wakes up and sees -1
            return;
        }
        tile_of[b] = tile;
        const int col0 = tile * 2 * G;
        uint8_t *st = base + b * STAGE_BYTES;
        mbar_arrive_expect_tx(full + b, TILE_BYTES + (LOAD_HS ? g_::HS_TX : 0));
#pragma unroll
        for (int ss = 0; ss < SUB; ss++) {
#pragma unroll
            for (int bx = 0; bx < NBOX; bx++)
                tma_load_3d(st + ss * g_::SUB_BYTES + bx * RB * RBY, &p.m_data, full + b, 2 * (col0 + 2 * CPW * ss), bx * RB, 0);
            if (LOAD_HS) {
                uint8_t *hs = st + TILE_BYTES + ss * g_::HS_SUB_BYTES;
#pragma unroll
                for (int bx = 0; bx < g_::NHBOX; bx++)
                    tma_load_3d(hs + bx * g_::HB * RBY, &p.m_hs, full + b, 2 * (col0 + 2 * CPW * ss), bx * g_::HB, 0);
                tma_load_3d(hs + (N / 2) * RBY, &p.m_hs_row, full + b, 2 * (col0 + 2 * CPW * ss), N / 2, 0);
            }
        }
    };
    if (tid == 0) {
        issue_load(0);
        if (more) issue_load(1);
    }
    LastTw<N> wres; // the last stage's hi/lo twiddles of the psi transforms stay in registers across tiles
    constexpr bool RES = MODE == P_H_NLKIN && res_tw_for(N);
    if (RES) wres.template load<true>(j, p.a.tw);
    const LastTw<N> *res = RES ? &wres : nullptr;

    for (int k = 0;; k++) {
        const int b = k % NST;
        const uint32_t par = (k / NST) & 1;
        uint8_t *st = base + b * STAGE_BYTES;
        float4 *sub = reinterpret_cast<float4 *>(st) + s * g_::SUB_F4;
        float4 *hsub = reinterpret_cast<float4 *>(st + TILE_BYTES) + s * g_::HS_SUB_F4;
        SmemSub<T, CPW> sm{sub, t, 1 + g};
        mbar_wait(full + b, par);
        const int tile = tile_of[b];
        if (tile < 0) break;

        const int jf = opaque(j), ji = opaque(j), jz = opaque(j); // per-tile copies: see opaque()
        float4 *mine = sub + nat_slot<CPW>(jf, t);
        {
            float2 z[P];
            // rows jz + T m (m < P/2) and N - jz - T m (m >= P/2): the mirrored rows step DOWN by CPW T slots
            const float4 *hup = hsub + nat_slot<CPW>(jz, t), *hdn = hsub + nat_slot<CPW>(N / 2 - jz, t);
#pragma unroll
            for (int m = 0; m < P; m++) {
                const float4 u = m < P / 2 ? hup[CPW * T * m] : hdn[-CPW * T * (m - P / 2)];
                z[m] = m < P / 2 ? make_float2(u.x - u.w, u.y + u.z) : make_float2(u.x + u.w, u.z - u.y);
            }
            SmemSubOne<T, CPW> sm1{reinterpret_cast<float2 *>(hsub), t, 1 + g};
            fft_single<N, -1, false>(z, jz, p.a.tw, sm1);
            // z[m] = (phi[col 2t], phi[col 2t+1]) at row j + T m.  The previous tile's store has had the
            // whole c2r to leave its stage: reload it now.
            if (tid == 0 && k >= 1 && more) {
                bulk_wait_read<0>();
                issue_load(k + 1);
            }
            if (MODE == P_H_BOHM) {
                float2 a[P], c[P];
                // z = W = lap sqrt(rho) of the thread's two columns: psi *= exp(-i s c_B W/(2 max(sqrt(rho), floor))),
                // eq. (15); each thread rewrites only its own slots
#pragma unroll
                for (int m = 0; m < P; m++) {
                    const float4 v = mine[CPW * T * m];
                    a[m] = rotate_half_angle(lo2(v), p.a.hbohm * z[m].x / fmaxf(sqrtf(abs2(lo2(v))), p.a.sfloor));
                    c[m] = rotate_half_angle(hi2(v), p.a.hbohm * z[m].y / fmaxf(sqrtf(abs2(hi2(v))), p.a.sfloor));
                    mine[CPW * T * m] = pack4(a[m], c[m]);
                }
            } else {
                cp2 x[P];
#pragma unroll
                for (int m = 0; m < P; m++) {
                    nl_phase_pair<EXTRA>(mine[CPW * T * m], z[m], p.a.nl, x[m].r, x[m].i);
                }
                fft_pair<N, +1, true>(x, jf, p.a.tw, sm, res);
                apply_phase<T, P>(x, jf, p.a.phase);
                fft_pair<N, -1, true>(x, ji, p.a.tw, sm, res);
                __syncwarp();
#pragma unroll
                for (int m = 0; m < P; m++) mine[CPW * T * m] = pack4(x[m]);
            }
        }
        warp_arrive_done(done + b);

        if (tid == 0) {
            mbar_wait(done + b, par);
            const int col0 = tile * 2 * G;
#pragma unroll
            for (int ss = 0; ss < SUB; ss++)
#pragma unroll
                for (int bx = 0; bx < NBOX; bx++)
                    tma_store_3d(&p.m_data, st + ss * g_::SUB_BYTES + bx * RB * RBY, 2 * (col0 + 2 * CPW * ss), bx * RB, 0);
            bulk_commit();
        }
    }
    if (tid == 0) {
        bulk_wait<0>();
        // the last CTA to leave rewinds the counters for the next launch on the stream
        if (dyn) {
            __threadfence();
            if (atomicAdd(p.sched + 1, 1) == (int)gridDim.x - 1) {
                p.sched[0] = 0;
                p.sched[1] = 0;
            }
        }
    }
}

// P_H_R2C (S4, S5): rho = |psi|^2 -> packed real-to-complex transform along axis 0 -> half spectrum.
// Memory-bound (12 B/cell, one single-line FFT per column pair), so the two rings are decoupled:
// a psi stage is reloaded as soon as every warp has pulled its values into registers, and the
// transform runs in the OUTPUT buffer (a group's N/2+1 output slots hold its N float2 positions).
template <int N, bool SQRT>
__global__ void __launch_bounds__(pipe_threads(N), 1) k_pipe_r2c(const __grid_constant__ PipeArgs p)
{
    using g_ = Geo<N>;
    constexpr int P = g_::P, TILE_BYTES = g_::TILE_BYTES, PIPE_WARPS = g_::NWARP, T = g_::T, G = g_::G, CPW = g_::CPW, RBY = g_::RBY, SUB = g_::SUB, RB = g_::RB, NBOX = g_::NBOX, NST = 2;
    constexpr int OUT_BYTES = SUB * g_::HS_SUB_BYTES;
    extern __shared__ uint8_t smem_raw[];
    uint8_t *base = align_1024(smem_raw);
    uint8_t *outb = base + NST * TILE_BYTES;
    uint64_t *full = reinterpret_cast<uint64_t *>(outb + NST * OUT_BYTES), *consumed = full + NST, *done = full + 2 * NST,
             *freeb = full + 3 * NST;
    const int tid = threadIdx.x, g = tid / T, j = tid % T, s = g / CPW, t = g % CPW;

    if (tid == 0) {
        for (int i = 0; i < NST; i++) {
            mbar_init(full + i, 1);
            mbar_init(consumed + i, PIPE_WARPS);
            mbar_init(done + i, PIPE_WARPS);
            mbar_init(freeb + i, 1);
        }
        mbar_fence_init();
    }
    __syncthreads();

    const int nk = (p.n_tiles - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x;
    auto issue_load = [&](int k) {
        const int col0 = (blockIdx.x + k * gridDim.x) * 2 * G;
        const int b = k % NST;
        mbar_arrive_expect_tx(full + b, TILE_BYTES);
#pragma unroll
        for (int ss = 0; ss < SUB; ss++)
#pragma unroll
            for (int bx = 0; bx < NBOX; bx++)
                tma_load_3d(base + b * TILE_BYTES + ss * g_::SUB_BYTES + bx * RB * RBY, &p.m_data, full + b,
                            2 * (col0 + 2 * CPW * ss), bx * RB, 0);
    };
    if (tid == 0) {
        if (nk > 0) issue_load(0);
        if (nk > 1) issue_load(1);
    }

    for (int k = 0; k < nk; k++) {
        const int b = k % NST;
        const uint32_t par = (k / NST) & 1;
        const float4 *sub = reinterpret_cast<const float4 *>(base + b * TILE_BYTES) + s * g_::SUB_F4;
        float4 *hsub = reinterpret_cast<float4 *>(outb + b * OUT_BYTES) + s * g_::HS_SUB_F4;
        const int jf = opaque(j);
        mbar_wait(full + b, par);
        float2 z[P];
        {
            const float4 *mine = sub + nat_slot<CPW>(jf, t);
#pragma unroll
            for (int m = 0; m < P; m++) {
                const float4 v = mine[CPW * T * m];
                z[m] = make_float2(abs2(lo2(v)), abs2(hi2(v)));
                if (SQRT) z[m] = make_float2(sqrtf(z[m].x), sqrtf(z[m].y)); // Bohm term: transform of sqrt(rho)
            }
        }
        __syncwarp();
        if ((tid & 31) == 0) mbar_arrive(consumed + b);
        if (k >= NST) mbar_wait(freeb + b, ((k / NST) - 1) & 1); // the store of tile k-2 has left this output buffer

        SmemSubOne<T, CPW> sm1{reinterpret_cast<float2 *>(hsub), t, 1 + g};
        fft_single<N, +1, false>(z, jf, p.a.tw, sm1);
        if (tid == 0 && k + NST < nk) {
            mbar_wait(consumed + b, par);
            issue_load(k + NST);
        }
        // X[k] and Y[k] from Z[k] and Z[N-k]: pass Z through the buffer once more
        float2 dummy = make_float2(0.f, 0.f), y[P / 2 + 1];
        sm1.sync();
#pragma unroll
        for (int m = 0; m < P; m++) sm1.st(jf + T * m, z[m], dummy);
        sm1.sync();
#pragma unroll
        for (int m = 0; m <= P / 2; m++)
            if (m < P / 2 || j == 0) sm1.ld((N - (jf + T * m)) % N, y[m], dummy);
        sm1.sync();
#pragma unroll
        for (int m = 0; m <= P / 2; m++)
            if (m < P / 2 || j == 0)
                hsub[nat_slot<CPW>(jf + T * m, t)] =
                    make_float4(z[m].x + y[m].x, z[m].y - y[m].y, z[m].y + y[m].y, y[m].x - z[m].x);
        warp_arrive_done(done + b);

        if (tid == 0) {
            mbar_wait(done + b, par);
            const int col0 = (blockIdx.x + k * gridDim.x) * 2 * G;
#pragma unroll
            for (int ss = 0; ss < SUB; ss++) {
                const uint8_t *hs = outb + b * OUT_BYTES + ss * g_::HS_SUB_BYTES;
#pragma unroll
                for (int bx = 0; bx < g_::NHBOX; bx++)
                    tma_store_3d(&p.m_hs, hs + bx * g_::HB * RBY, 2 * (col0 + 2 * CPW * ss), bx * g_::HB, 0);
                tma_store_3d(&p.m_hs_row, hs + (N / 2) * RBY, 2 * (col0 + 2 * CPW * ss), N / 2, 0);
            }
            bulk_commit();
            if (k >= 1) {
                bulk_wait_read<1>(); // the store of tile k-1 has drained: its buffer is free for tile k+1
                mbar_arrive(freeb + ((k + 1) % NST));
            }
        }
    }
    if (tid == 0) bulk_wait<0>();
}

// P_H_SRC (eq. (12); NEXT-1): the half spectrum holds F[lap rho].  Per tile: c2r along axis 0 ->
// s = gamma rho + beta lap rho from psi and the interleaved (beta, gamma) table -> packed r2c -> F[s], in place in
// the half-spectrum tile.  Memory-bound (4 + 8 + 8 + 4 B/cell), so both inputs are prefetched one tile ahead:
// two half-spectrum buffers (in/out in place) and ONE auxiliary stage (psi tile + table tile) that is reloaded as
// soon as every warp has turned it into registers.
template <int N>
__global__ void __launch_bounds__(pipe_threads(N), 1) k_pipe_src(const __grid_constant__ PipeArgs p)
{
    using g_ = Geo<N>;
    constexpr int P = g_::P, TILE_BYTES = g_::TILE_BYTES, PIPE_WARPS = g_::NWARP, T = g_::T, G = g_::G, CPW = g_::CPW,
                  RBY = g_::RBY, SUB = g_::SUB, RB = g_::RB, NBOX = g_::NBOX;
    constexpr int HS_BYTES = SUB * g_::HS_SUB_BYTES;
    extern __shared__ uint8_t smem_raw[];
    uint8_t *base = align_1024(smem_raw);       // [psi tile][bg tile][hs buffer 0][hs buffer 1][barriers]
    uint8_t *hsb = base + 2 * TILE_BYTES;
    uint64_t *hfull = reinterpret_cast<uint64_t *>(hsb + 2 * HS_BYTES), *done = hfull + 2, *afull = hfull + 4, *ause = hfull + 5;
    const int tid = threadIdx.x, g = tid / T, j = tid % T, s = g / CPW, t = g % CPW;

    if (tid == 0) {
        for (int i = 0; i < 2; i++) {
            mbar_init(hfull + i, 1);
            mbar_init(done + i, PIPE_WARPS);
        }
        mbar_init(afull, 1);
        mbar_init(ause, PIPE_WARPS);
        mbar_fence_init();
    }
    __syncthreads();

    const int nk = (p.n_tiles - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x;
    auto col_of = [&](int k) { return (int)(blockIdx.x + k * gridDim.x) * 2 * G; };
    auto issue_hs = [&](int k) {
        const int col0 = col_of(k), b = k & 1;
        mbar_arrive_expect_tx(hfull + b, g_::HS_TX);
#pragma unroll
        for (int ss = 0; ss < SUB; ss++) {
            uint8_t *hs = hsb + b * HS_BYTES + ss * g_::HS_SUB_BYTES;
#pragma unroll
            for (int bx = 0; bx < g_::NHBOX; bx++)
                tma_load_3d(hs + bx * g_::HB * RBY, &p.m_hs, hfull + b, 2 * (col0 + 2 * CPW * ss), bx * g_::HB, 0);
            tma_load_3d(hs + (N / 2) * RBY, &p.m_hs_row, hfull + b, 2 * (col0 + 2 * CPW * ss), N / 2, 0);
        }
    };
    auto issue_aux = [&](int k) {
        const int col0 = col_of(k);
        mbar_arrive_expect_tx(afull, 2 * TILE_BYTES);
#pragma unroll
        for (int ss = 0; ss < SUB; ss++)
#pragma unroll
            for (int bx = 0; bx < NBOX; bx++) {
                const int off = ss * g_::SUB_BYTES + bx * RB * RBY;
                tma_load_3d(base + off, &p.m_data, afull, 2 * (col0 + 2 * CPW * ss), bx * RB, 0);
                tma_load_3d(base + TILE_BYTES + off, &p.m_bg, afull, 2 * (col0 + 2 * CPW * ss), bx * RB, 0);
            }
    };
    if (tid == 0) {
        if (nk > 0) { issue_hs(0); issue_aux(0); }
        if (nk > 1) issue_hs(1);
    }

    for (int k = 0; k < nk; k++) {
        const int b = k & 1;
        const uint32_t hpar = (k >> 1) & 1, apar = k & 1;
        const float4 *psub = reinterpret_cast<const float4 *>(base) + s * g_::SUB_F4;
        const float4 *qsub = reinterpret_cast<const float4 *>(base + TILE_BYTES) + s * g_::SUB_F4;
        float4 *hsub = reinterpret_cast<float4 *>(hsb + b * HS_BYTES) + s * g_::HS_SUB_F4;
        const int jz = opaque(j), jf = opaque(j);
        SmemSubOne<T, CPW> sm1{reinterpret_cast<float2 *>(hsub), t, 1 + g};

        // c2r of F[lap rho] (two real columns as one complex line)
        mbar_wait(hfull + b, hpar);
        float2 z[P];
        {
            const float4 *hup = hsub + nat_slot<CPW>(jz, t), *hdn = hsub + nat_slot<CPW>(N / 2 - jz, t);
#pragma unroll
            for (int m = 0; m < P; m++) {
                const float4 u = m < P / 2 ? hup[CPW * T * m] : hdn[-CPW * T * (m - P / 2)];
                z[m] = m < P / 2 ? make_float2(u.x - u.w, u.y + u.z) : make_float2(u.x + u.w, u.z - u.y);
            }
        }
        fft_single<N, -1, false>(z, jz, p.a.tw, sm1);
        // the store of tile k-1 has had the whole c2r to drain: prefetch the half spectrum of tile k+1 into its buffer
        if (tid == 0 && k >= 1 && k + 1 < nk) {
            bulk_wait_read<0>();
            issue_hs(k + 1);
        }

        // s = gamma rho + beta lap rho for the thread's two columns at rows j + T m
        mbar_wait(afull, apar);
        {
            const float4 *pm = psub + nat_slot<CPW>(jf, t), *qm = qsub + nat_slot<CPW>(jf, t);
#pragma unroll
            for (int m = 0; m < P; m++) {
                const float4 v = pm[CPW * T * m], q = qm[CPW * T * m]; // q = (beta0, gamma0, beta1, gamma1)
                z[m] = make_float2(fmaf(q.y, abs2(lo2(v)), q.x * z[m].x), fmaf(q.w, abs2(hi2(v)), q.z * z[m].y));
            }
        }
        __syncwarp();
        if ((tid & 31) == 0) mbar_arrive(ause);

        // packed r2c of s, in place in the half-spectrum buffer
        fft_single<N, +1, false>(z, jf, p.a.tw, sm1);
        if (tid == 0 && k + 1 < nk) { // every warp has consumed the auxiliary stage: reload it for tile k+1
            mbar_wait(ause, apar);
            issue_aux(k + 1);
        }
        float2 dummy = make_float2(0.f, 0.f), y[P / 2 + 1];
        sm1.sync();
#pragma unroll
        for (int m = 0; m < P; m++) sm1.st(jf + T * m, z[m], dummy);
        sm1.sync();
#pragma unroll
        for (int m = 0; m <= P / 2; m++)
            if (m < P / 2 || j == 0) sm1.ld((N - (jf + T * m)) % N, y[m], dummy);
        sm1.sync();
#pragma unroll
        for (int m = 0; m <= P / 2; m++)
            if (m < P / 2 || j == 0)
                hsub[nat_slot<CPW>(jf + T * m, t)] =
                    make_float4(z[m].x + y[m].x, z[m].y - y[m].y, z[m].y + y[m].y, y[m].x - z[m].x);
        warp_arrive_done(done + b);

        if (tid == 0) {
            mbar_wait(done + b, hpar);
            const int col0 = col_of(k);
#pragma unroll
            for (int ss = 0; ss < SUB; ss++) {
                const uint8_t *hs = hsb + b * HS_BYTES + ss * g_::HS_SUB_BYTES;
#pragma unroll
                for (int bx = 0; bx < g_::NHBOX; bx++)
                    tma_store_3d(&p.m_hs, hs + bx * g_::HB * RBY, 2 * (col0 + 2 * CPW * ss), bx * g_::HB, 0);
                tma_store_3d(&p.m_hs_row, hs + (N / 2) * RBY, 2 * (col0 + 2 * CPW * ss), N / 2, 0);
            }
            bulk_commit();
        }
    }
    if (tid == 0) bulk_wait<0>();
}

// ---------------------------------------------------------------------------- contiguous axis
// P_X_KIN: forward -> kinetic phase -> inverse along the contiguous axis of psi; P_X_POISSON (S5-S7,
// eq. (2)): forward -> D/(C - k^2) -> inverse along the contiguous axis of the half
// spectrum.  A tile is 2G consecutive lines = one contiguous 64 KB run, moved with 1D bulk copies;
// a group owns two adjacent lines and exchanges inside its own 16*N bytes.  3-stage ring as above.

template <int N>
struct GeoX {
    static constexpr int P = pipe_ppt(N);
    static constexpr int NTHR = pipe_threads(N);
    static constexpr int T = N / P;
    static constexpr int G = NTHR / T;
    static constexpr int LINES = 2 * G;
    static constexpr int TILE_BYTES = LINES * N * 8;
};

// VEXT (P_X_KIN only): this is the last kinetic pass before an N sub-step, so psi is back in real space when
// the inverse transform ends: the phase exp(-i dtau V(x)) of a fixed external potential (phi_C of eq. (15),
// PAPER.md:102) commutes with the nonlinear phase and is applied here, where V arrives as contiguous lines
// (a second bulk copy per tile: 2 stages of 64 KB psi + 32 KB V instead of 3 stages of psi).
template <int N, int MODE, bool VEXT>
__global__ void __launch_bounds__(pipe_threads(N), 1) k_pipe_contig(const __grid_constant__ PipeArgs p)
{
    constexpr int P = GeoX<N>::P, TILE_BYTES = GeoX<N>::TILE_BYTES, PIPE_THREADS = GeoX<N>::NTHR, PIPE_WARPS = PIPE_THREADS / 32;
    constexpr int T = GeoX<N>::T, LINES = GeoX<N>::LINES, NST = VEXT ? 2 : 3;
    constexpr int STAGE_BYTES = VEXT ? TILE_BYTES + TILE_BYTES / 2 : TILE_BYTES;
    extern __shared__ uint8_t smem_raw[];
    uint8_t *base = align_1024(smem_raw);
    uint64_t *full = reinterpret_cast<uint64_t *>(base + NST * STAGE_BYTES), *done = full + NST;
    const int tid = threadIdx.x, g = tid / T, j = tid % T;

    if (tid == 0) {
        for (int i = 0; i < NST; i++) {
            mbar_init(full + i, 1);
            mbar_init(done + i, PIPE_WARPS);
        }
        mbar_fence_init();
    }
    __syncthreads();

    const int nk = (p.n_tiles - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x;
    auto tile_lines = [&](int k, long long &line0) {
        line0 = (long long)(blockIdx.x + k * gridDim.x) * LINES;
        const long long left = p.a.nlines - line0;
        return (int)(left < LINES ? left : LINES);
    };
    auto issue_load = [&](int k) {
        long long line0;
        const uint32_t bytes = (uint32_t)tile_lines(k, line0) * N * 8;
        const int b = k % NST;
        mbar_arrive_expect_tx(full + b, VEXT ? bytes + bytes / 2 : bytes);
        bulk_load_1d(base + b * STAGE_BYTES, p.a.data + line0 * N, bytes, full + b);
        if (VEXT) bulk_load_1d(base + b * STAGE_BYTES + TILE_BYTES, p.a.vext + line0 * N, bytes / 2, full + b);
    };
    if (tid == 0) {
        if (nk > 0) issue_load(0);
        if (nk > 1) issue_load(1);
    }
    LastTw<N> wres; // the last stage's twiddles stay in registers across tiles (sn_fft_core.cuh)
    constexpr bool RES = res_tw_for(N);
    if (RES) wres.template load<MODE == P_X_KIN>(j, p.a.tw);
    const LastTw<N> *res = RES ? &wres : nullptr;

    for (int k = 0; k < nk; k++) {
        const int b = k % NST;
        const uint32_t par = (k / NST) & 1;
        long long line0;
        const int nl = tile_lines(k, line0);
        float4 *grp = reinterpret_cast<float4 *>(base + b * STAGE_BYTES) + g * N; // two lines = N float4
        float2 *la = reinterpret_cast<float2 *>(grp), *lb = la + N;
        SmemLine<T> sm{grp, 1 + g, T == PIPE_THREADS};
        mbar_wait(full + b, par);

        if (2 * g < nl) {
            const int jf = opaque(j), ji = opaque(j); // per-tile copies: see opaque()
            cp2 x[P]; // the two lines, packed (sn_fft_core.cuh)
#pragma unroll
            for (int m = 0; m < P; m++) x[m] = pack_pair(la[jf + T * m], lb[jf + T * m]);
            if (MODE == P_X_KIN) {
                fft_pair<N, +1, true>(x, jf, p.a.tw, sm, res);
                if (NST == 2 && tid == 0 && k >= 1 && k + 1 < nk) { // reload the stage tile k-1 was stored from
                    bulk_wait_read<0>();
                    issue_load(k + 1);
                }
                apply_phase<T, P>(x, jf, p.a.phase);
                fft_pair<N, -1, true>(x, ji, p.a.tw, sm, res);
                if (VEXT) {
                    const float *va = reinterpret_cast<const float *>(base + b * STAGE_BYTES + TILE_BYTES) + 2 * g * N;
#pragma unroll
                    for (int m = 0; m < P; m++)
                        x[m] = pack_pair(rotate_half_angle(line_a(x[m]), p.a.nl.hv * va[ji + T * m]),
                                         rotate_half_angle(line_b(x[m]), p.a.nl.hv * va[N + ji + T * m]));
                }
            } else { // P_X_POISSON
                fft_pair<N, +1, false>(x, jf, p.a.tw, sm, res);
                const float2 ka = __ldg(p.a.dko + line0 + 2 * g), kb = __ldg(p.a.dko + line0 + 2 * g + 1);
#pragma unroll
                for (int m = 0; m < P; m++) {
                    const float2 kx = __ldg(p.a.ksq2 + jf + T * m);
                    x[m] = cscale(x[m], helmholtz_mult(ka, kx, p.a.pscale, p.a.lap), helmholtz_mult(kb, kx, p.a.pscale, p.a.lap));
                }
                fft_pair<N, -1, false>(x, ji, p.a.tw, sm, res);
            }
            sm.sync(); // exchange layout (float4 per position) != line layout: whole group must be done reading
#pragma unroll
            for (int m = 0; m < P; m++) {
                la[ji + T * m] = line_a(x[m]);
                lb[ji + T * m] = line_b(x[m]);
            }
        }
        warp_arrive_done(done + b);

        if (tid == 0) {
            mbar_wait(done + b, par);
            bulk_store_1d(p.a.data + line0 * N, base + b * STAGE_BYTES, (uint32_t)nl * N * 8);
            bulk_commit();
            if (NST == 3 && k + 2 < nk) {
                bulk_wait_read<1>(); // tile k+2 goes where tile k-1 was stored from
                issue_load(k + 2);
            }
            // two stages (VEXT): tile k+2 reuses THIS stage; it is reloaded from inside tile k+1's compute (below),
            // when this store has long drained, so the issuer never waits for it
        }
    }
    if (tid == 0) bulk_wait<0>();
}

// ---------------------------------------------------------------------------- launchers

template <class K>
static int launch_pipe_kernel(K kern, int threads, size_t smem_bytes, const PipeArgs &a)
{
    if (!smem_attr_done(reinterpret_cast<const void *>(kern))) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_bytes);
        if (e != cudaSuccess) return (int)e;
        smem_attr_mark(reinterpret_cast<const void *>(kern));
    }
    kern<<<a.grid, threads, smem_bytes, a.a.stream>>>(a);
    return (int)cudaGetLastError();
}

template <int N>
int launch_pipe(const PipeArgs &a)
{
    constexpr size_t SLACK = 1024 + 64; // alignment of the ring + the mbarriers
    constexpr int TILE_BYTES = Geo<N>::TILE_BYTES, NT = pipe_threads(N);
    constexpr size_t S3 = 3 * (size_t)TILE_BYTES + SLACK;
    if (a.a.kind == P_X_KIN)
        return a.a.vext ? launch_pipe_kernel(k_pipe_contig<N, P_X_KIN, true>, NT, S3, a)
                        : launch_pipe_kernel(k_pipe_contig<N, P_X_KIN, false>, NT, S3, a);
    if (a.a.kind == P_X_POISSON) return launch_pipe_kernel(k_pipe_contig<N, P_X_POISSON, false>, NT, S3, a);
    {
        constexpr size_t S2H = 2 * ((size_t)TILE_BYTES + Geo<N>::SUB * Geo<N>::HS_SUB_BYTES) + SLACK;
        switch (a.a.kind) {
        case P_S_KIN: return launch_pipe_kernel(k_pipe_strided<N, P_S_KIN, +1, true>, NT, S3, a);
        case P_S_FFT:
            if (a.a.dir > 0)
                return a.a.hilo ? launch_pipe_kernel(k_pipe_strided<N, P_S_FFT, +1, true>, NT, S3, a)
                                : launch_pipe_kernel(k_pipe_strided<N, P_S_FFT, +1, false>, NT, S3, a);
            return a.a.hilo ? launch_pipe_kernel(k_pipe_strided<N, P_S_FFT, -1, true>, NT, S3, a)
                            : launch_pipe_kernel(k_pipe_strided<N, P_S_FFT, -1, false>, NT, S3, a);
        case P_H_NLKIN:
            return (a.a.nl.flags & 1) ? launch_pipe_kernel(k_pipe_haxis<N, P_H_NLKIN, true>, NT, S2H, a)
                                      : launch_pipe_kernel(k_pipe_haxis<N, P_H_NLKIN, false>, NT, S2H, a);
        case P_H_R2C:
            return a.a.sqrt_rho ? launch_pipe_kernel(k_pipe_r2c<N, true>, NT, S2H, a)
                                : launch_pipe_kernel(k_pipe_r2c<N, false>, NT, S2H, a);
        case P_H_SRC: return launch_pipe_kernel(k_pipe_src<N>, NT, S2H + 0, a);
        case P_H_BOHM: return launch_pipe_kernel(k_pipe_haxis<N, P_H_BOHM, false>, NT, S2H, a);
        default: break;
        }
    }
    return (int)cudaErrorInvalidValue;
}

template int launch_pipe<SN_LEN>(const PipeArgs &a);

} // namespace snk
