// sn_resident.cu -- the whole Strang step of a small 2D system inside ONE thread-block cluster (sm_100a),
// compiled once per line length (-DSN_LEN=N, N in {64, 128}).
//
// Why: a 128 x 128 complex64 state is 128 KiB.  Run through the pass kernels, one step is four launches that each
// move the state L2 -> SM -> L2 for a few microseconds of latency and almost no work (C1: 25 us/step, 0.5 % of the
// HBM roofline).  Here the state never leaves the chip: a cluster of 8 CTAs holds it in its
// distributed shared memory, rank r owning rows [r N/8, (r+1) N/8), and ONE launch advances it by all n steps of an
// sn_step(n) call -- the state is read from HBM once and written once per call.
//
//   "row" sweeps (transforms along axis 1): each rank's own rows, in its own shared memory;
//   "column" sweeps (along axis 0): rank r takes the column pairs [r N/8, (r+1) N/8) and reads / writes its points in
//     place in the owners' shared memory (ld/st.shared::cluster, one float4 = both columns of a row; the row pitch of
//     N + 2 complex puts the 8 lanes of a quarter-warp on 8 different bank groups): no transposed copy exists;
//   a stored row keeps the two columns of a pair interleaved -- slot (row, c/2) = (re_c, re_c+1, im_c, im_c+1) -- which
//     IS the engine's packed register layout: a column sweep's 128-bit access and a row sweep's four 32-bit accesses per
//     point land in the register pairs directly (the first version stored complex values and spent 15 % of its
//     instructions re-packing);
//   between sweeps of different orientation: one hardware cluster barrier (barrier.cluster, release/acquire).
//
// One sub-step [N K] (S1-S13 of SURVEY.md 8(a); eq. (1),(2), method PAPER.md:113) is THREE sweeps, the
// orientation alternating (x = the axis of the sweep, y = the other one; the kinetic factors of the two axes commute
// and the transform of rho may start along either axis):
//   P   forward along x -> D/(C - k^2)/(N0 N1), phi^(0) = 0 if C = 0 -> inverse along x        on rho^ (forward along y done)
//   NK  inverse along y -> phi = Re; psi *= exp(-i dtau (B phi + G(rho))); forward -> kinetic phase -> inverse along y
//   KR  forward -> kinetic phase -> inverse along x on psi; rho = |psi|^2 -> forward along x   (the next step's P runs along y)
// rho is transformed as a COMPLEX field with zero imaginary part (no half spectrum: at this size the arithmetic is free
// and the data path is what is being shortened).  Same line-FFT engine, hi/lo arithmetic and nonlinear-phase routine as
// the pass kernels; the density / potential transforms use the plain twiddles like theirs.  Every table (twiddles,
// kinetic phases, the k^2 tables of eq. (2)) is copied into shared memory at kernel start: the acquire side of a
// cluster barrier invalidates L1 (SASS CCTL.IVALL), so table loads through L1 would miss after every barrier.
// Ensembles (sn_create_batch): one cluster per member.  The local terms of eq. (16) (logarithmic / power-law G) are a
// template variant of the nonlinear phase, and so is a fixed external potential V(x) (phi_C of eq. (15)), whose rows sit
// in the ranks' shared memory beside psi; contexts with source tables or the Bohm term take the pass kernels.
#include <cooperative_groups.h>
#include <stdint.h>

#define SN_TW_LOAD(p) (*(p)) // the engine's twiddle loads: the tables live in shared memory here
#define SN_NL_SLOW_OUTLINE   // the rare large-angle path of the nonlinear phase as a call (code size)
#include "sn_fft_core.cuh"
#include "sn_launch.h"
#include "sn_pointwise.cuh"

#ifndef SN_LEN
#error "compile with -DSN_LEN=<line length>"
#endif

namespace cg = cooperative_groups;

namespace snk {

template <int N>
struct RGeo {
    static constexpr int R = RES_CLUSTER;     // CTAs per cluster
    static constexpr int NL = N / R;          // rows owned by a rank = columns it transforms along axis 0
    static constexpr int P = 8, T = N / P;    // points per thread and line, threads per line pair
    static constexpr int G = NL / 2;          // line pairs per rank
    static constexpr int NTHR = G * T;        // 32 / 128 threads at N = 64 / 128
    static constexpr int PITCH = N + 2;       // complex per stored row
    static constexpr int NTW = twiddle_entries(N);
    // psi rows | rho rows | exchange buffers | twiddles (hi/lo + plain copy) | phases [slot][axis][N] | C - k0^2 [N] | k1^2 [N] | multipliers
    static constexpr size_t OFF_RHO = (size_t)NL * PITCH * 8;
    static constexpr size_t OFF_XCH = 2 * OFF_RHO;
    static constexpr size_t OFF_TW = OFF_XCH + (size_t)G * N * 16;
    static constexpr size_t OFF_PH = OFF_TW + (size_t)NTW * 24;
    static constexpr size_t OFF_DK0 = OFF_PH + 2 * RES_PH_SLOTS * (size_t)N * 16;
    static constexpr size_t OFF_K1 = OFF_DK0 + (size_t)N * 8;
    static constexpr size_t OFF_MUL = OFF_K1 + (size_t)N * 8; // multipliers of eq. (2) per thread: [orientation][m][thread] float2
    static constexpr size_t OFF_V = OFF_MUL + 2 * (size_t)P * NTHR * 8; // external potential rows: [NL][PITCH] floats, column pairs adjacent
    static constexpr size_t SMEM = OFF_V + (size_t)NL * PITCH * 4;
    static_assert(T == NL && T <= 32, "point j + T m of an axis-0 line lives in row j of rank m; a pair is one warp or less");
    static_assert(OFF_TW % 16 == 0 && OFF_PH % 16 == 0 && (NTW * 16) % 8 == 0, "table alignment");
};

// distributed shared memory through 32-bit shared::cluster addresses (a generic pointer per slot would cost 16 registers)
__device__ __forceinline__ uint32_t cluster_addr(const void *own_smem, uint32_t rank)
{
    uint32_t r;
    asm("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"((uint32_t)__cvta_generic_to_shared(own_smem)), "r"(rank));
    return r;
}
__device__ __forceinline__ float4 ld_cluster(uint32_t addr)
{
    float4 v;
    asm volatile("ld.shared::cluster.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(addr) : "memory");
    return v;
}
__device__ __forceinline__ void st_cluster(uint32_t addr, float4 v)
{
    asm volatile("st.shared::cluster.v4.f32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w) : "memory");
}

// a value the compiler cannot hoist out of the step loop (keeps it from precomputing per-thread address tables)
__device__ __forceinline__ int opaque(int v)
{
    asm volatile("" : "+r"(v));
    return v;
}

// Where the thread's line pair lives.  A stored row is N/2 + 1 slots of float4 = (re_c, re_c+1, im_c, im_c+1), one per
// column pair.  cols == false: the thread's two own rows; point p = j + T m of row r is the float at
// r * PF + 4 (p / 2) + (p & 1) (re) and 2 further (im): row0 points at it for m = 0 of the first row, the second row is PF
// floats further, consecutive m are 2 T floats apart (T is even).  cols == true: its column pair, point j + T m in row j
// of rank m (slot[m], one float4).  rho / phi^ sits at the same place in the rho rows (QB bytes further).
template <int N>
struct Lines {
    static constexpr int P = RGeo<N>::P, T = RGeo<N>::T, PF = 2 * RGeo<N>::PITCH;
    static constexpr uint32_t QB = (uint32_t)RGeo<N>::OFF_RHO;
    float *row0;
    uint32_t slot[P];

    template <bool RHO>
    __device__ __forceinline__ void load(cp2 (&x)[P], bool cols) const
    {
        if (cols) {
#pragma unroll
            for (int m = 0; m < P; m++) {
                const float4 v = ld_cluster(slot[m] + (RHO ? QB : 0u));
                x[m] = cp2{make_float2(v.x, v.y), make_float2(v.z, v.w)};
            }
        } else {
            const float *a = row0 + (RHO ? QB / 4 : 0), *b = a + PF;
#pragma unroll
            for (int m = 0; m < P; m++)
                x[m] = cp2{make_float2(a[2 * T * m], b[2 * T * m]), make_float2(a[2 * T * m + 2], b[2 * T * m + 2])};
        }
    }
    template <bool RHO>
    __device__ __forceinline__ void store(const cp2 (&x)[P], bool cols) const
    {
        if (cols) {
#pragma unroll
            for (int m = 0; m < P; m++) st_cluster(slot[m] + (RHO ? QB : 0u), make_float4(x[m].r.x, x[m].r.y, x[m].i.x, x[m].i.y));
        } else {
            float *a = row0 + (RHO ? QB / 4 : 0), *b = a + PF;
#pragma unroll
            for (int m = 0; m < P; m++) {
                a[2 * T * m] = x[m].r.x;
                b[2 * T * m] = x[m].r.y;
                a[2 * T * m + 2] = x[m].i.x;
                b[2 * T * m + 2] = x[m].i.y;
            }
        }
    }
};

template <int T, int P>
__device__ __forceinline__ void phase_mul(cp2 (&x)[P], int j, const float4 *phase)
{
#pragma unroll
    for (int m = 0; m < P; m++) x[m] = twmul<+1, true>(x[m], phase[j + T * m]);
}

// K along one axis: forward -> kinetic phase -> inverse.  with_rho: then rho = |psi|^2 -> forward along the same axis.
template <int N, class SM>
__device__ __forceinline__ void sweep_kin(const Lines<N> &ln, bool cols, bool with_rho, int j, const float4 *tw,
                                          const float4 *ph, SM &sm, const LastTw<N> *wpsi, const LastTw<N> *wrho)
{
    constexpr int P = RGeo<N>::P, T = RGeo<N>::T;
    cp2 x[P];
    ln.template load<false>(x, cols);
    fft_pair<N, +1, true>(x, j, tw, sm, wpsi);
    phase_mul<T, P>(x, j, ph);
    fft_pair<N, -1, true>(x, j, tw, sm, wpsi);
    ln.template store<false>(x, cols);
    if (with_rho) {
#pragma unroll
        for (int m = 0; m < P; m++) {
            x[m].r = __ffma2_rn(x[m].r, x[m].r, __fmul2_rn(x[m].i, x[m].i));
            x[m].i = make_float2(0.f, 0.f);
        }
        fft_pair<N, +1, false>(x, j, tw, sm, wrho);
        ln.template store<true>(x, cols);
    }
}

// PERIOD = the program's period (1: Strang, 3: fourth-order composition) as a compile-time constant: the Strang
// instantiation keeps constant table and coefficient indices (a run-time period costs C1 0.35 us/step)
// EXTRA: the logarithmic / power-law terms of eq. (16) (sn_set_local_terms) and / or an external potential
// (sn_set_external_potential) are in effect.
template <int N, int PERIOD, bool EXTRA>
__global__ void __cluster_dims__(RES_CLUSTER, 1, 1) __launch_bounds__(RGeo<N>::NTHR, 1)
    k_resident(const __grid_constant__ ResidentArgs a)
{
    using g_ = RGeo<N>;
    constexpr int R = g_::R, NL = g_::NL, P = g_::P, T = g_::T, NTHR = g_::NTHR, PITCH = g_::PITCH, NTW = g_::NTW;
    cg::cluster_group cluster = cg::this_cluster();
    const int rank = (int)cluster.block_rank();
    const int member = blockIdx.x / R;
    extern __shared__ __align__(16) uint8_t smem_raw[];
    float *psis = reinterpret_cast<float *>(smem_raw);                       // [NL][2 PITCH] this rank's rows of psi (slots, see Lines)
    float4 *xch = reinterpret_cast<float4 *>(smem_raw + g_::OFF_XCH);        // [G][N] exchange buffers of the line-FFT engine
    float4 *tw = reinterpret_cast<float4 *>(smem_raw + g_::OFF_TW);          // twiddles: hi/lo table, then the plain copy
    float4 *phs = reinterpret_cast<float4 *>(smem_raw + g_::OFF_PH);         // kinetic phases [slot][axis][N]
    float2 *dk0 = reinterpret_cast<float2 *>(smem_raw + g_::OFF_DK0);        // C - k0^2 per index of axis 0 (hi + lo)
    float2 *k1s = reinterpret_cast<float2 *>(smem_raw + g_::OFF_K1);         // k1^2 per index of axis 1 (hi + lo)
    float2 *mul = reinterpret_cast<float2 *>(smem_raw + g_::OFF_MUL);        // D/(C - k^2)/(N0 N1) of the thread's points, both orientations
    float *vrows = reinterpret_cast<float *>(smem_raw + g_::OFF_V);          // this rank's rows of the external potential
    const int tid = threadIdx.x, g = tid / T, j = tid % T;
    SmemLine<T> sm{xch + g * N, 1 + g, false};
    float2 *gpsi = a.psi + (long long)member * N; // storage [n0][batch][n1]

    // tables and state -> shared memory
    for (int e = tid; e < NTW; e += NTHR) tw[e] = __ldg(a.tw + e);
    {
        const float2 *src = reinterpret_cast<const float2 *>(a.tw + NTW);
        float2 *dst = reinterpret_cast<float2 *>(tw + NTW);
        for (int e = tid; e < NTW; e += NTHR) dst[e] = __ldg(src + e);
    }
    for (int e = tid; e < N; e += NTHR) {
#pragma unroll
        for (int sl = 0; sl < RES_PH_SLOTS; sl++)
            if (a.ph[sl][0] != nullptr) {
                phs[(2 * sl + 0) * N + e] = __ldg(a.ph[sl][0] + e);
                phs[(2 * sl + 1) * N + e] = __ldg(a.ph[sl][1] + e);
            }
        const int kf = e <= N / 2 ? e : N - e; // C - k0^2 is tabulated for the half spectrum's rows: [n0/2+1][batch]
        dk0[e] = __ldg(a.dk0 + (long long)kf * a.batch + member);
        k1s[e] = __ldg(a.ksq2_1 + e);
    }
    if (EXTRA && a.vext != nullptr)
        for (int e = tid; e < NL * N; e += NTHR) {
            const int l = e / N, p = e % N;
            vrows[l * PITCH + p] = __ldg(a.vext + (long long)member * N + (long long)(rank * NL + l) * a.row_stride + p);
        }
    for (int e = tid; e < NL * N; e += NTHR) {
        const int l = e / N, p = e % N;
        const float2 v = gpsi[(long long)(rank * NL + l) * a.row_stride + p];
        psis[l * 2 * PITCH + 4 * (p >> 1) + (p & 1)] = v.x;
        psis[l * 2 * PITCH + 4 * (p >> 1) + (p & 1) + 2] = v.y;
    }
    __syncthreads();

    // the last stage's twiddles stay in registers for the whole call: hi/lo for psi, plain for rho / phi
    LastTw<N> wpsi, wrho;
    wpsi.template load<true>(j, tw);
    wrho.template load<false>(j, tw);

    Lines<N> ln;
    ln.row0 = psis + 2 * g * 2 * PITCH + 4 * (j >> 1) + (j & 1);
    const int col = rank * NL + 2 * g; // first column of the pair (column sweeps); first row of the pair = the same number
#pragma unroll
    for (int m = 0; m < P; m++) ln.slot[m] = cluster_addr(psis + j * 2 * PITCH + 2 * col, m);

    uint32_t vslot[P]; // external potential of the column pair: (V_col, V_col+1) in row j of rank m
#pragma unroll
    for (int m = 0; m < P; m++) vslot[m] = EXTRA ? cluster_addr(vrows + j * PITCH + col, m) : 0u;
    const float *vrow0 = vrows + 2 * g * PITCH + j; // the row pair's values at point j (rows PITCH apart, points T apart)

    // multipliers of eq. (2) for the thread's 2 x 8 points, once per call: [0] column sweeps (lines = columns col, col + 1
    // = k1; points = k0), [1] row sweeps (lines = rows col, col + 1 = k0; points = k1)
    {
        const float2 ka = k1s[col], kb = k1s[col + 1], da = dk0[col], db = dk0[col + 1];
#pragma unroll
        for (int m = 0; m < P; m++) {
            const float2 d = dk0[j + T * m], kx = k1s[j + T * m];
            mul[(0 * P + m) * NTHR + tid] = make_float2(helmholtz_mult(d, ka, a.pscale, 0), helmholtz_mult(d, kb, a.pscale, 0));
            mul[(1 * P + m) * NTHR + tid] = make_float2(helmholtz_mult(da, kx, a.pscale, 0), helmholtz_mult(db, kx, a.pscale, 0));
        }
    }

    // it = -1, 0: the opening kinetic sweep K(ph_open) = K0 K1 as two K sweeps (rows, then columns with the density
    // transform of the first N); it >= 1: one sub-step [N K] = P, NK, KR.  One copy of each sweep's code.
    bool ycols = true; // orientation of the previous sweep = the axis rho^ has been transformed along
    for (long long it = -1; it <= a.nsub; it++) {
        const bool last = it == a.nsub;
        const bool xcols = !ycols;
        const int pos = PERIOD > 1 && it >= 1 ? (int)((it - 1) % PERIOD) : 0;
        // phase tables of this sub-step's K (Strang: slot 0 = dtau, slot 1 = dtau/2 for the opening and the closing sweep)
        const int slot = PERIOD == 1 ? ((it <= 0 || last) ? 1 : 0) : (it <= 0 ? a.ph_open : (last ? a.ph_last : a.ph_of[pos]));
        if (it >= 1) {
            // P: forward along x -> multiplier of eq. (2) -> inverse along x
            {
                const int jj = opaque(j);
                cp2 x[P];
                ln.template load<true>(x, xcols);
                fft_pair<N, +1, false>(x, jj, tw, sm, &wrho);
                const float2 *mm = mul + (xcols ? 0 : P * NTHR) + tid;
#pragma unroll
                for (int m = 0; m < P; m++) {
                    const float2 f = mm[m * NTHR];
                    x[m] = cscale(x[m], f.x, f.y);
                }
                fft_pair<N, -1, false>(x, jj, tw, sm, &wrho);
                ln.template store<true>(x, xcols);
            }
            // NK: inverse along y -> phi; nonlinear phase; K along y.  psi has not changed since the barrier before P:
            // its loads (remote ones every other step) are issued between the arrive and the wait of this barrier
            {
                const int jj = opaque(j);
                const float4 *ph = phs + (2 * slot + (ycols ? 0 : 1)) * N;
                const NLParams &nl = a.nl[PERIOD > 1 ? a.nl_of[pos] : 0];
                cp2 x[P], v[P];
                cluster.barrier_arrive();
                ln.template load<false>(v, ycols);
                cluster.barrier_wait();
                ln.template load<true>(x, ycols);
                fft_pair<N, -1, false>(x, jj, tw, sm, &wrho);
#pragma unroll
                for (int m = 0; m < P; m++) {
                    const float2 phi = x[m].r; // (phi of line a, phi of line b): the imaginary parts are rounding noise
                    float2 ve = make_float2(0.f, 0.f);
                    if (EXTRA && (nl.flags & 2)) {
                        if (ycols) asm volatile("ld.shared::cluster.v2.f32 {%0, %1}, [%2];" : "=f"(ve.x), "=f"(ve.y) : "r"(vslot[m]) : "memory");
                        else ve = make_float2(vrow0[T * m], vrow0[PITCH + T * m]);
                    }
                    nl_phase_pair_ri<EXTRA>(v[m].r, v[m].i, phi, nl, x[m].r, x[m].i, ve);
                }
                fft_pair<N, +1, true>(x, jj, tw, sm, &wpsi);
                phase_mul<T, P>(x, jj, ph);
                fft_pair<N, -1, true>(x, jj, tw, sm, &wpsi);
                ln.template store<false>(x, ycols);
            }
            cluster.sync();
        }
        // KR: K along x (+ the next step's density transform along x)
        sweep_kin<N>(ln, xcols, it >= 0 && !last, opaque(j), tw, phs + (2 * slot + (xcols ? 0 : 1)) * N, sm, &wpsi, &wrho);
        cluster.sync(); // (the last one also keeps every rank's shared memory alive until all remote accesses are done)
        ycols = xcols;
    }

    for (int e = tid; e < NL * N; e += NTHR) {
        const int l = e / N, p = e % N;
        gpsi[(long long)(rank * NL + l) * a.row_stride + p] =
            make_float2(psis[l * 2 * PITCH + 4 * (p >> 1) + (p & 1)], psis[l * 2 * PITCH + 4 * (p >> 1) + (p & 1) + 2]);
    }
}

template <class K>
static int launch_resident_kernel(K kern, int threads, size_t smem, const ResidentArgs &a)
{
    if (!smem_attr_done(reinterpret_cast<const void *>(kern))) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return (int)e;
        smem_attr_mark(reinterpret_cast<const void *>(kern));
    }
    kern<<<RES_CLUSTER * a.batch, threads, smem, a.stream>>>(a);
    return (int)cudaGetLastError();
}

template <int N>
int launch_resident(const ResidentArgs &a)
{
    const bool extra = a.nl[0].flags != 0; // log / power-law terms and / or an external potential
    if (a.period == 1)
        return extra ? launch_resident_kernel(k_resident<N, 1, true>, RGeo<N>::NTHR, RGeo<N>::SMEM, a)
                     : launch_resident_kernel(k_resident<N, 1, false>, RGeo<N>::NTHR, RGeo<N>::SMEM, a);
    if (a.period == 3)
        return extra ? launch_resident_kernel(k_resident<N, 3, true>, RGeo<N>::NTHR, RGeo<N>::SMEM, a)
                     : launch_resident_kernel(k_resident<N, 3, false>, RGeo<N>::NTHR, RGeo<N>::SMEM, a);
    return (int)cudaErrorInvalidValue;
}

// clusters of this kernel the device can hold at once (0: it cannot schedule one -- e.g. a partitioned GPU whose GPC
// slices are smaller than 8 SMs -- and the scheduler keeps the pass kernels); negative: -cudaError_t
template <int N>
int resident_max_clusters()
{
    auto kern = k_resident<N, 1, false>;
    constexpr size_t smem = RGeo<N>::SMEM;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return -(int)e;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(RES_CLUSTER, 1, 1);
    cfg.blockDim = dim3(RGeo<N>::NTHR, 1, 1);
    cfg.dynamicSmemBytes = smem;
    cudaLaunchAttribute attr;
    attr.id = cudaLaunchAttributeClusterDimension;
    attr.val.clusterDim.x = RES_CLUSTER;
    attr.val.clusterDim.y = 1;
    attr.val.clusterDim.z = 1;
    cfg.attrs = &attr;
    cfg.numAttrs = 1;
    int n = 0;
    e = cudaOccupancyMaxActiveClusters(&n, kern, &cfg);
    if (e != cudaSuccess) return -(int)e;
    return n;
}

template int launch_resident<SN_LEN>(const ResidentArgs &a);
template int resident_max_clusters<SN_LEN>();

} // namespace snk
