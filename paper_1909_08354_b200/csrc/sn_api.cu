// sn_api.cu -- C ABI (include/sn.h), table builder and Strang scheduler of libsn.so.
//
// Host-side only: builds the float64 -> hi/lo float tables, lays the caller's workspace out,
// and enqueues the pass list of one sn_step(n) call on the context's stream.  Every arithmetic
// step of the path runs in the kernels of sn_kernels.cu; there is no CPU fallback.
#include "../../include/sn.h"
#include "sn_launch.h"

#include <algorithm>
#include <climits>
#include <cmath>
#include <cstdlib>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <new>
#include <set>
#include <utility>
#include <vector>

namespace {

using snk::PassArgs;

// kinetic sub-step lengths (in units of dtau) and nonlinear sub-step lengths of the two integrators:
// Strang: K(1/2) N(1) K(1/2), merged K(1) between steps.  Order 4 (Yoshida composition of three
// Strang steps of lengths w1, w0, w1): w1 = 1/(2 - 2^(1/3)), w0 = 1 - 2 w1.
constexpr double YW1 = 1.3512071919596576340476878089715, YW0 = 1.0 - 2.0 * YW1;
enum { PH_FULL = 0, PH_HALF, PH_Y_END, PH_Y_MID, PH_Y_JOIN, PH_SLOTS };
const double PH_LEN[PH_SLOTS] = {1.0, 0.5, 0.5 * YW1, 0.5 * (YW1 + YW0), YW1};
enum { NL_MAIN = 0, NL_Y1, NL_Y0, NL_SLOTS };
const double NL_LEN[NL_SLOTS] = {1.0, YW1, YW0};

thread_local char g_cuda_msg[256] = "no CUDA error recorded";

// supported line lengths: 2^n in [32, 4096] and 3*2^a in [96, 3072]; keep in step with build.py LENGTHS
// (32: first-path kernels only -- a 64 KB pipelined tile would be 256 columns wide)
inline bool len_ok(int64_t n)
{
    if (n >= 32 && n <= 4096 && (n & (n - 1)) == 0) return true;
    return n == 96 || n == 192 || n == 384 || n == 768 || n == 1536 || n == 3072;
}
inline size_t align256(size_t x) { return (x + 255) & ~(size_t)255; }

// stage radices of the line-FFT engine (the same rule as snk::radix_for in sn_fft_core.cuh)
int radix_for(int N, int ns)
{
    const int rem = N / ns;
    if (N % 3 == 0) {
        if (rem == 6) return 6;
        int m = N / 6;
        while (m % 4 == 0) m /= 4;
        return (ns == 1 && m == 2) ? 2 : 4;
    }
    return rem >= 8 ? 8 : rem;
}

int twiddle_entries(int N)
{
    int total = 0, ns = 1;
    while (ns < N) {
        const int r = radix_for(N, ns);
        if (ns > 1) total += ns * (r - 1);
        ns *= r;
    }
    return total;
}

struct Layout {
    int ndim;
    int64_t batch;  // ensemble members (sn_create_batch): storage [n0][batch][n1]([n2]); no pass runs along the member index
    int64_t pcells; // cells of ONE system (cells = batch * pcells is the storage size)
    int64_t n[3];
    int64_t cells, cols0, nx, hs_lines, hs_elems;
    unsigned features; // SN_FEAT_*: which optional regions exist
    unsigned dtype;    // SN_DTYPE_*
    size_t esz;        // bytes of a complex value: 8 (complex64) or 16 (complex128)
    int ncomp;         // coupled wave functions (sn_create_mc): psi holds ncomp arrays one after the other; else 1
    // slab decomposition (sn_slab_create; 3D, complex64): rank `rank` of R.  n[] stay the GLOBAL dims (pcells too);
    // cells = the LOCAL cell count; "A" = the z-slab view [n0/R][n1][n2] (axis-1/2 passes; psi = psi_A, hs = hs_A with
    // h_cnt of the n0/2+1 half-spectrum rows, starting at h_lo), "B" = the y-slab view [n0][n1/R][n2] (axis-0 passes;
    // cols0 = (n1/R) n2 is its column count)
    int R, rank;
    int64_t rowsA, n1B, h_lo, h_cnt, hsB_elems;
    size_t off_psiB, off_hsB, off_stage;
    size_t off_psi, off_hs, off_phi, off_vext, off_bg, off_tw[3], off_ph[5][3], off_ksq[3], off_ksq2[3], off_kother[2],
        off_diag, total;
};

// rows [lo, lo + cnt) of the n0/2+1 half-spectrum rows owned by rank r of R in the z-slab view: (n0/2)/R each, the
// Nyquist row n0/2 goes to the last rank
inline void slab_hs_rows(int64_t n0, int R, int r, int64_t &lo, int64_t &cnt)
{
    const int64_t per = (n0 / 2) / R;
    lo = per * r;
    cnt = per + (r == R - 1 ? 1 : 0);
}

bool make_layout(int ndim, const int64_t *dims, Layout &L, int64_t batch = 1, unsigned features = 0,
                 unsigned dtype = SN_DTYPE_C64, int ncomp = 1, int R = 1, int rank = 0)
{
    if (ncomp < 1 || ncomp > 4) return false;
    L.ncomp = ncomp;
    if (R < 1 || rank < 0 || rank >= R) return false;
    if (R > 1 && (ndim != 3 || batch != 1 || features != 0 || dtype != SN_DTYPE_C64 || ncomp != 1)) return false;
    L.R = R;
    L.rank = rank;
    if (!dims || (ndim != 2 && ndim != 3)) return false;
    if (batch < 1 || batch > (1 << 20)) return false;
    if (features & ~SN_FEAT_ALL) return false;
    if (dtype != SN_DTYPE_C64 && dtype != SN_DTYPE_C128) return false;
    if (dtype == SN_DTYPE_C128 && features != 0) return false; // the NEXT-1 terms are complex64 only
    L.ndim = ndim;
    L.batch = batch;
    L.features = features;
    L.dtype = dtype;
    L.esz = dtype == SN_DTYPE_C128 ? 16 : 8;
    L.pcells = 1;
    for (int d = 0; d < ndim; d++) {
        if (!len_ok(dims[d])) return false;
        L.n[d] = dims[d];
        L.pcells *= dims[d];
    }
    L.cells = L.pcells * batch;
    L.cols0 = L.cells / L.n[0];
    L.nx = L.n[ndim - 1];
    L.hs_lines = (L.n[0] / 2 + 1) * L.cols0 / L.nx;
    if (L.hs_lines & 1) L.hs_lines++; // line pairs: one dummy line (2D)
    L.hs_elems = L.hs_lines * L.nx;
    L.rowsA = L.n[0]; L.n1B = L.n[1]; L.h_lo = 0; L.h_cnt = L.n[0] / 2 + 1; L.hsB_elems = 0;
    if (R > 1) {
        // every rank needs whole tiles in both views: n0/R rows and n1/R columns per rank, (n0/2)/R spectrum rows
        if (L.n[0] % R || L.n[1] % R || (L.n[0] / 2) % R) return false;
        L.rowsA = L.n[0] / R;
        L.n1B = L.n[1] / R;
        if ((L.n1B * L.n[2]) % 32) return false; // axis-0 tiles are up to 32 columns wide
        slab_hs_rows(L.n[0], R, rank, L.h_lo, L.h_cnt);
        L.cells = L.rowsA * L.n[1] * L.n[2];
        L.cols0 = L.n1B * L.n[2];
        L.hs_lines = L.h_cnt * L.n[1];              // lines of hs_A
        L.hs_elems = L.hs_lines * L.nx;
        L.hsB_elems = (L.n[0] / 2 + 1) * L.cols0;   // hs_B
    }
    // the kernels index columns, lines and outer blocks with 32-bit ints: reject ensembles that do not fit
    if (L.cols0 > INT_MAX || L.cells / L.nx > INT_MAX || L.hs_lines > INT_MAX || L.n[0] * batch > INT_MAX) return false;
    size_t o = 0;
    L.off_psi = o; o = align256(o + (size_t)L.cells * L.esz * (size_t)ncomp);
    L.off_hs = o; o = align256(o + (size_t)L.hs_elems * L.esz);
    // table entries have the same size in both precisions: twiddle / phase = float4 (hi + lo) or double2 (16 B),
    // + the plain float2 twiddle copy; k^2 = float + float2 (hi + lo) or double; denominators float2 or double (8 B)
    for (int d = 0; d < ndim; d++) {
        L.off_tw[d] = o; o = align256(o + (size_t)twiddle_entries((int)L.n[d]) * 24); // float4 hi/lo table + float2 plain copy
        for (int sl = 0; sl < 5; sl++) { L.off_ph[sl][d] = o; o = align256(o + (size_t)L.n[d] * 16 * (size_t)ncomp); } // one table per component
        L.off_ksq[d] = o; o = align256(o + (size_t)L.n[d] * 8);
        L.off_ksq2[d] = o; o = align256(o + (size_t)L.n[d] * 8);
    }
    for (int i = 0; i < 2; i++) { L.off_kother[i] = o; o = align256(o + (size_t)L.hs_lines * 8); }
    L.off_diag = o; o = align256(o + 8 * sizeof(double));
    // optional regions (sn_options.features)
    L.off_phi = o; if (features & SN_FEAT_STAGING) o = align256(o + (size_t)L.cells * 4);
    L.off_vext = o; if (features & SN_FEAT_VEXT) o = align256(o + (size_t)L.cells * 4);
    L.off_bg = o; if (features & SN_FEAT_SOURCE) o = align256(o + (size_t)L.cells * 8);
    L.off_psiB = L.off_hsB = L.off_stage = o;
    if (R > 1) {
        L.off_psiB = o; o = align256(o + (size_t)L.cells * 8);
        L.off_hsB = o; o = align256(o + (size_t)L.hsB_elems * 8);
        L.off_stage = o; o = align256(o + (size_t)L.cells * 8); // pack/unpack staging of the distributed exchange
    }
    L.total = o;
    return true;
}

struct f4 { float x, y, z, w; };

inline f4 split_hilo(double re, double im)
{
    f4 r;
    r.x = (float)re; r.y = (float)im;
    r.z = (float)(re - (double)r.x);
    r.w = (float)(im - (double)r.y);
    return r;
}

struct f2 { float x, y; };
inline f2 split_real(double v)
{
    f2 r;
    r.x = (float)v;
    r.y = (float)(v - (double)r.x);
    return r;
}

// complex128 contexts keep the same table slots (16 and 8 bytes per entry) filled with doubles
inline f4 as_double2(double re, double im)
{
    f4 r;
    const double v[2] = {re, im};
    std::memcpy(&r, v, 16);
    return r;
}
inline f2 as_double(double v)
{
    f2 r;
    std::memcpy(&r, &v, 8);
    return r;
}

inline double kval(int64_t j, int64_t n, double L)
{
    const int64_t jj = j < n / 2 ? j : j - n;
    return 2.0 * M_PI / L * (double)jj;
}

} // namespace

namespace snk {
// kernels whose dynamic-shared-memory limit has been raised, per device (key = device id, kernel address)
static std::mutex g_attr_mu;
static std::set<std::pair<int, const void *>> g_attr_set;
bool smem_attr_done(const void *kernel)
{
    int dev = 0;
    cudaGetDevice(&dev);
    std::lock_guard<std::mutex> lk(g_attr_mu);
    return g_attr_set.count({dev, kernel}) != 0;
}
void smem_attr_mark(const void *kernel)
{
    int dev = 0;
    cudaGetDevice(&dev);
    std::lock_guard<std::mutex> lk(g_attr_mu);
    g_attr_set.insert({dev, kernel});
}
} // namespace snk

struct sn_ctx {
    Layout lay;
    double L[3];
    double A, B, C, D, g[4], dtau;
    double g_log, rho_floor, g_pow, p_pow; // NEXT-1 local terms (eq. (16)); off when g_log == g_pow == 0
    bool has_vext;                          // external potential set (eq. (15) phi_C)
    bool v_in_xkin;                         // its phase is applied by the pipelined contiguous-axis kinetic pass
    float *vext;
    bool has_src;                           // position-dependent Poisson source of eq. (12) set
    double c_bohm, sqrt_floor;              // Bohm term of eq. (15): c_B V_B in the N sub-step (0 = off)
    float2 *bg;                             // interleaved (beta, gamma)
    int n_g;
    int device;                             // the device that owns the workspace: every entry point runs under it
    char *ws;
    cudaStream_t stream;
    bool has_state;
    int64_t launches;
    snk::NLParams nl;
    float2 *psi, *hs;
    float *phi;
    const float4 *tw[3], *ph[5][3]; // kinetic phase tables per slot (PH_*) and axis
    snk::NLParams nlv[3];           // nonlinear coefficients per slot (NL_*)
    // coupled wave functions (NEXT-4b; reading Q18): per-component constants; component c's state is
    // psi + c * cells, its kinetic phase tables ph[slot][axis] + c * n[axis]
    float2 *psiB, *hsB, *stage;             // slab contexts: the y-slab view buffers and the exchange staging
    int ncomp;
    bool is_mc; // created by sn_create_mc (also with ncomp == 1): sn_step runs the coupled scheduler
    double Ac[4], Bc[4], wc[4], gc[4][4];
    CUtensorMap m_psi_mc[4][2];
    bool f64;                       // SN_DTYPE_C128: every array and table below holds double2 / double instead
    snk::NLParamsD nlvd[3];
    const float *ksq[3];
    const float2 *ksq2[3];                  // k_a^2 as hi + lo (Helmholtz denominator, evaluated without cancellation)
    const float2 *kother[2];                // per half-spectrum line: [0] C - k_other^2, [1] -k_other^2 (Laplacian), hi + lo
    double *diag;
    int *sched;                             // tile counters of the dynamically scheduled pipelined kernels
    // pipelined (TMA) passes: tensor maps of psi / half spectrum seen along axis 0 and axis 1
    bool resident_ok;  // the device can schedule the resident kernel's cluster (checked once at create)
    bool use_resident; // SN_OPT_RESIDENT: small square 2D grids advance inside one cluster's shared memory (sn_resident.cu)
    bool use_pipe;  // SN_OPT_DISPATCH != 1
    bool pipe_all;  // SN_OPT_DISPATCH == 2: pipelined kernels wherever they are instantiated (tests, A/B runs)
    int sm_count;
    CUtensorMap m_psi[2], m_hs1, m_hs0, m_hs0_row, m_bg;
    bool m_ok[2];
    // CUDA graph of one interior step [N(dtau) K(dtau)] for launch-bound grids (<= 2^24 cells): captured once
    // on a private stream, replayed on the caller's stream
    bool use_graph;
    cudaStream_t cap_stream;
    cudaGraphExec_t step_graph;  // graph_steps interior steps
    cudaGraphExec_t step_graph1; // one interior step (the remainder of a call, when graph_steps > 1)
    int graph_launches, graph_launches1; // kernels inside each graph
    int graph_steps;    // interior steps [N(dtau) K(dtau)] captured per graph (SN_OPT_GRAPH_STEPS)
    // optional per-launch timing (sn_profile): event pairs around every launch, summed per pass kind
    bool profiling;
    std::vector<cudaEvent_t> *ev;       // pool, pairs (start, stop)
    std::vector<int> *ev_kind;          // pass kind of each recorded pair
    double prof_ms[SN_NUM_PASS_KINDS];
    int64_t prof_launches[SN_NUM_PASS_KINDS];
};

namespace {

int cuda_fail(cudaError_t e)
{
    std::snprintf(g_cuda_msg, sizeof(g_cuda_msg), "%s: %s", cudaGetErrorName(e), cudaGetErrorString(e));
    return SN_ERR_CUDA;
}
#define SN_CUDA(call)                                   \
    do {                                                \
        cudaError_t e_ = (call);                        \
        if (e_ != cudaSuccess) return cuda_fail(e_);    \
    } while (0)

// every entry point runs on the device that owns the workspace and restores the caller's device on return
struct DeviceGuard {
    int prev = -1;
    bool switched = false;
    explicit DeviceGuard(int dev)
    {
        if (cudaGetDevice(&prev) == cudaSuccess && prev != dev) switched = cudaSetDevice(dev) == cudaSuccess;
    }
    ~DeviceGuard()
    {
        if (switched) cudaSetDevice(prev);
    }
};

// fold the recorded event pairs into the per-kind sums (synchronises the stream)
int profile_flush(sn_ctx *c)
{
    if (!c->ev || c->ev_kind->empty()) return SN_OK;
    SN_CUDA(cudaStreamSynchronize(c->stream));
    for (size_t i = 0; i < c->ev_kind->size(); i++) {
        float ms = 0.f;
        SN_CUDA(cudaEventElapsedTime(&ms, (*c->ev)[2 * i], (*c->ev)[2 * i + 1]));
        c->prof_ms[(*c->ev_kind)[i]] += ms;
        c->prof_launches[(*c->ev_kind)[i]]++;
    }
    c->ev_kind->clear();
    return SN_OK;
}

// ---- TMA tensor maps (driver entry point fetched through the runtime: no libcuda link) ----
typedef CUresult (*encode_tiled_fn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                    const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                    CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

encode_tiled_fn get_encode_fn()
{
    static encode_tiled_fn fn = nullptr;
    if (!fn) {
        void *ptr = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &ptr, cudaEnableDefault, &q) == cudaSuccess &&
            q == cudaDriverEntryPointSuccess)
            fn = reinterpret_cast<encode_tiled_fn>(ptr);
    }
    return fn;
}

// complex64 array [outer][rows][cols] seen as float32 [outer][rows][2*cols]; box = 2*cpw complex x box_rows x 1
// (cpw column pairs = 16*cpw bytes per row, swizzled over exactly that width: 128B / 64B / 32B / none)
int make_map(CUtensorMap *m, void *ptr, int64_t outer, int64_t rows, int64_t cols, int box_rows, int cpw)
{
    encode_tiled_fn fn = get_encode_fn();
    if (!fn) {
        std::snprintf(g_cuda_msg, sizeof(g_cuda_msg), "cuTensorMapEncodeTiled entry point not available");
        return SN_ERR_CUDA;
    }
    const cuuint64_t gdim[3] = {(cuuint64_t)(2 * cols), (cuuint64_t)rows, (cuuint64_t)outer};
    const cuuint64_t gstr[2] = {(cuuint64_t)(cols * 8), (cuuint64_t)(rows * cols * 8)};
    const cuuint32_t box[3] = {(cuuint32_t)(4 * cpw), (cuuint32_t)box_rows, 1u};
    const CUtensorMapSwizzle swz = cpw == 8 ? CU_TENSOR_MAP_SWIZZLE_128B
                                 : cpw == 4 ? CU_TENSOR_MAP_SWIZZLE_64B
                                 : cpw == 2 ? CU_TENSOR_MAP_SWIZZLE_32B : CU_TENSOR_MAP_SWIZZLE_NONE;
    const cuuint32_t estr[3] = {1u, 1u, 1u};
    const CUresult r = fn(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, ptr, gdim, gstr, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                          swz, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                          CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
        std::snprintf(g_cuda_msg, sizeof(g_cuda_msg), "cuTensorMapEncodeTiled failed (CUresult %d)", (int)r);
        return SN_ERR_CUDA;
    }
    return SN_OK;
}

int make_tensor_maps(sn_ctx *c)
{
    const Layout &l = c->lay;
    int rc;
    c->m_ok[0] = c->m_ok[1] = false;
    // axis-0 views (slab contexts: the y-slab buffers psi_B / hs_B, n0 rows x (n1/R) n2 columns)
    float2 *p0 = l.R > 1 ? c->psiB : c->psi, *h0 = l.R > 1 ? c->hsB : c->hs;
    if (l.n[0] >= 64 && l.cols0 % (2 * snk::pipe_groups((int)l.n[0])) == 0) {
        const int n0 = (int)l.n[0], cpw = snk::pipe_cpw(n0);
        if ((rc = make_map(&c->m_psi[0], p0, 1, n0, l.cols0, snk::pipe_box_rows(n0), cpw))) return rc;
        if ((rc = make_map(&c->m_hs0, h0, 1, n0 / 2 + 1, l.cols0, snk::pipe_box_rows(n0 / 2), cpw))) return rc;
        if ((rc = make_map(&c->m_hs0_row, h0, 1, n0 / 2 + 1, l.cols0, 1, cpw))) return rc;
        if (c->bg && (rc = make_map(&c->m_bg, c->bg, 1, n0, l.cols0, snk::pipe_box_rows(n0), cpw))) return rc;
        c->m_ok[0] = true;
    }
    for (int k = 1; k < l.ncomp; k++) { // coupled components: their own views of psi_k (same geometry)
        float2 *pk = c->psi + (size_t)k * l.cells;
        if (c->m_ok[0] && (rc = make_map(&c->m_psi_mc[k][0], pk, 1, (int)l.n[0], l.cols0, snk::pipe_box_rows((int)l.n[0]), snk::pipe_cpw((int)l.n[0])))) return rc;
        if (l.ndim == 3 && l.n[1] >= 64 && l.n[2] % (2 * snk::pipe_groups((int)l.n[1])) == 0 &&
            (rc = make_map(&c->m_psi_mc[k][1], pk, l.n[0] * l.batch, (int)l.n[1], l.n[2], snk::pipe_box_rows((int)l.n[1]), snk::pipe_cpw((int)l.n[1])))) return rc;
    }
    if (l.ndim == 3 && l.n[1] >= 64 && l.n[2] % (2 * snk::pipe_groups((int)l.n[1])) == 0) {
        const int n1 = (int)l.n[1], cpw = snk::pipe_cpw(n1);
        // axis-1 views (slab contexts: the z-slab buffers, rowsA rows of psi and h_cnt rows of the half spectrum)
        if ((rc = make_map(&c->m_psi[1], c->psi, l.rowsA * l.batch, n1, l.n[2], snk::pipe_box_rows(n1), cpw))) return rc;
        if ((rc = make_map(&c->m_hs1, c->hs, l.h_cnt * l.batch, n1, l.n[2], snk::pipe_box_rows(n1), cpw))) return rc;
        c->m_ok[1] = true;
    }
    return SN_OK;
}

int run_pass_raw(sn_ctx *c, int N, PassArgs &a);

int run_pass(sn_ctx *c, int N, PassArgs &a)
{
    if (!c->profiling) return run_pass_raw(c, N, a);
    const size_t i = c->ev_kind->size();
    if (c->ev->size() < 2 * (i + 1)) {
        cudaEvent_t e0, e1;
        SN_CUDA(cudaEventCreate(&e0));
        SN_CUDA(cudaEventCreate(&e1));
        c->ev->push_back(e0);
        c->ev->push_back(e1);
    }
    SN_CUDA(cudaEventRecord((*c->ev)[2 * i], c->stream));
    const int rc = run_pass_raw(c, N, a);
    if (rc) return rc;
    SN_CUDA(cudaEventRecord((*c->ev)[2 * i + 1], c->stream));
    c->ev_kind->push_back(a.kind);
    if (c->ev_kind->size() >= 8192) return profile_flush(c);
    return SN_OK;
}

// complex128 context: the same pass descriptor, pointers reinterpreted (the scheduler only handles addresses), the
// scalars rebuilt in double from the context
int run_pass_f64(sn_ctx *c, int N, const PassArgs &a)
{
    snk::PassArgsD d;
    std::memset(&d, 0, sizeof(d));
    d.kind = a.kind; d.dir = a.dir;
    d.data = reinterpret_cast<double2 *>(a.data);
    d.hs = reinterpret_cast<double2 *>(a.hs);
    d.row_stride = a.row_stride; d.outer_stride = a.outer_stride;
    d.ncols = a.ncols; d.n_outer = a.n_outer; d.axis = a.axis; d.nlines = a.nlines;
    d.tw = reinterpret_cast<const double2 *>(a.tw);
    d.phase = reinterpret_cast<const double2 *>(a.phase);
    d.ksq = reinterpret_cast<const double *>(a.kind == snk::P_X_POISSON ? (const void *)a.ksq2 : (const void *)a.ksq);
    d.dko = reinterpret_cast<const double *>(a.dko);
    d.scale = a.scale == 1.f ? 1.0 : 1.0 / (double)N; // the only scales the scheduler uses: 1 and 1/N (sn_debug_fft inverse)
    d.lap = a.lap;
    d.pscale = (a.lap ? 1.0 : c->D) * 0.5 / (double)c->lay.pcells;
    d.nl = c->nlvd[a.kind == snk::P_H_NLKIN ? a.nl_slot : NL_MAIN];
    d.phi_out = reinterpret_cast<double *>(a.phi_out);
    d.diag = a.diag;
    d.stream = c->stream;
    int rc;
    switch (N) {
    case 96: rc = snk::launch_pass_d<96>(d); break;
    case 384: rc = snk::launch_pass_d<384>(d); break;
    case 1536: rc = snk::launch_pass_d<1536>(d); break;
    case 192: rc = snk::launch_pass_d<192>(d); break;
    case 768: rc = snk::launch_pass_d<768>(d); break;
    case 3072: rc = snk::launch_pass_d<3072>(d); break;
    case 32: rc = snk::launch_pass_d<32>(d); break;
    case 64: rc = snk::launch_pass_d<64>(d); break;
    case 128: rc = snk::launch_pass_d<128>(d); break;
    case 256: rc = snk::launch_pass_d<256>(d); break;
    case 512: rc = snk::launch_pass_d<512>(d); break;
    case 1024: rc = snk::launch_pass_d<1024>(d); break;
    case 2048: rc = snk::launch_pass_d<2048>(d); break;
    case 4096: rc = snk::launch_pass_d<4096>(d); break;
    default: return SN_ERR_DIMS;
    }
    if (rc != 0) return cuda_fail((cudaError_t)rc);
    c->launches++;
    return SN_OK;
}

int run_pass_raw(sn_ctx *c, int N, PassArgs &a)
{
    a.stream = c->stream;
    if (c->f64) return run_pass_f64(c, N, a);
    int rc;
    if (c->use_pipe) {
        const bool strided = a.kind == snk::P_S_FFT || a.kind == snk::P_S_KIN;
        const bool haxis = a.kind == snk::P_H_NLKIN || a.kind == snk::P_H_R2C || a.kind == snk::P_H_SRC ||
                           a.kind == snk::P_H_BOHM;
        const int axis = strided ? a.axis : 0;
        const bool maps = ((strided || haxis) ? c->m_ok[axis] : true) &&
                          !(a.kind == snk::P_H_NLKIN && c->has_vext && !c->v_in_xkin); // then the first-path kernel reads V
        // which kinds gain from the pipeline depends on the line length (measured): the heavy axis-0
        // pass always; the others at N = 512 and N >= 2048 (N <= 256 and N = 1024: two first-path CTAs per SM win)
        const bool worth = a.kind == snk::P_H_NLKIN || c->pipe_all || N == 512 || N >= 2048 ||
                           (a.kind == snk::P_H_R2C && (N == 256 || N == 384 || N == 1024)) || // measured per length: the
                           (a.kind == snk::P_S_FFT && N == 256) ||                             // light axis-0 / axis-1 passes too
                           (a.kind == snk::P_X_KIN && a.vext != nullptr); // V rides on the pipelined contiguous pass
        if (maps && worth && snk::pipe_supported(N, a.kind, a.ncols, a.nlines)) {
            snk::PipeArgs pa;
            std::memset(&pa, 0, sizeof(pa));
            pa.a = a;
            pa.sched = c->sched;
            if (strided) {
                const int comp = (a.data == c->hs || c->ncomp <= 1) ? 0 : (int)((a.data - c->psi) / c->lay.cells);
                pa.m_data = a.data == c->hs ? c->m_hs1 : (comp ? c->m_psi_mc[comp][axis] : c->m_psi[axis]);
                pa.tiles_per_outer = a.ncols / (2 * snk::pipe_groups(N));
                pa.n_tiles = pa.tiles_per_outer * a.n_outer;
            } else if (haxis) {
                pa.m_data = c->m_psi[0];
                pa.m_hs = c->m_hs0;
                pa.m_hs_row = c->m_hs0_row;
                pa.m_bg = c->m_bg;
                pa.tiles_per_outer = a.ncols / (2 * snk::pipe_groups(N));
                pa.n_tiles = pa.tiles_per_outer;
            } else {
                const int lines = 2 * snk::pipe_groups(N);
                pa.n_tiles = (int)((a.nlines + lines - 1) / lines);
            }
            pa.grid = pa.n_tiles < c->sm_count ? pa.n_tiles : c->sm_count;
            switch (N) {
            case 96: rc = snk::launch_pipe<96>(pa); break;
            case 384: rc = snk::launch_pipe<384>(pa); break;
            case 1536: rc = snk::launch_pipe<1536>(pa); break;
            case 192: rc = snk::launch_pipe<192>(pa); break;
            case 768: rc = snk::launch_pipe<768>(pa); break;
            case 3072: rc = snk::launch_pipe<3072>(pa); break;
            case 64: rc = snk::launch_pipe<64>(pa); break;
            case 128: rc = snk::launch_pipe<128>(pa); break;
            case 256: rc = snk::launch_pipe<256>(pa); break;
            case 512: rc = snk::launch_pipe<512>(pa); break;
            case 1024: rc = snk::launch_pipe<1024>(pa); break;
            case 2048: rc = snk::launch_pipe<2048>(pa); break;
            case 4096: rc = snk::launch_pipe<4096>(pa); break;
            default: return SN_ERR_DIMS;
            }
            if (rc != 0) return cuda_fail((cudaError_t)rc);
            c->launches++;
            return SN_OK;
        }
    }
    switch (N) {
    case 96: rc = snk::launch_pass<96>(a); break;
    case 384: rc = snk::launch_pass<384>(a); break;
    case 1536: rc = snk::launch_pass<1536>(a); break;
    case 192: rc = snk::launch_pass<192>(a); break;
    case 768: rc = snk::launch_pass<768>(a); break;
    case 3072: rc = snk::launch_pass<3072>(a); break;
    case 32: rc = snk::launch_pass<32>(a); break;
    case 64: rc = snk::launch_pass<64>(a); break;
    case 128: rc = snk::launch_pass<128>(a); break;
    case 256: rc = snk::launch_pass<256>(a); break;
    case 512: rc = snk::launch_pass<512>(a); break;
    case 1024: rc = snk::launch_pass<1024>(a); break;
    case 2048: rc = snk::launch_pass<2048>(a); break;
    case 4096: rc = snk::launch_pass<4096>(a); break;
    default: return SN_ERR_DIMS;
    }
    if (rc != 0) return cuda_fail((cudaError_t)rc);
    c->launches++;
    return SN_OK;
}

// kinetic phase tables exp(i A k_a^2 s)/N_a for s = dtau and dtau/2 (S2; reading Q2)
int upload_phase_tables(sn_ctx *c)
{
    const Layout &l = c->lay;
    for (int d = 0; d < l.ndim; d++) {
        const int64_t n = l.n[d];
        std::vector<f4> tab(n * l.ncomp); // 16 bytes per entry: (re hi, im hi, re lo, im lo) floats, or (re, im) doubles
        for (int sl = 0; sl < PH_SLOTS; sl++) {
            for (int64_t kc = 0; kc < n * l.ncomp; kc++) {
                const int64_t k = kc % n;
                const double Acomp = c->is_mc ? c->Ac[kc / n] : c->A;
                const double kk = kval(k, n, c->L[d]);
                const double th = Acomp * kk * kk * c->dtau * PH_LEN[sl];
                if (c->f64) {
                    const double v[2] = {std::cos(th) / (double)n, std::sin(th) / (double)n};
                    std::memcpy(&tab[kc], v, 16);
                } else {
                    tab[kc] = split_hilo(std::cos(th) / (double)n, std::sin(th) / (double)n);
                }
            }
            SN_CUDA(cudaMemcpyAsync(c->ws + l.off_ph[sl][d], tab.data(), tab.size() * 16, cudaMemcpyHostToDevice, c->stream));
            SN_CUDA(cudaStreamSynchronize(c->stream)); // the host vector is rewritten in the next iteration
        }
    }
    for (int sl = 0; sl < NL_SLOTS; sl++) {
        snk::NLParams &nl = c->nlv[sl];
        const double h = -0.5 * c->dtau * NL_LEN[sl]; // half-angle factor of this sub-step
        nl.hb = (float)(h * c->B);
        nl.flags = ((c->g_log != 0.0 || c->g_pow != 0.0) ? 1 : 0) | (c->has_vext ? 2 : 0);
        nl.hlog = (float)(h * c->g_log);
        nl.hpow = (float)(h * c->g_pow);
        nl.floor_ = (float)c->rho_floor;
        nl.ppow = (float)c->p_pow;
        nl.hv = (float)h;
        nl.flog = (float)c->g_log;
        nl.fpow = (float)(c->g_pow / (c->p_pow + 1.0));
        snk::NLParamsD &nd = c->nlvd[sl];
        nd.hb = 2.0 * h * c->B; // full angle: theta = -s (B phi + G)
        for (int j = 0; j < 4; j++) {
            nl.hg[j] = j < c->n_g ? (float)(h * c->g[j]) : 0.f;
            nl.fg[j] = j < c->n_g ? (float)(c->g[j] / (double)(j + 2)) : 0.f;
            nd.hg[j] = j < c->n_g ? 2.0 * h * c->g[j] : 0.0;
            nd.fg[j] = j < c->n_g ? c->g[j] / (double)(j + 2) : 0.0;
        }
    }
    c->nl = c->nlv[NL_MAIN];
    return SN_OK;
}

int upload_static_tables(sn_ctx *c)
{
    const Layout &l = c->lay;
    for (int d = 0; d < l.ndim; d++) {
        const int N = (int)l.n[d];
        // twiddles: for each stage (NS, R) with NS > 1: entry [r-1][kp] = exp(-2 pi i r kp/(NS R))
        std::vector<f4> tw;
        tw.reserve(twiddle_entries(N));
        for (int ns = 1; ns < N;) {
            const int r = radix_for(N, ns);
            if (ns > 1)
                for (int q = 1; q < r; q++)
                    for (int kp = 0; kp < ns; kp++) {
                        const double th = -2.0 * M_PI * (double)((q * kp) % (ns * r)) / (double)(ns * r);
                        tw.push_back(c->f64 ? as_double2(std::cos(th), std::sin(th)) : split_hilo(std::cos(th), std::sin(th)));
                    }
            ns *= r;
        }
        std::vector<float> ksq(N);
        std::vector<f2> ksq2(N); // complex128: k^2 as double, in the slot of the float table too
        for (int k = 0; k < N; k++) {
            const double kk = kval(k, N, c->L[d]);
            ksq[k] = (float)(kk * kk);
            ksq2[k] = c->f64 ? as_double(kk * kk) : split_real(kk * kk);
        }
        std::vector<f2> twp(tw.size()); // the same entries, hi part only (stages / transforms that apply them plainly)
        for (size_t i = 0; i < tw.size(); i++) twp[i] = f2{tw[i].x, tw[i].y};
        SN_CUDA(cudaMemcpyAsync(c->ws + l.off_tw[d], tw.data(), tw.size() * 16, cudaMemcpyHostToDevice, c->stream));
        SN_CUDA(cudaMemcpyAsync(c->ws + l.off_tw[d] + tw.size() * 16, twp.data(), twp.size() * 8, cudaMemcpyHostToDevice, c->stream));
        if (c->f64) SN_CUDA(cudaMemcpyAsync(c->ws + l.off_ksq[d], ksq2.data(), (size_t)N * 8, cudaMemcpyHostToDevice, c->stream));
        else SN_CUDA(cudaMemcpyAsync(c->ws + l.off_ksq[d], ksq.data(), (size_t)N * 4, cudaMemcpyHostToDevice, c->stream));
        SN_CUDA(cudaMemcpyAsync(c->ws + l.off_ksq2[d], ksq2.data(), (size_t)N * 8, cudaMemcpyHostToDevice, c->stream));
        SN_CUDA(cudaStreamSynchronize(c->stream));
    }
    // Denominator of eq. (2) per contiguous line of the half spectrum, without the contiguous axis' own k^2:
    // table 0 holds C - k_other^2, table 1 (Laplacian passes of eq. (12),(15)) -k_other^2, both as hi + lo floats
    // built in double, so that the kernel's (hi - kx_hi) + (lo - kx_lo) is C - k^2 to ~1e-7 RELATIVE even where C > 0
    // nearly cancels k^2 (a plain float C - k^2 has an absolute error of 1e-7 k^2 there).
    // Lines of the half spectrum are indexed (k0, member[, k1]); the member index carries no wavenumber.
    std::vector<f2> ko(l.hs_lines);
    const int64_t h0 = l.h_cnt; // slab contexts: the rows h_lo .. h_lo + h_cnt of the half spectrum
    for (int tab = 0; tab < 2; tab++) {
        const double c0 = tab == 0 ? c->C : 0.0;
        auto enc = [&](double v) { return c->f64 ? as_double(v) : split_real(v); };
        std::fill(ko.begin(), ko.end(), enc(tab == 0 && c->C != 0.0 ? c->C : -1.0)); // padding line: any finite non-zero value
        for (int64_t k0 = 0; k0 < h0; k0++) {
            const double a = kval(l.h_lo + k0, l.n[0], c->L[0]);
            for (int64_t b = 0; b < l.batch; b++) {
                if (l.ndim == 2) {
                    ko[k0 * l.batch + b] = enc(c0 - a * a);
                } else {
                    for (int64_t k1 = 0; k1 < l.n[1]; k1++) {
                        const double q = kval(k1, l.n[1], c->L[1]);
                        ko[(k0 * l.batch + b) * l.n[1] + k1] = enc(c0 - (a * a + q * q));
                    }
                }
            }
        }
        SN_CUDA(cudaMemcpyAsync(c->ws + l.off_kother[tab], ko.data(), ko.size() * 8, cudaMemcpyHostToDevice, c->stream));
        SN_CUDA(cudaStreamSynchronize(c->stream));
    }
    SN_CUDA(cudaMemsetAsync(c->ws + l.off_hs, 0, (size_t)l.hs_elems * l.esz, c->stream));
    SN_CUDA(cudaStreamSynchronize(c->stream));
    return SN_OK;
}

PassArgs base_args(const sn_ctx *c)
{
    PassArgs a;
    std::memset(&a, 0, sizeof(a));
    a.hilo = 1;
    a.dir = +1;
    a.scale = 1.f;
    a.nl = c->nl;
    a.diag = c->diag;
    a.vext = c->has_vext ? c->vext : nullptr;
    return a;
}

// geometry of a pass along `axis` of an array shaped like psi but with n0 rows on axis 0
void set_axis_geometry(const sn_ctx *c, PassArgs &a, int axis, int64_t n0)
{
    const Layout &l = c->lay;
    a.axis = axis;
    if (axis == 0) {
        a.n_outer = 1; a.outer_stride = 0; a.ncols = (int)l.cols0; a.row_stride = l.cols0;
    } else { // axis 1 of a 3D array
        a.n_outer = (int)(n0 * l.batch); a.outer_stride = l.n[1] * l.n[2]; a.ncols = (int)l.n[2]; a.row_stride = l.n[2];
    }
}

// one kinetic sweep over all axes; with_nl fuses the nonlinear phase (and the c2r of phi^) into axis 0
// ph_slot: which kinetic phase table (PH_*); with_nl: the axis-0 pass first applies the nonlinear phase of the N
// sub-step just solved, with the coefficients of nl_slot; before_n / next_nl_slot: the sweep is followed by an N
// sub-step of that slot (the external-potential phase of THAT sub-step may ride on the sweep's last pass)
int kinetic_sweep(sn_ctx *c, int ph_slot, bool with_nl, bool before_n, int nl_slot = NL_MAIN, int next_nl_slot = NL_MAIN)
{
    const Layout &l = c->lay;
    int rc;
    for (int d = 0; d < l.ndim; d++) {
        PassArgs a = base_args(c);
        a.data = c->psi;
        a.hs = c->hs;
        a.tw = c->tw[d];
        a.phase = c->ph[ph_slot][d];
        a.nl = c->nlv[nl_slot];
        a.nl_slot = nl_slot;
        if (c->v_in_xkin) a.nl.flags &= ~2; // the axis-0 pass leaves V to the contiguous pass
        a.vext = nullptr;
        if (d == l.ndim - 1) {
            a.kind = snk::P_X_KIN;
            a.nlines = (int)(l.cells / l.nx);
            if (c->v_in_xkin && before_n) {
                a.vext = c->vext;
                a.nl.hv = c->nlv[next_nl_slot].hv;
            }
        } else {
            a.kind = (d == 0 && with_nl) ? snk::P_H_NLKIN : snk::P_S_KIN;
            if (a.kind == snk::P_H_NLKIN && c->has_vext && !c->v_in_xkin) a.vext = c->vext;
            set_axis_geometry(c, a, d, l.n[0]);
        }
        if ((rc = run_pass(c, (int)l.n[d], a))) return rc;
    }
    return SN_OK;
}

// half-spectrum passes along the non-zero axes: forward (axis 1 in 3D) -> fused forward-multiply-inverse along
// the contiguous axis -> inverse (axis 1).  lap: multiply by -k^2/prod(N) (Laplacian) instead of D/(C - k^2)/prod(N).
int spectrum_chain(sn_ctx *c, bool lap)
{
    const Layout &l = c->lay;
    int rc;
    if (l.ndim == 3) {
        PassArgs a = base_args(c);
        a.kind = snk::P_S_FFT; a.dir = +1; a.hilo = 0; a.data = c->hs; a.tw = c->tw[1];
        set_axis_geometry(c, a, 1, l.n[0] / 2 + 1);
        if ((rc = run_pass(c, (int)l.n[1], a))) return rc;
    }
    {
        const int dx = l.ndim - 1;
        PassArgs a = base_args(c);
        a.kind = snk::P_X_POISSON; a.data = c->hs; a.tw = c->tw[dx]; a.ksq2 = c->ksq2[dx]; a.dko = c->kother[lap ? 1 : 0];
        a.nlines = (int)l.hs_lines;
        a.lap = lap ? 1 : 0;
        const double npts = (double)l.pcells; // points of ONE system: the 1/prod(N) of its transforms
        a.pscale = (float)((lap ? 1.0 : c->D) * 0.5 / npts); // 0.5: the packed r2c carries a factor 2
        if ((rc = run_pass(c, (int)l.n[dx], a))) return rc;
    }
    if (l.ndim == 3) {
        PassArgs a = base_args(c);
        a.kind = snk::P_S_FFT; a.dir = -1; a.hilo = 0; a.data = c->hs; a.tw = c->tw[1]; a.scale = 1.f;
        set_axis_geometry(c, a, 1, l.n[0] / 2 + 1);
        if ((rc = run_pass(c, (int)l.n[1], a))) return rc;
    }
    return SN_OK;
}

// phi^ (half spectrum, all scales folded in, ready for the axis-0 c2r) from the current psi.
// With source tables (eq. (12)): rho -> F[rho] -> -k^2 -> lap rho -> s = gamma rho + beta lap rho -> F[s] -> phi^.
int density_r2c(sn_ctx *c, bool sqrt_rho)
{
    const Layout &l = c->lay;
    PassArgs a = base_args(c);
    a.kind = snk::P_H_R2C; a.data = c->psi; a.hs = c->hs; a.tw = c->tw[0];
    a.sqrt_rho = sqrt_rho ? 1 : 0;
    set_axis_geometry(c, a, 0, l.n[0]);
    return run_pass(c, (int)l.n[0], a);
}

int potential_spectrum(sn_ctx *c)
{
    const Layout &l = c->lay;
    int rc;
    if ((rc = density_r2c(c, false))) return rc;
    if (c->has_src) {
        if ((rc = spectrum_chain(c, /*lap=*/true))) return rc;
        PassArgs a = base_args(c);
        a.kind = snk::P_H_SRC; a.data = c->psi; a.hs = c->hs; a.tw = c->tw[0];
        a.bg = c->bg;
        set_axis_geometry(c, a, 0, l.n[0]);
        if ((rc = run_pass(c, (int)l.n[0], a))) return rc;
    }
    return spectrum_chain(c, /*lap=*/false);
}

// What an N sub-step of length dtau * NL_LEN[nl_slot] needs before the axis-0 pass of the next sweep: the Bohm
// phase (eq. (15): psi *= exp(-i s c_B lap sqrt(rho)/(2 sqrt(rho))), a pass of its own since it commutes with the
// rest of the N phase and leaves rho unchanged), then phi^.
int prepare_n(sn_ctx *c, int nl_slot)
{
    const Layout &l = c->lay;
    int rc;
    if (c->c_bohm != 0.0) {
        if ((rc = density_r2c(c, true))) return rc;
        if ((rc = spectrum_chain(c, /*lap=*/true))) return rc;
        PassArgs a = base_args(c);
        a.kind = snk::P_H_BOHM; a.data = c->psi; a.hs = c->hs; a.tw = c->tw[0];
        a.hbohm = (float)(-0.25 * c->dtau * NL_LEN[nl_slot] * c->c_bohm);
        a.sfloor = (float)c->sqrt_floor;
        set_axis_geometry(c, a, 0, l.n[0]);
        if ((rc = run_pass(c, (int)l.n[0], a))) return rc;
    }
    return potential_spectrum(c);
}

// ---- coupled wave functions (NEXT-4b, reading Q18 of DESIGN.md) ----
// K(s): every component on its own, one forward -> phase -> inverse pass per axis with the component's phase tables
int kinetic_sweep_mc(sn_ctx *c, int ph_slot)
{
    const Layout &l = c->lay;
    int rc;
    for (int k = 0; k < l.ncomp; k++)
        for (int d = 0; d < l.ndim; d++) {
            PassArgs a = base_args(c);
            a.data = c->psi + (size_t)k * l.cells;
            a.tw = c->tw[d];
            a.phase = c->ph[ph_slot][d] + (size_t)k * l.n[d];
            a.vext = nullptr;
            if (d == l.ndim - 1) {
                a.kind = snk::P_X_KIN;
                a.nlines = (int)(l.cells / l.nx);
            } else {
                a.kind = snk::P_S_KIN;
                set_axis_geometry(c, a, d, l.n[0]);
            }
            if ((rc = run_pass(c, (int)l.n[d], a))) return rc;
        }
    return SN_OK;
}

snk::MCParams mc_params(const sn_ctx *c, double s)
{
    snk::MCParams m;
    std::memset(&m, 0, sizeof(m));
    m.ncomp = c->lay.ncomp;
    m.comp_stride = c->lay.cells;
    for (int a = 0; a < m.ncomp; a++) {
        m.w[a] = (float)c->wc[a];
        m.hb[a] = (float)(-0.5 * s * c->Bc[a]);
        for (int b = 0; b < m.ncomp; b++) m.hg[a][b] = (float)(-0.5 * s * c->gc[a][b]);
    }
    return m;
}

// N(s): rho = sum_c w_c |psi_c|^2 -> phi^ (same half-spectrum chain as one component) -> every component's phase
int nonlinear_mc(sn_ctx *c, double s)
{
    const Layout &l = c->lay;
    int rc;
    PassArgs a = base_args(c);
    a.kind = snk::P_H_R2C_MC; a.data = c->psi; a.hs = c->hs; a.tw = c->tw[0];
    a.mc = mc_params(c, s);
    set_axis_geometry(c, a, 0, l.n[0]);
    if ((rc = run_pass(c, (int)l.n[0], a))) return rc;
    if ((rc = spectrum_chain(c, /*lap=*/false))) return rc;
    a.kind = snk::P_H_NL_MC;
    return run_pass(c, (int)l.n[0], a);
}

// ---- slab-decomposed step (NEXT-2): the LOCAL passes of rank `rank` of R ----
// Lines along axis 0 are whole in the y-slab view B = [n0][n1/R][n2], lines along axes 1 and 2 in the z-slab view
// A = [n0/R][n1][n2]; between the stages below the caller moves psi (8 B/cell) or the half spectrum (4 B/cell) from
// one view to the other with an all-to-all (sn_slab_exchange_local for R contexts on one device; pack / all_to_all /
// unpack for one process per GPU).  The kernels are the ones of the single-GPU step, on the local geometry.
void slab_axis1(const sn_ctx *c, PassArgs &a, int64_t rows)
{
    const Layout &l = c->lay;
    a.axis = 1; a.n_outer = (int)rows; a.outer_stride = l.n[1] * l.n[2]; a.ncols = (int)l.n[2]; a.row_stride = l.n[2];
}
void slab_axis0(const sn_ctx *c, PassArgs &a)
{
    const Layout &l = c->lay;
    a.axis = 0; a.n_outer = 1; a.outer_stride = 0; a.ncols = (int)l.cols0; a.row_stride = l.cols0;
}

int slab_stage(sn_ctx *c, int stage, int ph_slot)
{
    const Layout &l = c->lay;
    int rc;
    switch (stage) {
    case SN_SLAB_KIN_A: { // kinetic passes along axes 1 and 2 on psi_A
        PassArgs a = base_args(c);
        a.kind = snk::P_S_KIN; a.data = c->psi; a.tw = c->tw[1]; a.phase = c->ph[ph_slot][1]; a.vext = nullptr;
        slab_axis1(c, a, l.rowsA);
        if ((rc = run_pass(c, (int)l.n[1], a))) return rc;
        PassArgs b = base_args(c);
        b.kind = snk::P_X_KIN; b.data = c->psi; b.tw = c->tw[2]; b.phase = c->ph[ph_slot][2]; b.vext = nullptr;
        b.nlines = (int)(l.cells / l.nx);
        return run_pass(c, (int)l.n[2], b);
    }
    case SN_SLAB_KIN0_B: { // kinetic pass along axis 0 on psi_B, no nonlinear phase (opening sweep of a call)
        PassArgs a = base_args(c);
        a.kind = snk::P_S_KIN; a.data = c->psiB; a.tw = c->tw[0]; a.phase = c->ph[ph_slot][0]; a.vext = nullptr;
        slab_axis0(c, a);
        return run_pass(c, (int)l.n[0], a);
    }
    case SN_SLAB_R2C_B: { // rho = |psi_B|^2 -> packed r2c along axis 0 -> hs_B
        PassArgs a = base_args(c);
        a.kind = snk::P_H_R2C; a.data = c->psiB; a.hs = c->hsB; a.tw = c->tw[0];
        slab_axis0(c, a);
        return run_pass(c, (int)l.n[0], a);
    }
    case SN_SLAB_CHAIN_A: { // hs_A: forward along axis 1 -> forward, D/(C - k^2), inverse along axis 2 -> inverse along axis 1
        PassArgs a = base_args(c);
        a.kind = snk::P_S_FFT; a.dir = +1; a.hilo = 0; a.data = c->hs; a.tw = c->tw[1];
        slab_axis1(c, a, l.h_cnt);
        if ((rc = run_pass(c, (int)l.n[1], a))) return rc;
        PassArgs x = base_args(c);
        x.kind = snk::P_X_POISSON; x.data = c->hs; x.tw = c->tw[2]; x.ksq2 = c->ksq2[2]; x.dko = c->kother[0];
        x.nlines = (int)l.hs_lines;
        x.pscale = (float)(c->D * 0.5 / (double)l.pcells);
        if ((rc = run_pass(c, (int)l.n[2], x))) return rc;
        a.dir = -1;
        return run_pass(c, (int)l.n[1], a);
    }
    case SN_SLAB_NLKIN_B: { // c2r of hs_B -> nonlinear phase -> kinetic pass along axis 0, on psi_B
        PassArgs a = base_args(c);
        a.kind = snk::P_H_NLKIN; a.data = c->psiB; a.hs = c->hsB; a.tw = c->tw[0]; a.phase = c->ph[ph_slot][0];
        a.nl = c->nlv[NL_MAIN]; a.nl_slot = NL_MAIN; a.vext = nullptr;
        slab_axis0(c, a);
        return run_pass(c, (int)l.n[0], a);
    }
    default:
        return SN_ERR_PARAM;
    }
}

// block of the exchange between the y-slab buffer of rank s and the z-slab buffer of rank r: rows [lo, lo + cnt) of
// s's B array (contiguous there), columns s (n1/R) n2 ... of r's A array (pitch n1 n2)
int slab_copy_block(const Layout &l, float2 *A_r, float2 *B_s, int64_t lo, int64_t cnt, int s, bool b2a, cudaStream_t st)
{
    const size_t width = (size_t)l.cols0 * 8;                       // bytes of one row of a block
    float2 *bp = B_s + (size_t)lo * l.cols0;                        // contiguous in B
    float2 *ap = A_r + (size_t)s * l.cols0;                         // strided in A
    const size_t apitch = (size_t)l.n[1] * l.n[2] * 8;
    const cudaError_t e = b2a ? cudaMemcpy2DAsync(ap, apitch, bp, width, width, (size_t)cnt, cudaMemcpyDeviceToDevice, st)
                              : cudaMemcpy2DAsync(bp, width, ap, apitch, width, (size_t)cnt, cudaMemcpyDeviceToDevice, st);
    return e == cudaSuccess ? SN_OK : cuda_fail(e);
}

// ---- cluster-resident step (sn_resident.cu): the whole sn_step(n) call of a small square 2D grid in ONE launch ----
// Served: complex64, 2D, n0 == n1 in {64, 128}, local nonlinearities (polynomial G and the log / power-law terms of
// eq. (16), an external potential; no source tables or Bohm term), the default
// dispatch (SN_OPT_DISPATCH 1 / 2 ask for the pass kernels by name), ensembles of up to RESIDENT_MAX_BATCH members
// (one cluster per member; measured on B200, 128^2: 16 members 13 vs 25 us/step, 32 members 14 vs 26, 64 members 28 vs 28 -- a large
// ensemble fills the machine through the pass kernels, which are the faster ones per cell).  Everything else takes the
// pass kernels.
// member limits, measured on B200 (us/step resident vs pass kernels): 128^2: 16 members 13 vs 25, 32 members 14 vs 26, 64
// members 28 vs 28; 64^2 (32-thread CTAs, 25 KB of shared memory: many more clusters at once): 64 members 6.5 vs 19.2, 148
// members 13.5 vs 19.7, 296 members 21.9 vs 23.6, 1024 members 70 vs 54
#ifndef SN_RES_MAXB64
#define SN_RES_MAXB64 256
#endif
constexpr int64_t RESIDENT_MAX_BATCH = 32;
bool resident_eligible(const sn_ctx *c)
{
    const Layout &l = c->lay;
    return c->use_resident && c->use_pipe && !c->pipe_all && !c->f64 && !c->is_mc && l.R == 1 && l.ndim == 2 &&
           snk::resident_supported((int)l.n[0], (int)l.n[1]) && !c->has_src && c->c_bohm == 0.0 &&
           l.batch <= (l.n[0] == 64 ? (int64_t)SN_RES_MAXB64 : RESIDENT_MAX_BATCH);
}

int run_resident(sn_ctx *c, int64_t nsteps, bool order4 = false)
{
    const Layout &l = c->lay;
    snk::ResidentArgs a;
    std::memset(&a, 0, sizeof(a));
    a.psi = c->psi;
    a.row_stride = l.batch * l.n[1];
    a.batch = (int)l.batch;
    a.tw = c->tw[0]; // n0 == n1: one table serves both axes
    // the call's program: phase slots and nonlinear-coefficient sets in the order the kernel indexes them
    const int ph_slots[2][snk::RES_PH_SLOTS] = {{PH_FULL, PH_HALF, -1, -1}, {PH_Y_END, PH_Y_MID, PH_Y_JOIN, -1}};
    for (int sl = 0; sl < snk::RES_PH_SLOTS; sl++)
        for (int d = 0; d < 2; d++) a.ph[sl][d] = ph_slots[order4][sl] >= 0 ? c->ph[ph_slots[order4][sl]][d] : nullptr;
    if (!order4) { // K(dtau/2) [N(dtau) K(dtau)]^(n-1) N(dtau) K(dtau/2)
        a.nsub = nsteps; a.period = 1;
        a.nl_of[0] = 0; a.ph_of[0] = 0; a.ph_open = a.ph_last = 1;
        a.nl[0] = c->nlv[NL_MAIN];
    } else { // K(w1/2) [N(w1) K((w1+w0)/2) N(w0) K((w0+w1)/2) N(w1) K(w1 or w1/2)]^n
        a.nsub = 3 * nsteps; a.period = 3;
        a.nl_of[0] = 0; a.nl_of[1] = 1; a.nl_of[2] = 0;
        a.ph_of[0] = 1; a.ph_of[1] = 1; a.ph_of[2] = 2; a.ph_open = a.ph_last = 0;
        a.nl[0] = c->nlv[NL_Y1]; a.nl[1] = c->nlv[NL_Y0];
    }
    a.ksq2_1 = c->ksq2[1];
    a.dk0 = c->kother[0];
    a.pscale = (float)(c->D / (double)l.pcells);
    a.vext = c->has_vext ? c->vext : nullptr;
    for (int k = 0; k < 3; k++) // the pass kernels may leave V to the contiguous pass (v_in_xkin); here it rides on the nonlinear phase
        if (c->has_vext) a.nl[k].flags |= 2;
    a.stream = c->stream;
    size_t ev = 0;
    if (c->profiling) {
        ev = c->ev_kind->size();
        if (c->ev->size() < 2 * (ev + 1)) {
            cudaEvent_t e0, e1;
            SN_CUDA(cudaEventCreate(&e0));
            SN_CUDA(cudaEventCreate(&e1));
            c->ev->push_back(e0);
            c->ev->push_back(e1);
        }
        SN_CUDA(cudaEventRecord((*c->ev)[2 * ev], c->stream));
    }
    int rc;
    switch ((int)l.n[0]) {
    case 64: rc = snk::launch_resident<64>(a); break;
    case 128: rc = snk::launch_resident<128>(a); break;
    default: return SN_ERR_DIMS;
    }
    if (rc != 0) return cuda_fail((cudaError_t)rc);
    c->launches++;
    if (c->profiling) {
        SN_CUDA(cudaEventRecord((*c->ev)[2 * ev + 1], c->stream));
        c->ev_kind->push_back(snk::P_R_STEPS);
    }
    return SN_OK;
}

// capture one interior step N(dtau) K(dtau) (the pass list of potential_spectrum + a full kinetic sweep)
int build_step_graph(sn_ctx *c, int steps, cudaGraphExec_t *exec, int *launches_out)
{
    if (!c->cap_stream) SN_CUDA(cudaStreamCreateWithFlags(&c->cap_stream, cudaStreamNonBlocking));
    const cudaStream_t user = c->stream;
    const int64_t before = c->launches;
    SN_CUDA(cudaStreamBeginCapture(c->cap_stream, cudaStreamCaptureModeThreadLocal));
    c->stream = c->cap_stream;
    int rc = SN_OK;
    for (int s = 0; rc == SN_OK && s < steps; s++) {
        rc = prepare_n(c, NL_MAIN);
        if (rc == SN_OK) rc = kinetic_sweep(c, PH_FULL, /*with_nl=*/true, /*before_n=*/true);
    }
    c->stream = user;
    cudaGraph_t g = nullptr;
    const cudaError_t e = cudaStreamEndCapture(c->cap_stream, &g);
    *launches_out = (int)(c->launches - before);
    c->launches = before;
    if (rc != SN_OK) {
        if (g) cudaGraphDestroy(g);
        return rc;
    }
    if (e != cudaSuccess) return cuda_fail(e);
    const cudaError_t e2 = cudaGraphInstantiate(exec, g, 0);
    cudaGraphDestroy(g);
    if (e2 != cudaSuccess) {
        *exec = nullptr;
        return cuda_fail(e2);
    }
    return SN_OK;
}

void drop_step_graph(sn_ctx *c)
{
    if (c->step_graph) cudaGraphExecDestroy(c->step_graph);
    if (c->step_graph1) cudaGraphExecDestroy(c->step_graph1);
    c->step_graph = c->step_graph1 = nullptr;
}

} // namespace

namespace snk {
// for translation units with entry points of their own (sn_static.cu): record the text of a CUDA error for sn_strerror
void record_cuda_error(int cuda_error) { cuda_fail((cudaError_t)cuda_error); }
} // namespace snk

// ============================================================================ C ABI

extern "C" {

struct MCInit { // constants of the coupled-component system handed from sn_create_mc to create_impl
    int n;
    const double *A, *B, *w, *g;
};

static bool options_ok(const sn_options *opt) { return opt && opt->struct_size == sizeof(sn_options); }

size_t sn_workspace_bytes(int ndim, const int64_t *dims)
{
    Layout l;
    return make_layout(ndim, dims, l) ? l.total : 0;
}

size_t sn_workspace_bytes_batch(int ndim, const int64_t *dims, int64_t batch)
{
    Layout l;
    return make_layout(ndim, dims, l, batch) ? l.total : 0;
}

size_t sn_workspace_bytes_opt(int ndim, const int64_t *dims, const sn_options *opt)
{
    Layout l;
    if (!options_ok(opt)) return 0;
    return make_layout(ndim, dims, l, opt->batch, opt->features, opt->dtype) ? l.total : 0;
}

static int create_impl(sn_ctx **out, int ndim, const int64_t *dims, const double *L, double A, double B, double C, double D,
                       const double *g, int n_g, double dtau, void *d_workspace, size_t workspace_bytes, void *cuda_stream,
                       int64_t batch, unsigned features, unsigned dtype = SN_DTYPE_C64, const MCInit *mc = nullptr, int R = 1,
                       int rank = 0);

int sn_create(sn_ctx **out, int ndim, const int64_t *dims, const double *L, double A, double B, double C, double D,
              const double *g, int n_g, double dtau, void *d_workspace, size_t workspace_bytes, void *cuda_stream)
{
    return create_impl(out, ndim, dims, L, A, B, C, D, g, n_g, dtau, d_workspace, workspace_bytes, cuda_stream, 1, 0);
}

int sn_create_batch(sn_ctx **out, int ndim, const int64_t *dims, int64_t batch, const double *L, double A, double B,
                    double C, double D, const double *g, int n_g, double dtau, void *d_workspace, size_t workspace_bytes,
                    void *cuda_stream)
{
    return create_impl(out, ndim, dims, L, A, B, C, D, g, n_g, dtau, d_workspace, workspace_bytes, cuda_stream, batch, 0);
}

int sn_create_opt(sn_ctx **out, int ndim, const int64_t *dims, const double *L, double A, double B, double C, double D,
                  const double *g, int n_g, double dtau, void *d_workspace, size_t workspace_bytes, void *cuda_stream,
                  const sn_options *opt)
{
    if (!opt) return SN_ERR_NULL;
    if (!options_ok(opt)) return SN_ERR_PARAM;
    if (opt->features & ~SN_FEAT_ALL) return SN_ERR_PARAM;
    if (opt->dtype != SN_DTYPE_C64 && opt->dtype != SN_DTYPE_C128) return SN_ERR_PARAM;
    if (opt->dtype == SN_DTYPE_C128 && opt->features != 0) return SN_ERR_PARAM;
    return create_impl(out, ndim, dims, L, A, B, C, D, g, n_g, dtau, d_workspace, workspace_bytes, cuda_stream, opt->batch,
                       opt->features, opt->dtype);
}

// reading Q5: C > 0 within 1e-12 (relative) of k^2 of a grid mode makes eq. (2) unsolvable.  Per axis: the distinct
// k_a^2 values are sorted once, and for every pair (k0^2, k1^2) the remainder C - k0^2 - k1^2 is looked up among the
// last axis' values (O(N0 N1 log N2) instead of a sweep over all modes).
static bool helmholtz_singular(const Layout &l, const double *L, double C)
{
    const double tol = 1e-12 * std::fmax(1.0, std::fabs(C));
    std::vector<double> k2[3];
    for (int d = 0; d < 3; d++) {
        if (d >= l.ndim) {
            k2[d].push_back(0.0);
            continue;
        }
        for (int64_t i = 0; i <= l.n[d] / 2; i++) {
            const double k = kval(i, l.n[d], L[d]);
            k2[d].push_back(k * k);
        }
    }
    const std::vector<double> &last = k2[l.ndim - 1]; // ascending in i
    const std::vector<double> &a0 = k2[0], &a1 = l.ndim == 3 ? k2[1] : k2[2];
    for (double x : a0)
        for (double y : a1) {
            const double want = C - x - y;
            if (want < -tol) break; // y ascending: the remainder only decreases
            auto it = std::lower_bound(last.begin(), last.end(), want - tol);
            if (it != last.end() && std::fabs(*it - want) < tol) return true;
        }
    return false;
}

static int create_impl(sn_ctx **out, int ndim, const int64_t *dims, const double *L, double A, double B, double C, double D,
                       const double *g, int n_g, double dtau, void *d_workspace, size_t workspace_bytes, void *cuda_stream,
                       int64_t batch, unsigned features, unsigned dtype, const MCInit *mc, int R, int rank)
{
    if (!out || !dims || !L || !d_workspace || (n_g > 0 && !g)) return SN_ERR_NULL;
    Layout l;
    if (!make_layout(ndim, dims, l, batch, features, dtype, mc ? mc->n : 1, R, rank)) return SN_ERR_DIMS;
    if (n_g < 0 || n_g > 4) return SN_ERR_PARAM;
    if (!std::isfinite(A) || !std::isfinite(B) || !std::isfinite(C) || !std::isfinite(D) || !std::isfinite(dtau))
        return SN_ERR_PARAM;
    for (int d = 0; d < ndim; d++)
        if (!std::isfinite(L[d]) || L[d] <= 0.0) return SN_ERR_PARAM;
    for (int j = 0; j < n_g; j++)
        if (!std::isfinite(g[j])) return SN_ERR_PARAM;
    if (workspace_bytes < l.total || ((uintptr_t)d_workspace & 255) != 0) return SN_ERR_WORKSPACE;
    if (C > 0.0 && helmholtz_singular(l, L, C)) return SN_ERR_SINGULAR;
    sn_ctx *c = new (std::nothrow) sn_ctx;
    if (!c) return SN_ERR_NOMEM;
    std::memset(c, 0, sizeof(*c));
    c->lay = l;
    for (int d = 0; d < ndim; d++) c->L[d] = L[d];
    c->A = A; c->B = B; c->C = C; c->D = D; c->dtau = dtau; c->n_g = n_g;
    for (int j = 0; j < n_g; j++) c->g[j] = g[j];
    c->ws = static_cast<char *>(d_workspace);
    c->stream = static_cast<cudaStream_t>(cuda_stream);
    c->psi = reinterpret_cast<float2 *>(c->ws + l.off_psi);
    c->hs = reinterpret_cast<float2 *>(c->ws + l.off_hs);
    c->phi = (features & SN_FEAT_STAGING) ? reinterpret_cast<float *>(c->ws + l.off_phi) : nullptr;
    c->vext = (features & SN_FEAT_VEXT) ? reinterpret_cast<float *>(c->ws + l.off_vext) : nullptr;
    c->bg = (features & SN_FEAT_SOURCE) ? reinterpret_cast<float2 *>(c->ws + l.off_bg) : nullptr;
    // one rank: the two views coincide
    c->psiB = l.R > 1 ? reinterpret_cast<float2 *>(c->ws + l.off_psiB) : c->psi;
    c->hsB = l.R > 1 ? reinterpret_cast<float2 *>(c->ws + l.off_hsB) : c->hs;
    c->stage = l.R > 1 ? reinterpret_cast<float2 *>(c->ws + l.off_stage) : nullptr;
    c->rho_floor = 1e-30; c->p_pow = 1.0; c->sqrt_floor = 1e-30;
    for (int d = 0; d < ndim; d++) {
        c->tw[d] = reinterpret_cast<const float4 *>(c->ws + l.off_tw[d]);
        for (int sl = 0; sl < PH_SLOTS; sl++) c->ph[sl][d] = reinterpret_cast<const float4 *>(c->ws + l.off_ph[sl][d]);
        c->ksq[d] = reinterpret_cast<const float *>(c->ws + l.off_ksq[d]);
        c->ksq2[d] = reinterpret_cast<const float2 *>(c->ws + l.off_ksq2[d]);
    }
    for (int i = 0; i < 2; i++) c->kother[i] = reinterpret_cast<const float2 *>(c->ws + l.off_kother[i]);
    c->diag = reinterpret_cast<double *>(c->ws + l.off_diag);
    c->sched = reinterpret_cast<int *>(c->ws + l.off_diag + 128); // inside the 256-byte block of the diagnostics
    c->f64 = dtype == SN_DTYPE_C128;
    c->ncomp = l.ncomp;
    c->is_mc = mc != nullptr;
    if (mc)
        for (int a = 0; a < mc->n; a++) {
            c->Ac[a] = mc->A[a]; c->Bc[a] = mc->B[a]; c->wc[a] = mc->w[a];
            for (int b = 0; b < mc->n; b++) c->gc[a][b] = mc->g[a * mc->n + b];
        }
    c->use_graph = l.cells <= ((int64_t)1 << 24) && !c->is_mc && l.R == 1;
    c->graph_steps = 8; // measured on B200 (1 -> 8 steps per replay): C2 39.0 -> 36.5, 64^3 28.8 -> 27.3, 128^3 61.9 -> 59.9 us/step
    c->use_pipe = !c->f64; // the TMA-pipelined kernels are complex64 only
    c->use_resident = c->resident_ok = false; // decided below, on the context's device
    c->pipe_all = false;
    // the device that owns the workspace is the context's device
    int rc = SN_OK;
    {
        cudaPointerAttributes pat;
        const cudaError_t e = cudaPointerGetAttributes(&pat, d_workspace);
        if (e != cudaSuccess) rc = cuda_fail(e);
        else if (pat.type != cudaMemoryTypeDevice && pat.type != cudaMemoryTypeManaged) {
            cudaGetLastError();
            rc = SN_ERR_WORKSPACE;
        } else c->device = pat.device;
    }
    if (rc == SN_OK) {
        DeviceGuard guard(c->device);
        rc = upload_static_tables(c);
        if (rc == SN_OK) rc = upload_phase_tables(c);
        if (rc == SN_OK && cudaMemsetAsync(c->sched, 0, 2 * sizeof(int), c->stream) != cudaSuccess) rc = cuda_fail(cudaGetLastError());
        if (rc == SN_OK) {
            if (cudaDeviceGetAttribute(&c->sm_count, cudaDevAttrMultiProcessorCount, c->device) != cudaSuccess || c->sm_count < 1)
                rc = cuda_fail(cudaGetLastError());
            else if (c->use_pipe)
                rc = make_tensor_maps(c);
        }
        // the cluster-resident kernel serves the context where the grid qualifies and this device can schedule its cluster
        if (rc == SN_OK && !c->f64 && !c->is_mc && l.R == 1 && l.ndim == 2 &&
            snk::resident_supported((int)l.n[0], (int)l.n[1])) {
            const int nc = l.n[0] == 64 ? snk::resident_max_clusters<64>() : snk::resident_max_clusters<128>();
            if (nc < 0) cudaGetLastError(); // not an error of the context: the pass kernels serve it
            c->use_resident = c->resident_ok = nc > 0;
        }
    }
    if (rc != SN_OK) {
        delete c;
        return rc;
    }
    *out = c;
    return SN_OK;
}

size_t sn_workspace_bytes_mc(int ndim, const int64_t *dims, int n_comp)
{
    Layout l;
    return make_layout(ndim, dims, l, 1, 0, SN_DTYPE_C64, n_comp) ? l.total : 0;
}

int sn_create_mc(sn_ctx **out, int ndim, const int64_t *dims, const double *L, int n_comp, const double *A, const double *B,
                 double C, double D, const double *w, const double *g, double dtau, void *d_workspace,
                 size_t workspace_bytes, void *cuda_stream)
{
    if (!A || !B || !w || !g) return SN_ERR_NULL;
    if (n_comp < 1 || n_comp > 4) return SN_ERR_PARAM;
    for (int a = 0; a < n_comp; a++) {
        if (!std::isfinite(A[a]) || !std::isfinite(B[a]) || !std::isfinite(w[a])) return SN_ERR_PARAM;
        for (int b = 0; b < n_comp; b++)
            if (!std::isfinite(g[a * n_comp + b])) return SN_ERR_PARAM;
    }
    MCInit mc;
    mc.n = n_comp; mc.A = A; mc.B = B; mc.w = w; mc.g = g;
    return create_impl(out, ndim, dims, L, A[0], B[0], C, D, nullptr, 0, dtau, d_workspace, workspace_bytes, cuda_stream, 1, 0,
                       SN_DTYPE_C64, &mc);
}

int sn_mc_norms(sn_ctx *c, double *norms)
{
    if (!c || !norms) return SN_ERR_NULL;
    if (!c->has_state) return SN_ERR_STATE;
    DeviceGuard guard(c->device);
    const Layout &l = c->lay;
    SN_CUDA(cudaMemsetAsync(c->diag, 0, 8 * sizeof(double), c->stream));
    for (int k = 0; k < l.ncomp; k++) {
        const int rc = snk::launch_norm(c->psi + (size_t)k * l.cells, l.cells, c->diag + k, c->stream);
        if (rc != 0) return cuda_fail((cudaError_t)rc);
        c->launches++;
    }
    double h[4];
    SN_CUDA(cudaMemcpyAsync(h, c->diag, sizeof(h), cudaMemcpyDeviceToHost, c->stream));
    SN_CUDA(cudaStreamSynchronize(c->stream));
    double dV = 1.0;
    for (int d = 0; d < l.ndim; d++) dV *= c->L[d] / (double)l.n[d];
    for (int k = 0; k < l.ncomp; k++) norms[k] = h[k] * dV;
    return SN_OK;
}

size_t sn_slab_workspace_bytes(const int64_t *dims, int nranks, int rank)
{
    Layout l;
    return make_layout(3, dims, l, 1, 0, SN_DTYPE_C64, 1, nranks, rank) ? l.total : 0;
}

int sn_slab_create(sn_ctx **out, const int64_t *dims, const double *L, double A, double B, double C, double D,
                   const double *g, int n_g, double dtau, int nranks, int rank, void *d_workspace, size_t workspace_bytes,
                   void *cuda_stream)
{
    if (nranks < 1 || rank < 0 || rank >= nranks) return SN_ERR_PARAM;
    return create_impl(out, 3, dims, L, A, B, C, D, g, n_g, dtau, d_workspace, workspace_bytes, cuda_stream, 1, 0,
                       SN_DTYPE_C64, nullptr, nranks, rank);
}

int sn_slab_stage(sn_ctx *c, int stage, int half_phase)
{
    if (!c) return SN_ERR_NULL;
    if (c->lay.R < 1 || c->lay.ndim != 3 || c->is_mc || c->f64 || c->lay.batch != 1) return SN_ERR_FEATURE;
    if (!c->has_state) return SN_ERR_STATE;
    DeviceGuard guard(c->device);
    return slab_stage(c, stage, half_phase ? PH_HALF : PH_FULL);
}

int sn_slab_buffer(sn_ctx *c, int which, void **ptr, int64_t *elems)
{
    if (!c || !ptr || !elems) return SN_ERR_NULL;
    const Layout &l = c->lay;
    if (l.ndim != 3 || c->is_mc || c->f64 || l.batch != 1) return SN_ERR_FEATURE;
    switch (which) {
    case SN_SLAB_PSI_A: *ptr = c->psi; *elems = l.cells; break;
    case SN_SLAB_PSI_B: *ptr = c->psiB; *elems = l.cells; break;
    case SN_SLAB_HS_A: *ptr = c->hs; *elems = l.hs_elems; break;
    case SN_SLAB_HS_B: *ptr = c->hsB; *elems = l.R > 1 ? l.hsB_elems : l.hs_elems; break;
    case SN_SLAB_STAGING: *ptr = c->stage; *elems = l.cells; break;
    default: return SN_ERR_PARAM;
    }
    return SN_OK;
}

// staging <-> z-slab view: staging holds, for each peer s, the block (rows of this rank) x (columns of s) contiguously
int sn_slab_pack(sn_ctx *c, int what, int unpack)
{
    if (!c) return SN_ERR_NULL;
    const Layout &l = c->lay;
    if (what != SN_SLAB_PSI_A && what != SN_SLAB_HS_A) return SN_ERR_PARAM;
    if (l.R <= 1) return SN_OK; // one rank: view A is view B
    DeviceGuard guard(c->device);
    float2 *A = what == SN_SLAB_PSI_A ? c->psi : c->hs;
    const int64_t rows = what == SN_SLAB_PSI_A ? l.rowsA : l.h_cnt;
    for (int s = 0; s < l.R; s++) {
        // the staging area seen as a B-like array of R blocks of `rows` rows: block s starts at row s * rows
        const int rc = slab_copy_block(l, A, c->stage, (int64_t)s * rows, rows, s, /*b2a=*/unpack != 0, c->stream);
        if (rc) return rc;
    }
    return SN_OK;
}

int sn_slab_exchange_local(sn_ctx **ctxs, int nranks, int what, int to_a)
{
    if (!ctxs) return SN_ERR_NULL;
    if (what != SN_SLAB_PSI_A && what != SN_SLAB_HS_A) return SN_ERR_PARAM;
    for (int r = 0; r < nranks; r++)
        if (!ctxs[r] || ctxs[r]->lay.R != nranks || ctxs[r]->lay.rank != r || ctxs[r]->device != ctxs[0]->device ||
            ctxs[r]->stream != ctxs[0]->stream)
            return SN_ERR_PARAM; // R contexts of one decomposition, on one device and one stream
    if (nranks == 1) return SN_OK;
    DeviceGuard guard(ctxs[0]->device);
    for (int r = 0; r < nranks; r++)     // destination (to_a) / source (!to_a) of the z-slab side
        for (int s = 0; s < nranks; s++) {
            const Layout &lr = ctxs[r]->lay;
            int64_t lo = (int64_t)r * lr.rowsA, cnt = lr.rowsA;
            if (what == SN_SLAB_HS_A) { lo = lr.h_lo; cnt = lr.h_cnt; }
            float2 *A_r = what == SN_SLAB_PSI_A ? ctxs[r]->psi : ctxs[r]->hs;
            float2 *B_s = what == SN_SLAB_PSI_A ? ctxs[s]->psiB : ctxs[s]->hsB;
            const int rc = slab_copy_block(lr, A_r, B_s, lo, cnt, s, to_a != 0, ctxs[0]->stream);
            if (rc) return rc;
        }
    return SN_OK;
}

int sn_slab_local_norm(sn_ctx *c, double *sum_abs2_dv)
{
    if (!c || !sum_abs2_dv) return SN_ERR_NULL;
    if (!c->has_state) return SN_ERR_STATE;
    DeviceGuard guard(c->device);
    const Layout &l = c->lay;
    SN_CUDA(cudaMemsetAsync(c->diag, 0, 8 * sizeof(double), c->stream));
    const int rc = snk::launch_norm(c->psi, l.cells, c->diag, c->stream);
    if (rc != 0) return cuda_fail((cudaError_t)rc);
    c->launches++;
    double h = 0.0;
    SN_CUDA(cudaMemcpyAsync(&h, c->diag, sizeof(h), cudaMemcpyDeviceToHost, c->stream));
    SN_CUDA(cudaStreamSynchronize(c->stream));
    double dV = 1.0;
    for (int d = 0; d < l.ndim; d++) dV *= c->L[d] / (double)l.n[d];
    *sum_abs2_dv = h * dV;
    return SN_OK;
}

int sn_set_option(sn_ctx *c, int option, int value)
{
    if (!c) return SN_ERR_NULL;
    if (option == SN_OPT_GRAPH) {
        if (value != 0 && value != 1) return SN_ERR_PARAM;
    } else if (option == SN_OPT_GRAPH_STEPS) {
        if (value < 1 || value > 64) return SN_ERR_PARAM;
    } else if (option == SN_OPT_DISPATCH) {
        if (value < 0 || value > 2) return SN_ERR_PARAM;
    } else if (option == SN_OPT_RESIDENT) {
        if (value != 0 && value != 1) return SN_ERR_PARAM;
    } else {
        return SN_ERR_PARAM;
    }
    DeviceGuard guard(c->device);
    SN_CUDA(cudaStreamSynchronize(c->stream));
    drop_step_graph(c);
    if (option == SN_OPT_RESIDENT) {
        c->use_resident = value == 1 && c->resident_ok;
    } else if (option == SN_OPT_GRAPH_STEPS) {
        c->graph_steps = value;
    } else if (option == SN_OPT_GRAPH) {
        c->use_graph = value == 1 && c->lay.cells <= ((int64_t)1 << 24) && !c->is_mc && c->lay.R == 1;
    } else {
        c->use_pipe = value != 1 && !c->f64;
        c->pipe_all = value == 2 && !c->f64;
        c->v_in_xkin = c->has_vext && c->use_pipe && c->lay.nx % 3 != 0 && c->lay.nx >= 64;
        return upload_phase_tables(c); // the external-potential flag of the nonlinear coefficients follows v_in_xkin
    }
    return SN_OK;
}

int sn_destroy(sn_ctx *c)
{
    if (!c) return SN_ERR_NULL;
    DeviceGuard guard(c->device);
    cudaStreamSynchronize(c->stream);
    drop_step_graph(c);
    if (c->cap_stream) cudaStreamDestroy(c->cap_stream);
    if (c->ev) {
        for (cudaEvent_t e : *c->ev) cudaEventDestroy(e);
        delete c->ev;
        delete c->ev_kind;
    }
    delete c;
    return SN_OK;
}

int sn_set_dtau(sn_ctx *c, double dtau)
{
    if (!c) return SN_ERR_NULL;
    DeviceGuard guard(c->device);
    if (!std::isfinite(dtau)) return SN_ERR_PARAM;
    SN_CUDA(cudaStreamSynchronize(c->stream));
    drop_step_graph(c); // the nonlinear-phase coefficients are kernel arguments baked into the graph
    const double old = c->dtau;
    c->dtau = dtau;
    const int rc = upload_phase_tables(c);
    if (rc != SN_OK) c->dtau = old; // SN_ERR_CUDA: the tables are undefined (sn.h), the context must be destroyed
    return rc;
}

int sn_set_local_terms(sn_ctx *c, double g_log, double rho_floor, double g_pow, double p_pow)
{
    if (!c) return SN_ERR_NULL;
    DeviceGuard guard(c->device);
    if (c->is_mc || c->lay.R > 1) return SN_ERR_FEATURE; // coupled-component / slab contexts: sn_step, state copies, sn_mc_norms, sn_set_dtau
    if (!std::isfinite(g_log) || !std::isfinite(rho_floor) || !std::isfinite(g_pow) || !std::isfinite(p_pow))
        return SN_ERR_PARAM;
    if (rho_floor <= 0.0 || p_pow == -1.0) return SN_ERR_PARAM;
    if (c->f64 && (g_log != 0.0 || g_pow != 0.0)) return SN_ERR_FEATURE; // NEXT-1 terms: complex64 contexts only
    SN_CUDA(cudaStreamSynchronize(c->stream));
    drop_step_graph(c);
    c->g_log = g_log; c->rho_floor = rho_floor; c->g_pow = g_pow; c->p_pow = p_pow;
    return upload_phase_tables(c);
}

int sn_set_external_potential(sn_ctx *c, const float *v, int src_on_device)
{
    if (!c) return SN_ERR_NULL;
    DeviceGuard guard(c->device);
    if (c->is_mc || c->lay.R > 1) return SN_ERR_FEATURE; // coupled-component / slab contexts: sn_step, state copies, sn_mc_norms, sn_set_dtau
    if (v && !c->vext) return SN_ERR_FEATURE; // SN_FEAT_VEXT not requested at create
    SN_CUDA(cudaStreamSynchronize(c->stream));
    drop_step_graph(c);
    if (v) {
        SN_CUDA(cudaMemcpyAsync(c->vext, v, (size_t)c->lay.cells * 4,
                                src_on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, c->stream));
        SN_CUDA(cudaStreamSynchronize(c->stream));
    }
    c->has_vext = v != nullptr;
    c->v_in_xkin = c->has_vext && c->use_pipe && c->lay.nx % 3 != 0 && c->lay.nx >= 64; // the pipelined contiguous pass serves 2^n >= 64 only
    return upload_phase_tables(c);
}

int sn_set_bohm(sn_ctx *c, double c_bohm, double sqrt_floor)
{
    if (!c) return SN_ERR_NULL;
    DeviceGuard guard(c->device);
    if (c->is_mc || c->lay.R > 1) return SN_ERR_FEATURE; // coupled-component / slab contexts: sn_step, state copies, sn_mc_norms, sn_set_dtau
    if (!std::isfinite(c_bohm) || !std::isfinite(sqrt_floor) || sqrt_floor <= 0.0) return SN_ERR_PARAM;
    if (c->f64 && c_bohm != 0.0) return SN_ERR_FEATURE;
    SN_CUDA(cudaStreamSynchronize(c->stream));
    drop_step_graph(c);
    c->c_bohm = c_bohm;
    c->sqrt_floor = sqrt_floor;
    return SN_OK;
}

int sn_set_source_tables(sn_ctx *c, const float *beta, const float *gamma, int src_on_device)
{
    if (!c) return SN_ERR_NULL;
    DeviceGuard guard(c->device);
    if (c->is_mc || c->lay.R > 1) return SN_ERR_FEATURE; // coupled-component / slab contexts: sn_step, state copies, sn_mc_norms, sn_set_dtau
    if ((beta == nullptr) != (gamma == nullptr)) return SN_ERR_NULL;
    if (beta && (!c->bg || (!src_on_device && !c->phi))) return SN_ERR_FEATURE; // SN_FEAT_SOURCE (+ SN_FEAT_STAGING for host tables)
    SN_CUDA(cudaStreamSynchronize(c->stream));
    drop_step_graph(c);
    if (beta) {
        const cudaMemcpyKind k = src_on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice;
        // stored interleaved; host tables pass through two scratch regions (phi scratch, half spectrum) that hold
        // nothing between calls
        const float *db = beta, *dg = gamma;
        if (!src_on_device) {
            float *sb = c->phi, *sg = reinterpret_cast<float *>(c->hs);
            SN_CUDA(cudaMemcpyAsync(sb, beta, (size_t)c->lay.cells * 4, k, c->stream));
            SN_CUDA(cudaMemcpyAsync(sg, gamma, (size_t)c->lay.cells * 4, k, c->stream));
            db = sb; dg = sg;
        }
        const int rc = snk::launch_interleave(db, dg, c->bg, c->lay.cells, c->stream);
        if (rc != 0) return cuda_fail((cudaError_t)rc);
        if (!src_on_device) // the padding line of the half spectrum (2D, odd line count) must stay finite: clear the scratch
            SN_CUDA(cudaMemsetAsync(c->hs, 0, (size_t)c->lay.hs_elems * 8, c->stream));
        SN_CUDA(cudaStreamSynchronize(c->stream));
    }
    c->has_src = beta != nullptr;
    return SN_OK;
}

int sn_set_state(sn_ctx *c, const void *psi, int src_on_device)
{
    if (!c || !psi) return SN_ERR_NULL;
    DeviceGuard guard(c->device);
    SN_CUDA(cudaMemcpyAsync(c->psi, psi, (size_t)c->lay.cells * c->lay.esz * (size_t)c->lay.ncomp,
                            src_on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, c->stream));
    if (!src_on_device) SN_CUDA(cudaStreamSynchronize(c->stream)); // caller may reuse its host buffer
    c->has_state = true;
    return SN_OK;
}

int sn_get_state(sn_ctx *c, void *psi_out, int dst_on_device)
{
    if (!c || !psi_out) return SN_ERR_NULL;
    DeviceGuard guard(c->device);
    if (!c->has_state) return SN_ERR_STATE;
    SN_CUDA(cudaMemcpyAsync(psi_out, c->psi, (size_t)c->lay.cells * c->lay.esz * (size_t)c->lay.ncomp,
                            dst_on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, c->stream));
    if (!dst_on_device) SN_CUDA(cudaStreamSynchronize(c->stream));
    return SN_OK;
}

int sn_step(sn_ctx *c, int64_t nsteps)
{
    if (!c) return SN_ERR_NULL;
    DeviceGuard guard(c->device);
    if (!c->has_state) return SN_ERR_STATE;
    if (nsteps < 0) return SN_ERR_PARAM;
    if (c->lay.R > 1) return SN_ERR_FEATURE; // a slab context advances through sn_slab_stage + the caller's exchanges
    if (nsteps == 0) return SN_OK;
    if (c->is_mc) { // coupled components: same merged schedule, component-wise sweeps
        int rc = kinetic_sweep_mc(c, PH_HALF);
        for (int64_t i = 1; rc == SN_OK && i <= nsteps; i++) {
            rc = nonlinear_mc(c, c->dtau);
            if (rc == SN_OK) rc = kinetic_sweep_mc(c, i == nsteps ? PH_HALF : PH_FULL);
        }
        return rc;
    }
    if (resident_eligible(c)) return run_resident(c, nsteps); // same schedule, one launch, state held on chip
    // K(dtau/2) [N(dtau) K(dtau)]^(n-1) N(dtau) K(dtau/2): adjacent half kinetics merged
    int rc = kinetic_sweep(c, PH_HALF, /*with_nl=*/false, /*before_n=*/true);
    int64_t i = 1;
    if (rc == SN_OK && c->use_graph && !c->profiling && nsteps >= 4) {
        // each replay advances graph_steps interior steps; the interior steps left over replay the one-step graph; the
        // closing step (half kinetic sweep) runs as plain launches
        if (c->graph_steps > 1) {
            if (!c->step_graph && i + c->graph_steps <= nsteps)
                rc = build_step_graph(c, c->graph_steps, &c->step_graph, &c->graph_launches);
            for (; rc == SN_OK && i + c->graph_steps <= nsteps; i += c->graph_steps) {
                SN_CUDA(cudaGraphLaunch(c->step_graph, c->stream));
                c->launches += c->graph_launches;
            }
        }
        if (rc == SN_OK && !c->step_graph1 && i + 1 <= nsteps) rc = build_step_graph(c, 1, &c->step_graph1, &c->graph_launches1);
        for (; rc == SN_OK && i + 1 <= nsteps; i++) {
            SN_CUDA(cudaGraphLaunch(c->step_graph1, c->stream));
            c->launches += c->graph_launches1;
        }
    }
    for (; rc == SN_OK && i <= nsteps; i++) {
        rc = prepare_n(c, NL_MAIN);
        if (rc == SN_OK) rc = kinetic_sweep(c, i == nsteps ? PH_HALF : PH_FULL, /*with_nl=*/true, /*before_n=*/i < nsteps);
    }
    return rc;
}

int sn_step_order4(sn_ctx *c, int64_t nsteps)
{
    if (!c) return SN_ERR_NULL;
    DeviceGuard guard(c->device);
    if (c->is_mc || c->lay.R > 1) return SN_ERR_FEATURE; // coupled-component / slab contexts: sn_step, state copies, sn_mc_norms, sn_set_dtau
    if (!c->has_state) return SN_ERR_STATE;
    if (nsteps < 0) return SN_ERR_PARAM;
    if (nsteps == 0) return SN_OK;
    if (resident_eligible(c)) return run_resident(c, nsteps, /*order4=*/true); // same schedule, one launch
    // one step = S2(w1 h) S2(w0 h) S2(w1 h) with S2 the Strang step; adjacent kinetic halves merged:
    // K(w1/2) [N(w1) K((w1+w0)/2) N(w0) K((w0+w1)/2) N(w1) K(w1 or w1/2)]^n
    int rc = kinetic_sweep(c, PH_Y_END, /*with_nl=*/false, /*before_n=*/true, NL_MAIN, NL_Y1);
    for (int64_t i = 1; rc == SN_OK && i <= nsteps; i++) {
        rc = prepare_n(c, NL_Y1);
        if (rc == SN_OK) rc = kinetic_sweep(c, PH_Y_MID, true, true, NL_Y1, NL_Y0);
        if (rc == SN_OK) rc = prepare_n(c, NL_Y0);
        if (rc == SN_OK) rc = kinetic_sweep(c, PH_Y_MID, true, true, NL_Y0, NL_Y1);
        if (rc == SN_OK) rc = prepare_n(c, NL_Y1);
        if (rc == SN_OK) rc = kinetic_sweep(c, i == nsteps ? PH_Y_END : PH_Y_JOIN, true, /*before_n=*/i < nsteps, NL_Y1, NL_Y1);
    }
    return rc;
}

int sn_debug_fft(sn_ctx *c, int direction)
{
    if (!c) return SN_ERR_NULL;
    DeviceGuard guard(c->device);
    if (c->is_mc || c->lay.R > 1) return SN_ERR_FEATURE; // coupled-component / slab contexts: sn_step, state copies, sn_mc_norms, sn_set_dtau
    if (!c->has_state) return SN_ERR_STATE;
    if (direction != 1 && direction != -1) return SN_ERR_PARAM;
    const Layout &l = c->lay;
    for (int d = 0; d < l.ndim; d++) {
        PassArgs a = base_args(c);
        a.data = c->psi; a.tw = c->tw[d]; a.dir = direction; a.hilo = 1;
        a.scale = direction < 0 ? (float)(1.0 / (double)l.n[d]) : 1.f;
        if (d == l.ndim - 1) {
            a.kind = snk::P_X_FFT;
            a.nlines = (int)(l.cells / l.nx);
        } else {
            a.kind = snk::P_S_FFT;
            set_axis_geometry(c, a, d, l.n[0]);
        }
        const int rc = run_pass(c, (int)l.n[d], a);
        if (rc) return rc;
    }
    return SN_OK;
}

int sn_debug_potential(sn_ctx *c, float *phi_out, int dst_on_device)
{
    if (!c || !phi_out) return SN_ERR_NULL;
    DeviceGuard guard(c->device);
    if (c->is_mc || c->lay.R > 1) return SN_ERR_FEATURE; // coupled-component / slab contexts: sn_step, state copies, sn_mc_norms, sn_set_dtau
    if (!c->has_state) return SN_ERR_STATE;
    if (!dst_on_device && !c->phi) return SN_ERR_FEATURE; // a host destination is staged through the SN_FEAT_STAGING scratch
    int rc = potential_spectrum(c);
    if (rc) return rc;
    PassArgs a = base_args(c);
    a.kind = snk::P_H_POT; a.data = c->psi; a.hs = c->hs; a.tw = c->tw[0];
    a.phi_out = dst_on_device ? phi_out : c->phi;
    set_axis_geometry(c, a, 0, c->lay.n[0]);
    if ((rc = run_pass(c, (int)c->lay.n[0], a))) return rc;
    if (!dst_on_device) {
        SN_CUDA(cudaMemcpyAsync(phi_out, c->phi, (size_t)c->lay.cells * 4, cudaMemcpyDeviceToHost, c->stream));
        SN_CUDA(cudaStreamSynchronize(c->stream));
    }
    return SN_OK;
}

int sn_diagnostics(sn_ctx *c, sn_diag *out)
{
    if (!c || !out) return SN_ERR_NULL;
    DeviceGuard guard(c->device);
    if (c->is_mc || c->lay.R > 1) return SN_ERR_FEATURE; // coupled-component / slab contexts: sn_step, state copies, sn_mc_norms, sn_set_dtau
    if (!c->has_state) return SN_ERR_STATE;
    const Layout &l = c->lay;
    SN_CUDA(cudaMemsetAsync(c->diag, 0, 8 * sizeof(double), c->stream));
    int rc = potential_spectrum(c);
    if (rc) return rc;
    {
        PassArgs a = base_args(c);
        a.kind = snk::P_H_DIAG; a.data = c->psi; a.hs = c->hs; a.tw = c->tw[0];
        set_axis_geometry(c, a, 0, l.n[0]);
        if ((rc = run_pass(c, (int)l.n[0], a))) return rc;
    }
    // kinetic energy axis by axis: sum_k k_a^2 |psi^_k|^2 / prod N = sum_lines sum_ka k_a^2 |F_a psi|^2 / N_a
    // (Parseval along the other axes), so one forward line transform per axis suffices.
    for (int d = 0; d < l.ndim; d++) {
        PassArgs a = base_args(c);
        a.data = c->psi; a.tw = c->tw[d]; a.ksq = c->ksq[d]; a.diag = c->diag + 3 + d;
        if (d == l.ndim - 1) {
            a.kind = snk::P_X_KDIAG;
            a.nlines = (int)(l.cells / l.nx);
        } else {
            a.kind = snk::P_S_KDIAG;
            set_axis_geometry(c, a, d, l.n[0]);
        }
        if ((rc = run_pass(c, (int)l.n[d], a))) return rc;
    }
    double h[8];
    SN_CUDA(cudaMemcpyAsync(h, c->diag, sizeof(h), cudaMemcpyDeviceToHost, c->stream));
    SN_CUDA(cudaStreamSynchronize(c->stream));
    double dV = 1.0;
    for (int d = 0; d < l.ndim; d++)
        dV *= c->L[d] / (double)l.n[d];
    double ek = 0.0;
    for (int d = 0; d < l.ndim; d++)
        ek += h[3 + d] / (double)l.n[d];
    out->norm = h[0] * dV;
    out->e_kin = -c->A * ek * dV;
    out->e_nonlocal = 0.5 * c->B * h[1] * dV;
    out->e_local = h[2] * dV;
    out->e_total = out->e_kin + out->e_nonlocal + out->e_local;
    return SN_OK;
}

int64_t sn_launch_count(const sn_ctx *c) { return c ? c->launches : 0; }

int sn_profile(sn_ctx *c, int enable)
{
    if (!c) return SN_ERR_NULL;
    DeviceGuard guard(c->device);
    if (enable && !c->ev) {
        c->ev = new (std::nothrow) std::vector<cudaEvent_t>();
        c->ev_kind = new (std::nothrow) std::vector<int>();
        if (!c->ev || !c->ev_kind) return SN_ERR_NOMEM;
    }
    if (!enable && c->profiling) {
        const int rc = profile_flush(c);
        if (rc) return rc;
    }
    c->profiling = enable != 0;
    return SN_OK;
}

int sn_profile_read(sn_ctx *c, double *ms_by_kind, int64_t *launches_by_kind, int reset)
{
    if (!c || !ms_by_kind || !launches_by_kind) return SN_ERR_NULL;
    DeviceGuard guard(c->device);
    const int rc = profile_flush(c);
    if (rc) return rc;
    for (int k = 0; k < SN_NUM_PASS_KINDS; k++) {
        ms_by_kind[k] = c->prof_ms[k];
        launches_by_kind[k] = c->prof_launches[k];
        if (reset) {
            c->prof_ms[k] = 0.0;
            c->prof_launches[k] = 0;
        }
    }
    return SN_OK;
}

const char *sn_strerror(int code)
{
    switch (code) {
    case SN_OK: return "ok";
    case SN_ERR_NULL: return "null pointer argument";
    case SN_ERR_DIMS: return "unsupported dimensions (ndim 2 or 3; axis lengths 2^n in [32, 4096] or 3*2^a in [96, 3072])";
    case SN_ERR_PARAM: return "invalid parameter";
    case SN_ERR_SINGULAR: return "C > 0 coincides with k^2 of a grid mode: eq. (2) is singular";
    case SN_ERR_WORKSPACE: return "workspace too small or not 256-byte aligned";
    case SN_ERR_STATE: return "no state set";
    case SN_ERR_CUDA: return g_cuda_msg;
    case SN_ERR_NOMEM: return "host allocation failed";
    case SN_ERR_FEATURE: return "the call needs a workspace region that was not requested at create (sn_options.features)";
    case SN_ERR_TOO_LARGE:
        return "sn_norm_static: n_cells exceeds SN_STATIC_NORM_MAX_CELLS = 2^28 (the 256 KiB static scratch holds one partial sum "
               "per 8192 cells, 32768 slots); use a context (sn_create + sn_diagnostics) for larger arrays";
    default: return "unknown error code";
    }
}

} // extern "C"
