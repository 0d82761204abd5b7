// sn_static.cu -- the one entry point of libsn.so that needs no caller workspace and allocates nothing:
// sn_norm_static (include/sn.h).
//
// Why: some callers cannot allocate device memory at the call site -- code under CUDA graph capture, tight serving
// loops, harnesses that forbid cudaMalloc.  Every other entry point of the library works on a caller-owned workspace
// (sn_create); this one is the norm reduction of the diagnostics (S12 of SURVEY.md 8(a): norm = sum |psi|^2 dV, fp32
// data, fp64 accumulation) as a variant of the existing kernel k_norm (sn_kernels.cu; used by sn_mc_norms and
// sn_slab_local_norm), whose accumulator lives in the context's workspace and is cleared by a memset before each
// launch.  Here the scratch is a file-scope __device__ array: SN_STATIC_NORM_SCRATCH_DOUBLES doubles = 256 KiB, held by
// every GPU that loads the library until the process exits.
//
// Scratch protocol.  Block b of the first kernel sums the squares of its own 8192 cells in a fixed order and WRITES
// partial[b]; the second kernel (one block) adds partial[0 .. nblocks) in a fixed order, scales by dV and writes the
// caller's output.  A call reads only slots it has written itself, so nothing has to start at zero; slots beyond
// nblocks keep an earlier call's values and are never read.  The result is bitwise reproducible (no atomics).
// All calls on a device share the array: two calls that OVERLAP on the GPU (different streams, or graphs replayed
// concurrently) race on it -- keep them on one stream or order them with events.
//
// The array's name is a host-side stand-in in host code, not a device address: the address the kernels get is taken
// with cudaGetSymbolAddress, once per device, with that device current (scratch_for_device below).
#include "../../include/sn.h"

#include <cuda_runtime.h>
#include <mutex>

namespace {

constexpr int CELLS_PER_BLOCK = 8192; // one partial per 8192 cells
constexpr int THREADS = 256;
static_assert(SN_STATIC_NORM_MAX_CELLS == (long long)SN_STATIC_NORM_SCRATCH_DOUBLES * CELLS_PER_BLOCK, "limit = scratch slots x cells per slot");

static __device__ __align__(256) double g_norm_scratch[SN_STATIC_NORM_SCRATCH_DOUBLES];

// partial[b] = sum over the block's cells of |psi|^2: fp32 squares, fp64 sums, fixed order
__global__ void __launch_bounds__(THREADS) k_norm_partial(const float2 *__restrict__ psi, long long n, double *__restrict__ partial)
{
    __shared__ double red[THREADS / 32];
    const long long base = (long long)blockIdx.x * CELLS_PER_BLOCK;
    double s = 0.0;
#pragma unroll 8
    for (int i = 0; i < CELLS_PER_BLOCK / THREADS; i++) {
        const long long c = base + (long long)i * THREADS + threadIdx.x;
        if (c < n) {
            const float2 v = psi[c];
            s += (double)fmaf(v.x, v.x, v.y * v.y);
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0;
#pragma unroll
        for (int w = 0; w < THREADS / 32; w++) t += red[w];
        partial[blockIdx.x] = t;
    }
}

// *out = dv * sum partial[0 .. nb), one block, fixed order
__global__ void __launch_bounds__(1024) k_norm_final(const double *__restrict__ partial, int nb, double dv, double *__restrict__ out)
{
    __shared__ double red[32];
    double s = 0.0;
    for (int i = threadIdx.x; i < nb; i += 1024) s += partial[i];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0;
#pragma unroll
        for (int w = 0; w < 32; w++) t += red[w];
        *out = t * dv;
    }
}

// device address of the scratch array on `dev` (which must be the current device): taken once per device
constexpr int MAX_DEVICES = 64;
std::mutex g_mu;
double *g_scratch_ptr[MAX_DEVICES] = {};

cudaError_t scratch_for_device(int dev, double **ptr)
{
    std::lock_guard<std::mutex> lk(g_mu);
    if (!g_scratch_ptr[dev]) {
        double *p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress((void **)&p, g_norm_scratch);
        if (e != cudaSuccess) return e;
        g_scratch_ptr[dev] = p;
    }
    *ptr = g_scratch_ptr[dev];
    return cudaSuccess;
}

} // namespace

namespace snk {
void record_cuda_error(int cuda_error); // sn_api.cu: the text sn_strerror(SN_ERR_CUDA) returns on this thread
}

extern "C" {

int sn_norm_static(const void *psi, int64_t n_cells, double dv, double *norm_out, void *cuda_stream)
{
    if (!psi || !norm_out) return SN_ERR_NULL;
    if (n_cells < 0 || !(dv == dv)) return SN_ERR_PARAM;
    if (n_cells > SN_STATIC_NORM_MAX_CELLS) return SN_ERR_TOO_LARGE; // text: sn_strerror (states the limit)
    // run on the device that owns psi; restore the caller's device on return
    cudaPointerAttributes pat;
    cudaError_t e = cudaPointerGetAttributes(&pat, psi);
    if (e != cudaSuccess || (pat.type != cudaMemoryTypeDevice && pat.type != cudaMemoryTypeManaged)) {
        cudaGetLastError();
        return SN_ERR_PARAM; // psi is not a device pointer
    }
    const int dev = pat.device;
    if (dev < 0 || dev >= MAX_DEVICES) return SN_ERR_PARAM;
    int prev = -1;
    if ((e = cudaGetDevice(&prev)) != cudaSuccess) goto fail;
    if (prev != dev && (e = cudaSetDevice(dev)) != cudaSuccess) goto fail;
    {
        double *scratch = nullptr;
        e = scratch_for_device(dev, &scratch);
        if (e == cudaSuccess) {
            cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
            const int nb = (int)((n_cells + CELLS_PER_BLOCK - 1) / CELLS_PER_BLOCK);
            if (nb > 0) k_norm_partial<<<nb, THREADS, 0, st>>>(static_cast<const float2 *>(psi), n_cells, scratch);
            k_norm_final<<<1, 1024, 0, st>>>(scratch, nb, dv, norm_out);
            e = cudaGetLastError();
        }
        if (prev != dev) cudaSetDevice(prev);
        if (e == cudaSuccess) return SN_OK;
    }
fail:
    snk::record_cuda_error((int)e);
    return SN_ERR_CUDA;
}

} // extern "C"
