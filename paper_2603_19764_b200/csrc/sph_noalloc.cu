// sph_noalloc.cu -- sph_diagnostics_noalloc: the S8 conservation sums (total mass, linear and
// angular momentum, kinetic + internal energy) of a particle state the CALLER holds on the device, for callers
// that cannot give this library a workspace.
//
// Who that is.  Everything else in libsph.so works out of a device workspace the caller allocates (sph_init).
// Two kinds of host program cannot do that for a quick conservation check: (1) a simulation code that, at
// start-up, hands all of the GPU's memory to its own particle pool (the way tree codes of pkdgrav3's kind size
// their particle store) -- a later cudaMalloc there simply fails with out-of-memory; (2) a time-step loop that
// must not stall: cudaMalloc and cudaFree synchronise the whole device, so one allocation in the loop serialises
// every stream the program has in flight.  For them the per-block partial sums of the reduction -- the only
// global memory the reduction needs besides its inputs and its 8 outputs -- live in a file-scope __device__
// array below, which the CUDA runtime places in device memory when the library's module is loaded.  The entry
// point calls no cudaMalloc, no cudaFree and no library routine that allocates.
//
// What that costs.  g_diag_rows is SPH_DIAG_NOALLOC_ROWS x 8 doubles = 512 KiB; every GPU on which the library's
// module gets loaded keeps that much until the process exits, whether or not the entry point is ever called.  One
// row per 4 096 particles bounds the particle count at SPH_DIAG_NOALLOC_MAX_N = 2^25 (BASELINE.json's largest
// configuration has 31 998 174).
//
// Sharing.  There is one array per device, not one per call.  A call writes rows 0 .. ceil(n/4096)-1 and then
// reads exactly those rows, so nothing in the array has to start at zero and the previous call's rows (which
// stay in it) are never read.  Two calls that run on the GPU at the same time -- different streams of one device,
// from one host thread or several -- write the same rows and race: their results are undefined.  Calls on ONE
// stream are ordered and safe, as are calls on different devices (each device has its own copy of the array).
//
// The array's name in HOST code is not a device address (it is the host-side handle the runtime registered for
// the symbol): a kernel given `g_diag_rows` from host code would fault or touch unrelated memory.  The host side
// therefore asks the runtime for the address once per device (cudaGetSymbolAddress with that device current)
// and hands the kernels that pointer.
#include <cuda_runtime.h>

#include <mutex>

#include "../../include/sph.h"

#define NOALLOC_SPAN 4096                                          // particles per row (one CTA of 256 threads, 16 each)
#define NOALLOC_ROWS (SPH_DIAG_NOALLOC_MAX_N / NOALLOC_SPAN)       // 8 192
#define NOALLOC_MAX_DEVICES 64

static_assert(SPH_DIAG_NOALLOC_MAX_N % NOALLOC_SPAN == 0, "whole rows");

static __device__ __align__(256) double g_diag_rows[NOALLOC_ROWS * 8];

// device address of g_diag_rows per device ordinal; nullptr = not asked yet
static double *g_rows_addr[NOALLOC_MAX_DEVICES];
static std::mutex g_rows_mutex;

// One CTA per span of 4 096 particles, a fixed summation order that depends on n only (not on the GPU):
// thread t of the CTA adds particles base + t, base + t + 256, ...; lanes by a shuffle tree, warps in order.
__global__ void __launch_bounds__(256) k_diag_rows(const float *__restrict__ x, const float *__restrict__ y,
                                                   const float *__restrict__ z, const float *__restrict__ m,
                                                   const float *__restrict__ vx, const float *__restrict__ vy,
                                                   const float *__restrict__ vz, const float *__restrict__ u,
                                                   long long n, double *__restrict__ rows)
{
    const long long base = (long long)blockIdx.x * NOALLOC_SPAN;
    const long long end = base + NOALLOC_SPAN < n ? base + NOALLOC_SPAN : n;
    double s[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    for (long long i = base + threadIdx.x; i < end; i += 256) {
        const double mi = m[i], xi = x[i], yi = y[i], zi = z[i];
        const double vxi = vx[i], vyi = vy[i], vzi = vz[i], ui = u[i];
        s[0] += mi;
        s[1] += mi * vxi; s[2] += mi * vyi; s[3] += mi * vzi;
        s[4] += mi * (yi * vzi - zi * vyi); s[5] += mi * (zi * vxi - xi * vzi); s[6] += mi * (xi * vyi - yi * vxi);
        s[7] += mi * (0.5 * (vxi * vxi + vyi * vyi + vzi * vzi) + ui);
    }
    __shared__ double sh[8][8];
#pragma unroll
    for (int k = 0; k < 8; ++k) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) s[k] += __shfl_xor_sync(0xffffffffu, s[k], o);
        if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5][k] = s[k];
    }
    __syncthreads();
    if (threadIdx.x < 8) {
        double t = 0.0;
        for (int w = 0; w < 8; ++w) t += sh[w][threadIdx.x];
        rows[(long long)blockIdx.x * 8 + threadIdx.x] = t;
    }
}

// 8 warps, one per quantity; a lane adds rows lane, lane + 32, ...; then a shuffle tree.  nrows = 0 writes zeros.
__global__ void __launch_bounds__(256) k_diag_rows_sum(const double *__restrict__ rows, int nrows, double *__restrict__ out)
{
    const int k = threadIdx.x >> 5, lane = threadIdx.x & 31;
    double t = 0.0;
    for (int b = lane; b < nrows; b += 32) t += rows[b * 8 + k];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
    if (lane == 0) out[k] = t;
}

// Set-up, once per device: the device address of g_diag_rows on the CURRENT device.
static cudaError_t rows_address(double **addr)
{
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= NOALLOC_MAX_DEVICES) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_rows_mutex);
    if (!g_rows_addr[dev]) {
        double *p = nullptr;
        e = cudaGetSymbolAddress((void **)&p, g_diag_rows);
        if (e != cudaSuccess) return e;
        if (!p) return cudaErrorInvalidSymbol;
        g_rows_addr[dev] = p;
    }
    *addr = g_rows_addr[dev];
    return cudaSuccess;
}

extern "C" int sph_diagnostics_noalloc(const sph_state *state, long long n, double *out, void *cuda_stream, int *cuda_error)
{
    if (cuda_error) *cuda_error = 0;
    if (!state || !out || n < 0) return SPH_EINVAL;
    if (n > (long long)SPH_DIAG_NOALLOC_MAX_N) return SPH_ECAPACITY;    // more rows than g_diag_rows has
    if (n > 0 && (!state->x || !state->y || !state->z || !state->m || !state->vx || !state->vy || !state->vz || !state->u))
        return SPH_EINVAL;
    double *rows = nullptr;
    cudaError_t e = rows_address(&rows);
    if (e == cudaSuccess) {
        cudaStream_t st = (cudaStream_t)cuda_stream;
        const int nrows = (int)((n + NOALLOC_SPAN - 1) / NOALLOC_SPAN);
        if (nrows > 0)
            k_diag_rows<<<nrows, 256, 0, st>>>(state->x, state->y, state->z, state->m, state->vx, state->vy, state->vz,
                                               state->u, n, rows);
        k_diag_rows_sum<<<1, 256, 0, st>>>(rows, nrows, out);
        e = cudaGetLastError();
    }
    if (e != cudaSuccess) {
        if (cuda_error) *cuda_error = (int)e;
        return SPH_ECUDA;
    }
    return SPH_OK;
}
