// sph_bench.cu -- measurement aid: the FP32 CUDA-core rate of this device on independent FFMA chains.
// "measure an FMA-chain microbenchmark and the sustained SM clock, and quote %
// against both the nominal and the measured peak".  No memory traffic, 8 independent chains per thread
// (FFMA latency is 4 cycles; 4 warps per scheduler x 8 chains keep every issue slot busy), 2 flop per FFMA.
#include "sph_internal.cuh"

#define PEAK_CHAINS 8
#define PEAK_ITERS 4096

__global__ void __launch_bounds__(512) k_fma_chains(float *out, float a, float b)
{
    float x[PEAK_CHAINS];
#pragma unroll
    for (int k = 0; k < PEAK_CHAINS; ++k) x[k] = (float)(threadIdx.x + k) * 1.0e-3f;
    for (int it = 0; it < PEAK_ITERS / 8; ++it) {
#pragma unroll
        for (int u = 0; u < 8; ++u) {
#pragma unroll
            for (int k = 0; k < PEAK_CHAINS; ++k) x[k] = fmaf(x[k], a, b);
        }
    }
    float s = 0.f;
#pragma unroll
    for (int k = 0; k < PEAK_CHAINS; ++k) s += x[k];
    if (s == 123.456f) out[0] = s;          // never true: keeps the chains alive
}

extern "C" int sph_fp32_peak(void *cuda_stream, int repeats, double *tflops)
{
    if (!tflops || repeats < 1) return SPH_EINVAL;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int dev = 0, nsm = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess)
        return SPH_ECUDA;
    float *out = nullptr;
    if (cudaMalloc(&out, sizeof(float)) != cudaSuccess) return SPH_ECUDA;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    const int blocks = nsm * 4 * 8, threads = 512;       // 4 resident CTAs of 16 warps per SM, 8 waves
    const double flop = 2.0 * PEAK_CHAINS * (double)PEAK_ITERS * (double)blocks * threads;
    double best = 0.0;
    int rc = SPH_OK;
    for (int r = 0; r < repeats + 1; ++r) {              // the first launch is a warm-up
        cudaEventRecord(e0, st);
        k_fma_chains<<<blocks, threads, 0, st>>>(out, 0.999f, 1.0e-3f);
        cudaEventRecord(e1, st);
        if (cudaEventSynchronize(e1) != cudaSuccess) { rc = SPH_ECUDA; break; }
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        if (r > 0 && ms > 0.f) best = fmax(best, flop / (ms * 1.0e-3) / 1.0e12);
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(out);
    if (rc == SPH_OK && cudaGetLastError() != cudaSuccess) rc = SPH_ECUDA;
    *tflops = best;
    return rc;
}

// ------------------------------------------------------------------------------------------
// Shared-memory scatter rate (see include/sph.h): every thread adds NACC values to the accumulators of a
// pseudo-random target of its tile, SCATTER_ITERS times; shared-memory float atomicAdd is a CAS loop on sm_100a.
// ------------------------------------------------------------------------------------------
#define SCATTER_ITERS 2048
template <int NACC>
__global__ void __launch_bounds__(256, 2) k_shared_scatter(float *out)
{
    __shared__ float acc[NACC][256];
    for (int k = threadIdx.x; k < NACC * 256; k += 256) (&acc[0][0])[k] = 0.f;
    __syncthreads();
    unsigned x = (blockIdx.x * 256u + threadIdx.x) * 2654435761u + 12345u;
    float v = 1.0f + (float)threadIdx.x * 1.0e-3f;
    for (int it = 0; it < SCATTER_ITERS; ++it) {
        x = x * 1664525u + 1013904223u;
        const int j = (int)(x >> 24);
#pragma unroll
        for (int c = 0; c < NACC; ++c) atomicAdd(&acc[c][j], v);
        v += 1.0e-6f;
    }
    __syncthreads();
    float s = 0.f;
    for (int c = 0; c < NACC; ++c) s += acc[c][threadIdx.x];
    if (s == -1.f) out[0] = s;
}

extern "C" int sph_shared_scatter_rate(void *cuda_stream, int accumulators, double *pairs_per_s)
{
    if (!pairs_per_s || (accumulators != 5 && accumulators != 20)) return SPH_EINVAL;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int dev = 0, nsm = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess)
        return SPH_ECUDA;
    float *out = nullptr;
    if (cudaMalloc(&out, sizeof(float)) != cudaSuccess) return SPH_ECUDA;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    const int blocks = nsm * 2 * 4;
    double best = 0.0;
    int rc = SPH_OK;
    for (int r = 0; r < 4; ++r) {
        cudaEventRecord(e0, st);
        if (accumulators == 20) k_shared_scatter<20><<<blocks, 256, 0, st>>>(out);
        else k_shared_scatter<5><<<blocks, 256, 0, st>>>(out);
        cudaEventRecord(e1, st);
        if (cudaEventSynchronize(e1) != cudaSuccess) { rc = SPH_ECUDA; break; }
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        if (r > 0 && ms > 0.f) best = fmax(best, (double)blocks * 256.0 * SCATTER_ITERS / (ms * 1.0e-3));
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(out);
    if (rc == SPH_OK && cudaGetLastError() != cudaSuccess) rc = SPH_ECUDA;
    *pairs_per_s = best;
    return rc;
}
