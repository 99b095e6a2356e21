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
// sph_fp32_rate: the same measurement for the instruction FORMS a real kernel is made of (round 3; the question behind it:
// k_pair_l is issue-bound with scalar FP32 instructions, sm_100a has packed fma/mul/add.rn.f32x2 -- SASS FFMA2 -- that
// do two lanes' worth of work per issue slot).  Variants:
//   0  scalar FFMA, multiplier and addend from the constant bank (k_fma_chains above, the roofline's denominator)
//   1  scalar FFMA, three REGISTER operands (what the pair kernels issue almost everywhere)
//   2  packed FFMA2 (__ffma2_rn), three 64-bit register operands
//   3  variant 1 with one independent integer ALU instruction (PRMT) per FFMA  -- 8 FFMA + 8 PRMT per round
//   4  variant 2 with one independent integer ALU instruction (PRMT) per FFMA2 -- 8 FFMA2 + 8 PRMT per round
// 3 against 1 and 4 against 2 show what an issue slot taken by something else costs each form.
// ------------------------------------------------------------------------------------------
template <int VARIANT>
__global__ void __launch_bounds__(512) k_fp32_forms(float *out, float seed)
{
    constexpr bool PACKED = VARIANT == 2 || VARIANT == 4, WITH_ALU = VARIANT >= 3;
    float2 x[PEAK_CHAINS], y[PEAK_CHAINS], z[PEAK_CHAINS];
    unsigned q[PEAK_CHAINS];
#pragma unroll
    for (int k = 0; k < PEAK_CHAINS; ++k) {
        const float t = (float)(threadIdx.x + k) * 1.0e-3f + seed;       // run-time values: nothing folds into an immediate
        x[k] = make_float2(t, t + 0.5f);
        y[k] = make_float2(0.999f - t * 1.0e-6f, 0.998f + t * 1.0e-6f);
        z[k] = make_float2(1.0e-3f + t * 1.0e-7f, 2.0e-3f - t * 1.0e-7f);
        q[k] = __float_as_uint(t) * 2654435761u + (unsigned)k;
    }
    const unsigned m1 = __float_as_uint(seed) + threadIdx.x, m2 = 0x4321u + (blockIdx.x & 1u);   // two run-time registers
    for (int it = 0; it < PEAK_ITERS / 8; ++it) {
#pragma unroll
        for (int u = 0; u < 8; ++u) {
#pragma unroll
            for (int k = 0; k < PEAK_CHAINS; ++k) {
                if (PACKED) x[k] = __ffma2_rn(x[k], y[k], z[k]);
                else x[k].x = fmaf(x[k].x, y[k].x, z[k].x);
                if (WITH_ALU) q[k] = __byte_perm(q[k], m1, m2);          // one PRMT on three registers (ALU pipe)
            }
        }
    }
    float s = 0.f;
    unsigned qs = 0u;
#pragma unroll
    for (int k = 0; k < PEAK_CHAINS; ++k) { s += x[k].x + (PACKED ? x[k].y : 0.f); qs ^= q[k]; }
    if (s == 123.456f || (WITH_ALU && qs == 0x12345u)) out[0] = s;       // never true: keeps the chains alive
}

extern "C" int sph_fp32_rate(void *cuda_stream, int variant, int repeats, double *tflops)
{
    if (!tflops || repeats < 1 || variant < 0 || variant > 4) return SPH_EINVAL;
    if (variant == 0) return sph_fp32_peak(cuda_stream, repeats, tflops);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int dev = 0, nsm = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess)
        return SPH_ECUDA;
    float *out = nullptr;
    if (cudaMalloc(&out, sizeof(float)) != cudaSuccess) return SPH_ECUDA;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    const int blocks = nsm * 2 * 8, threads = 512;       // 2 resident CTAs of 16 warps per SM (the register budget), 8 waves
    const double per = (variant == 2 || variant == 4) ? 4.0 : 2.0;
    const double flop = per * PEAK_CHAINS * (double)PEAK_ITERS * (double)blocks * threads;
    double best = 0.0;
    int rc = SPH_OK;
    for (int r = 0; r < repeats + 1; ++r) {              // the first launch is a warm-up
        cudaEventRecord(e0, st);
        switch (variant) {
        case 1: k_fp32_forms<1><<<blocks, threads, 0, st>>>(out, 0.25f); break;
        case 2: k_fp32_forms<2><<<blocks, threads, 0, st>>>(out, 0.25f); break;
        case 3: k_fp32_forms<3><<<blocks, threads, 0, st>>>(out, 0.25f); break;
        default: k_fp32_forms<4><<<blocks, threads, 0, st>>>(out, 0.25f); break;
        }
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
