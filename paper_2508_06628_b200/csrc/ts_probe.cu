/*
 * ts_probe.cu -- register-only FMA microbenchmark ("the builder measures both [FP32 and FP64 peaks]
 * with a register-only FMA microbenchmark and uses the measured value").  bench.py reports the ALU roofline of the
 * pair kernels against these numbers instead of the nominal 148 x 128 x 2 x clock.
 *
 * Every thread runs eight independent FMA chains (enough to cover the pipe latency at full occupancy) for `iters`
 * rounds; nothing touches memory inside the loop.  FLOP = 2 x 8 x iters x threads.
 */
#include <stdint.h>

#include "ts_internal.cuh"

template <typename T>
__global__ void __launch_bounds__(1024) k_fma_probe(T *out, int iters, T a, T b)
{
    T x0 = (T)threadIdx.x, x1 = x0 + (T)1, x2 = x0 + (T)2, x3 = x0 + (T)3, x4 = x0 + (T)4, x5 = x0 + (T)5, x6 = x0 + (T)6, x7 = x0 + (T)7;
#pragma unroll 4
    for (int k = 0; k < iters; ++k) {
        x0 = x0 * a + b; x1 = x1 * a + b; x2 = x2 * a + b; x3 = x3 * a + b;
        x4 = x4 * a + b; x5 = x5 * a + b; x6 = x6 * a + b; x7 = x7 * a + b;
    }
    const T s = ((x0 + x1) + (x2 + x3)) + ((x4 + x5) + (x6 + x7));
    if (s == (T)-1.2345) out[blockIdx.x] = s;          /* never true: keeps the chains alive */
}

/* packed variant: fma.rn.f32x2 (two FMAs per instruction on Blackwell), the form the resident LJ loop issues */
__global__ void __launch_bounds__(1024) k_fma2_probe(float *out, int iters, float a, float b)
{
    unsigned long long x[8], A, B;
    asm("mov.b64 %0, {%1, %1};" : "=l"(A) : "f"(a));
    asm("mov.b64 %0, {%1, %1};" : "=l"(B) : "f"(b));
#pragma unroll
    for (int k = 0; k < 8; ++k) { const float v = (float)(threadIdx.x + k); asm("mov.b64 %0, {%1, %1};" : "=l"(x[k]) : "f"(v)); }
#pragma unroll 4
    for (int k = 0; k < iters; ++k)
#pragma unroll
        for (int c = 0; c < 8; ++c) asm("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(x[c]) : "l"(A), "l"(B));
    unsigned long long s = 0ull;
#pragma unroll
    for (int c = 0; c < 8; ++c) s ^= x[c];
    if (s == 0x123456789abcdefull) out[blockIdx.x] = 1.f;
}

/* kind 0: fp32 FFMA, 1: fp64 DFMA, 2: packed fp32 (FFMA2).  *tflops = measured rate; scratch: device, >= 4096 bytes.
 * Synchronises `stream` (CUDA events around the launch, best of three). */
extern "C" ts_status ts_measure_fma_tflops(int32_t kind, void *scratch, double *tflops, void *stream)
{
    if (!scratch || !tflops || kind < 0 || kind > 2) return TS_ERR_INVALID_ARG;
    cudaStream_t q = (cudaStream_t)stream;
    int dev = 0, nsm = 148;
    if (cudaGetDevice(&dev) != cudaSuccess) return TS_ERR_CUDA;
    cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev);
    const int blocks = nsm * 2, threads = 1024, iters = kind == 1 ? 1 << 13 : 1 << 15;
    cudaEvent_t e0, e1;
    if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) return TS_ERR_CUDA;
    double best = 0.0;
    for (int rep = 0; rep < 4; ++rep) {
        cudaEventRecord(e0, q);
        if (kind == 0) k_fma_probe<float><<<blocks, threads, 0, q>>>((float *)scratch, iters, 0.999f, 0.001f);
        else if (kind == 1) k_fma_probe<double><<<blocks, threads, 0, q>>>((double *)scratch, iters, 0.999, 0.001);
        else k_fma2_probe<<<blocks, threads, 0, q>>>((float *)scratch, iters, 0.999f, 0.001f);
        cudaEventRecord(e1, q);
        if (cudaEventSynchronize(e1) != cudaSuccess) { cudaEventDestroy(e0); cudaEventDestroy(e1); return TS_ERR_CUDA; }
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        const double flop = 2.0 * 8.0 * (kind == 2 ? 2.0 : 1.0) * (double)iters * (double)blocks * (double)threads;
        if (rep > 0 && ms > 0.f && flop / (ms * 1e-3) / 1e12 > best) best = flop / (ms * 1e-3) / 1e12;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    *tflops = best;
    return cudaGetLastError() == cudaSuccess ? TS_OK : TS_ERR_CUDA;
}
