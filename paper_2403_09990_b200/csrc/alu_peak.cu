// Measured CUDA-core FMA peak of the device: the roofline denominator of the walker kernel.
// MEASURED_PEAKS.json carries only HBM and bf16 tensor peaks; the walk is bound by the plain
// FP64 (or FP32) pipes, so the library times a register-resident FMA chain itself
// (DESIGN.md "Roofline").
#include <cuda_runtime.h>

#include "closure_internal.h"

namespace closure {
namespace {

constexpr int kChains = 8;
constexpr int kIters = 4096;
constexpr int kUnroll = 16;

template <typename T>
__global__ void __launch_bounds__(256) fma_chain_kernel(T *sink, T a, T b)
{
    T x[kChains];
#pragma unroll
    for (int c = 0; c < kChains; ++c) x[c] = (T)(threadIdx.x + c) * (T)1e-3;
    for (int it = 0; it < kIters / kUnroll; ++it) {
#pragma unroll
        for (int u = 0; u < kUnroll; ++u)
#pragma unroll
            for (int c = 0; c < kChains; ++c) x[c] = fma(x[c], a, b);
    }
    T s = 0;
#pragma unroll
    for (int c = 0; c < kChains; ++c) s += x[c];
    if (s == (T)123456789) sink[0] = s;      // never true; keeps the chain live
}

template <typename T>
cudaError_t run(double *flops_per_s, double *seconds, cudaStream_t stream)
{
    int dev = 0, sms = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess) return e;
    T *sink = nullptr;
    e = cudaMalloc(&sink, sizeof(T));
    if (e != cudaSuccess) return e;
    cudaEvent_t t0, t1;
    cudaEventCreate(&t0);
    cudaEventCreate(&t1);
    const int blocks = sms * 16;
    float best_ms = 1e30f;
    for (int rep = 0; rep < 5; ++rep) {      // first repetitions warm the clocks up
        cudaEventRecord(t0, stream);
        fma_chain_kernel<T><<<blocks, 256, 0, stream>>>(sink, (T)0.999, (T)1e-3);
        cudaEventRecord(t1, stream);
        e = cudaEventSynchronize(t1);
        if (e != cudaSuccess) break;
        float ms = 0.f;
        cudaEventElapsedTime(&ms, t0, t1);
        if (rep >= 2 && ms < best_ms) best_ms = ms;
    }
    cudaEventDestroy(t0);
    cudaEventDestroy(t1);
    cudaFree(sink);
    if (e != cudaSuccess) return e;
    e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    const double flops = 2.0 * (double)blocks * 256.0 * (double)kIters * (double)kChains;
    *seconds = best_ms * 1e-3;
    *flops_per_s = flops / (best_ms * 1e-3);
    return cudaSuccess;
}

// Philox4x32-10 calls per second: 4 independent counters per thread, nothing else (the integer work of an
// iteration that a flop count does not see: 150 calls per walker-step at the paper's N_P).
constexpr int kPhiloxIters = 512;

__global__ void __launch_bounds__(256) philox_rate_kernel(unsigned int *sink, unsigned int k0, unsigned int k1)
{
    unsigned int acc = 0;
    for (int it = 0; it < kPhiloxIters; ++it) {
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            unsigned int c0 = threadIdx.x + blockIdx.x * 256u, c1 = it, c2 = q, c3 = 1u, a0 = k0, a1 = k1;
#pragma unroll
            for (int r = 0; r < 10; ++r) {
                const unsigned int hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
                const unsigned int hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
                c0 = hi1 ^ c1 ^ a0; c1 = lo1; c2 = hi0 ^ c3 ^ a1; c3 = lo0;
                a0 += 0x9E3779B9u; a1 += 0xBB67AE85u;
            }
            acc ^= c0 ^ c1 ^ c2;
        }
    }
    if (acc == 0x12345678u) sink[0] = acc;       // practically never true; keeps the calls live
}

cudaError_t run_philox(double *calls_per_s, double *seconds, cudaStream_t stream)
{
    int dev = 0, sms = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess) return e;
    unsigned int *sink = nullptr;
    e = cudaMalloc(&sink, sizeof(unsigned int));
    if (e != cudaSuccess) return e;
    cudaEvent_t t0, t1;
    cudaEventCreate(&t0);
    cudaEventCreate(&t1);
    const int blocks = sms * 16;
    float best_ms = 1e30f;
    for (int rep = 0; rep < 5; ++rep) {
        cudaEventRecord(t0, stream);
        philox_rate_kernel<<<blocks, 256, 0, stream>>>(sink, 1u + rep, 2u);
        cudaEventRecord(t1, stream);
        e = cudaEventSynchronize(t1);
        if (e != cudaSuccess) break;
        float ms = 0.f;
        cudaEventElapsedTime(&ms, t0, t1);
        if (rep >= 2 && ms < best_ms) best_ms = ms;
    }
    cudaEventDestroy(t0);
    cudaEventDestroy(t1);
    cudaFree(sink);
    if (e != cudaSuccess) return e;
    e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    *seconds = best_ms * 1e-3;
    *calls_per_s = (double)blocks * 256.0 * kPhiloxIters * 4.0 / (best_ms * 1e-3);
    return cudaSuccess;
}

}  // namespace

cudaError_t measure_alu_peak(int precision, double *flops_per_s, double *seconds, cudaStream_t stream)
{
    if (precision == 64) return run<double>(flops_per_s, seconds, stream);
    if (precision == 32) return run<float>(flops_per_s, seconds, stream);
    if (precision == 4) return run_philox(flops_per_s, seconds, stream);
    return cudaErrorInvalidValue;
}

}  // namespace closure
