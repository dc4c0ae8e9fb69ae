// Measurement-only entry point (include/numa_b200_measure.h): the FP64 FMA ceiling of the
// device, the denominator of bench.py's FP64 roofline leg.
#include <algorithm>

#include "numa_internal.cuh"

namespace {

constexpr int kChains = 8;       // independent accumulators per thread
constexpr int kIters = 1024;     // FMAs per accumulator per launch
constexpr int kThreads = 256;

__global__ void __launch_bounds__(kThreads)
k_dfma_peak(double *out, double a, double b)
{
    double x[kChains];
#pragma unroll
    for (int c = 0; c < kChains; ++c) x[c] = (double)(threadIdx.x + c) * 1e-3;
#pragma unroll 1
    for (int it = 0; it < kIters / 8; ++it) {
#pragma unroll
        for (int u = 0; u < 8; ++u) {
#pragma unroll
            for (int c = 0; c < kChains; ++c) x[c] = fma(x[c], a, b);
        }
    }
    double s = 0.0;
#pragma unroll
    for (int c = 0; c < kChains; ++c) s += x[c];
    if (s == 123.456) out[0] = s;  // never true for the arguments used: keeps the chains alive
}

}  // namespace

extern "C" numa_status numa_measure_fp64_peak(int32_t repeats, double *tflops, void *stream)
{
    if (!tflops || repeats < 1) return NUMA_ERR_ARG;
    cudaStream_t s = (cudaStream_t)stream;
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess ||
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) {
        cudaGetLastError();
        return NUMA_ERR_CUDA;
    }
    const int blocks = sms * 8 * 16;   // 16 waves of 8 resident 256-thread blocks per SM
    double *d_out = nullptr;
    cudaEvent_t e0, e1;
    if (cudaMalloc(&d_out, 8) != cudaSuccess) { cudaGetLastError(); return NUMA_ERR_CUDA; }
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    double best = 0.0;
    numa_status st = NUMA_OK;
    for (int r = 0; r <= repeats; ++r) {   // r = 0 is the warm-up
        cudaEventRecord(e0, s);
        k_dfma_peak<<<blocks, kThreads, 0, s>>>(d_out, 0.999999, 1e-7);
        cudaEventRecord(e1, s);
        float ms = 0.f;
        if (cudaEventSynchronize(e1) != cudaSuccess || cudaEventElapsedTime(&ms, e0, e1) != cudaSuccess) {
            cudaGetLastError();
            st = NUMA_ERR_CUDA;
            break;
        }
        const double fl = 2.0 * kChains * kIters * (double)kThreads * blocks;
        if (r > 0) best = std::max(best, fl / (ms * 1e-3) / 1e12);
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaFree(d_out);
    *tflops = best;
    return st;
}
