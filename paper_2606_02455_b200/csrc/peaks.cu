// Measured arithmetic peaks of the device this process runs on: plain FMA throughput in fp32 and fp64 (the roofline
// denominators of the fp32 MLIP path and of the fp64 cfg1 path; MEASURED_PEAKS.json only carries HBM and bf16 tensor figures).
// A grid of resident warps runs 16 independent FMA chains per thread; timed with CUDA events on the caller's stream.
#include <algorithm>
#include "lsd_internal.h"

namespace {

template <typename T>
__global__ void __launch_bounds__(256) k_fma_chain(T* out, int iters, T a, T b)
{
    T x[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) x[i] = (T)(threadIdx.x + i) * (T)1e-3;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 16; ++i) x[i] = fma(x[i], a, b);
    }
    T s = (T)0;
#pragma unroll
    for (int i = 0; i < 16; ++i) s += x[i];
    out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = s;
}

template <typename T> double measure(cudaStream_t st, int iters)
{
    const int blocks = lsd_sm_count() * 8, threads = 256;
    T* out = nullptr;
    if (cudaMalloc(&out, sizeof(T) * (size_t)blocks * threads) != cudaSuccess) return -1.0;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    double best = 0.0;
    for (int rep = 0; rep < 4; ++rep) {                     // first repetition warms up; best of the rest
        cudaEventRecord(e0, st);
        k_fma_chain<T><<<blocks, threads, 0, st>>>(out, iters, (T)0.999, (T)1e-3);
        cudaEventRecord(e1, st);
        cudaEventSynchronize(e1);
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        const double flops = 2.0 * 16.0 * (double)iters * (double)blocks * threads;
        if (rep > 0 && ms > 0.f) best = std::max(best, flops / (ms * 1e-3) / 1e12);
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaFree(out);
    return cudaGetLastError() == cudaSuccess ? best : -1.0;
}

}  // namespace

extern "C" lsd_status lsd_measure_fma_peak(int32_t kind, void* stream, double* tflops)
{
    if (!tflops || kind < 0 || kind > 1) return LSD_ERR_INVALID_ARG;
    const double v = kind == 0 ? measure<float>((cudaStream_t)stream, 1 << 15) : measure<double>((cudaStream_t)stream, 1 << 13);
    if (v <= 0.0) return LSD_ERR_CUDA;
    *tflops = v;
    return LSD_OK;
}
