// Measured arithmetic peaks of the device this process runs on: plain FMA throughput in fp32 and fp64 (the roofline
// denominators of the fp32 MLIP path and of the fp64 cfg1 path; MEASURED_PEAKS.json only carries HBM and bf16 tensor figures).
// A grid of resident warps runs 16 independent FMA chains per thread; timed with CUDA events on the caller's stream.
// Also two design measurements that DESIGN.md cites: the tensor-memory load / store bandwidth of an SM, and the cost of the
// second delivery of a half-list schedule (one bf16 feature row per undirected pair scattered to the partner's slot, then
// summed per atom in slot order).
#include <algorithm>
#include <cuda_bf16.h>
#include "lsd_internal.h"
#include "tc_ptx.cuh"

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

// ---- tensor memory: `warps` warps of one CTA per SM move 2 KB (32 lanes x 16 columns) per tcgen05.ld / tcgen05.st
template <int STORE>
__global__ void __launch_bounds__(512, 1) k_tmem_bw(int iters, long long* cycles, uint32_t* sink)
{
    __shared__ uint32_t tb_s;
    const int warp = threadIdx.x >> 5;
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(tcp::smem_u32(&tb_s)), "n"(512));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
    }
    tcp::tc_fence_before();
    __syncthreads();
    tcp::tc_fence_after();
    const uint32_t tl = tb_s + ((uint32_t)((warp & 3) * 32) << 16) + (uint32_t)((warp >> 2) * 64);
    uint32_t v[16], acc = 0;
#pragma unroll
    for (int i = 0; i < 16; ++i) v[i] = threadIdx.x + i;
    __syncthreads();
    const long long t0 = clock64();
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            if (STORE) tcp::tmem_st16(tl + u * 16, v);
            else { tcp::tmem_ld16(tl + u * 16, v); tcp::tmem_wait_ld(); acc += v[0] ^ v[7] ^ v[15]; }
        }
        if (STORE) tcp::tmem_wait_st();
    }
    const long long t1 = clock64();
    if (threadIdx.x == 0) cycles[blockIdx.x] = t1 - t0;
    if (acc == 0x12345678u) sink[0] = acc;
    tcp::tc_fence_before();
    __syncthreads();
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tb_s), "n"(512));
}

// ---- half-list delivery: rows of 128 bf16 channels (256 B), `per_atom` incoming rows per atom
__global__ void k_partner(int n, int atoms, int per_atom, int* __restrict__ partner)
{
    const long t = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= (long)atoms * per_atom) return;
    const int a = (int)(t / per_atom), k = (int)(t % per_atom);
    const int st = a / n, i = a % n;
    const int off = (k + 1) * 37 + ((k * 7919) % 1024);             // partners a few hundred rows away: neighbouring cells of a cell-sorted crystal
    partner[t] = (st * n + (i + off) % n) * per_atom + k;           // the reverse edge's slot
}
__global__ void k_pair_scatter(const int* __restrict__ partner, uint2* __restrict__ scratch, long pairs)
{
    const long w = ((long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (w >= pairs) return;
    scratch[(size_t)partner[w] * 32 + lane] = make_uint2((uint32_t)w * 2654435761u + lane, lane);     // stands in for bf16(lin . mbar_i)
}
__global__ void k_pair_gather(const uint2* __restrict__ scratch, uint2* __restrict__ out, int atoms, int per_atom)
{
    const int a = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    if (a >= atoms) return;
    float acc[4] = {0.f, 0.f, 0.f, 0.f};
    for (int s = 0; s < per_atom; ++s) {                           // fixed slot order: deterministic, batch-invariant
        const uint2 v = scratch[((size_t)a * per_atom + s) * 32 + lane];
        const __nv_bfloat162 p0 = *reinterpret_cast<const __nv_bfloat162*>(&v.x), p1 = *reinterpret_cast<const __nv_bfloat162*>(&v.y);
        acc[0] += __low2float(p0); acc[1] += __high2float(p0); acc[2] += __low2float(p1); acc[3] += __high2float(p1);
    }
    const __nv_bfloat162 r0 = __floats2bfloat162_rn(acc[0], acc[1]), r1 = __floats2bfloat162_rn(acc[2], acc[3]);
    out[(size_t)a * 32 + lane] = make_uint2(*reinterpret_cast<const uint32_t*>(&r0), *reinterpret_cast<const uint32_t*>(&r1));
}

}  // namespace

extern "C" lsd_status lsd_measure_tmem_bandwidth(int32_t warps, int32_t store, void* stream, double* bytes_per_clk)
{
    if (!bytes_per_clk || (warps != 1 && warps != 4 && warps != 8 && warps != 16)) return LSD_ERR_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    const int blocks = lsd_sm_count(), iters = 2000;
    long long* cyc = nullptr; uint32_t* sink = nullptr;
    if (cudaMalloc(&cyc, sizeof(long long) * blocks) != cudaSuccess || cudaMalloc(&sink, 4) != cudaSuccess) return LSD_ERR_OOM;
    for (int rep = 0; rep < 2; ++rep) {
        if (store) k_tmem_bw<1><<<blocks, warps * 32, 0, st>>>(iters, cyc, sink);
        else k_tmem_bw<0><<<blocks, warps * 32, 0, st>>>(iters, cyc, sink);
    }
    long long h = 0;
    cudaStreamSynchronize(st);
    cudaMemcpy(&h, cyc, sizeof h, cudaMemcpyDeviceToHost);
    cudaFree(cyc); cudaFree(sink);
    if (cudaGetLastError() != cudaSuccess || h <= 0) return LSD_ERR_CUDA;
    *bytes_per_clk = (double)iters * warps * 4 * 2048.0 / (double)h;
    return LSD_OK;
}

extern "C" lsd_status lsd_measure_half_list_delivery(int32_t n_atoms, int32_t n_states, int32_t rows_per_atom, void* stream,
                                                      double* scatter_ms, double* gather_ms)
{
    if (!scatter_ms || !gather_ms || n_atoms < 1 || n_states < 1 || rows_per_atom < 1) return LSD_ERR_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    const int atoms = n_atoms * n_states;
    const long pairs = (long)atoms * rows_per_atom;
    int* partner = nullptr; uint2 *scratch = nullptr, *out = nullptr;
    if (cudaMalloc(&partner, pairs * 4) != cudaSuccess || cudaMalloc(&scratch, (size_t)pairs * 256) != cudaSuccess ||
        cudaMalloc(&out, (size_t)atoms * 256) != cudaSuccess) { cudaFree(partner); cudaFree(scratch); cudaFree(out); cudaGetLastError(); return LSD_ERR_OOM; }
    k_partner<<<(int)((pairs + 255) / 256), 256, 0, st>>>(n_atoms, atoms, rows_per_atom, partner);
    cudaEvent_t e0, e1, e2;
    cudaEventCreate(&e0); cudaEventCreate(&e1); cudaEventCreate(&e2);
    float best_s = 1e30f, best_g = 1e30f;
    for (int rep = 0; rep < 3; ++rep) {
        cudaEventRecord(e0, st);
        k_pair_scatter<<<(int)((pairs * 32 + 255) / 256), 256, 0, st>>>(partner, scratch, pairs);
        cudaEventRecord(e1, st);
        k_pair_gather<<<(int)(((long)atoms * 32 + 255) / 256), 256, 0, st>>>(scratch, out, atoms, rows_per_atom);
        cudaEventRecord(e2, st);
        cudaEventSynchronize(e2);
        float a = 0.f, b = 0.f;
        cudaEventElapsedTime(&a, e0, e1); cudaEventElapsedTime(&b, e1, e2);
        if (rep > 0) { best_s = std::min(best_s, a); best_g = std::min(best_g, b); }
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1); cudaEventDestroy(e2);
    cudaFree(partner); cudaFree(scratch); cudaFree(out);
    if (cudaGetLastError() != cudaSuccess) return LSD_ERR_CUDA;
    *scatter_ms = best_s; *gather_ms = best_g;
    return LSD_OK;
}

extern "C" lsd_status lsd_measure_fma_peak(int32_t kind, void* stream, double* tflops)
{
    if (!tflops || kind < 0 || kind > 1) return LSD_ERR_INVALID_ARG;
    const double v = kind == 0 ? measure<float>((cudaStream_t)stream, 1 << 15) : measure<double>((cudaStream_t)stream, 1 << 13);
    if (v <= 0.0) return LSD_ERR_CUDA;
    *tflops = v;
    return LSD_OK;
}
