// lsd_transport_window_noalloc (include/lsd.h): the accept / reflect decisions of a drafted window (Eq. 8, PAPER.md:108-111;
// first-reject scan :424) for forces the caller already holds on the device, without a context and WITHOUT ANY ALLOCATION.
//
// Who needs this: code that runs where the process must not call cudaMalloc.  Two cases we know of.  (1) An MD engine or a
// PyTorch program that has handed (nearly) all of the GPU's memory to its own pool: a cudaMalloc from inside this library can
// then fail although the pool has room, and the pool cannot give the memory back in the middle of a step.  (2) A force
// callback inside somebody else's time-step loop: cudaMalloc and cudaFree synchronise the whole device, which stalls every
// other stream of the host program, so such callbacks are usually forbidden to allocate.  The context API (lsd_init) owns
// device buffers and is of no use to these callers; this one entry point is.
//
// The two-stage reduction of the transport map needs a place for the per-block partial sums of S1 and S2.  In the context
// path that is ctx->partial (cudaMalloc in lsd_init).  Here it is the file-scope array g_noalloc_partial below: 64 steps x 148
// blocks x 2 doubles = 151,552 bytes of device memory that every GPU holds from the moment it loads this library until the
// process exits.  That size is what fixes the limits LSD_NOALLOC_MAX_K / LSD_NOALLOC_MAX_ATOMS.
//
// Host code must not hand the NAME of a __device__ array to a kernel: on the host the name is only a stand-in symbol, not a
// device address (a kernel given it faults, or quietly uses the wrong memory where the GPU can reach host memory).  The
// device address comes from cudaGetSymbolAddress, asked once per device with that device current (noalloc_partial_ptr).
//
// The kernels are the arithmetic of k_transport_partial / k_transport_final (integrator.cu) in the same order and with the
// same block decomposition (transport_blocks), so the results equal the context path's; that path is not touched.
#include <cmath>
#include <mutex>

#include "lsd_internal.h"
#include "philox.cuh"

constexpr int kThreads = 256;          // as k_transport_partial
constexpr int kMaxBlocks = 148;        // transport_blocks() never returns more

// The scratch.  Shared by every call on this device and never cleared: each call's first kernel overwrites every slot its
// second kernel reads (slots [j][blk], j < K, blk < nblk), so nothing has to start at zero, and what an earlier call left in
// the other slots is never looked at.  Two calls that run on the GPU at the same time would overwrite each other's sums.
static __device__ __align__(256) double g_noalloc_partial[LSD_NOALLOC_MAX_K * kMaxBlocks * 2];

namespace {

using namespace lsdrng;

thread_local std::string g_noalloc_error;

lsd_status nfail(lsd_status s, const std::string& msg) { g_noalloc_error = msg; return s; }

// Device address of g_noalloc_partial on the CURRENT device; looked up on the first call per device, then cached.
lsd_status noalloc_partial_ptr(double** out)
{
    static std::mutex mu;
    static double* ptr[64] = {};
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return nfail(LSD_ERR_CUDA, "cudaGetDevice failed (no CUDA device?)");
    if (dev < 0 || dev >= 64) return nfail(LSD_ERR_UNSUPPORTED, "device ordinal >= 64");
    std::lock_guard<std::mutex> lock(mu);
    if (!ptr[dev]) {
        double* p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress((void**)&p, g_noalloc_partial);
        if (e != cudaSuccess || !p)
            return nfail(LSD_ERR_CUDA, std::string("cudaGetSymbolAddress(g_noalloc_partial): ") + cudaGetErrorString(e));
        ptr[dev] = p;
    }
    *out = ptr[dev];
    return LSD_OK;
}

// Stage 1, grid (nblk, K): S1 = xi.d and S2 = d.d of step j + 1 summed over this block's atoms, d = (b / sigma)(F~ - F),
// sigma_i = sqrt(m_i kT (1 - c1^2)) (Eq. 7 covariance), xi regenerated from Philox(seed; n0 + j + 1, atom).  Fixed order:
// thread-serial over a strided slice, xor-shuffle tree in the warp, warps summed in index order.
__global__ void __launch_bounds__(kThreads)
k_transport_partial_noalloc(int n, uint64_t seed, uint64_t n0, const double* __restrict__ Ft, const double* __restrict__ Fg,
                            const double* __restrict__ mass_amu, double temperature_K, double one_minus_c1sq, double b,
                            double* __restrict__ partial)
{
    const int j = blockIdx.y;
    const size_t base = (size_t)j * 3 * n;
    double s1 = 0.0, s2 = 0.0;
    for (int i = blockIdx.x * kThreads + threadIdx.x; i < n; i += gridDim.x * kThreads) {
        double xi[3];
        normals3(seed, n0 + (uint64_t)j + 1, (uint32_t)i, 0u, xi);
        const double sigma = sqrt(mass_amu[i] * LSD_AMU_EV * LSD_KB_EV * temperature_K * one_minus_c1sq);   // products only: rounds as lsd_init's host expression
        const double bs = b / sigma;
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            const double d = bs * (Ft[base + (size_t)c * n + i] - Fg[base + (size_t)c * n + i]);
            s1 += xi[c] * d;
            s2 += d * d;
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        s1 += __shfl_xor_sync(0xffffffffu, s1, o);
        s2 += __shfl_xor_sync(0xffffffffu, s2, o);
    }
    __shared__ double sh1[kThreads / 32], sh2[kThreads / 32];
    if ((threadIdx.x & 31) == 0) { sh1[threadIdx.x >> 5] = s1; sh2[threadIdx.x >> 5] = s2; }
    __syncthreads();
    if (threadIdx.x == 0) {
        double a = 0.0, c = 0.0;
        for (int w = 0; w < kThreads / 32; ++w) { a += sh1[w]; c += sh2[w]; }
        partial[((size_t)j * gridDim.x + blockIdx.x) * 2 + 0] = a;
        partial[((size_t)j * gridDim.x + blockIdx.x) * 2 + 1] = c;
    }
}

// Stage 2, one block: blocks summed in index order; ell = -S1 - S2/2; u_j from Philox; reject iff S2 > 0 and ln u > min(0, ell);
// l = min{j : rejected}.  stats [4][K] = S1 | S2 | ell | ln u;  verdict = {l (0: none), n_commit, non-finite sum among the committed}.
__global__ void k_transport_final_noalloc(int K, int nblk, uint64_t seed, uint64_t n0, const double* __restrict__ partial,
                                          double* __restrict__ stats, int32_t* __restrict__ reject, int32_t* __restrict__ verdict)
{
    __shared__ int rej[LSD_NOALLOC_MAX_K], bad[LSD_NOALLOC_MAX_K];
    const int j = threadIdx.x;
    if (j < K) {
        double a = 0.0, c = 0.0;
        for (int blk = 0; blk < nblk; ++blk) { a += partial[((size_t)j * nblk + blk) * 2]; c += partial[((size_t)j * nblk + blk) * 2 + 1]; }
        const double l = -a - 0.5 * c;
        const double lu = log(uniform53(seed, n0 + (uint64_t)j + 1));
        const int r = (c > 0.0 && lu > fmin(0.0, l)) ? 1 : 0;
        stats[j] = a; stats[K + j] = c; stats[2 * K + j] = l; stats[3 * K + j] = lu;
        reject[j] = r;
        rej[j] = r;
        bad[j] = !(isfinite(a) && isfinite(c));
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        int l = 0;
        for (int t = 0; t < K; ++t) if (rej[t]) { l = t + 1; break; }
        const int nc = l ? l : K;
        int nonfinite = 0;
        for (int t = 0; t < nc; ++t) nonfinite |= bad[t];
        verdict[0] = l; verdict[1] = nc; verdict[2] = nonfinite;
    }
}

bool on_device(const void* p)
{
    cudaPointerAttributes at;
    if (cudaPointerGetAttributes(&at, p) != cudaSuccess) { cudaGetLastError(); return false; }
    return at.type == cudaMemoryTypeDevice || at.type == cudaMemoryTypeManaged;
}

}  // namespace

extern "C" const char* lsd_noalloc_last_error(void) { return g_noalloc_error.c_str(); }

extern "C" lsd_status lsd_transport_window_noalloc(int32_t n_atoms, int32_t K, uint64_t seed, uint64_t n0, double temperature_K,
                                                   double friction_per_fs, double dt_fs, const double* mass_amu,
                                                   const double* F_draft, const double* F_target, double* stats, int32_t* reject,
                                                   int32_t* verdict, void* stream)
{
    if (K < 1 || K > LSD_NOALLOC_MAX_K)
        return nfail(LSD_ERR_INVALID_ARG, "lsd_transport_window_noalloc: K = " + std::to_string(K) + " is outside 1.." +
                                              std::to_string(LSD_NOALLOC_MAX_K) + " (LSD_NOALLOC_MAX_K: the static scratch holds that many steps)");
    if (n_atoms < 1 || n_atoms > LSD_NOALLOC_MAX_ATOMS)
        return nfail(LSD_ERR_INVALID_ARG, "lsd_transport_window_noalloc: n_atoms = " + std::to_string(n_atoms) + " is outside 1.." +
                                              std::to_string(LSD_NOALLOC_MAX_ATOMS) + " (LSD_NOALLOC_MAX_ATOMS)");
    if (!(temperature_K > 0.0) || !(friction_per_fs > 0.0) || !(dt_fs > 0.0))
        return nfail(LSD_ERR_INVALID_ARG, "lsd_transport_window_noalloc: temperature, friction and time step must be positive");
    if (!mass_amu || !F_draft || !F_target || !stats || !reject || !verdict)
        return nfail(LSD_ERR_INVALID_ARG, "lsd_transport_window_noalloc: null pointer");
    if (!on_device(mass_amu) || !on_device(F_draft) || !on_device(F_target) || !on_device(stats) || !on_device(reject) || !on_device(verdict))
        return nfail(LSD_ERR_INVALID_ARG, "lsd_transport_window_noalloc: every array must be DEVICE memory of the current device");
    double* partial = nullptr;
    const lsd_status st = noalloc_partial_ptr(&partial);
    if (st != LSD_OK) return st;

    const double c1 = std::exp(-friction_per_fs * dt_fs);            // as lsd_init
    const double b = (1.0 + c1) * dt_fs / 2.0;
    const double one_minus_c1sq = 1.0 - c1 * c1;
    const int nblk = transport_blocks(n_atoms);                      // <= kMaxBlocks; the context path's decomposition
    cudaStream_t s = (cudaStream_t)stream;
    k_transport_partial_noalloc<<<dim3(nblk, K), kThreads, 0, s>>>(n_atoms, seed, n0, F_draft, F_target, mass_amu, temperature_K,
                                                                  one_minus_c1sq, b, partial);
    k_transport_final_noalloc<<<1, LSD_NOALLOC_MAX_K, 0, s>>>(K, nblk, seed, n0, partial, stats, reject, verdict);
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return nfail(LSD_ERR_CUDA, std::string("lsd_transport_window_noalloc: launch failed: ") + cudaGetErrorString(e));
    return LSD_OK;
}
