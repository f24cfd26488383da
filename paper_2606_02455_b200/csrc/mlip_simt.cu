// SchNet-style MLIP (M1-M9): forward pass and hand-derived analytic force backward, fp32 on the FMA pipes.
// No autograd, no float atomics: every per-atom sum runs in the order of the atom's sorted neighbour row, inside
// one warp, so results are bit-reproducible and independent of the batch size (draft == target => F~ == F bitwise).
//
// Structure of every kernel: persistent CTAs, the block's weight matrices resident in shared memory, each warp
// loops over work items and multiplies an 8-row tile by the resident matrix (rows = edges of one atom for the
// filter MLP, rows = atoms for the atom-wise layers).
//
//   forward block t :  y = W_in x ;  m_a = sum_j y_j . w_aj ;  h = W_o1 m ;  x += W_o2 ssp(h)
//   filter          :  w(r) = (W_f2 ssp(W_f1 g(r))) f_c(r)
//   backward block t:  hbar = logistic(h) . (W_o2^T xbar) ;  mbar = W_o1^T hbar ;
//                      ybar_a = sum_j mbar_j . w_aj ;
//                      F_a   += sum_j [ sum_f (mbar_a y_j + mbar_j y_a)_f w'_aj,f ] rhat_aj ;   xbar += W_in^T ybar
#include <cuda_bf16.h>
#include <algorithm>
#include <cstdlib>
#include "lsd_internal.h"

namespace {

constexpr int kMaxWarps = 16;          // warps per CTA: 16 for batches that fill the device, 8 for small ones (run_fp32)
constexpr int kMaxThreads = kMaxWarps * 32;
constexpr float kLn2 = 0.69314718055994530942f;

__device__ __forceinline__ float ssp(float x) { return fmaxf(x, 0.f) + log1pf(expf(-fabsf(x))) - kLn2; }          // M3
__device__ __forceinline__ float logistic(float x) { return 1.f / (1.f + expf(-x)); }

template <int CPT> struct Vec;
template <> struct Vec<4> { using T = float4; };
template <> struct Vec<2> { using T = float2; };
template <> struct Vec<1> { using T = float; };

template <int CPT> __device__ __forceinline__ void ldv(const float* p, float (&v)[CPT])
{
    typename Vec<CPT>::T t = *reinterpret_cast<const typename Vec<CPT>::T*>(p);
    const float* f = reinterpret_cast<const float*>(&t);
#pragma unroll
    for (int c = 0; c < CPT; ++c) v[c] = f[c];
}
template <int CPT> __device__ __forceinline__ void stv(float* p, const float (&v)[CPT])
{
    typename Vec<CPT>::T t;
    float* f = reinterpret_cast<float*>(&t);
#pragma unroll
    for (int c = 0; c < CPT; ++c) f[c] = v[c];
    *reinterpret_cast<typename Vec<CPT>::T*>(p) = t;
}

// bf16 (round to nearest even) copy of a lane's channels
__device__ __forceinline__ uint32_t bf16x2(float lo, float hi) { const __nv_bfloat162 v = __floats2bfloat162_rn(lo, hi); return *reinterpret_cast<const uint32_t*>(&v); }
__device__ __forceinline__ void st16(uint16_t* p, const float (&v)[4]) { *reinterpret_cast<uint2*>(p) = make_uint2(bf16x2(v[0], v[1]), bf16x2(v[2], v[3])); }
__device__ __forceinline__ void st16(uint16_t* p, const float (&v)[2]) { *reinterpret_cast<uint32_t*>(p) = bf16x2(v[0], v[1]); }
__device__ __forceinline__ void st16(uint16_t* p, const float (&v)[1]) { const __nv_bfloat16 h = __float2bfloat16_rn(v[0]); *p = *reinterpret_cast<const uint16_t*>(&h); }

// acc[8][CPT] = A[8][KD] (shared, row-major, leading dimension lda) * W[KD][F] (shared); lane owns channels lane*CPT..
template <int KD, int F>
__device__ __forceinline__ void warp_gemm8(const float* __restrict__ As, int lda, const float* __restrict__ Ws, int lane, float (&acc)[8][F / 32])
{
    constexpr int CPT = F / 32;
#pragma unroll
    for (int r = 0; r < 8; ++r)
#pragma unroll
        for (int c = 0; c < CPT; ++c) acc[r][c] = 0.f;
#pragma unroll 2
    for (int k4 = 0; k4 < KD / 4; ++k4) {
        float4 a[8];
#pragma unroll
        for (int r = 0; r < 8; ++r) a[r] = *reinterpret_cast<const float4*>(As + r * lda + 4 * k4);
#pragma unroll
        for (int kk = 0; kk < 4; ++kk) {
            float w[CPT];
            ldv<CPT>(Ws + (4 * k4 + kk) * F + lane * CPT, w);
#pragma unroll
            for (int r = 0; r < 8; ++r) {
                const float av = kk == 0 ? a[r].x : kk == 1 ? a[r].y : kk == 2 ? a[r].z : a[r].w;
#pragma unroll
                for (int c = 0; c < CPT; ++c) acc[r][c] = fmaf(av, w[c], acc[r][c]);
            }
        }
    }
}

__device__ __forceinline__ void load_weights(float* dst, const float* __restrict__ src, int count)
{
    for (int i = threadIdx.x * 4; i < count; i += blockDim.x * 4) *reinterpret_cast<float4*>(dst + i) = *reinterpret_cast<const float4*>(src + i);
}

// ------------------------------------------------------------------------------------------------ embedding (M4)

// x = Emb[s] and the first block's y = W_in(0) Emb[s] from the per-species table (M4, M5): no contraction needed
__global__ void k_embed_y(int total, int n, int F, const int* __restrict__ species, const float* __restrict__ emb, const float* __restrict__ ytab,
                          float* __restrict__ x, float* __restrict__ y, uint16_t* __restrict__ y16)
{
    const size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= (size_t)total * F) return;
    const int g = (int)(t / F), f = (int)(t % F);
    const int s = species[g % n];
    x[t] = emb[s * F + f];
    const float yv = ytab[s * F + f];
    y[t] = yv;
    if (y16) { const __nv_bfloat16 b = __float2bfloat16_rn(yv); y16[t] = *reinterpret_cast<const uint16_t*>(&b); }
}

// ------------------------------------------------------------------------------------------------ atom-wise layers
enum DenseMode { DENSE_IN = 0, DENSE_OUT = 1, BWD_OUT = 2, BWD_IN = 3 };

// DENSE_IN : out = in * W0                                   (y = W_in x)
// DENSE_OUT: aux = in * W0 ; io += ssp(aux) * W1             (h = W_o1 m ; x += W_o2 ssp(h))
// BWD_OUT  : out = (logistic(aux) . (in * W0)) * W1          (mbar = W_o1^T (logistic(h) . W_o2^T xbar))
// BWD_IN   : io += in * W0                                   (xbar += W_in^T ybar)
template <int F, int MODE>
__global__ void __launch_bounds__(kMaxThreads, 1)
k_dense(int total, const float* __restrict__ in, const float* __restrict__ W0, const float* __restrict__ W1,
        float* __restrict__ aux, float* __restrict__ out, uint16_t* __restrict__ out16,
        const uint16_t* __restrict__ pair16 = nullptr, uint32_t* __restrict__ outpair = nullptr)
{
    constexpr int CPT = F / 32, LDA = F + 4;
    constexpr bool TWO = (MODE == DENSE_OUT || MODE == BWD_OUT);
    extern __shared__ __align__(16) float smem[];
    float* Ws0 = smem;
    float* Ws1 = Ws0 + F * F;
    float* Asw = Ws0 + (TWO ? 2 : 1) * F * F + (threadIdx.x >> 5) * 8 * LDA;
    load_weights(Ws0, W0, F * F);
    if (TWO) load_weights(Ws1, W1, F * F);
    __syncthreads();
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int ntiles = (total + 7) / 8;
    for (int tile = blockIdx.x * (blockDim.x >> 5) + warp; tile < ntiles; tile += gridDim.x * (blockDim.x >> 5)) {
        const int g0 = tile * 8;
#pragma unroll
        for (int r = 0; r < 8; ++r) {
            float v[CPT];
#pragma unroll
            for (int c = 0; c < CPT; ++c) v[c] = 0.f;
            if (g0 + r < total) ldv<CPT>(in + (size_t)(g0 + r) * F + lane * CPT, v);
            stv<CPT>(Asw + r * LDA + lane * CPT, v);
        }
        __syncwarp();
        float acc[8][CPT];
        warp_gemm8<F, F>(Asw, LDA, Ws0, lane, acc);
        if (MODE == DENSE_IN) {
#pragma unroll
            for (int r = 0; r < 8; ++r) if (g0 + r < total) {
                stv<CPT>(out + (size_t)(g0 + r) * F + lane * CPT, acc[r]);
                if (out16) st16(out16 + (size_t)(g0 + r) * F + lane * CPT, acc[r]);
            }
        } else if (MODE == BWD_IN) {
#pragma unroll
            for (int r = 0; r < 8; ++r) if (g0 + r < total) {
                float v[CPT];
                ldv<CPT>(out + (size_t)(g0 + r) * F + lane * CPT, v);
#pragma unroll
                for (int c = 0; c < CPT; ++c) v[c] += acc[r][c];
                stv<CPT>(out + (size_t)(g0 + r) * F + lane * CPT, v);
            }
        } else {
            __syncwarp();
#pragma unroll
            for (int r = 0; r < 8; ++r) {
                float v[CPT];
                if (MODE == DENSE_OUT) {
                    if (g0 + r < total) stv<CPT>(aux + (size_t)(g0 + r) * F + lane * CPT, acc[r]);      // keep h for the backward
#pragma unroll
                    for (int c = 0; c < CPT; ++c) v[c] = ssp(acc[r][c]);
                } else {
                    float hv[CPT];
#pragma unroll
                    for (int c = 0; c < CPT; ++c) hv[c] = 0.f;
                    if (g0 + r < total) ldv<CPT>(aux + (size_t)(g0 + r) * F + lane * CPT, hv);
#pragma unroll
                    for (int c = 0; c < CPT; ++c) v[c] = logistic(hv[c]) * acc[r][c];
                }
                stv<CPT>(Asw + r * LDA + lane * CPT, v);
            }
            __syncwarp();
            float acc2[8][CPT];
            warp_gemm8<F, F>(Asw, LDA, Ws1, lane, acc2);
#pragma unroll
            for (int r = 0; r < 8; ++r) if (g0 + r < total) {
                if (MODE == DENSE_OUT) {
                    float v[CPT];
                    ldv<CPT>(out + (size_t)(g0 + r) * F + lane * CPT, v);
#pragma unroll
                    for (int c = 0; c < CPT; ++c) v[c] += acc2[r][c];
                    stv<CPT>(out + (size_t)(g0 + r) * F + lane * CPT, v);
                } else {
                    stv<CPT>(out + (size_t)(g0 + r) * F + lane * CPT, acc2[r]);
                    if (out16) st16(out16 + (size_t)(g0 + r) * F + lane * CPT, acc2[r]);
                    if (outpair) {
                        // rows gathered by the edges-as-rows backward kernel (mlip_edge_rows.cu), pair layout: per channel pair
                        // (f, f+1) the words (y_f | y_f+1 << 16), (mbar_f | mbar_f+1 << 16)
                        const size_t o = (size_t)(g0 + r) * F + lane * CPT;
                        if constexpr (CPT >= 2) {
#pragma unroll
                            for (int c = 0; c < CPT; c += 2)
                                *reinterpret_cast<uint2*>(outpair + o + c) = make_uint2(*reinterpret_cast<const uint32_t*>(pair16 + o + c), bf16x2(acc2[r][c], acc2[r][c + 1]));
                        } else {
                            const float nxt = __shfl_down_sync(0xffffffffu, acc2[r][0], 1);
                            if ((lane & 1) == 0) *reinterpret_cast<uint2*>(outpair + o) = make_uint2(*reinterpret_cast<const uint32_t*>(pair16 + o), bf16x2(acc2[r][0], nxt));
                        }
                    }
                }
            }
        }
        __syncwarp();
    }
}

// ------------------------------------------------------------------------------------------------ readout (M6) + xbar seed
// z = W_r1 x ; e = alpha w_r2 . ssp(z) ; xbar = alpha W_r1^T (logistic(z) . w_r2).  One warp per atom.
template <int F>
__global__ void __launch_bounds__(kMaxThreads)
k_readout(int total, float alpha, const float* __restrict__ x, const float* __restrict__ Wr1, const float* __restrict__ wr2,
          float* __restrict__ xbar, double* __restrict__ e_atom)
{
    constexpr int H = F / 2, LD = F + 1;
    extern __shared__ __align__(16) float smem[];
    float* Ws = smem;                       // [H][F+1]
    float* w2 = Ws + H * LD;                // [H]
    float* xs = w2 + H + (threadIdx.x >> 5) * (F + H);   // per warp: x[F], s[H]
    for (int i = threadIdx.x; i < H * F; i += blockDim.x) Ws[(i / F) * LD + (i % F)] = Wr1[i];
    for (int i = threadIdx.x; i < H; i += blockDim.x) w2[i] = wr2[i];
    __syncthreads();
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    float* ss = xs + F;
    for (int g = blockIdx.x * (blockDim.x >> 5) + warp; g < total; g += gridDim.x * (blockDim.x >> 5)) {
        for (int f = lane; f < F; f += 32) xs[f] = x[(size_t)g * F + f];
        __syncwarp();
        float e = 0.f;
        for (int k = lane; k < H; k += 32) {
            float z = 0.f;
            for (int f = 0; f < F; ++f) z = fmaf(Ws[k * LD + f], xs[f], z);
            e += w2[k] * ssp(z);
            ss[k] = logistic(z) * w2[k];
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) e += __shfl_xor_sync(0xffffffffu, e, o);
        __syncwarp();
        for (int f = lane; f < F; f += 32) {
            float v = 0.f;
            for (int k = 0; k < H; ++k) v = fmaf(Ws[k * LD + f], ss[k], v);
            xbar[(size_t)g * F + f] = alpha * v;
        }
        if (lane == 0 && e_atom) e_atom[g] = (double)(alpha * e);
        __syncwarp();
    }
}

// ------------------------------------------------------------------------------------------------ one-block networks (the drafts)
// With T = 1 everything between the two edge kernels is local to an atom: h = W_o1 m; x = Emb + W_o2 ssp(h); readout
// z = W_r1 x, e = alpha w_r2 . ssp(z); xbar = alpha W_r1^T (logistic(z) . w_r2); hbar = logistic(h) . W_o2^T xbar; mbar = W_o1^T hbar
// (M5, M6, M9).  One warp per atom, lane = channel (F = 32), the six small matrices resident in shared memory: one launch
// instead of k_dense<DENSE_OUT>, k_readout and k_dense<BWD_OUT>, and nothing but mbar leaves the kernel.
// out[lane] = sum_k in[k] W[k][lane], in[k] held by lane k; four interleaved chains, summed in a fixed order
__device__ __forceinline__ float warp_matvec32(float in, const float* __restrict__ W, int lane, int K = 32)
{
    float acc[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll 8
    for (int k = 0; k < K; k += 4) {
#pragma unroll
        for (int u = 0; u < 4; ++u) acc[u] = fmaf(__shfl_sync(0xffffffffu, in, k + u), W[(k + u) * 32 + lane], acc[u]);
    }
    return (acc[0] + acc[1]) + (acc[2] + acc[3]);
}

__global__ void __launch_bounds__(512)
k_atom_chain1(int total, int n, const int* __restrict__ species, float alpha, const float* __restrict__ m, const float* __restrict__ emb,
              const float* __restrict__ Wo1T, const float* __restrict__ Wo2T, const float* __restrict__ Wo2, const float* __restrict__ Wo1,
              const float* __restrict__ Wr1, const float* __restrict__ wr2, float* __restrict__ mbar, uint16_t* __restrict__ mbar16,
              const uint16_t* __restrict__ y16, uint32_t* __restrict__ ympair, double* __restrict__ e_atom)
{
    constexpr int F = 32, H = F / 2;
    __shared__ __align__(16) float W[4 * F * F + H * F + H];
    float* const sWo1T = W; float* const sWo2T = W + F * F; float* const sWo2 = W + 2 * F * F; float* const sWo1 = W + 3 * F * F;
    float* const sWr1 = W + 4 * F * F; float* const sw2 = sWr1 + H * F;
    for (int i = threadIdx.x; i < F * F; i += blockDim.x) { sWo1T[i] = Wo1T[i]; sWo2T[i] = Wo2T[i]; sWo2[i] = Wo2[i]; sWo1[i] = Wo1[i]; }
    for (int i = threadIdx.x; i < H * F; i += blockDim.x) sWr1[i] = Wr1[i];
    if (threadIdx.x < H) sw2[threadIdx.x] = wr2[threadIdx.x];
    __syncthreads();
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, nw = blockDim.x >> 5;
    for (int g = blockIdx.x * nw + warp; g < total; g += gridDim.x * nw) {
        const float h = warp_matvec32(m[(size_t)g * F + lane], sWo1T, lane);
        const float x = emb[species[g % n] * F + lane] + warp_matvec32(ssp(h), sWo2T, lane);
        float z0 = 0.f, z1 = 0.f;
#pragma unroll 8
        for (int f = 0; f < F; f += 2) {
            const float x0 = __shfl_sync(0xffffffffu, x, f), x1 = __shfl_sync(0xffffffffu, x, f + 1);
            if (lane < H) { z0 = fmaf(sWr1[lane * F + f], x0, z0); z1 = fmaf(sWr1[lane * F + f + 1], x1, z1); }
        }
        const float z = z0 + z1;
        float e = lane < H ? sw2[lane] * ssp(z) : 0.f;
        const float s = lane < H ? logistic(z) * sw2[lane] : 0.f;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) e += __shfl_xor_sync(0xffffffffu, e, o);
        const float xb = alpha * warp_matvec32(s, sWr1, lane, H);
        const float hb = logistic(h) * warp_matvec32(xb, sWo2, lane);
        const float mb = warp_matvec32(hb, sWo1, lane);
        const size_t o = (size_t)g * F + lane;
        if (mbar) mbar[o] = mb;
        if (mbar16) { const __nv_bfloat16 b = __float2bfloat16_rn(mb); mbar16[o] = *reinterpret_cast<const uint16_t*>(&b); }
        if (ympair) {                                  // pair rows of the edges-as-rows backward kernel (see k_dense)
            const float nxt = __shfl_down_sync(0xffffffffu, mb, 1);
            if ((lane & 1) == 0) *reinterpret_cast<uint2*>(ympair + o) = make_uint2(*reinterpret_cast<const uint32_t*>(y16 + o), bf16x2(mb, nxt));
        }
        if (lane == 0 && e_atom) e_atom[g] = (double)(alpha * e);
    }
}

// ------------------------------------------------------------------------------------------------ continuous-filter convolution

template <int F, bool BWD>
__global__ void __launch_bounds__(kMaxThreads, 1)
k_edge(EdgeArgs a)
{
    constexpr int CPT = F / 32, LDA = F + 4, LDG = LSD_NRBF + 4, SPW = BWD ? 4 : 8;
    extern __shared__ __align__(16) float smem[];
    float* Wf1 = smem;                                   // [32][F]
    float* Wf2 = Wf1 + LSD_NRBF * F;                     // [F][F]
    float* Gs = Wf2 + F * F + (threadIdx.x >> 5) * (8 * LDG + 8 * LDA);
    float* As = Gs + 8 * LDG;
    load_weights(Wf1, a.Wf1, LSD_NRBF * F);
    load_weights(Wf2, a.Wf2, F * F);
    __syncthreads();
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int n = a.n;
    for (int g = blockIdx.x * (blockDim.x >> 5) + warp; g < a.total; g += gridDim.x * (blockDim.x >> 5)) {
        const int b = g / n, i = g % n;
        const int cnt = a.count[g];
        float part[CPT], ya[CPT], mba[CPT];
#pragma unroll
        for (int c = 0; c < CPT; ++c) part[c] = 0.f;
        if (BWD) { ldv<CPT>(a.y + (size_t)g * F + lane * CPT, ya); ldv<CPT>(a.mbar + (size_t)g * F + lane * CPT, mba); }
        double fx = 0.0, fy = 0.0, fz = 0.0;
        for (int u0 = 0; u0 < cnt; u0 += SPW) {
            // --- geometry of the unit's slots (lanes 0..SPW-1): edge records written by k_compact (fp64 -> fp32 once)
            const int slot = u0 + lane;
            const bool valid = lane < SPW && slot < cnt;
            float r = 0.f, fc = 0.f, fcp = 0.f, ux = 0.f, uy = 0.f, uz = 0.f;
            int jrow = g;
            if (valid) {
                const float* e = a.recs + lsd_rec_index((size_t)g, a.cap, slot, 0);
                r = e[LSD_REC_R * 16]; fc = e[LSD_REC_FC * 16]; jrow = __float_as_int(e[LSD_REC_JROW * 16]);
                if (BWD) { fcp = e[LSD_REC_FCP * 16]; ux = e[LSD_REC_UX * 16]; uy = e[LSD_REC_UY * 16]; uz = e[LSD_REC_UZ * 16]; }
            }
            // --- radial basis rows (M1): lane k holds basis k; BWD interleaves value / r-derivative rows
#pragma unroll
            for (int e = 0; e < SPW; ++e) {
                const float re = __shfl_sync(0xffffffffu, r, e);
                const bool ve = (u0 + e) < cnt;
                const float x = re - (float)lane * a.delta;
                const float gk = ve ? expf(-0.5f * x * x * a.inv_delta2) : 0.f;
                if (BWD) { Gs[(2 * e) * LDG + lane] = gk; Gs[(2 * e + 1) * LDG + lane] = -gk * x * a.inv_delta2; }
                else Gs[e * LDG + lane] = gk;
            }
            __syncwarp();
            float acc[8][CPT];
            warp_gemm8<LSD_NRBF, F>(Gs, LDG, Wf1, lane, acc);
            // --- activation (M3) -> A operand of the second layer
            if (BWD) {
#pragma unroll
                for (int e = 0; e < 4; ++e) {
                    float v0[CPT], v1[CPT];
#pragma unroll
                    for (int c = 0; c < CPT; ++c) { v0[c] = ssp(acc[2 * e][c]); v1[c] = logistic(acc[2 * e][c]) * acc[2 * e + 1][c]; }
                    stv<CPT>(As + (2 * e) * LDA + lane * CPT, v0);
                    stv<CPT>(As + (2 * e + 1) * LDA + lane * CPT, v1);
                }
            } else {
#pragma unroll
                for (int e = 0; e < 8; ++e) {
                    float v0[CPT];
#pragma unroll
                    for (int c = 0; c < CPT; ++c) v0[c] = ssp(acc[e][c]);
                    stv<CPT>(As + e * LDA + lane * CPT, v0);
                }
            }
            __syncwarp();
            warp_gemm8<F, F>(As, LDA, Wf2, lane, acc);
            // --- epilogue: cfconv gather (and its adjoints)
#pragma unroll
            for (int e = 0; e < SPW; ++e) {
                const int jr = __shfl_sync(0xffffffffu, jrow, e);
                const float fce = __shfl_sync(0xffffffffu, fc, e);
                float yj[CPT];
                if (!BWD) {
                    ldv<CPT>(a.y + (size_t)jr * F + lane * CPT, yj);
#pragma unroll
                    for (int c = 0; c < CPT; ++c) part[c] = fmaf(yj[c], acc[e][c] * fce, part[c]);
                } else {
                    const float fcpe = __shfl_sync(0xffffffffu, fcp, e);
                    const float uxe = __shfl_sync(0xffffffffu, ux, e), uye = __shfl_sync(0xffffffffu, uy, e), uze = __shfl_sync(0xffffffffu, uz, e);
                    float mbj[CPT];
                    ldv<CPT>(a.y + (size_t)jr * F + lane * CPT, yj);
                    ldv<CPT>(a.mbar + (size_t)jr * F + lane * CPT, mbj);
                    float gp = 0.f;
#pragma unroll
                    for (int c = 0; c < CPT; ++c) {
                        const float w = acc[2 * e][c] * fce;
                        const float wp = acc[2 * e + 1][c] * fce + acc[2 * e][c] * fcpe;
                        part[c] = fmaf(mbj[c], w, part[c]);
                        gp = fmaf(fmaf(mba[c], yj[c], mbj[c] * ya[c]), wp, gp);
                    }
#pragma unroll
                    for (int o = 16; o > 0; o >>= 1) gp += __shfl_xor_sync(0xffffffffu, gp, o);
                    fx += (double)(gp * uxe); fy += (double)(gp * uye); fz += (double)(gp * uze);
                }
            }
            __syncwarp();
        }
        if (!BWD) stv<CPT>(a.m_out + (size_t)g * F + lane * CPT, part);
        else {
            if (a.ybar) stv<CPT>(a.ybar + (size_t)g * F + lane * CPT, part);
            if (lane == 0) {
                double* Fb = a.Fout + (size_t)b * 3 * n;
                Fb[i] += fx; Fb[n + i] += fy; Fb[2 * n + i] += fz;
            }
        }
    }
}

template <int F> size_t smem_dense(bool two, int kWarps) { return sizeof(float) * ((two ? 2 : 1) * F * F + kWarps * 8 * (F + 4)); }
template <int F> size_t smem_edge(int kWarps) { return sizeof(float) * (LSD_NRBF * F + F * F + kWarps * (8 * (LSD_NRBF + 4) + 8 * (F + 4))); }
template <int F> size_t smem_readout(int kWarps) { return sizeof(float) * ((F / 2) * (F + 1) + F / 2 + kWarps * (F + F / 2)); }

int g_num_sms = 0;
int num_sms() { if (!g_num_sms) { int dev = 0; cudaGetDevice(&dev); cudaDeviceGetAttribute(&g_num_sms, cudaDevAttrMultiProcessorCount, dev); if (g_num_sms <= 0) g_num_sms = 148; } return g_num_sms; }

template <typename K> void set_smem(K kernel, size_t bytes) { cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes); }

template <int F>
void run_fp32(Launcher L, const SysDev& sys, const MlipDev& net, MlipWork& w, int B, const double* q, const int* img,
              const CompactList& cl, double* Fout, double* e_atom, bool use_tc)
{
    const int total = B * sys.n;
    static bool configured_dev[64] = {};
    bool& configured = configured_dev[lsd_current_device()];
    if (!configured) {
        set_smem(k_dense<F, DENSE_IN>, smem_dense<F>(false, kMaxWarps)); set_smem(k_dense<F, BWD_IN>, smem_dense<F>(false, kMaxWarps));
        set_smem(k_dense<F, DENSE_OUT>, smem_dense<F>(true, kMaxWarps)); set_smem(k_dense<F, BWD_OUT>, smem_dense<F>(true, kMaxWarps));
        set_smem(k_edge<F, false>, smem_edge<F>(kMaxWarps)); set_smem(k_edge<F, true>, smem_edge<F>(kMaxWarps));
        set_smem(k_readout<F>, smem_readout<F>(kMaxWarps));
        configured = true;
    }
    const int sms = num_sms();
    // widths 32 / 64 on the tcgen05 path: the edges-as-rows kernels of mlip_edge_rows_narrow.cu (width 128 has its own driver,
    // mlip_forward_backward_tc128)
    static_assert(F == 32 || F == 64 || F == 128, "network widths");
    if (use_tc && F == 128) return;                    // never reached: mlip_forward_backward_bf16tc routes width 128 elsewhere
    // 16 warps per CTA once every SM has at least 16 atoms to work on (occupancy: +8 % at cfg4 fp32); 8 for small batches,
    // whose kernels are latency-bound (a bigger CTA only adds to the weight-load and barrier time).  Same arithmetic either way.
    const int kWarps = total >= sms * kMaxWarps ? kMaxWarps : 8;
    const int kThreads = kWarps * 32;
    const int grid_tiles = std::max(1, std::min(sms, (total + kWarps * 8 - 1) / (kWarps * 8)));
    const int grid_atoms = std::max(1, std::min(sms, (total + kWarps - 1) / kWarps));
    // one-block width-32 network of a small system: k_atom_chain1 between the two edge kernels (three launches less per evaluation;
    // cfg4: draft network 2.32 -> 1.76 ms per window).  Large systems keep the tiled kernels, which are faster there (cfg5: 6.1 vs
    // 6.5 ms).  The choice depends on the atoms of ONE state, never on the batch: the same network gives the same bits alone and batched.
    const bool chain1 = F == 32 && net.T == 1 && sys.n <= 16384;
    // y of the first block depends on the species only (M4, M5): for a one-block network nothing else is read from the embedding
    // kernel's outputs, so its rows are written once per context (and again when a larger batch needs more of them)
    if (!chain1 || w.y0_rows < total) {
        k_embed_y<<<(int)(((size_t)total * F + 255) / 256), 256, 0, L.s>>>(total, sys.n, F, sys.species, net.emb, net.ytab0, w.x, w.y[0], use_tc ? w.y16[0] : nullptr); LSD_COUNT(L);
        if (chain1) w.y0_rows = total;
    }
    EdgeArgs ea{};
    ea.total = total; ea.n = sys.n; ea.cap = cl.cap; ea.count = cl.count; ea.keys = cl.keys; ea.recs = cl.recs; ea.rec_zero = cl.rec_zero;
    ea.rc = net.rc; ea.inv_rc = 1.f / net.rc; ea.delta = net.rc / (float)(net.R - 1); ea.inv_delta2 = 1.f / (ea.delta * ea.delta);
    for (int t = 0; t < net.T; ++t) {
        int pid = -1;
        if (t > 0) {
            pid = prof_begin(L, PROF_DENSE);
            k_dense<F, DENSE_IN><<<grid_tiles, kThreads, smem_dense<F>(false, kWarps), L.s>>>(total, w.x, net.WinT[t], nullptr, nullptr, w.y[t], use_tc ? w.y16[t] : nullptr); LSD_COUNT(L);
            prof_end(L, pid);
        }
        ea.Wf1 = net.Wf1T[t]; ea.Wf2 = net.Wf2T[t]; ea.y = w.y[t]; ea.m_out = w.m; ea.mbar = nullptr; ea.ybar = nullptr; ea.Fout = nullptr;
        pid = prof_begin(L, PROF_EDGE_FWD);
        if (use_tc) {
            ea.Wf1_tc = net.Wf1_bf16[t]; ea.Wf2_tc = net.Wf2_bf16[t]; ea.y16 = w.y16[t];
            launch_edge_rows_narrow(L, ea, F, false);
        }
        else { k_edge<F, false><<<grid_atoms, kThreads, smem_edge<F>(kWarps), L.s>>>(ea); LSD_COUNT(L); }
        prof_end(L, pid);
        if (chain1) continue;
        pid = prof_begin(L, PROF_DENSE);
        k_dense<F, DENSE_OUT><<<grid_tiles, kThreads, smem_dense<F>(true, kWarps), L.s>>>(total, w.m, net.Wo1T[t], net.Wo2T[t], w.h[t], w.x, nullptr); LSD_COUNT(L);
        prof_end(L, pid);
    }
    const bool pairs = use_tc;                                  // (y, mbar) pair rows for k_edge_rows
    if (chain1) {
        const int pidc = prof_begin(L, PROF_DENSE);
        const int cw = 16, grid_c = std::max(1, std::min(sms * 2, (total + cw - 1) / cw));
        k_atom_chain1<<<grid_c, cw * 32, 0, L.s>>>(total, sys.n, sys.species, net.alpha, w.m, net.emb, net.Wo1T[0], net.Wo2T[0], net.Wo2[0], net.Wo1[0], net.Wr1, net.wr2,
                                                   w.mbar, use_tc && !pairs ? w.mbar16 : nullptr, pairs ? w.y16[0] : nullptr, pairs ? w.ym16 : nullptr, e_atom); LSD_COUNT(L);
        prof_end(L, pidc);
    } else {
        int pidr = prof_begin(L, PROF_DENSE);
        k_readout<F><<<grid_atoms, kThreads, smem_readout<F>(kWarps), L.s>>>(total, net.alpha, w.x, net.Wr1, net.wr2, w.xbar, e_atom); LSD_COUNT(L);
        prof_end(L, pidr);
    }
    for (int t = net.T - 1; t >= 0; --t) {
        int pid = -1;
        if (!chain1) {
        pid = prof_begin(L, PROF_DENSE);
        k_dense<F, BWD_OUT><<<grid_tiles, kThreads, smem_dense<F>(true, kWarps), L.s>>>(total, w.xbar, net.Wo2[t], net.Wo1[t], w.h[t], w.mbar, use_tc && !pairs ? w.mbar16 : nullptr,
                                                                                 pairs ? w.y16[t] : nullptr, pairs ? w.ym16 : nullptr); LSD_COUNT(L);
        prof_end(L, pid);
        }
        ea.Wf1 = net.Wf1T[t]; ea.Wf2 = net.Wf2T[t]; ea.y = w.y[t]; ea.m_out = nullptr; ea.mbar = w.mbar; ea.ybar = t > 0 ? w.ybar : nullptr; ea.Fout = Fout;
        pid = prof_begin(L, PROF_EDGE_BWD);
        if (use_tc) {
            ea.Wf1_tc = net.Wf1_bf16[t]; ea.Wf2_tc = net.Wf2_bf16[t]; ea.y16 = w.y16[t]; ea.mbar16 = w.mbar16; ea.ym16 = w.ym16;
            launch_edge_rows_narrow(L, ea, F, true);
        }
        else { k_edge<F, true><<<grid_atoms, kThreads, smem_edge<F>(kWarps), L.s>>>(ea); LSD_COUNT(L); }
        prof_end(L, pid);
        if (t > 0) { pid = prof_begin(L, PROF_DENSE); k_dense<F, BWD_IN><<<grid_tiles, kThreads, smem_dense<F>(false, kWarps), L.s>>>(total, w.ybar, net.Win[t], nullptr, nullptr, w.xbar, nullptr); LSD_COUNT(L); prof_end(L, pid); }
    }
}

}  // namespace

size_t mlip_work_bytes(const MlipDev& net, int n, int bmax)
{
    return sizeof(float) * (size_t)n * bmax * net.F * (5 + 2 * net.T) + sizeof(double) * (size_t)n * bmax;
}

void mlip_forward_backward_fp32(Launcher L, const SysDev& sys, const MlipDev& net, MlipWork& w, int B, const double* q,
                                const int* img, const CompactList& cl, double* F, double* e_atom)
{
    switch (net.F) {
        case 32:  run_fp32<32>(L, sys, net, w, B, q, img, cl, F, e_atom, false); break;
        case 64:  run_fp32<64>(L, sys, net, w, B, q, img, cl, F, e_atom, false); break;
        case 128: run_fp32<128>(L, sys, net, w, B, q, img, cl, F, e_atom, false); break;
        default: break;
    }
}

// bf16 tcgen05 variant: same sequence, the two edge kernels replaced by k_edge_tc (mlip_tc.cu); atom-wise layers stay fp32.
void mlip_forward_backward_bf16tc(Launcher L, const SysDev& sys, const MlipDev& net, MlipWork& w, int B, const double* q,
                                  const int* img, const CompactList& cl, double* F, double* e_atom)
{
    switch (net.F) {
        case 32:  run_fp32<32>(L, sys, net, w, B, q, img, cl, F, e_atom, true); break;
        case 64:  run_fp32<64>(L, sys, net, w, B, q, img, cl, F, e_atom, true); break;
        case 128: mlip_forward_backward_tc128(L, sys, net, w, B, q, img, cl, F, e_atom); break;
        default: break;
    }
}
