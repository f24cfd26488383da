// ABOBA half-steps, counter-based Philox noise, and the reflection-coupling transport map.
// PAPER.md:60-66 (Eq. 2), :101-111 (Eq. 7, 8), :421-425 (Alg. 1), :584-604 (DRAFT_STEP / VERIFY_STEP).
// State is fp64, component-major [3][n].
#include "lsd_internal.h"
#include "philox.cuh"

namespace {

using namespace lsdrng;

// A(1/2): q_half = q + (dt/2) p / m  (Eq. 2 first line; map f of Thm 3.1).  Also checks the Verlet skin.
__global__ void k_half_a(int n, const double* __restrict__ q, const double* __restrict__ p, const double* __restrict__ mass,
                         double hdt, double* __restrict__ qhalf, const double* __restrict__ qref, double skin_half2, int* flags)
{
    pdl_sync();
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const double m = mass[i];
    double d2 = 0.0;
    bool bad = false;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const double v = q[c * n + i] + hdt * p[c * n + i] / m;
        qhalf[c * n + i] = v;
        if (qref) { const double d = v - qref[c * n + i]; d2 += d * d; }
        bad |= !isfinite(v);
    }
    if (qref && d2 > skin_half2) atomicOr(flags, LSD_FLAG_SKIN);
    if (bad) atomicOr(flags, LSD_FLAG_NONFINITE);
}

// B O B (= Eq. 7 Gaussian draw) followed by A(1/2):  p' = c1 p + b F + sigma xi;  q' = q_half + (dt/2) p'/m
__global__ void k_bob_a(int n, uint64_t seed, const uint64_t* __restrict__ n0p, uint64_t j, const double* __restrict__ p_prev, const double* __restrict__ Ft,
                        const double* __restrict__ qhalf, const double* __restrict__ mass, const double* __restrict__ sigma,
                        double c1, double b, double hdt, double* __restrict__ q_new, double* __restrict__ p_new,
                        const double* __restrict__ dF, double* __restrict__ qhalf_next, const double* __restrict__ qref,
                        double skin_half2, int* flags)
{
    pdl_sync();
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    double xi[3];
    normals3(seed, *n0p + j, (uint32_t)i, 0u, xi);          // step index n0 + j; n0 lives in device memory so that a captured graph can be replayed
    const double m = mass[i], sg = sigma[i];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const double Fe = dF ? Ft[c * n + i] + dF[c * n + i] : Ft[c * n + i];      // EC (Alg. 3): <p~> = [Eq. 7](F~ + dF)
        const double pn = c1 * p_prev[c * n + i] + b * Fe + sg * xi[c];
        p_new[c * n + i] = pn;
        q_new[c * n + i] = qhalf[c * n + i] + hdt * pn / m;
    }
    if (qhalf_next) {                                // first A(1/2) of the next step of a rollout (the same arithmetic as k_half_a): one launch less per step
        double d2 = 0.0;
        bool bad = false;
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            const double v = q_new[c * n + i] + hdt * p_new[c * n + i] / m;
            qhalf_next[c * n + i] = v;
            const double d = v - qref[c * n + i]; d2 += d * d;
            bad |= !isfinite(v);
        }
        if (d2 > skin_half2) atomicOr(flags, LSD_FLAG_SKIN);
        if (bad) atomicOr(flags, LSD_FLAG_NONFINITE);
    }
}

__global__ void k_initial_momenta(int n, uint64_t seed, const double* __restrict__ mass, double kT, double* __restrict__ p)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    double xi[3];
    normals3(seed, 0, (uint32_t)i, 2u, xi);
    const double s = sqrt(mass[i] * kT);
#pragma unroll
    for (int c = 0; c < 3; ++c) p[c * n + i] = s * xi[c];
}

// ---- transport, stage 1: per-block partial sums of S1 = xi.d and S2 = d.d, d = (b/sigma)(F~ - F)  (Eq. 8; R6, R13).
// grid (nblk, K).  Fixed-order reduction: thread-serial over a strided slice, xor-shuffle tree in the warp,
// warps summed in index order by thread 0.  fp64 throughout.
constexpr int kTrThreads = 256;

__global__ void __launch_bounds__(kTrThreads)
k_transport_partial(int n, uint64_t seed, const uint64_t* __restrict__ n0p, const double* __restrict__ Ft, const double* __restrict__ Fg,
                    const double* __restrict__ sigma, double b, double* __restrict__ partial, double* __restrict__ xi_dbg,
                    const double* __restrict__ dF, double slack)
{
    pdl_sync();
    const int j = blockIdx.y;                      // step j+1 of the window
    const uint64_t n0 = *n0p;
    const size_t base = (size_t)j * 3 * n;
    double s1 = 0.0, s2 = 0.0;
    for (int i = blockIdx.x * kTrThreads + threadIdx.x; i < n; i += gridDim.x * kTrThreads) {
        double xi[3];
        normals3(seed, n0 + (uint64_t)j + 1, (uint32_t)i, 0u, xi);
        const double bs = b / sigma[i];
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            const double Fe = dF ? Ft[base + (size_t)c * n + i] + dF[c * n + i] : Ft[base + (size_t)c * n + i];   // EC: the draft was drawn around F~ + dF
            double dFo = Fe - Fg[base + (size_t)c * n + i];
            if (slack > 0.0) dFo -= fmin(fmax(dFo, -slack), slack);       // force slack (App. H :779): F_(eps) = F + clip(-eps; F~ - F; eps) in the place of F
            const double d = bs * dFo;
            s1 += xi[c] * d;
            s2 += d * d;
            if (xi_dbg) xi_dbg[base + (size_t)c * n + i] = xi[c];
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        s1 += __shfl_xor_sync(0xffffffffu, s1, o);
        s2 += __shfl_xor_sync(0xffffffffu, s2, o);
    }
    __shared__ double sh1[kTrThreads / 32], sh2[kTrThreads / 32];
    if ((threadIdx.x & 31) == 0) { sh1[threadIdx.x >> 5] = s1; sh2[threadIdx.x >> 5] = s2; }
    __syncthreads();
    if (threadIdx.x == 0) {
        double a = 0.0, c = 0.0;
        for (int w = 0; w < kTrThreads / 32; ++w) { a += sh1[w]; c += sh2[w]; }
        partial[((size_t)j * gridDim.x + blockIdx.x) * 2 + 0] = a;
        partial[((size_t)j * gridDim.x + blockIdx.x) * 2 + 1] = c;
    }
}

// ---- stage 2: ell_j = -S1 - S2/2, u_j, accept iff S2 == 0 or ln u <= min(0, ell) (R7, R8); first-reject scan (:424).
__global__ void k_transport_final(int K, int nblk, uint64_t seed, const uint64_t* __restrict__ n0p, const double* __restrict__ partial,
                                  double* S1, double* S2, double* ell, double* lnu, int* reject, const int* flags,
                                  TransportResult* result)
{
    pdl_sync();
    __shared__ int rej[LSD_MAX_K], bad[LSD_MAX_K];
    __shared__ double beta[LSD_MAX_K];
    const int j = threadIdx.x;
    const uint64_t n0 = *n0p;
    if (j < K) {
        double a = 0.0, c = 0.0;
        for (int blk = 0; blk < nblk; ++blk) { a += partial[((size_t)j * nblk + blk) * 2]; c += partial[((size_t)j * nblk + blk) * 2 + 1]; }
        const double l = -a - 0.5 * c;
        const double lu = log(uniform53(seed, n0 + (uint64_t)j + 1));
        const int r = (c > 0.0 && lu > fmin(0.0, l)) ? 1 : 0;
        S1[j] = a; S2[j] = c; ell[j] = l; lnu[j] = lu; reject[j] = r;
        rej[j] = r;
        bad[j] = !(isfinite(a) && isfinite(c));      // a non-finite draft or target force (r -> 0 pair, overflow): comparisons with NaN are false,
                                                     // i.e. the step would read as accepted
        beta[j] = erf(sqrt(c) / sqrt(8.0));           // Eq. 9
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        int l = 0;
        for (int t = 0; t < K; ++t) if (rej[t]) { l = t + 1; break; }   // l = min{j : x_j != y_j}
        const int nc = l ? l : K;                                      // R3 (no bonus step), R4 (x_l counts)
        double bs = 0.0;
        int fl = *flags;
        for (int t = 0; t < nc; ++t) { bs += beta[t]; if (bad[t]) fl |= LSD_FLAG_NONFINITE; }   // k_commit then commits nothing
        result->first_reject = l; result->n_commit = nc; result->flags = fl; result->beta_sum = bs;
    }
}

// ---- stage 3: override of the first rejected step and map g (Eq. 8 else-branch; :602), or commit of y_K.
__global__ void k_commit(int n, int K, uint64_t seed, const uint64_t* __restrict__ n0p, const TransportResult* __restrict__ result,
                         const double* __restrict__ S1, const double* __restrict__ S2, const double* __restrict__ Ft,
                         const double* __restrict__ Fg, const double* __restrict__ qhalf, const double* __restrict__ pstart,
                         double* __restrict__ yq, double* __restrict__ yp, const double* __restrict__ mass,
                         const double* __restrict__ sigma, double c1, double b, double hdt, double* __restrict__ q_base,
                         double* __restrict__ p_base, const double* __restrict__ dF, double* __restrict__ dF_out, double slack)
{
    pdl_sync();
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    if (result->flags != 0) return;                  // skin / overflow / non-finite: nothing is committed
    const int l = result->first_reject;
    if (dF_out) {                                    // EC cache <- F - F~ (bare draft output) of the last committed step
        const size_t cb = (size_t)((l ? l : K) - 1) * 3 * n;
#pragma unroll
        for (int c = 0; c < 3; ++c) dF_out[c * n + i] = Fg[cb + (size_t)c * n + i] - Ft[cb + (size_t)c * n + i];
    }
    if (l == 0) {
        const size_t base = (size_t)(K - 1) * 3 * n;
#pragma unroll
        for (int c = 0; c < 3; ++c) { q_base[c * n + i] = yq[base + (size_t)c * n + i]; p_base[c * n + i] = yp[base + (size_t)c * n + i]; }
        return;
    }
    const size_t base = (size_t)(l - 1) * 3 * n;
    const double* pprev = (l == 1) ? pstart : yp + (size_t)(l - 2) * 3 * n;
    double xi[3];
    normals3(seed, *n0p + (uint64_t)l, (uint32_t)i, 0u, xi);
    const double sg = sigma[i], m = mass[i], ratio = S1[l - 1] / S2[l - 1];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        double F = Fg[base + (size_t)c * n + i];
        const double Fe = dF ? Ft[base + (size_t)c * n + i] + dF[c * n + i] : Ft[base + (size_t)c * n + i];
        if (slack > 0.0) F += fmin(fmax(Fe - F, -slack), slack);          // F_(eps) of App. H replaces the target force in the override too
        const double d = b / sg * (Fe - F);
        const double ps = c1 * pprev[c * n + i] + b * F + sg * (xi[c] - 2.0 * ratio * d);
        const double qs = qhalf[base + (size_t)c * n + i] + hdt * ps / m;
        p_base[c * n + i] = ps; q_base[c * n + i] = qs;
        yp[base + (size_t)c * n + i] = ps; yq[base + (size_t)c * n + i] = qs;     // x_l replaces y_l in the committed window
    }
}

// (OBABO) output momentum of committed step j of the window by time staggering (App. F Eq. 26-30, :700-753):
// w = Sigma_half^{-1/2}(p_new - c1 p_prev - (1 + c1)(dt/2) F);  xi1* = ch/(1 + c1) w + (1 + c1)^{-1/2} zeta (zeta: Philox tag 3);
// p_mid = ch (p_prev + (dt/2) F) + Sigma_half^{1/2} xi1*,  Sigma_half = m kT (1 - c1), ch = e^{-gamma dt/2}, c1 = e^{-gamma dt}.
__global__ void k_obabo(int n, uint64_t seed, const uint64_t* __restrict__ n0p, uint64_t j, const double* __restrict__ p_prev,
                        const double* __restrict__ p_new, const double* __restrict__ F, const double* __restrict__ mass,
                        double kT, double c1, double ch, double hdt, double* __restrict__ p_mid)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    double zeta[3];
    normals3(seed, *n0p + j, (uint32_t)i, 3u, zeta);
    const double sh = sqrt(mass[i] * kT * (1.0 - c1));
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const double pp = p_prev[c * n + i], f = F[c * n + i];
        const double w = (p_new[c * n + i] - c1 * pp - (1.0 + c1) * hdt * f) / sh;
        const double xi1 = ch / (1.0 + c1) * w + sqrt(1.0 / (1.0 + c1)) * zeta[c];
        p_mid[c * n + i] = ch * (pp + hdt * f) + sh * xi1;
    }
}

}  // namespace

void launch_obabo(Launcher L, int n, uint64_t seed, const uint64_t* n0_dev, uint64_t j, const double* p_prev, const double* p_new,
                  const double* F, const double* mass, double kT, double c1, double ch, double hdt, double* p_mid)
{
    k_obabo<<<(n + 127) / 128, 128, 0, L.s>>>(n, seed, n0_dev, j, p_prev, p_new, F, mass, kT, c1, ch, hdt, p_mid);
    LSD_COUNT(L);
}

int transport_blocks(int n)
{
    int nb = (n + kTrThreads * 4 - 1) / (kTrThreads * 4);
    if (nb < 1) nb = 1;
    if (nb > 148) nb = 148;
    return nb;
}

void launch_half_a(Launcher L, int n, const double* q, const double* p, const double* mass, double hdt,
                   double* qhalf, const double* qref, double skin_half2, int* flags)
{
    const int pid = prof_begin(L, PROF_INTEG);
    launch_pdl(L, k_half_a, dim3((n + 255) / 256), dim3(256), 0, n, q, p, mass, hdt, qhalf, qref, skin_half2, flags);
    LSD_COUNT(L);
    prof_end(L, pid);
}

void launch_bob_a(Launcher L, int n, uint64_t seed, const uint64_t* n0_dev, uint64_t j, const double* p_prev, const double* Ft,
                  const double* qhalf, const double* mass, const double* sigma, double c1, double b, double hdt,
                  double* q_new, double* p_new, const double* dF, double* qhalf_next, const double* qref, double skin_half2, int* flags)
{
    const int pid = prof_begin(L, PROF_INTEG);
    launch_pdl(L, k_bob_a, dim3((n + 127) / 128), dim3(128), 0, n, seed, n0_dev, j, p_prev, Ft, qhalf, mass, sigma, c1, b, hdt, q_new, p_new, dF, qhalf_next, qref, skin_half2, flags);
    LSD_COUNT(L);
    prof_end(L, pid);
}

__global__ void k_set_u64(uint64_t* dst, uint64_t v) { pdl_sync(); *dst = v; }
void launch_set_u64(Launcher L, uint64_t* dst, uint64_t v)
{
    launch_pdl(L, k_set_u64, dim3(1), dim3(1), 0, dst, v);
    LSD_COUNT(L);
}

void launch_initial_momenta(Launcher L, int n, uint64_t seed, const double* mass, double kT, double* p)
{
    k_initial_momenta<<<(n + 127) / 128, 128, 0, L.s>>>(n, seed, mass, kT, p);
    LSD_COUNT(L);
}

void launch_transport(Launcher L, int n, int K, uint64_t seed, const uint64_t* n0, const double* Ft, const double* Fg,
                      const double* sigma, double b, double* partial, int nblk, double* S1, double* S2, double* ell,
                      double* lnu, int* reject, const int* flags, TransportResult* result, double* xi_dbg, const double* dF, double slack)
{
    const int pid = prof_begin(L, PROF_TRANSPORT);
    launch_pdl(L, k_transport_partial, dim3(nblk, K), dim3(kTrThreads), 0, n, seed, n0, Ft, Fg, sigma, b, partial, xi_dbg, dF, slack);
    LSD_COUNT(L);
    launch_pdl(L, k_transport_final, dim3(1), dim3(LSD_MAX_K), 0, K, nblk, seed, n0, partial, S1, S2, ell, lnu, reject, flags, result);
    LSD_COUNT(L);
    prof_end(L, pid);
}

void launch_commit(Launcher L, int n, int K, uint64_t seed, const uint64_t* n0, const TransportResult* result,
                   const double* S1, const double* S2, const double* Ft, const double* Fg, const double* qhalf,
                   const double* pstart, double* yq, double* yp, const double* mass, const double* sigma,
                   double c1, double b, double hdt, double* q_base, double* p_base, const double* dF, double* dF_out, double slack)
{
    const int pid = prof_begin(L, PROF_TRANSPORT);
    launch_pdl(L, k_commit, dim3((n + 127) / 128), dim3(128), 0, n, K, seed, n0, result, S1, S2, Ft, Fg, qhalf, pstart, yq, yp, mass, sigma,
                                               c1, b, hdt, q_base, p_base, dF, dF_out, slack);
    LSD_COUNT(L);
    prof_end(L, pid);
}
