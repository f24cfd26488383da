// Draft rollout of a TINY system as ONE kernel launch (a0; PAPER.md:584-593 DRAFT_STEP, Eq. 2, Eq. 7, launch-bound
// regime).  The general rollout (rollout_body in lsd_api.cu) spends ~10 dependent launches of 4-10 us per draft step; for a
// system of <= 64 atoms every one of them is a fraction of one SM's work and the chain is pure latency.  Here ONE thread-block
// cluster of 8 CTAs (8 SMs: a single CTA is itself latency-bound, 41 us per step at cfg2 against 12 us for the cluster) keeps
// the state (fp64, replicated), the draft network's weights and the per-step neighbour rows of the atoms it owns in shared
// memory and loops over the K steps of the window; per step the owners push mbar and the total forces into every CTA's shared
// memory (distributed shared memory) and two cluster barriers order them:  A(1/2) -> neighbour rows by brute force (no skin, no Verlet list) -> prior forces (fp64) ->
// width-32, one-block network forward and analytic backward (fp32 FMA, M1-M9) -> B O B + A(1/2) with Philox noise.
// The step's q_half, F~, y are written to the window slot exactly as the general rollout writes them.
//
// Same formulas as prior.cu / mlip_simt.cu / integrator.cu, but its own summation orders (per atom: neighbours in ascending
// index order inside one warp), so the forces agree with the batched kernels to fp32 round-off, not bit for bit: lsd_api.cu
// uses this kernel only when the draft differs from the target (draft == target must reproduce the target bitwise, R8).
#include <algorithm>
#include "lsd_internal.h"
#include "philox.cuh"

namespace {

using namespace lsdrng;

constexpr int kNMax = LSD_TINY_MAX_ATOMS;              // atoms
constexpr int kF = 32;                                 // width of the draft network
constexpr int kR = LSD_NRBF;
constexpr int kWarps = 16, kThreads = kWarps * 32;
constexpr int kLD = kF + 4;                            // leading dimension of the per-warp operand tiles
constexpr int kMaxSpecies = 8;
constexpr float kLn2 = 0.69314718055994530942f;

__device__ __forceinline__ float ssp(float x) { return fmaxf(x, 0.f) + log1pf(expf(-fabsf(x))) - kLn2; }          // M3
__device__ __forceinline__ float logistic(float x) { return 1.f / (1.f + expf(-x)); }

struct TinyArgs {
    int n, ns, K, periodic;
    double box[3];
    const int* species; const double* mass; const double* sigma;
    // prior
    const double* pair; const double* pair_rc2; const double* tether;
    int has_pair, use_bonded, n_bonds;
    const int *bt_start, *bt_term, *bonds, *angles;
    const double *bond_k, *bond_r0, *angle_k, *angle_t0;
    // network (F = 32, T = 1) or has_net = 0
    int has_net;
    float rc, alpha, delta, inv_delta2, inv_rc;
    const float *emb, *ytab0, *Wf1T, *Wf2T, *Wo1T, *Wo2T, *Wo2, *Wo1, *Wr1, *wr2;
    // integrator
    uint64_t seed; const uint64_t* n0_dev;
    double c1, b, hdt, skin_half2;
    const double *qstart, *pstart, *dF;
    double *qhalf, *Ft, *yq, *yp;                      // [K][3][n]
    int* flags;
};

constexpr int kNC = LSD_TINY_CLUSTER;                 // CTAs of the cluster (one SM each); atom i is owned by CTA i % kNC
constexpr int kOwnMax = (kNMax + kNC - 1) / kNC;       // owned atoms per CTA
constexpr int kItemMax = kOwnMax * (kNMax / 4);        // (atom, unit of 4 edges) work items per CTA

// shared-memory plan of a CTA (floats unless noted)
struct Plan {
    // weights
    static constexpr int oWf1 = 0, oWf2 = oWf1 + kR * kF, oWo1T = oWf2 + kF * kF, oWo2T = oWo1T + kF * kF, oWo2 = oWo2T + kF * kF,
                         oWo1 = oWo2 + kF * kF, oWr1 = oWo1 + kF * kF, oWr2 = oWr1 + (kF / 2) * kF, oEmb = oWr2 + kF / 2,
                         oYtab = oEmb + kMaxSpecies * kF, oScratch = oYtab + kMaxSpecies * kF;
    static constexpr int ScratchPerWarp = 8 * (kR + 4) + 8 * kLD;
    static constexpr int oMbar = oScratch + kWarps * ScratchPerWarp;          // [n][F], every atom (pushed by its owner)
    static constexpr int oMpart = oMbar + kNMax * kF;                          // [items][F] partial sums m of the forward units
    static constexpr int oRec = oMpart + kItemMax * kF;                        // 6 fields [owned][64]: r, fc, fc', ux, uy, uz
    static constexpr int oEnd = oRec + 6 * kOwnMax * kNMax;
    static constexpr int oD = ((oEnd * 4 + 15) / 16) * 16;                     // bytes: fp64 q, p, qh [3][n], F [2][3][n] (by step parity), mass, sigma [n], prior force [owned][3], unit forces [items][3]
    static constexpr int nD = (5 * 3 + 2) * kNMax + 3 * kOwnMax + 3 * kItemMax;
    static constexpr int oNbr = oD + nD * 8;                                   // bytes: neighbour rows [owned][64] uint8
    static constexpr int oInt = oNbr + kOwnMax * kNMax;                        // ints: cnt [owned], species [n], item tables (fwd, bwd) [items] each, counters
    static constexpr int Bytes = oInt + (kOwnMax + kNMax + 2 * kItemMax + 4) * 4;
};
static_assert(Plan::Bytes <= 200 * 1024, "shared memory budget");

// acc[8] = A[8][KD] (shared, leading dimension lda) * W[KD][32] (shared, k-major); lane owns output channel `lane`
template <int KD>
__device__ __forceinline__ void warp_gemm8(const float* __restrict__ As, int lda, const float* __restrict__ Ws, int lane, float (&acc)[8])
{
#pragma unroll
    for (int r = 0; r < 8; ++r) acc[r] = 0.f;
#pragma unroll 2
    for (int k4 = 0; k4 < KD / 4; ++k4) {
        float4 a[8];
#pragma unroll
        for (int r = 0; r < 8; ++r) a[r] = *reinterpret_cast<const float4*>(As + r * lda + 4 * k4);
#pragma unroll
        for (int kk = 0; kk < 4; ++kk) {
            const float w = Ws[(4 * k4 + kk) * kF + lane];
#pragma unroll
            for (int r = 0; r < 8; ++r) {
                const float av = kk == 0 ? a[r].x : kk == 1 ? a[r].y : kk == 2 ? a[r].z : a[r].w;
                acc[r] = fmaf(av, w, acc[r]);
            }
        }
    }
}
// out[lane] = sum_k in[k] W[k][lane], in[k] held by lane k; four interleaved chains (k mod 4), summed in a fixed order
__device__ __forceinline__ float warp_matvec(float in, const float* __restrict__ W, int lane, int K = kF)
{
    float acc[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll 8
    for (int k = 0; k < K; k += 4) {
#pragma unroll
        for (int u = 0; u < 4; ++u) acc[u] = fmaf(__shfl_sync(0xffffffffu, in, k + u), W[(k + u) * kF + lane], acc[u]);
    }
    return (acc[0] + acc[1]) + (acc[2] + acc[3]);
}

__device__ __forceinline__ void cluster_sync()
{
    asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");
    asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");
}
__device__ __forceinline__ uint32_t cluster_rank() { uint32_t r; asm("mov.u32 %0, %%cluster_ctarank;" : "=r"(r)); return r; }
// address of the same shared-memory location in CTA `rank` of the cluster
__device__ __forceinline__ uint32_t map_rank(const void* p, uint32_t rank)
{
    uint32_t local = (uint32_t)__cvta_generic_to_shared(p), remote;
    asm("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(remote) : "r"(local), "r"(rank));
    return remote;
}
__device__ __forceinline__ void st_cluster(uint32_t addr, float v) { asm volatile("st.shared::cluster.f32 [%0], %1;" ::"r"(addr), "f"(v) : "memory"); }
__device__ __forceinline__ void st_cluster(uint32_t addr, double v) { asm volatile("st.shared::cluster.f64 [%0], %1;" ::"r"(addr), "d"(v) : "memory"); }

__global__ void __cluster_dims__(kNC, 1, 1) __launch_bounds__(kThreads, 1)
k_tiny_rollout(TinyArgs a)
{
    extern __shared__ __align__(16) uint8_t smem_raw[];
    float* const sf = reinterpret_cast<float*>(smem_raw);
    double* const sd = reinterpret_cast<double*>(smem_raw + Plan::oD);
    const int n = a.n, tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int rank = (int)cluster_rank();
    const int n_own = rank < n ? (n - rank + kNC - 1) / kNC : 0;          // atoms rank, rank + kNC, ...
    double* const q = sd, * const p = sd + 3 * kNMax, * const qh = sd + 6 * kNMax, * const Fs2 = sd + 9 * kNMax, * const ms = sd + 15 * kNMax, * const sg = sd + 16 * kNMax;
    double* const Fp = sd + 17 * kNMax;                                    // [owned][3] prior force of the owned atoms
    double* const fpart = Fp + 3 * kOwnMax;                                // [items][3] force of a backward unit
    uint8_t* const nbr = smem_raw + Plan::oNbr;
    int* const cnt = reinterpret_cast<int*>(smem_raw + Plan::oInt);
    int* const spc = cnt + kOwnMax;
    int* const itf = spc + kNMax;                                          // forward units: (owned atom << 8) | unit
    int* const itb = itf + kItemMax;                                       // backward units
    int* const nit = itb + kItemMax;                                       // [0]: forward units, [1]: backward units
    float* const rec = sf + Plan::oRec;
    float* const mbar_s = sf + Plan::oMbar;
    float* const mpart = sf + Plan::oMpart;
    float* const Gs = sf + Plan::oScratch + warp * Plan::ScratchPerWarp;
    float* const As = Gs + 8 * (kR + 4);
    constexpr int LDG = kR + 4, RS = kOwnMax * kNMax;                      // RS: stride between record fields

    if (a.has_net) {                                   // the whole network stays resident for the K steps
        auto cp = [&](int off, const float* src, int count) { for (int i = tid; i < count; i += kThreads) sf[off + i] = src[i]; };
        cp(Plan::oWf1, a.Wf1T, kR * kF); cp(Plan::oWf2, a.Wf2T, kF * kF); cp(Plan::oWo1T, a.Wo1T, kF * kF); cp(Plan::oWo2T, a.Wo2T, kF * kF);
        cp(Plan::oWo2, a.Wo2, kF * kF); cp(Plan::oWo1, a.Wo1, kF * kF); cp(Plan::oWr1, a.Wr1, (kF / 2) * kF); cp(Plan::oWr2, a.wr2, kF / 2);
        cp(Plan::oEmb, a.emb, a.ns * kF); cp(Plan::oYtab, a.ytab0, a.ns * kF);
    }
    for (int i = tid; i < n; i += kThreads) {
#pragma unroll
        for (int c = 0; c < 3; ++c) { q[c * kNMax + i] = a.qstart[c * n + i]; p[c * kNMax + i] = a.pstart[c * n + i]; }
        ms[i] = a.mass[i]; sg[i] = a.sigma[i]; spc[i] = a.species[i];
    }
    const uint64_t n0 = *a.n0_dev;
    const double rc2 = (double)a.rc * (double)a.rc;
    cluster_sync();                                    // every CTA of the cluster is running before anyone writes into its shared memory

    for (int j = 1; j <= a.K; ++j) {
        // ---- A(1/2): q_half = q + (dt/2) p / m; skin of the window-shared lists the verification will use (k_half_a).  Every CTA
        // keeps the whole state (the update is the same arithmetic everywhere); rank 0 reports.
        if (tid < n) {
            const int i = tid;
            double d2 = 0.0; bool bad = false;
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                const double v = q[c * kNMax + i] + a.hdt * p[c * kNMax + i] / ms[i];
                qh[c * kNMax + i] = v;
                const double d = v - a.qstart[c * n + i]; d2 += d * d;
                bad |= !isfinite(v);
            }
            if (rank == 0 && d2 > a.skin_half2) atomicOr(a.flags, LSD_FLAG_SKIN);
            if (rank == 0 && bad) atomicOr(a.flags, LSD_FLAG_NONFINITE);
        }
        __syncthreads();
        // ---- per owned atom (one warp): neighbour row of the network (ascending j), pair prior, bonded prior
        for (int k = warp; k < n_own; k += kWarps) {
            const int i = rank + k * kNC;
            const int si = spc[i];
            double f[3] = {0.0, 0.0, 0.0};
            int c_i = 0;
            for (int j0 = 0; j0 < n; j0 += 32) {
                const int jj = j0 + lane;
                bool keep = false;
                double d[3] = {0.0, 0.0, 0.0}, r2 = 0.0;
                if (jj < n && jj != i) {
#pragma unroll
                    for (int c = 0; c < 3; ++c) {
                        double x = __dsub_rn(qh[c * kNMax + jj], qh[c * kNMax + i]);
                        if (a.periodic) x = __dadd_rn(x, __dmul_rn(-rint(x / a.box[c]), a.box[c]));       // nearest image (R10)
                        d[c] = x;
                    }
                    r2 = __dadd_rn(__dadd_rn(__dmul_rn(d[0], d[0]), __dmul_rn(d[1], d[1])), __dmul_rn(d[2], d[2]));
                    keep = a.has_net && r2 < rc2;
                    if (a.has_pair && r2 < a.pair_rc2[si * a.ns + spc[jj]]) {                              // O-4 pair terms, fp64
                        const double r = sqrt(r2);
                        const double* pp = a.pair + 8 * (si * a.ns + spc[jj]);
                        double du = 0.0;
                        if (pp[0] != 0.0 && r < pp[2]) { const double sr = pp[1] / r, s2 = sr * sr, s6 = s2 * s2 * s2; du += -24.0 * pp[0] / r * (2.0 * s6 * s6 - s6); }
                        if (pp[3] != 0.0 && r < pp[6]) { const double x = exp(-pp[4] * (r - pp[5])); du += 2.0 * pp[3] * pp[4] * x * (1.0 - x); }
                        const double g = du / r;
                        f[0] += g * d[0]; f[1] += g * d[1]; f[2] += g * d[2];
                    }
                }
                const unsigned m = __ballot_sync(0xffffffffu, keep);
                if (keep) {                                                 // record: fp64 geometry rounded once to fp32 (k_compact)
                    const int pos = c_i + __popc(m & ((1u << lane) - 1));
                    const double rd = sqrt(r2);
                    const float rf = (float)rd;
                    float fc = 0.f, fcp = 0.f;
                    const float t = rf * a.inv_rc;
                    if (t < 1.f) { float sn, cs; sincospif(t, &sn, &cs); fc = 0.5f * (cs + 1.f); fcp = -0.5f * 3.14159265358979323846f * a.inv_rc * sn; }   // M2
                    float* o = rec + k * kNMax + pos;
                    o[0] = rf; o[RS] = fc; o[2 * RS] = fcp;
                    o[3 * RS] = (float)(d[0] / rd); o[4 * RS] = (float)(d[1] / rd); o[5 * RS] = (float)(d[2] / rd);
                    nbr[k * kNMax + pos] = (uint8_t)jj;
                }
                c_i += __popc(m);
            }
            if (a.use_bonded) {
                auto mi = [&](int from, int to, double (&d)[3]) {
#pragma unroll
                    for (int c = 0; c < 3; ++c) {
                        double x = qh[c * kNMax + to] - qh[c * kNMax + from];
                        if (a.periodic) x -= rint(x / a.box[c]) * a.box[c];
                        d[c] = x;
                    }
                };
                for (int t = a.bt_start[i] + lane; t < a.bt_start[i + 1]; t += 32) {
                    const int term = a.bt_term[t];
                    if (term < a.n_bonds) {                                  // U = k/2 (r - r0)^2
                        const int a0 = a.bonds[2 * term], a1 = a.bonds[2 * term + 1];
                        const int other = (a0 == i) ? a1 : a0;
                        double d[3]; mi(i, other, d);
                        const double r = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
                        const double g = a.bond_k[term] * (r - a.bond_r0[term]) / r;
                        f[0] += g * d[0]; f[1] += g * d[1]; f[2] += g * d[2];
                    } else {                                                 // U = k/2 (theta - theta0)^2, apex = middle index
                        const int an = term - a.n_bonds;
                        const int ia = a.angles[3 * an], ib = a.angles[3 * an + 1], ic = a.angles[3 * an + 2];
                        double u[3], v[3];
                        mi(ib, ia, u); mi(ib, ic, v);
                        const double nu = sqrt(u[0] * u[0] + u[1] * u[1] + u[2] * u[2]), nv = sqrt(v[0] * v[0] + v[1] * v[1] + v[2] * v[2]);
                        double ct = (u[0] * v[0] + u[1] * v[1] + u[2] * v[2]) / (nu * nv);
                        ct = fmin(1.0, fmax(-1.0, ct));
                        const double th = acos(ct), st = fmax(sqrt(1.0 - ct * ct), 1e-12);   // collinear arms: bounded (R19)
                        const double dU = a.angle_k[an] * (th - a.angle_t0[an]);
#pragma unroll
                        for (int c = 0; c < 3; ++c) {
                            const double uh = u[c] / nu, vh = v[c] / nv;
                            const double da = -(vh - ct * uh) / (nu * st), dc = -(uh - ct * vh) / (nv * st);
                            double contrib;
                            if (i == ia) contrib = -dU * da; else if (i == ic) contrib = -dU * dc; else contrib = dU * (da + dc);
                            f[c] += contrib;
                        }
                    }
                }
            }
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                f[0] += __shfl_xor_sync(0xffffffffu, f[0], o);
                f[1] += __shfl_xor_sync(0xffffffffu, f[1], o);
                f[2] += __shfl_xor_sync(0xffffffffu, f[2], o);
            }
            if (lane == 0) {
                if (a.tether) { const double kt = a.tether[si]; f[0] -= kt * qh[i]; f[1] -= kt * qh[kNMax + i]; f[2] -= kt * qh[2 * kNMax + i]; }
                Fp[3 * k] = f[0]; Fp[3 * k + 1] = f[1]; Fp[3 * k + 2] = f[2];
                cnt[k] = c_i;
            }
        }
        __syncthreads();
        if (a.has_net) {
            const float* Wf1 = sf + Plan::oWf1; const float* Wf2 = sf + Plan::oWf2;
            const float* ytab = sf + Plan::oYtab;
            if (tid == 0) {                            // work items of this CTA: (owned atom, unit of 8 edges) forward, (owned atom, unit of 4 edges) backward
                int nf = 0, nb = 0;
                for (int k = 0; k < n_own; ++k) {
                    for (int u = 0; u < (cnt[k] + 7) / 8; ++u) itf[nf++] = (k << 8) | u;
                    for (int u = 0; u < (cnt[k] + 3) / 4; ++u) itb[nb++] = (k << 8) | u;
                }
                nit[0] = nf; nit[1] = nb;
            }
            __syncthreads();
            // ---- forward units: partial m over the unit's 8 edges (M5), lane = channel
            for (int it = warp; it < nit[0]; it += kWarps) {
                const int k = itf[it] >> 8, u0 = (itf[it] & 255) * 8, ci = cnt[k];
#pragma unroll
                for (int e = 0; e < 8; ++e) {                              // radial basis rows (M1): lane k holds basis k
                    const bool ve = (u0 + e) < ci;
                    const float re = ve ? rec[k * kNMax + u0 + e] : 0.f;
                    const float x = re - (float)lane * a.delta;
                    Gs[e * LDG + lane] = ve ? expf(-0.5f * x * x * a.inv_delta2) : 0.f;
                }
                __syncwarp();
                float acc[8];
                warp_gemm8<kR>(Gs, LDG, Wf1, lane, acc);
#pragma unroll
                for (int e = 0; e < 8; ++e) As[e * kLD + lane] = ssp(acc[e]);
                __syncwarp();
                warp_gemm8<kF>(As, kLD, Wf2, lane, acc);
                float m_u = 0.f;
#pragma unroll
                for (int e = 0; e < 8; ++e) {
                    if (u0 + e < ci) {
                        const int jn = nbr[k * kNMax + u0 + e];
                        m_u = fmaf(ytab[spc[jn] * kF + lane], acc[e] * rec[RS + k * kNMax + u0 + e], m_u);
                    }
                }
                mpart[it * kF + lane] = m_u;
                __syncwarp();
            }
            __syncthreads();
            // ---- atom-wise layers, readout and their adjoints (M5, M6, M9) of the owned atoms: one warp per atom, lane = channel;
            //      mbar goes to every CTA of the cluster
            for (int k = warp; k < n_own; k += kWarps) {
                const int i = rank + k * kNC;
                float m_i = 0.f;
                for (int it = 0; it < nit[0]; ++it) if ((itf[it] >> 8) == k) m_i += mpart[it * kF + lane];     // units in list order
                const float h = warp_matvec(m_i, sf + Plan::oWo1T, lane);                  // h = W_o1 m
                const float x = sf[Plan::oEmb + spc[i] * kF + lane] + warp_matvec(ssp(h), sf + Plan::oWo2T, lane);   // x = Emb + W_o2 ssp(h)
                float s = 0.f;                                                             // readout: z = W_r1 x (lanes 0..15)
                {
                    float z0 = 0.f, z1 = 0.f;
#pragma unroll 8
                    for (int f = 0; f < kF; f += 2) {
                        const float x0 = __shfl_sync(0xffffffffu, x, f), x1 = __shfl_sync(0xffffffffu, x, f + 1);
                        if (lane < kF / 2) { z0 = fmaf(sf[Plan::oWr1 + lane * kF + f], x0, z0); z1 = fmaf(sf[Plan::oWr1 + lane * kF + f + 1], x1, z1); }
                    }
                    if (lane < kF / 2) s = logistic(z0 + z1) * sf[Plan::oWr2 + lane];
                }
                const float xb = a.alpha * warp_matvec(s, sf + Plan::oWr1, lane, kF / 2);  // xbar = alpha W_r1^T (logistic(z) . w_r2)
                const float hb = logistic(h) * warp_matvec(xb, sf + Plan::oWo2, lane);     // hbar = logistic(h) . (W_o2^T xbar)
                const float mb = warp_matvec(hb, sf + Plan::oWo1, lane);                   // mbar = W_o1^T hbar
#pragma unroll
                for (int r = 0; r < kNC; ++r) st_cluster(map_rank(mbar_s + i * kF + lane, (uint32_t)r), mb);
            }
            cluster_sync();
            // ---- backward units: adjoint of the continuous-filter convolution over the unit's 4 edges -> force of the unit
            for (int it = warp; it < nit[1]; it += kWarps) {
                const int k = itb[it] >> 8, u0 = (itb[it] & 255) * 4, ci = cnt[k];
                const int i = rank + k * kNC;
                const float ya = ytab[spc[i] * kF + lane], mba = mbar_s[i * kF + lane];
                double fx = 0.0, fy = 0.0, fz = 0.0;
#pragma unroll
                for (int e = 0; e < 4; ++e) {                              // value / r-derivative rows interleaved
                    const bool ve = (u0 + e) < ci;
                    const float re = ve ? rec[k * kNMax + u0 + e] : 0.f;
                    const float x = re - (float)lane * a.delta;
                    const float gk = ve ? expf(-0.5f * x * x * a.inv_delta2) : 0.f;
                    Gs[(2 * e) * LDG + lane] = gk; Gs[(2 * e + 1) * LDG + lane] = -gk * x * a.inv_delta2;
                }
                __syncwarp();
                float acc[8];
                warp_gemm8<kR>(Gs, LDG, Wf1, lane, acc);
#pragma unroll
                for (int e = 0; e < 4; ++e) {
                    As[(2 * e) * kLD + lane] = ssp(acc[2 * e]);
                    As[(2 * e + 1) * kLD + lane] = logistic(acc[2 * e]) * acc[2 * e + 1];
                }
                __syncwarp();
                warp_gemm8<kF>(As, kLD, Wf2, lane, acc);
#pragma unroll
                for (int e = 0; e < 4; ++e) {
                    if (u0 + e < ci) {                                     // (warp-uniform)
                        const int o = k * kNMax + u0 + e;
                        const int jn = nbr[o];
                        const float fce = rec[RS + o], fcpe = rec[2 * RS + o];
                        const float yj = ytab[spc[jn] * kF + lane], mbj = mbar_s[jn * kF + lane];
                        const float wp = acc[2 * e + 1] * fce + acc[2 * e] * fcpe;
                        float gp = fmaf(mba, yj, mbj * ya) * wp;
#pragma unroll
                        for (int sh = 16; sh > 0; sh >>= 1) gp += __shfl_xor_sync(0xffffffffu, gp, sh);
                        fx += (double)(gp * rec[3 * RS + o]); fy += (double)(gp * rec[4 * RS + o]); fz += (double)(gp * rec[5 * RS + o]);
                    }
                }
                if (lane == 0) { fpart[3 * it] = fx; fpart[3 * it + 1] = fy; fpart[3 * it + 2] = fz; }
                __syncwarp();
            }
            __syncthreads();
        }
        // ---- total force of the owned atoms (prior + units in list order) -> every CTA of the cluster.  Two copies by step parity: a
        // CTA may still read step j's forces in its B O B while a faster one already pushes those of step j + 1
        double* const Fs = Fs2 + (j & 1) * 3 * kNMax;
        if (tid < n_own) {
            const int k = tid, i = rank + k * kNC;
            double f0 = Fp[3 * k], f1 = Fp[3 * k + 1], f2 = Fp[3 * k + 2];
            if (a.has_net) for (int it = 0; it < nit[1]; ++it) if ((itb[it] >> 8) == k) { f0 += fpart[3 * it]; f1 += fpart[3 * it + 1]; f2 += fpart[3 * it + 2]; }
#pragma unroll
            for (int r = 0; r < kNC; ++r) {
                st_cluster(map_rank(Fs + i, (uint32_t)r), f0); st_cluster(map_rank(Fs + kNMax + i, (uint32_t)r), f1); st_cluster(map_rank(Fs + 2 * kNMax + i, (uint32_t)r), f2);
            }
        }
        cluster_sync();
        // ---- B O B (= Eq. 7 Gaussian draw) + A(1/2) (k_bob_a) on every CTA's copy of the state; rank 0 writes the step's rows of the window slot
        if (tid < n) {
            const int i = tid;
            double xi[3];
            normals3(a.seed, n0 + (uint64_t)j, (uint32_t)i, 0u, xi);
            const size_t row = (size_t)(j - 1) * 3 * n;
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                const double Fd = Fs[c * kNMax + i];
                const double Fe = a.dF ? Fd + a.dF[c * n + i] : Fd;            // EC (Alg. 3)
                const double pn = a.c1 * p[c * kNMax + i] + a.b * Fe + sg[i] * xi[c];
                const double qn = qh[c * kNMax + i] + a.hdt * pn / ms[i];
                if (rank == 0) {
                    a.qhalf[row + c * n + i] = qh[c * kNMax + i];
                    a.Ft[row + c * n + i] = Fd;
                    a.yp[row + c * n + i] = pn; a.yq[row + c * n + i] = qn;
                }
                p[c * kNMax + i] = pn; q[c * kNMax + i] = qn;
            }
        }
        __syncthreads();
    }
    cluster_sync();                                    // nobody leaves while a neighbour may still write into its shared memory
}

}  // namespace

bool tiny_rollout_supported(const SysDev& sys, const PotDev& pot)
{
    if (sys.n > kNMax || sys.ns > kMaxSpecies) return false;
    const MlipDev& m = pot.mlip;
    return m.F == 0 || (m.F == kF && m.T == 1 && m.R == kR);
}

void launch_tiny_rollout(Launcher L, const SysDev& sys, const PotDev& pot, int K, uint64_t seed, const uint64_t* n0_dev,
                         double c1, double b, double hdt, double skin_half2, const double* qstart, const double* pstart,
                         const double* dF, double* qhalf, double* Ft, double* yq, double* yp, int* flags)
{
    TinyArgs a{};
    a.n = sys.n; a.ns = sys.ns; a.K = K; a.periodic = sys.periodic;
    for (int c = 0; c < 3; ++c) a.box[c] = sys.box[c];
    a.species = sys.species; a.mass = sys.mass; a.sigma = sys.sigma;
    a.pair = pot.pair; a.pair_rc2 = pot.pair_rc2; a.tether = pot.has_tether ? pot.tether : nullptr;
    a.has_pair = pot.pair_rcmax > 0; a.use_bonded = pot.use_bonded && (sys.n_bonds + sys.n_angles) > 0; a.n_bonds = sys.n_bonds;
    a.bt_start = sys.bt_start; a.bt_term = sys.bt_term; a.bonds = sys.bonds; a.angles = sys.angles;
    a.bond_k = sys.bond_k; a.bond_r0 = sys.bond_r0; a.angle_k = sys.angle_k; a.angle_t0 = sys.angle_t0;
    const MlipDev& m = pot.mlip;
    a.has_net = m.F > 0;
    if (a.has_net) {
        a.rc = m.rc; a.alpha = m.alpha; a.delta = m.rc / (float)(m.R - 1); a.inv_delta2 = 1.f / (a.delta * a.delta); a.inv_rc = 1.f / m.rc;
        a.emb = m.emb; a.ytab0 = m.ytab0; a.Wf1T = m.Wf1T[0]; a.Wf2T = m.Wf2T[0]; a.Wo1T = m.Wo1T[0]; a.Wo2T = m.Wo2T[0];
        a.Wo2 = m.Wo2[0]; a.Wo1 = m.Wo1[0]; a.Wr1 = m.Wr1; a.wr2 = m.wr2;
    }
    a.seed = seed; a.n0_dev = n0_dev; a.c1 = c1; a.b = b; a.hdt = hdt; a.skin_half2 = skin_half2;
    a.qstart = qstart; a.pstart = pstart; a.dF = dF; a.qhalf = qhalf; a.Ft = Ft; a.yq = yq; a.yp = yp; a.flags = flags;
    static bool configured_dev[64] = {};
    bool& configured = configured_dev[lsd_current_device()];
    if (!configured) { cudaFuncSetAttribute(k_tiny_rollout, cudaFuncAttributeMaxDynamicSharedMemorySize, Plan::Bytes); configured = true; }
    const int pid = prof_begin(L, PROF_DRAFT_MLIP);
    k_tiny_rollout<<<kNC, kThreads, Plan::Bytes, L.s>>>(a);     // one cluster (__cluster_dims__)
    LSD_COUNT(L);
    prof_end(L, pid);
}
