// bf16 tcgen05 filter path (LSD_BF16_TC): the continuous-filter convolution of the SchNet-style MLIP (M5, M9)
// with the two per-edge filter contractions on the 5th-generation tensor cores (sm_100a), fp32 accumulation in TMEM.
//
// Orientation ("channels are rows"): for one tile of NT edges
//     D1[F x N] = W_f1[F x R] * G^T[R x N]          G   = radial basis rows (and, backward, their r-derivatives)
//     D2[F x N] = W_f2[F x F] * A^T[F x N]          A   = ssp(D1) (and, backward, logistic(D1) . D1')
// so TMEM lane = channel f = thread, TMEM column = edge.  The per-atom sums over edges (m_a, ybar_a, F_a) are then
// serial sums inside one thread in the order of the atom's sorted neighbour row (deterministic, independent of the
// batch and of the tiling), and the gathers y_j[f], mbar_j[f] are coalesced 128-byte rows per warp.
//
// One persistent CTA per SM, 4 teams of 128 threads.  The weights (A operands, K-major canonical no-swizzle layout,
// packed on the host) are resident in shared memory and shared by the teams; each team owns 128 TMEM columns, one
// B-operand buffer, and walks chunks of kCH consecutive atoms in tiles of 128 MMA columns
// (forward: 128 edges; backward: 64 edges = 64 value + 64 tangent columns).  Per tile and team:
//     geometry + radial basis -> smem (B1, K-major)      | MMA1 (2 x K16)  -> TMEM
//     TMEM -> activation -> smem (B2, MN-major, bf16)    | MMA2 (8 x K16)  -> TMEM (same columns)
//     TMEM -> cutoff, cfconv products, gathers, per-atom accumulation in registers.
// The phases of different teams overlap (MUFU-bound activation of one team with the LSU/FMA-bound epilogue of another).
#include <cuda_bf16.h>
#include <algorithm>
#include "lsd_internal.h"

namespace {

constexpr int kF = 128;                 // channels = MMA M
constexpr int kR = LSD_NRBF;            // 32 = K of the first contraction
constexpr int kTeams = 4;
constexpr int kTT = 128;                // threads per team
constexpr int kThreadsTC = kTeams * kTT;
constexpr int kNCOL = 128;              // MMA N per tile and team
constexpr int kCH = 64;                 // atoms per chunk
constexpr int kW1Bytes = kF * kR * 2;   // 8 KB
constexpr int kW2Bytes = kF * kF * 2;   // 32 KB
constexpr int kB2Bytes = kNCOL * kF * 2;  // 32 KB (B1 aliases its first 8 KB)
constexpr int kEsBytes = 2048;          // per-edge scalars: 64 x 32 B (backward) or 128 x 16 B (forward)
constexpr int kPrefBytes = 272;         // (kCH + 1) ints, padded
constexpr int kFpartBytes = kCH * 4 * 3 * 4;
constexpr int kTeamBytes = kB2Bytes + kEsBytes + kPrefBytes + kFpartBytes;
constexpr int kSmemTC = kW1Bytes + kW2Bytes + kTeams * kTeamBytes;
static_assert(kSmemTC <= 227 * 1024, "shared memory budget");
static_assert(kTeamBytes % 16 == 0, "team regions stay 16-byte aligned");

constexpr float kLn2 = 0.69314718055994530942f;
constexpr float kLog2e = 1.44269504088896340736f;

struct __align__(16) EdgeB { float fc, fcp, ux, uy, uz; int jrow, arow, pad; };   // backward, 32 B
struct __align__(16) EdgeF { float fc; int jrow, arow, pad; };                    // forward, 16 B

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ float ex2f(float x) { float y; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float lg2f(float x) { float y; asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float rcpf(float x) { float y; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ uint32_t pack_bf16(float lo, float hi)
{
    __nv_bfloat162 v = __floats2bfloat162_rn(lo, hi);
    return *reinterpret_cast<uint32_t*>(&v);
}
__device__ __forceinline__ void img_unpack(int v, int& ix, int& iy, int& iz) { ix = (v & 1023) - 512; iy = ((v >> 10) & 1023) - 512; iz = ((v >> 20) & 1023) - 512; }

// shared-memory matrix descriptor, canonical layout without swizzle (8 x 16-byte core matrices):
// start address, leading-dimension byte offset, stride-dimension byte offset (all >> 4), descriptor version 1.
__device__ __forceinline__ uint64_t make_desc(uint32_t saddr, uint32_t lbo, uint32_t sbo)
{
    uint64_t d = 0;
    d |= (uint64_t)((saddr >> 4) & 0x3FFF);
    d |= (uint64_t)((lbo >> 4) & 0x3FFF) << 16;
    d |= (uint64_t)((sbo >> 4) & 0x3FFF) << 32;
    d |= (uint64_t)1 << 46;
    return d;
}
// instruction descriptor, kind::f16: D = fp32, A = B = bf16, A K-major, B K-major or MN-major, M x N
__device__ __forceinline__ uint32_t make_idesc(int M, int N, int b_mn_major)
{
    uint32_t d = 0;
    d |= 1u << 4;
    d |= 1u << 7;
    d |= 1u << 10;
    d |= (uint32_t)(b_mn_major ? 1 : 0) << 16;
    d |= (uint32_t)(N >> 3) << 17;
    d |= (uint32_t)(M >> 4) << 24;
    return d;
}
__device__ __forceinline__ void umma(uint32_t tmem_d, uint64_t da, uint64_t db, uint32_t idesc, uint32_t accumulate)
{
    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                 "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}" ::"r"(tmem_d), "l"(da), "l"(db), "r"(idesc), "r"(accumulate) : "memory");
}
__device__ __forceinline__ void umma_commit(uint32_t bar) { asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory"); }
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity)
{
    uint32_t ok = 0;
    while (!ok) {
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    }
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void fence_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void team_bar(int team) { asm volatile("bar.sync %0, %1;" ::"r"(team + 1), "n"(kTT) : "memory"); }
__device__ __forceinline__ void tmem_ld16(uint32_t taddr, uint32_t (&v)[16])
{
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
                 : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]), "=r"(v[8]), "=r"(v[9]),
                   "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15])
                 : "r"(taddr) : "memory");
}
__device__ __forceinline__ void tmem_ld8(uint32_t taddr, uint32_t (&v)[8])
{
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                 : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7])
                 : "r"(taddr) : "memory");
}
__device__ __forceinline__ void tmem_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }

// geometry of one directed edge (slot of atom row g), identical arithmetic to the fp32 kernel: fp64 displacement -> fp32
struct EdgeGeom { float r, fc, fcp, ux, uy, uz; int jrow; };
__device__ __forceinline__ EdgeGeom edge_geometry(const EdgeArgs& a, int g, int slot)
{
    const int n = a.n, b = g / n, i = g - b * n;
    const double* qb = a.q + (size_t)b * 3 * n;
    const uint32_t key = a.keys[(size_t)g * a.cap + slot];
    const int j = (int)(key >> 5), code = (int)(key & 31u);
    int iix, iiy, iiz, jx, jy, jz;
    img_unpack(a.img[i], iix, iiy, iiz);
    img_unpack(a.img[j], jx, jy, jz);
    const double d0 = (qb[j] - qb[i]) + (double)(code / 9 - 1 + iix - jx) * a.box[0];
    const double d1 = (qb[n + j] - qb[n + i]) + (double)((code / 3) % 3 - 1 + iiy - jy) * a.box[1];
    const double d2 = (qb[2 * n + j] - qb[2 * n + i]) + (double)(code % 3 - 1 + iiz - jz) * a.box[2];
    const double rd = sqrt(d0 * d0 + d1 * d1 + d2 * d2);
    EdgeGeom o;
    o.r = (float)rd; o.ux = (float)(d0 / rd); o.uy = (float)(d1 / rd); o.uz = (float)(d2 / rd);
    o.fc = 0.f; o.fcp = 0.f;
    const float t = o.r * a.inv_rc;
    if (t < 1.f) {                                                                        // M2
        float sn, cs; sincospif(t, &sn, &cs);
        o.fc = 0.5f * (cs + 1.f); o.fcp = -0.5f * 3.14159265358979323846f * a.inv_rc * sn;
    }
    o.jrow = b * n + j;
    return o;
}

template <bool BWD>
__global__ void __launch_bounds__(kThreadsTC, 1)
k_edge_tc(EdgeArgs a, int nchunks)
{
    constexpr int NT = BWD ? 64 : 128;                 // edges per tile
    extern __shared__ __align__(1024) uint8_t smem[];
    __shared__ __align__(8) uint64_t mbar[kTeams];
    __shared__ uint32_t tmem_base_s;
    __shared__ int next_chunk, s_chunk[kTeams];
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31, team = tid >> 7, tt = tid & (kTT - 1);

    {   // resident A operands (already in the canonical K-major layout)
        const uint4* s1 = reinterpret_cast<const uint4*>(a.Wf1_tc);
        const uint4* s2 = reinterpret_cast<const uint4*>(a.Wf2_tc);
        uint4* d1 = reinterpret_cast<uint4*>(smem);
        uint4* d2 = reinterpret_cast<uint4*>(smem + kW1Bytes);
        for (int i = tid; i < kW1Bytes / 16; i += kThreadsTC) d1[i] = s1[i];
        for (int i = tid; i < kW2Bytes / 16; i += kThreadsTC) d2[i] = s2[i];
    }
    if (tid == 0) {
        for (int t = 0; t < kTeams; ++t) asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(smem_u32(&mbar[t])));
        asm volatile("fence.mbarrier_init.release.cluster;");
        next_chunk = 0;
    }
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&tmem_base_s)), "n"(512));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
    }
    fence_async_smem();
    tc_fence_before();
    __syncthreads();
    tc_fence_after();

    uint8_t* const tb = smem + kW1Bytes + kW2Bytes + team * kTeamBytes;
    uint8_t* const Bop = tb;                                           // B2 [128 cols][128 k] MN-major; B1 aliases its head
    EdgeB* const esb = reinterpret_cast<EdgeB*>(tb + kB2Bytes);
    EdgeF* const esf = reinterpret_cast<EdgeF*>(tb + kB2Bytes);
    int* const pref = reinterpret_cast<int*>(tb + kB2Bytes + kEsBytes);
    float* const fpart = reinterpret_cast<float*>(tb + kB2Bytes + kEsBytes + kPrefBytes);
    const uint32_t sW1 = smem_u32(smem), sW2 = smem_u32(smem + kW1Bytes), sB = smem_u32(Bop), bar = smem_u32(&mbar[team]);
    const uint32_t tmem = tmem_base_s + (uint32_t)(team * kNCOL);
    const uint32_t tlane = tmem + ((uint32_t)((warp & 3) * 32) << 16);
    const uint32_t idesc1 = make_idesc(kF, kNCOL, 0), idesc2 = make_idesc(kF, kNCOL, 1);
    uint32_t phase = 0;
    const int n = a.n;

    for (;;) {
        if (tt == 0) s_chunk[team] = atomicAdd(&next_chunk, 1);
        team_bar(team);
        const int chunk = blockIdx.x + s_chunk[team] * gridDim.x;
        if (chunk >= nchunks) break;
        const int g0 = chunk * kCH;
        if (tt < kCH) pref[tt + 1] = (g0 + tt < a.total) ? a.count[g0 + tt] : 0;
        team_bar(team);
        if (tt == 0) { int s = 0; pref[0] = 0; for (int i = 1; i <= kCH; ++i) { s += pref[i]; pref[i] = s; } }
        team_bar(team);
        const int E = pref[kCH];
        {   // atoms without neighbours: their sums are empty
            float* out = BWD ? a.ybar : a.m_out;
            if (out) for (int i = 0; i < kCH; ++i) if (g0 + i < a.total && pref[i + 1] == pref[i]) out[(size_t)(g0 + i) * kF + tt] = 0.f;
        }
        int cur = -1;
        float part = 0.f, ya = 0.f, mba = 0.f, fx = 0.f, fy = 0.f, fz = 0.f;
        auto flush = [&]() {
            if (cur < 0) return;
            if (!BWD) a.m_out[(size_t)cur * kF + tt] = part;
            else {
                if (a.ybar) a.ybar[(size_t)cur * kF + tt] = part;
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) {
                    fx += __shfl_xor_sync(0xffffffffu, fx, o); fy += __shfl_xor_sync(0xffffffffu, fy, o); fz += __shfl_xor_sync(0xffffffffu, fz, o);
                }
                if (lane == 0) { float* fp = fpart + ((cur - g0) * 4 + (warp & 3)) * 3; fp[0] = fx; fp[1] = fy; fp[2] = fz; }
            }
        };

        for (int base = 0; base < E; base += NT) {
            // ---- phase 1: geometry and radial basis rows (M1) -> B1, K-major: (n, k) at (n/8)*512 + (k/8)*128 + (n%8)*16 + (k%8)*2
            {
                const int col = BWD ? (tt & 63) : tt;
                const bool tang = BWD && tt >= 64;
                const int e = base + col;
                uint32_t gp[16];
#pragma unroll
                for (int k = 0; k < 16; ++k) gp[k] = 0u;
                if (e < E) {
                    int lo = 0, hi = kCH;
                    while (hi - lo > 1) { const int mid = (lo + hi) >> 1; if (pref[mid] <= e) lo = mid; else hi = mid; }
                    const int g = g0 + lo;
                    const EdgeGeom ge = edge_geometry(a, g, e - pref[lo]);
                    if (!tang) {
                        if (BWD) { EdgeB s; s.fc = ge.fc; s.fcp = ge.fcp; s.ux = ge.ux; s.uy = ge.uy; s.uz = ge.uz; s.jrow = ge.jrow; s.arow = g; s.pad = 0; esb[col] = s; }
                        else { EdgeF s; s.fc = ge.fc; s.jrow = ge.jrow; s.arow = g; s.pad = 0; esf[col] = s; }
                    }
                    const float c2 = -0.5f * kLog2e * a.inv_delta2;
#pragma unroll
                    for (int k = 0; k < kR; k += 2) {
                        const float x0 = ge.r - (float)k * a.delta, x1 = ge.r - (float)(k + 1) * a.delta;
                        float v0 = ex2f(c2 * x0 * x0), v1 = ex2f(c2 * x1 * x1);
                        if (tang) { v0 = -v0 * x0 * a.inv_delta2; v1 = -v1 * x1 * a.inv_delta2; }
                        gp[k >> 1] = pack_bf16(v0, v1);
                    }
                }
                const int row = tang ? NT + col : col;
                uint8_t* dst = Bop + (row >> 3) * 512 + (row & 7) * 16;
#pragma unroll
                for (int kc = 0; kc < 4; ++kc) *reinterpret_cast<uint4*>(dst + kc * 128) = make_uint4(gp[4 * kc], gp[4 * kc + 1], gp[4 * kc + 2], gp[4 * kc + 3]);
            }
            fence_async_smem();
            team_bar(team);
            if (tt == 0) {
                tc_fence_after();
#pragma unroll
                for (int k16 = 0; k16 < kR / 16; ++k16)
                    umma(tmem, make_desc(sW1 + k16 * 256, 128, (kR / 8) * 128), make_desc(sB + k16 * 256, 128, (kR / 8) * 128), idesc1, k16 > 0);
                umma_commit(bar);
            }
            mbar_wait(bar, phase); phase ^= 1u;
            tc_fence_after();
            const int nval = min(NT, E - base);
            // ---- phase 2: activation (M3) -> B2, MN-major: (n, k) at (n/8)*2048 + (k/8)*128 + (k%8)*16 + (n%8)*2, k = this thread's channel
            for (int c0 = 0; c0 < nval; c0 += 16) {
                uint32_t v[16], vp[16];
                tmem_ld16(tlane + c0, v);
                if (BWD) tmem_ld16(tlane + NT + c0, vp);
                tmem_wait_ld();
                uint32_t pa[8], pt[8];
#pragma unroll
                for (int c = 0; c < 16; c += 2) {
                    float s[2], d[2];
#pragma unroll
                    for (int h = 0; h < 2; ++h) {
                        const float x = __uint_as_float(v[c + h]);
                        const float t = ex2f(-fabsf(x) * kLog2e);
                        const float l = lg2f(1.f + t);
                        s[h] = fmaf(kLn2, l, fmaxf(x, 0.f)) - kLn2;
                        if (BWD) {
                            const float rr = rcpf(1.f + t);
                            const float sig = x >= 0.f ? rr : t * rr;
                            d[h] = sig * __uint_as_float(vp[c + h]);
                        }
                    }
                    pa[c >> 1] = pack_bf16(s[0], s[1]);
                    if (BWD) pt[c >> 1] = pack_bf16(d[0], d[1]);
                }
                uint8_t* d0 = Bop + (c0 >> 3) * 2048 + tt * 16;
                *reinterpret_cast<uint4*>(d0) = make_uint4(pa[0], pa[1], pa[2], pa[3]);
                *reinterpret_cast<uint4*>(d0 + 2048) = make_uint4(pa[4], pa[5], pa[6], pa[7]);
                if (BWD) {
                    uint8_t* d1 = Bop + ((NT + c0) >> 3) * 2048 + tt * 16;
                    *reinterpret_cast<uint4*>(d1) = make_uint4(pt[0], pt[1], pt[2], pt[3]);
                    *reinterpret_cast<uint4*>(d1 + 2048) = make_uint4(pt[4], pt[5], pt[6], pt[7]);
                }
            }
            tc_fence_before();
            fence_async_smem();
            team_bar(team);
            if (tt == 0) {
                tc_fence_after();
#pragma unroll
                for (int k16 = 0; k16 < kF / 16; ++k16)
                    umma(tmem, make_desc(sW2 + k16 * 256, 128, (kF / 8) * 128), make_desc(sB + k16 * 256, 128, (kF / 8) * 128), idesc2, k16 > 0);
                umma_commit(bar);
            }
            mbar_wait(bar, phase); phase ^= 1u;
            tc_fence_after();
            // ---- phase 3: cutoff, cfconv products and their adjoints; per-atom sums stay in this thread's registers
            for (int c0 = 0; c0 < nval; c0 += 8) {
                uint32_t v[8], vp[8];
                tmem_ld8(tlane + c0, v);
                if (BWD) tmem_ld8(tlane + NT + c0, vp);
                tmem_wait_ld();
#pragma unroll
                for (int c = 0; c < 8; ++c) {
                    if (c0 + c < nval) {
                        if (!BWD) {
                            const EdgeF s = esf[c0 + c];
                            if (s.arow != cur) { flush(); cur = s.arow; part = 0.f; }
                            const float yj = a.y[(size_t)s.jrow * kF + tt];
                            part = fmaf(yj, __uint_as_float(v[c]) * s.fc, part);
                        } else {
                            const EdgeB s = esb[c0 + c];
                            if (s.arow != cur) {
                                flush(); cur = s.arow; part = 0.f; fx = fy = fz = 0.f;
                                ya = a.y[(size_t)cur * kF + tt]; mba = a.mbar[(size_t)cur * kF + tt];
                            }
                            const float yj = a.y[(size_t)s.jrow * kF + tt], mbj = a.mbar[(size_t)s.jrow * kF + tt];
                            const float lin = __uint_as_float(v[c]), linp = __uint_as_float(vp[c]);
                            const float w = lin * s.fc, wp = fmaf(linp, s.fc, lin * s.fcp);
                            part = fmaf(mbj, w, part);
                            const float gq = fmaf(mba, yj, mbj * ya) * wp;
                            fx = fmaf(gq, s.ux, fx); fy = fmaf(gq, s.uy, fy); fz = fmaf(gq, s.uz, fz);
                        }
                    }
                }
            }
            tc_fence_before();
            team_bar(team);
        }
        flush();
        if (BWD) {
            team_bar(team);
            if (tt < kCH && pref[tt + 1] > pref[tt]) {
                const int g = g0 + tt, b = g / n, i = g - b * n;
                const float* fp = fpart + tt * 12;
                double* Fb = a.Fout + (size_t)b * 3 * n;
                Fb[i] += (((double)fp[0] + (double)fp[3]) + (double)fp[6]) + (double)fp[9];
                Fb[n + i] += (((double)fp[1] + (double)fp[4]) + (double)fp[7]) + (double)fp[10];
                Fb[2 * n + i] += (((double)fp[2] + (double)fp[5]) + (double)fp[8]) + (double)fp[11];
            }
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base_s), "n"(512));
}

int tc_num_sms()
{
    static int sms = 0;
    if (!sms) { int dev = 0; cudaGetDevice(&dev); cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev); if (sms <= 0) sms = 148; }
    return sms;
}

uint16_t bf16_rne(double x)
{
    float f = (float)x;
    uint32_t u; memcpy(&u, &f, 4);
    if ((u & 0x7F800000u) == 0x7F800000u) return (uint16_t)(u >> 16);
    u += 0x7FFFu + ((u >> 16) & 1u);
    return (uint16_t)(u >> 16);
}

}  // namespace

bool mlip_tc_supported(const MlipDev& net) { return net.F == kF && net.R == kR; }

// A operands: (m, k) at byte (m/8)*SBO + (k/8)*128 + (m%8)*16 + (k%8)*2, SBO = (K/8)*128
void tc_pack_weights(const double* Wf1, const double* Wf2, int F, int R, std::vector<uint16_t>& out1, std::vector<uint16_t>& out2)
{
    out1.assign((size_t)F * R, 0); out2.assign((size_t)F * F, 0);
    for (int m = 0; m < F; ++m)
        for (int k = 0; k < R; ++k)
            out1[((size_t)(m / 8) * (R / 8) * 128 + (k / 8) * 128 + (m % 8) * 16 + (k % 8) * 2) / 2] = bf16_rne(Wf1[(size_t)m * R + k]);
    for (int m = 0; m < F; ++m)
        for (int k = 0; k < F; ++k)
            out2[((size_t)(m / 8) * (F / 8) * 128 + (k / 8) * 128 + (m % 8) * 16 + (k % 8) * 2) / 2] = bf16_rne(Wf2[(size_t)m * F + k]);
}

void launch_edge_tc(Launcher L, const EdgeArgs& a, bool backward)
{
    static bool configured = false;
    if (!configured) {
        cudaFuncSetAttribute(k_edge_tc<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemTC);
        cudaFuncSetAttribute(k_edge_tc<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemTC);
        configured = true;
    }
    const int nchunks = (a.total + kCH - 1) / kCH;
    const int grid = std::max(1, std::min(tc_num_sms(), nchunks));
    if (backward) k_edge_tc<true><<<grid, kThreadsTC, kSmemTC, L.s>>>(a, nchunks);
    else k_edge_tc<false><<<grid, kThreadsTC, kSmemTC, L.s>>>(a, nchunks);
    LSD_COUNT(L);
}
