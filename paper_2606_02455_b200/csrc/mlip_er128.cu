// bf16 tcgen05 filter path for width F = 128, "edges are rows" schedule (M5, M9).
//
// Every contraction of a tile of 128 directed edges has the edges on the 128 accumulator rows, so a thread owns ONE edge
// (TMEM lane = edge = thread) and walks along its 128 channels:
//   D  = G  W_f1^T      G  [128 e x 32]  radial basis of the thread's edge          (A operand, K-major, written by the thread)
//   D  = A2 W_f2^T      A2 [128 e x 128] = ssp(D)  (packed pairs of adjacent channels; D is overwritten)
//   D3 = P^T S^T        P  [128 e x 128] = bf16(w fc) . y_j   (A operand, MN-major: the thread writes 8 channels = 16 bytes)
//                       S^T[128 e x 16]  = 1 where edge e belongs to atom a of the chunk (B operand)
// The sum over the edges of an atom -- a sum ACROSS threads in this orientation -- is the third contraction: the tensor
// core adds the rows of P into D3[channel][atom], in fp32, in a fixed order.  Per element the thread issues no shared-
// memory gather, no bf16 unpack and no per-edge broadcast: the row y_j is loaded straight from L2 as 16-byte pieces and
// multiplied as packed bf16x2.  A chunk is 16 atoms (one D3 tile of 16 columns, accumulated in TMEM over the chunk's
// tiles); 3 teams of 128 threads per SM, each with 128 + 16 TMEM columns (D1 and D2 share theirs) and one MMA-issuing warp.
// Measured alternatives (profiles/r1_edge_er128_fwd_cfg5.md): 2 teams with separate D1 / D2 (GEMM1 of tile t+1 under the
// epilogue of tile t) and 2 teams x 2 threads per edge were both slower; the binding units are all within a factor two of
// each other (MUFU 1280, shared-memory traffic ~1500, tensor ~700, issue ~1200 cycles per tile and SM).
#include <algorithm>
#include "lsd_internal.h"
#include "tc_ptx.cuh"

namespace {
using namespace tcp;

constexpr int kF = 128;
constexpr int kR = LSD_NRBF;
constexpr int kTeams = 3;
constexpr int kTT = 128;                               // edges of a tile
constexpr int kSplit = 1;                              // threads per edge (2: each owns 64 of the 128 channels; measured slower)
constexpr int kTeamThreads = kTT * kSplit;
constexpr int kThreads = kTeams * kTeamThreads + kTeams * 32;
constexpr int kCH = 16;                                // atoms per chunk = columns of D3
constexpr int kGE = 16;                                // edge slots per record group
constexpr int kGPT = kTT / kGE;                        // groups per tile
constexpr int kMaxGroups = kCH * (512 / kGE);
constexpr int kW1Bytes = kF * kR * 2, kW2Bytes = kF * kF * 2;
constexpr int kA1Bytes = kTT * kR * 2, kA2Bytes = kTT * kF * 2, kSTBytes = kCH * kTT * 2;
constexpr int kTeamBytes = kA1Bytes + kA2Bytes + kSTBytes + kMaxGroups + 128;
constexpr int kSmem = kW1Bytes + kW2Bytes + kTeams * kTeamBytes;
constexpr int kBars = 6;                               // per team: GEMM1 / GEMM2 / GEMM3 complete, A1 / A2 / P published
static_assert(kSmem + 1024 <= 227 * 1024, "shared memory budget");
static_assert(kTeamBytes % 16 == 0, "regions stay 16-byte aligned");

constexpr float kLog2e = 1.44269504088896340736f;
// -ln(1 + a) / (2 a) on [0, 1] (weighted minimax fit of a P(a), |error| < 3.6e-5)
constexpr float kP0 = -0.49872449040412903f, kP1 = 0.2356506735086441f, kP2 = -0.11284290254116058f, kP3 = 0.02937859483063221f;

__device__ __forceinline__ void team_bar(int team) { asm volatile("bar.sync %0, %1;" ::"r"(team + 1), "n"(kTeamThreads) : "memory"); }
__device__ __forceinline__ void tmem_ld32(uint32_t taddr, uint32_t (&v)[32])
{
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x32.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,"
                 "%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31}, [%32];"
                 : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]), "=r"(v[8]), "=r"(v[9]),
                   "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15]), "=r"(v[16]), "=r"(v[17]), "=r"(v[18]),
                   "=r"(v[19]), "=r"(v[20]), "=r"(v[21]), "=r"(v[22]), "=r"(v[23]), "=r"(v[24]), "=r"(v[25]), "=r"(v[26]), "=r"(v[27]),
                   "=r"(v[28]), "=r"(v[29]), "=r"(v[30]), "=r"(v[31])
                 : "r"(taddr) : "memory");
}
__device__ __forceinline__ uint32_t hmul2_bf16(uint32_t a, uint32_t b)
{
    uint32_t r;
    asm("mul.rn.bf16x2 %0, %1, %2;" : "=r"(r) : "r"(a), "r"(b));
    return r;
}
// instruction descriptor, kind::f16, D = fp32, A = B = bf16, M = 128, chosen major-ness of A and B
__device__ __forceinline__ uint32_t make_idesc2(int N, int a_mn_major, int b_mn_major)
{
    return make_idesc(128, N, b_mn_major) | ((uint32_t)(a_mn_major ? 1 : 0) << 15);
}

__global__ void __launch_bounds__(kThreads, 1)
k_edge_er128_fwd(EdgeArgs a, int chunks_per_state, int nchunks)
{
    extern __shared__ __align__(128) uint8_t smem[];
    __shared__ __align__(8) uint64_t mbar[kBars * kTeams];
    __shared__ uint32_t tmem_base_s;
    __shared__ volatile int s_nt[kTeams];
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;

    {   // resident B operand images (K-major): W_f1 / 2 [128 x 32], 2 W_f2 [128 x 128]; every other buffer starts as zeros
        const uint4* s1 = reinterpret_cast<const uint4*>(a.Wf1_tc);
        const uint4* s2 = reinterpret_cast<const uint4*>(a.Wf2_tc);
        uint4* d1 = reinterpret_cast<uint4*>(smem);
        uint4* d2 = reinterpret_cast<uint4*>(smem + kW1Bytes);
        for (int i = tid; i < kW1Bytes / 16; i += kThreads) d1[i] = s1[i];
        for (int i = tid; i < kW2Bytes / 16; i += kThreads) d2[i] = s2[i];
        uint4* z = reinterpret_cast<uint4*>(smem + kW1Bytes + kW2Bytes);
        for (int i = tid; i < kTeams * kTeamBytes / 16; i += kThreads) z[i] = make_uint4(0u, 0u, 0u, 0u);
    }
    if (tid == 0) {
        for (int t = 0; t < kTeams; ++t) {
            for (int b = 0; b < 3; ++b) mbar_init(smem_u32(&mbar[kBars * t + b]), 1);
            for (int b = 3; b < kBars; ++b) mbar_init(smem_u32(&mbar[kBars * t + b]), kTeamThreads / 32);   // one arrival per warp
        }
        asm volatile("fence.mbarrier_init.release.cluster;");
    }
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&tmem_base_s)), "n"(512));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
    }
    fence_async_smem();
    tc_fence_before();
    __syncthreads();
    tc_fence_after();

    constexpr int kTeamWarps = kTeamThreads / 32;
    const int team = warp >= kTeams * kTeamWarps ? warp - kTeams * kTeamWarps : warp / kTeamWarps;
    uint8_t* const tb = smem + kW1Bytes + kW2Bytes + team * kTeamBytes;
    const uint32_t sW1 = smem_u32(smem), sW2 = sW1 + kW1Bytes;
    const uint32_t sA1 = smem_u32(tb), sA2 = sA1 + kA1Bytes, sP = sA2, sST = sP + kA2Bytes;   // P re-uses A2's buffer
    const uint32_t bar1 = smem_u32(&mbar[kBars * team]), bar2 = bar1 + 8, bar3 = bar1 + 16, rdyA1 = bar1 + 24, rdyA2 = bar1 + 32, rdyP = bar1 + 40;
    const uint32_t tD1 = tmem_base_s + (uint32_t)(team * 160), tD2 = tD1, tD3 = tD1 + 128;   // D1 and D2 share their columns

    if (warp >= kTeams * kTeamWarps) {
        // ---- MMA warp of the team
        if (lane == 0) {
            const uint32_t id12 = make_idesc2(128, 0, 0), id3 = make_idesc2(kCH, 1, 0);
            uint32_t ph = 0;
            for (;;) {
                mbar_wait(rdyA1, ph);
                const int nt = s_nt[team];
                if (nt < 0) break;
                for (int t = 0; t < nt; ++t) {
                    if (t > 0) mbar_wait(rdyA1, ph);
                    tc_fence_after();
#pragma unroll
                    for (int k16 = 0; k16 < kR / 16; ++k16)
                        umma(tD1, make_desc(sA1 + k16 * 256, 128, 512), make_desc(sW1 + k16 * 256, 128, 512), id12, k16 > 0);
                    umma_commit(bar1);
                    mbar_wait(rdyA2, ph);
                    tc_fence_after();
#pragma unroll
                    for (int k16 = 0; k16 < kF / 16; ++k16)
                        umma(tD2, make_desc(sA2 + k16 * 256, 128, 2048), make_desc(sW2 + k16 * 256, 128, 2048), id12, k16 > 0);
                    umma_commit(bar2);
                    mbar_wait(rdyP, ph);
                    tc_fence_after();
#pragma unroll
                    for (int k16 = 0; k16 < kTT / 16; ++k16)
                        umma(tD3, make_desc(sP + k16 * 256, 128, 2048), make_desc(sST + k16 * 256, 128, 2048), id3, (t > 0 || k16 > 0) ? 1u : 0u);
                    umma_commit(bar3);
                    ph ^= 1u;
                }
            }
        }
    } else {
        const int e = tid & (kTT - 1), wq = warp & 3, half = (tid / kTT) % kSplit;   // warp % 4 selects the TMEM lane quarter
        uint8_t* const A1 = tb;
        uint8_t* const A2 = A1 + kA1Bytes;
        uint8_t* const Pb = A2;
        uint8_t* const ST = A2 + kA2Bytes;
        uint8_t* const gatom = ST + kSTBytes;                                     // group -> atom of the chunk
        int* const pref = reinterpret_cast<int*>(gatom + kMaxGroups);             // first group of every atom (17 entries)
        const uint32_t tl1 = tD1 + ((uint32_t)(wq * 32) << 16), tl2 = tD2 + ((uint32_t)(wq * 32) << 16), tl3 = tD3 + ((uint32_t)(wq * 32) << 16);
        const int n = a.n;
        const float c2 = -0.5f * kLog2e * a.inv_delta2;
        const int my_g = e >> 4, my_s = e & 15;
        uint8_t* const a1row = A1 + (e >> 3) * 512 + (e & 7) * 16;
        uint8_t* const a2row = A2 + (e >> 3) * 2048 + (e & 7) * 16;
        uint8_t* const prow = Pb + e * 16;
        uint32_t ph = 0;

        for (int chunk = blockIdx.x * kTeams + team; chunk < nchunks; chunk += gridDim.x * kTeams) {
            const int b = chunk / chunks_per_state, ci = chunk - b * chunks_per_state;
            const int g0 = b * n + ci * kCH;                                       // first feature row of the chunk
            const int natoms = min(kCH, n - ci * kCH);
            if (e < 32 && half == 0) {                                            // groups per atom, exclusive scan over the 16 atoms
                const int c = e < natoms ? a.count[g0 + e] : 0;
                int v = (c + kGE - 1) / kGE;
#pragma unroll
                for (int o = 1; o < 16; o <<= 1) { const int u = __shfl_up_sync(0xffffffffu, v, o); if (e >= o) v += u; }
                if (e < kCH) pref[e + 1] = v;
                if (e == 0) pref[0] = 0;
            }
            team_bar(team);
            const int G = pref[kCH];
            if (e < kCH && half == 0) for (int g = pref[e]; g < pref[e + 1]; ++g) gatom[g] = (uint8_t)e;
            const int ntiles = (G + kGPT - 1) / kGPT;
            if (ntiles == 0) {                                                     // no edges at all: empty sums
                if (half == 0) for (int i = 0; i < natoms; ++i) a.m16_out[(size_t)(g0 + i) * kF + e] = 0;
                team_bar(team);
                continue;
            }
            if (e == 0 && half == 0) s_nt[team] = ntiles;
            team_bar(team);

            // record fields of this thread's edge slot in tile t (zero record behind the chunk's last group)
            float r_n, fc_n; int jrow_n, at_n;
            auto load_record = [&](int t) {
                const int gl = t * kGPT + my_g;
                r_n = 0.f; fc_n = 0.f; jrow_n = g0; at_n = -1;
                if (gl < G) {
                    at_n = gatom[gl];
                    const float* rp = a.recs + lsd_rec_index((size_t)(g0 + at_n), a.cap, (gl - pref[at_n]) * kGE + my_s, 0);
                    r_n = rp[LSD_REC_R * 16]; fc_n = rp[LSD_REC_FC * 16]; jrow_n = __float_as_int(rp[LSD_REC_JROW * 16]);
                }
            };
            // radial basis (M1) of the thread's edge -> its row of A1
            auto stage_basis = [&](float r) {
                constexpr int KH = kR / kSplit;                                    // basis functions per thread
                uint32_t gv[KH / 2];
                const f32x2 c22 = pk2(c2, c2);
                const float rh = r - (float)(half * KH) * a.delta;
#pragma unroll
                for (int k = 0; k < KH; k += 2) {
                    const float x0 = rh - (float)k * a.delta, x1 = x0 - a.delta;
                    const f32x2 x2 = pk2(x0, x1);
                    float e0, e1;
                    un2(mul2(mul2(x2, x2), c22), e0, e1);
                    gv[k >> 1] = pack_bf16(ex2f(e0), ex2f(e1));
                }
#pragma unroll
                for (int kc = 0; kc < KH / 8; ++kc) *reinterpret_cast<uint4*>(a1row + (half * (KH / 8) + kc) * 128) = make_uint4(gv[4 * kc], gv[4 * kc + 1], gv[4 * kc + 2], gv[4 * kc + 3]);
                fence_async_smem();
                warp_arrive(rdyA1, lane);
            };

            load_record(0);
            stage_basis(r_n);
            int at_prev = -1;
            constexpr int AH = kCH / kSplit;                                       // atoms whose sums this thread reads (its channel = e)
            for (int t = 0; t < ntiles; ++t) {
                const float fc = fc_n; const int jrow = jrow_n, at = at_n;
                const uint4* yrow = reinterpret_cast<const uint4*>(a.y16 + (size_t)jrow * kF);
                constexpr int QPT = 4 / kSplit;                                    // 32-channel quarters per thread
                const uint4* ymine = yrow + half * (QPT * 4);
                uint4 y[8];                                                        // first two quarters of this thread's part of y_j (land under the activation)
#pragma unroll
                for (int i = 0; i < 8; ++i) y[i] = __ldg(ymine + i);
                if (t + 1 < ntiles) load_record(t + 1);
                // ---- activation (M3): D1 -> A2, K-major row of this edge
                mbar_wait(bar1, ph);                                               // implies GEMM3 of tile t-1: P's buffer and the S^T entry are free
                tc_fence_after();
                if (at_prev >= 0 && half == 0) *reinterpret_cast<uint16_t*>(ST + (at_prev >> 3) * 2048 + (e >> 3) * 128 + (at_prev & 7) * 16 + (e & 7) * 2) = 0;
                const f32x2 p3 = pk2(kP3, kP3), p2 = pk2(kP2, kP2), p1 = pk2(kP1, kP1), p0 = pk2(kP0, kP0);
                uint32_t v[32];
#pragma unroll
                for (int qq = 0; qq < QPT; ++qq) {
                    const int q = half * QPT + qq;
                    tmem_ld32(tl1 + q * 32, v);
                    tmem_wait_ld();
                    uint32_t pa[16];
#pragma unroll
                    for (int c = 0; c < 32; c += 2) {
                        // W_f1 is packed as W_f1 / 2 and W_f2 as 2 W_f2 (exact in bf16): the accumulator holds x / 2 and the
                        // operand written here is ssp(x) / 2 = max(x/2, 0) + a P(a), a = tanh(|x| / 2)
                        const float h0 = __uint_as_float(v[c]), h1 = __uint_as_float(v[c + 1]);
                        const f32x2 a2 = pk2(tanhf_approx(fabsf(h0)), tanhf_approx(fabsf(h1)));
                        f32x2 r2 = fma2(p3, a2, p2);
                        r2 = fma2(r2, a2, p1);
                        r2 = fma2(r2, a2, p0);
                        pa[c >> 1] = pack_bf16(fma2(r2, a2, pk2(fmaxf(h0, 0.f), fmaxf(h1, 0.f))));
                    }
#pragma unroll
                    for (int kc = 0; kc < 4; ++kc)
                        *reinterpret_cast<uint4*>(a2row + (q * 4 + kc) * 128) = make_uint4(pa[4 * kc], pa[4 * kc + 1], pa[4 * kc + 2], pa[4 * kc + 3]);
                }
                tc_fence_before();
                fence_async_smem();
                warp_arrive(rdyA2, lane);
                // ---- radial basis of tile t+1 while GEMM2 runs (A1 is free: GEMM1 of tile t is complete)
                if (t + 1 < ntiles) stage_basis(r_n);
                // ---- epilogue: P = bf16(w fc) . y_j, MN-major (8 channels of this edge = 16 bytes)
                mbar_wait(bar2, ph);
                tc_fence_after();
                const f32x2 fc2 = pk2(fc, fc);
#pragma unroll
                for (int qq = 0; qq < QPT; ++qq) {
                    const int q = half * QPT + qq;
                    tmem_ld32(tl2 + q * 32, v);
                    tmem_wait_ld();
                    uint4 o[4];
#pragma unroll
                    for (int kc = 0; kc < 4; ++kc) {
                        const uint4 yy = y[(qq & 1) * 4 + kc];
                        o[kc].x = hmul2_bf16(pack_bf16(mul2(pk2u(v[8 * kc], v[8 * kc + 1]), fc2)), yy.x);
                        o[kc].y = hmul2_bf16(pack_bf16(mul2(pk2u(v[8 * kc + 2], v[8 * kc + 3]), fc2)), yy.y);
                        o[kc].z = hmul2_bf16(pack_bf16(mul2(pk2u(v[8 * kc + 4], v[8 * kc + 5]), fc2)), yy.z);
                        o[kc].w = hmul2_bf16(pack_bf16(mul2(pk2u(v[8 * kc + 6], v[8 * kc + 7]), fc2)), yy.w);
                    }
                    if (qq + 2 < QPT) {                                            // the quarter after next, two quarters ahead of its use
#pragma unroll
                        for (int kc = 0; kc < 4; ++kc) y[(qq & 1) * 4 + kc] = __ldg(ymine + 8 + qq * 4 + kc);
                    }
#pragma unroll
                    for (int kc = 0; kc < 4; ++kc) *reinterpret_cast<uint4*>(prow + (q * 4 + kc) * 2048) = o[kc];
                }
                if (at >= 0 && half == 0) *reinterpret_cast<uint16_t*>(ST + (at >> 3) * 2048 + (e >> 3) * 128 + (at & 7) * 16 + (e & 7) * 2) = 0x3F80;   // S^T[e][at] = 1
                at_prev = at;
                tc_fence_before();
                fence_async_smem();
                warp_arrive(rdyP, lane);
                ph ^= 1u;
            }
            // ---- sums of the chunk: D3[channel][atom] -> m (bf16 rows)
            mbar_wait(bar3, ph ^ 1u);
            tc_fence_after();
            if (at_prev >= 0 && half == 0) *reinterpret_cast<uint16_t*>(ST + (at_prev >> 3) * 2048 + (e >> 3) * 128 + (at_prev & 7) * 16 + (e & 7) * 2) = 0;
            {
                uint32_t v[16];
                tmem_ld16(tl3, v);
                tmem_wait_ld();
#pragma unroll
                for (int i = 0; i < AH; ++i) {
                    if (half * AH + i < natoms) {
                        const __nv_bfloat16 pb = __float2bfloat16_rn(__uint_as_float(v[half * AH + i]));
                        a.m16_out[(size_t)(g0 + half * AH + i) * kF + e] = *reinterpret_cast<const uint16_t*>(&pb);
                    }
                }
            }
            tc_fence_before();
        }
        if (e == 0 && half == 0) s_nt[team] = -1;
        team_bar(team);
        warp_arrive(rdyA1, lane);
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base_s), "n"(512));
}

int sm_count() { return lsd_sm_count(); }

}  // namespace

void launch_edge_er128(Launcher L, const EdgeArgs& a, bool backward)
{
    static bool configured_dev[64] = {};
    bool& configured = configured_dev[lsd_current_device()];
    if (!configured) {
        cudaFuncSetAttribute(k_edge_er128_fwd, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmem);
        configured = true;
    }
    const int cps = (a.n + kCH - 1) / kCH;
    const int nchunks = cps * (a.total / a.n);
    const int grid = std::max(1, std::min(sm_count(), (nchunks + kTeams - 1) / kTeams));
    if (!backward) k_edge_er128_fwd<<<grid, kThreads, kSmem, L.s>>>(a, cps, nchunks);
    note_edge_launch(backward, 3, kCH, kThreads, grid, kF);
    LSD_COUNT(L);
}
