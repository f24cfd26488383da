// bf16 tcgen05 filter path for width F = 128, third generation: the "edges are rows" tile algebra of mlip_edge_rows.cu run
// as a warp-specialised pipeline (M5, M9, section 4.1).
//
// One persistent CTA per SM, 16 warps.  A tile is 128 edge slots (8 record groups of 16 slots; a chunk is 16 atoms); TMEM
// lane = edge.  Two groups of 8 warps (2 threads per edge, each owning half of the channels of a quarter) work on DIFFERENT
// tiles at the same time:
//   ACT group (warps 0-7):  radial basis g(r), g'(r) -> TMEM;  per channel quarter q (32 channels): wait for
//                           [x | x'] = [G | G'] W_f1[q]^T, write ssp(x) and logistic(x) x' as packed bf16 into the A operand
//                           buffer A2[tile & 1] in TMEM.  Bound by the special-function unit (one tanh per edge and channel).
//   EPI group (warps 8-15): gathers the neighbour rows (cp.async, one tile ahead), per output channel quarter o: wait for
//                           [lin | lin'] = [A2v | A2t] W_f2[o]^T, form the cfconv products in registers, write the segment-sum
//                           operand P in place over the gather stage; force term of the edge, group and atom sums; third
//                           contraction D3 = P^T S; running sums per atom.  Bound by shared-memory traffic.
// The last warp of each group issues that group's contractions through one elected lane (warp-uniform operands): the ACT
// issuer the first contraction (its inputs and its accumulator slots are all ACT-internal), the EPI issuer the second and
// third (it waits for "A2 complete" from the ACT group).  Accumulators are double-buffered at quarter granularity
// (2 x 64 columns each for the first and the second contraction), so a group never waits for a round trip in steady state;
// A2 is double-buffered per tile (2 x 128 columns), which is what lets the activation of tile t + 1 run under the epilogue
// of tile t.  TMEM: 128 + 128 + 256 = 512 columns; G / G' alias the last quarter of their tile's A2 buffer (dead until the
// last quarter's activation, which waits for the contraction that read them), D3 aliases its first 16 columns (A2 is dead
// when the third contraction is issued behind the second).
// Determinism / batch invariance: as in mlip_edge_rows.cu (fixed orders that depend only on the atom's own sorted row and on
// the 16-atom chunking of its state).
#include <algorithm>
#include <cstdio>
#include <cstdlib>
#include <vector>
#include "lsd_internal.h"
#include "tc_ptx.cuh"

namespace {
using namespace tcp;

constexpr int kF = 128;
constexpr int kR = LSD_NRBF;
constexpr int kTT = 128;                               // edge slots of a tile
constexpr int kCH = 16;                                // atoms per chunk = columns of D3
constexpr int kGE = 16;                                // edge slots per record group
constexpr int kGPT = kTT / kGE;                        // groups per tile
constexpr int kMaxGroups = kCH * (512 / kGE);
constexpr int kGT = 256;                               // threads of a group (2 per edge)
constexpr int kThreads = 2 * kGT;
constexpr int kW1Bytes = kF * kR * 2, kW2Bytes = kF * kF * 2;
constexpr int kSlab = 2048 + 16;                       // bytes between slabs of the gather stage (16 B x 128 edges + one bank group)
constexpr int kSTBytes = kCH * kTT * 2;
constexpr int kBookBytes = kMaxGroups + 128;           // group -> atom map and first group of every atom, one copy per warp group

template <bool BWD> struct Lay {
    static constexpr int NSLAB = BWD ? 32 : 16;        // 16-byte pieces of a gathered row (bwd: 4 channels x (y, y, mbar, mbar); fwd: 8 channels)
    static constexpr int StageBytes = ((NSLAB * kSlab + 127) / 128) * 128;
    static constexpr int OwnBytes = BWD ? kCH * 512 : 0;
    static constexpr int AccBytes = kTT * kCH * 4;     // running per (channel, atom) sums of the chunk
    static constexpr int RecBytes = 5 * kTT * 4;       // fc, fc', ux, uy, uz of a tile's slots
    static constexpr int oStage = kW1Bytes + kW2Bytes;
    static constexpr int oOwn = oStage + 2 * StageBytes;
    static constexpr int oST = oOwn + OwnBytes;
    static constexpr int oAcc = oST + kSTBytes;
    static constexpr int oRec = oAcc + AccBytes;
    static constexpr int oGx = oRec + 2 * RecBytes;    // [128][2] partial channel sums of the second part
    static constexpr int oGpart = oGx + 1024;          // [2 tile parities][2 parts][8 groups][4] force sums of the tile's groups
    static constexpr int oFsum = oGpart + 512;         // [16 atoms][4]
    static constexpr int oBook = oFsum + 256;          // ACT copy, EPI copy
    static constexpr int Smem = oBook + 2 * kBookBytes;
    static_assert(Smem + 1024 <= 227 * 1024, "shared memory budget");
};

constexpr float kLog2e = 1.44269504088896340736f;
// -ln(1 + a) / (2 a) on [0, 1] (weighted minimax fit of a P(a), |error| < 3.6e-5)
constexpr float kP0 = -0.49872449040412903f, kP1 = 0.2356506735086441f, kP2 = -0.11284290254116058f, kP3 = 0.02937859483063221f;

// TMEM columns
constexpr uint32_t kColD1 = 0, kColD2 = 128, kColA2 = 256;       // D1 / D2: two slots of [v 32 | t 32]; A2: two buffers of [A2v 64 | A2t 64]
constexpr uint32_t kOffG = 48, kOffGt = 64 + 48;                 // G, G' inside their tile's A2 buffer (channels 96..127 of A2v / A2t)

// mbarriers
enum { B_D1FULL = 0, B_D1FREE = 2, B_GREADY = 4, B_A2FULL = 5, B_A2FREE = 7, B_D2FULL = 9, B_D2FREE = 11, B_PREADY = 13, B_D3FULL = 14, B_STFULL = 15 /* [buffer][quarter] */, B_STFREE = 23, B_COUNT = 25 };

__device__ __forceinline__ void group_bar(int id) { asm volatile("bar.sync %0, %1;" ::"r"(id), "n"(kGT) : "memory"); }

// ssp(2h)/2 and (backward) logistic(2h) hp for a pair of channels; h = x/2 comes out of the first contraction because W_f1 is
// packed halved (and W_f2 doubled): ssp(x)/2 = max(h, 0) + a P(a), a = tanh|h|;  logistic(x) = (1 + tanh h)/2
template <bool BWD>
__device__ __forceinline__ void act_pair(uint32_t h0u, uint32_t h1u, uint32_t hp0u, uint32_t hp1u, uint32_t& pv, uint32_t& pt)
{
    const float h0 = __uint_as_float(h0u), h1 = __uint_as_float(h1u);
    const f32x2 p3 = pk2(kP3, kP3), p2 = pk2(kP2, kP2), p1 = pk2(kP1, kP1), p0 = pk2(kP0, kP0);
    float t0, t1, a0, a1;
    if (BWD) { t0 = tanhf_approx(h0); t1 = tanhf_approx(h1); a0 = fabsf(t0); a1 = fabsf(t1); }
    else { a0 = tanhf_approx(fabsf(h0)); a1 = tanhf_approx(fabsf(h1)); }
    const f32x2 a2 = pk2(a0, a1);
    f32x2 r2 = fma2(p3, a2, p2);
    r2 = fma2(r2, a2, p1);
    r2 = fma2(r2, a2, p0);
    pv = pack_bf16(fma2(r2, a2, pk2(fmaxf(h0, 0.f), fmaxf(h1, 0.f))));
    if (BWD) {
        const f32x2 half2 = pk2(0.5f, 0.5f);
        pt = pack_bf16(mul2(fma2(pk2(t0, t1), half2, half2), pk2u(hp0u, hp1u)));
    }
}

// groups of the chunk: per atom ceil(count / 16), exclusive scan -> pref[0..16], group -> atom map; returns the group count.
// Called by all threads of a warp group with their own copy of the book-keeping arrays.
__device__ __forceinline__ int chunk_book(const EdgeArgs& a, int g0, int natoms, int gt, int bar_id, uint8_t* gatom, int* pref)
{
    if (gt < 32) {
        const int c = gt < natoms ? a.count[g0 + gt] : 0;
        int v = (c + kGE - 1) / kGE;
#pragma unroll
        for (int o = 1; o < 16; o <<= 1) { const int u = __shfl_up_sync(0xffffffffu, v, o); if (gt >= o) v += u; }
        if (gt < kCH) pref[gt + 1] = v;
        if (gt == 0) pref[0] = 0;
    }
    group_bar(bar_id);
    if (gt < kCH) for (int g = pref[gt]; g < pref[gt + 1]; ++g) gatom[g] = (uint8_t)gt;
    group_bar(bar_id);
    return pref[kCH];
}

template <bool BWD>
__global__ void __launch_bounds__(kThreads, 1)
k_edge_pipe(EdgeArgs a, int chunks_per_state, int nchunks)
{
    using L = Lay<BWD>;
    extern __shared__ __align__(128) uint8_t smem[];
    __shared__ __align__(8) uint64_t mbar[B_COUNT];
    __shared__ uint32_t tmem_base_s;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;

    {   // resident B operand images (K-major): W_f1 / 2 [128 x 32], 2 W_f2 [128 x 128]; every other buffer starts as zeros
        const uint4* s1 = reinterpret_cast<const uint4*>(a.Wf1_tc);
        const uint4* s2 = reinterpret_cast<const uint4*>(a.Wf2_tc);
        uint4* d1 = reinterpret_cast<uint4*>(smem);
        uint4* d2 = reinterpret_cast<uint4*>(smem + kW1Bytes);
        for (int i = tid; i < kW1Bytes / 16; i += kThreads) d1[i] = s1[i];
        for (int i = tid; i < kW2Bytes / 16; i += kThreads) d2[i] = s2[i];
        uint4* z = reinterpret_cast<uint4*>(smem + L::oStage);
        for (int i = tid; i < (L::Smem - L::oStage) / 16; i += kThreads) z[i] = make_uint4(0u, 0u, 0u, 0u);
    }
    if (tid == 0) {
        const int cnt[B_COUNT] = {1, 1, 8, 8, 8, 8, 8, 8, 8, 1, 1, 8, 8, 8, 1, kGT, kGT, kGT, kGT, kGT, kGT, kGT, kGT, 8, 8};
        for (int i = 0; i < B_COUNT; ++i) mbar_init(smem_u32(&mbar[i]), cnt[i]);
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

    const int grp = __shfl_sync(0xffffffffu, warp, 0) >> 3;            // warp-uniform: 0 = ACT, 1 = EPI
    const bool issuer = (__shfl_sync(0xffffffffu, warp, 0) & 7) == 7;  // the group's last warp issues its contractions
    const uint32_t tmem = __shfl_sync(0xffffffffu, tmem_base_s, 0);
    const uint32_t sW1 = smem_u32(smem), sW2 = sW1 + kW1Bytes, bar0 = smem_u32(&mbar[0]);
    auto bar = [&](int i) { return bar0 + (uint32_t)i * 8u; };
    const uint32_t id32 = make_idesc(128, 32, 0), id3 = make_idesc(128, kCH, 0) | (1u << 15);
    const uint64_t dW1 = make_desc(sW1, 128, 512), dW2 = make_desc(sW2, 128, 2048);
    const int gt = tid & (kGT - 1), e = gt & (kTT - 1), part = gt >> 7, wq = warp & 3;   // group thread, edge slot, channel part, TMEM lane quarter
    const uint32_t tl = tmem + ((uint32_t)(wq * 32) << 16);
    const int my_g = e >> 4, my_s = e & 15;
    const int n = a.n;
    const bool need_sum = BWD ? (a.ybar16_out != nullptr) : true;      // the adjoint of the first block needs the forces only
    const uint8_t* const rows = reinterpret_cast<const uint8_t*>(BWD ? (const void*)a.ym16 : (const void*)a.y16);
    constexpr int ROWB = BWD ? 512 : 256;
    uint32_t T = 0, nq = 0;                                            // tiles and quarters this group has started (buffer / slot parities)
#ifdef LSD_EDGE_TRACE_BUILD
    int tr_n = 0;
    const bool tr_on = a.trace != nullptr && blockIdx.x == 0 && gt == 0;
#define TRACE(tag) do { if (tr_on && T >= 40 && tr_n < 500) { a.trace[grp * 1024 + tr_n++] = ((unsigned long long)(tag) << 48) | (clock64() & 0xFFFFFFFFFFFFull); } } while (0)
#else
#define TRACE(tag) do { } while (0)
#endif

    if (grp == 0) {
        // =========================================================== ACT group
        uint8_t* const gatom = smem + L::oBook;
        int* const pref = reinterpret_cast<int*>(gatom + kMaxGroups);
        const float c2 = -0.5f * kLog2e * a.inv_delta2;
        // first contraction of quarter q of the current tile into slot (nq + q) & 1 (waits until every warp has read the slot's last result)
        auto issue_g1 = [&](int q, uint32_t tA2) {
            const uint32_t nn = nq + (uint32_t)q, s = nn & 1u, k = nn >> 1;
            mbar_wait(bar(B_D1FREE + s), (k & 1u) ^ 1u);
            tc_fence_after();
            if (elect_one()) {
#pragma unroll
                for (int k16 = 0; k16 < kR / 16; ++k16) {
                    const uint64_t db = dW1 + (uint64_t)((q * 2048 + k16 * 256) >> 4);
                    umma_ts(tmem + kColD1 + 64 * s, tmem + tA2 + kOffG + 8 * k16, db, id32, k16 > 0);
                    if (BWD) umma_ts(tmem + kColD1 + 64 * s + 32, tmem + tA2 + kOffGt + 8 * k16, db, id32, k16 > 0);
                }
                umma_commit(bar(B_D1FULL + s));
            }
            __syncwarp();
        };
        for (int chunk = blockIdx.x; chunk < nchunks; chunk += gridDim.x) {
            const int b = chunk / chunks_per_state, ci = chunk - b * chunks_per_state;
            const int g0 = b * n + ci * kCH, natoms = min(kCH, n - ci * kCH);
            const int G = chunk_book(a, g0, natoms, gt, 1, gatom, pref);
            const int ntiles = (G + kGPT - 1) / kGPT;
            // distance, gathered row and record of this thread's edge slot in tile t (the zero group behind the chunk's last group)
            float r_n = 0.f; int jrow_n = g0; const float* rp_n = a.rec_zero + my_s;
            auto load_rec = [&](int t) {
                const int gl = t * kGPT + my_g;
                rp_n = a.rec_zero + my_s; jrow_n = g0;
                if (gl < G) {
                    const int at = gatom[gl];
                    rp_n = a.recs + lsd_rec_index((size_t)(g0 + at), a.cap, (gl - pref[at]) * kGE + my_s, 0);
                    jrow_n = __float_as_int(rp_n[LSD_REC_JROW * 16]);
                }
                r_n = rp_n[LSD_REC_R * 16];
            };
            // neighbour rows of the current tile, the 16-byte pieces that output quarter q of the epilogue consumes -> slabs of stage
            // buffer sb (bwd: 8 lanes = 128 contiguous bytes of a row, 4 rows per instruction; fwd: 4 lanes = 64 bytes, 8 rows); with quarter
            // 0 also cutoff / slope / unit vector of the slots -> recS[sb].  The EPI group waits for the copies on B_STFULL[sb][q].
            // Issued quarter by quarter between the activation work: a burst of 16 copies per thread stalls the warp on the LSU queue.
            auto issue_gathers = [&](int q, uint32_t sb, int jrow, const float* rp) {
                const uint32_t sStage = smem_u32(smem) + (uint32_t)(L::oStage + sb * L::StageBytes);
                if (BWD) {
#pragma unroll
                    for (int i = 0; i < 4; ++i) {
                        const int el = 16 * part + 4 * i + (lane >> 3), s = 8 * q + (lane & 7);
                        const int jr = __shfl_sync(0xffffffffu, jrow, el);
                        cp_async16_ca(sStage + (uint32_t)(s * kSlab + (32 * wq + el) * 16), rows + (size_t)jr * ROWB + s * 16);
                    }
                } else {
#pragma unroll
                    for (int i = 0; i < 2; ++i) {
                        const int el = 16 * part + 8 * i + (lane >> 2), s = 4 * q + (lane & 3);
                        const int jr = __shfl_sync(0xffffffffu, jrow, el);
                        cp_async16_ca(sStage + (uint32_t)(s * kSlab + (32 * wq + el) * 16), rows + (size_t)jr * ROWB + s * 16);
                    }
                }
                if (q == 0 && part == 0) {
                    const uint32_t d = smem_u32(smem) + (uint32_t)(L::oRec + sb * L::RecBytes) + (uint32_t)e * 4;
                    cp_async4(d, rp + LSD_REC_FC * 16);
                    if (BWD) {
                        cp_async4(d + kTT * 4, rp + LSD_REC_FCP * 16); cp_async4(d + 2 * kTT * 4, rp + LSD_REC_UX * 16);
                        cp_async4(d + 3 * kTT * 4, rp + LSD_REC_UY * 16); cp_async4(d + 4 * kTT * 4, rp + LSD_REC_UZ * 16);
                    }
                }
                asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];" ::"r"(bar(B_STFULL + 4 * (int)sb + q)) : "memory");
            };
            if (ntiles > 0) load_rec(0);
            for (int t = 0; t < ntiles; ++t) {
                const uint32_t sb = T & 1u, tA2 = kColA2 + 128u * sb;
                const int jrow_t = jrow_n; const float* const rp_t = rp_n;
                TRACE(1);
                mbar_wait(bar(B_A2FREE + sb), ((T >> 1) & 1u) ^ 1u);    // the epilogue of tile T - 2 is done with this A2 buffer and this stage
                tc_fence_after();
                TRACE(2);
                TRACE(3);
                {   // radial basis (M1) of the thread's edge and its r-derivative -> TMEM, packed bf16 pairs along k (16 of the 32 per part)
                    constexpr int KH = kR / 2;
                    uint32_t gv[KH / 2], gd[KH / 2];
                    const f32x2 c22 = pk2(c2, c2), nid = pk2(-a.inv_delta2, -a.inv_delta2);
                    const float rh = r_n - (float)(part * KH) * a.delta;
#pragma unroll
                    for (int k = 0; k < KH; k += 2) {
                        const float x0 = rh - (float)k * a.delta, x1 = x0 - a.delta;
                        const f32x2 x2 = pk2(x0, x1);
                        float e0, e1;
                        un2(mul2(mul2(x2, x2), c22), e0, e1);
                        const float v0 = ex2f(e0), v1 = ex2f(e1);
                        gv[k >> 1] = pack_bf16(v0, v1);
                        if (BWD) gd[k >> 1] = pack_bf16(mul2(mul2(pk2(v0, v1), x2), nid));
                    }
                    tmem_st8(tl + tA2 + kOffG + 8 * part, gv);
                    if (BWD) tmem_st8(tl + tA2 + kOffGt + 8 * part, gd);
                    tmem_wait_st();
                }
                tc_fence_before();
                warp_arrive(bar(B_GREADY), lane);
                TRACE(4);
                if (t + 1 < ntiles) load_rec(t + 1);
                if (issuer) {
                    mbar_wait(bar(B_GREADY), T & 1u);
                    tc_fence_after();
                    issue_g1(0, tA2);
                    issue_g1(1, tA2);
                }
#pragma unroll 1
                for (int q = 0; q < 4; ++q) {
                    const uint32_t nn = nq + (uint32_t)q, s = nn & 1u, k = nn >> 1;
                    mbar_wait(bar(B_D1FULL + s), k & 1u);
                    tc_fence_after();
                    TRACE(5);
                    uint32_t v[16], vp[16], pv[8], pt[8];
                    tmem_ld16(tl + kColD1 + 64 * s + 16 * part, v);
                    if (BWD) tmem_ld16(tl + kColD1 + 64 * s + 32 + 16 * part, vp);
                    tmem_wait_ld();
                    tc_fence_before();
                    warp_arrive(bar(B_D1FREE + s), lane);          // the slot is read: the contraction of quarter q + 2 may overwrite it
                    if (issuer && q + 2 < 4) issue_g1(q + 2, tA2);
                    if (q == 0) {                                  // the third contraction of tile T - 2 has read P from this stage buffer
                        mbar_wait(bar(B_STFREE + sb), ((T >> 1) & 1u) ^ 1u);
                        issue_gathers(0, sb, jrow_t, rp_t);
                    }
                    if (q < 3) issue_gathers(q + 1, sb, jrow_t, rp_t);
#pragma unroll
                    for (int c = 0; c < 16; c += 2) act_pair<BWD>(v[c], v[c + 1], BWD ? vp[c] : 0u, BWD ? vp[c + 1] : 0u, pv[c >> 1], pt[c >> 1]);
                    tmem_st8(tl + tA2 + 16 * q + 8 * part, pv);
                    if (BWD) tmem_st8(tl + tA2 + 64 + 16 * q + 8 * part, pt);
                    tmem_wait_st();
                    TRACE(6);
                }
                tc_fence_before();
                warp_arrive(bar(B_A2FULL + sb), lane);             // the tile's A2 buffer is complete
                nq += 4; ++T;
            }
            group_bar(1);                                          // the book-keeping arrays are rewritten by the next chunk
        }
    } else {
        // =========================================================== EPI group
        uint8_t* const gatom = smem + L::oBook + kBookBytes;
        int* const pref = reinterpret_cast<int*>(gatom + kMaxGroups);
        uint8_t* const own = smem + L::oOwn;                       // bwd: [16 atoms][512 B] (y, mbar) rows of the chunk's atoms
        uint8_t* const ST = smem + L::oST;
        float4* const accs = reinterpret_cast<float4*>(smem + L::oAcc);           // [4][128]: sums of channel e for atoms 4 j .. 4 j + 3
        float* const gpart = reinterpret_cast<float*>(smem + L::oGpart);
        float* const fsum = reinterpret_cast<float*>(smem + L::oFsum);
        const uint64_t dS = make_desc(smem_u32(ST), 128, 2048);
        // second contraction of output quarter o of the current tile into slot (nq + o) & 1
        auto issue_g2 = [&](int o, uint32_t tA2) {
            const uint32_t nn = nq + (uint32_t)o, s = nn & 1u, k = nn >> 1;
            mbar_wait(bar(B_D2FREE + s), (k & 1u) ^ 1u);
            tc_fence_after();
            if (elect_one()) {
#pragma unroll
                for (int k16 = 0; k16 < kF / 16; ++k16) {
                    const uint64_t db = dW2 + (uint64_t)((o * 8192 + k16 * 256) >> 4);
                    umma_ts(tmem + kColD2 + 64 * s, tmem + tA2 + 8 * k16, db, id32, k16 > 0);
                    if (BWD) umma_ts(tmem + kColD2 + 64 * s + 32, tmem + tA2 + 64 + 8 * k16, db, id32, k16 > 0);
                }
                umma_commit(bar(B_D2FULL + s));
            }
            __syncwarp();
        };
        uint16_t* scell_pend = nullptr;                            // S^T entry of the tile whose third contraction has not been consumed yet
        uint32_t pendT = 0; bool pending = false;
        // consume D3 of tile pendT: running sums, clear the S^T entry, release the tile's stage buffer to the ACT group
        auto consume_d3 = [&]() {
            const uint32_t pb = pendT & 1u;
            if (need_sum) {
                mbar_wait(bar(B_D3FULL), pendT & 1u);
                tc_fence_after();
                uint32_t v[8];
                tmem_ld8(tl + kColD2 + 8 * part, v);               // lane = channel e, columns = atoms 8 part .. 8 part + 7
                tmem_wait_ld();
#pragma unroll
                for (int j = 0; j < 2; ++j) {
                    float4 s4 = accs[(2 * part + j) * kTT + e];
                    s4.x += __uint_as_float(v[4 * j]); s4.y += __uint_as_float(v[4 * j + 1]); s4.z += __uint_as_float(v[4 * j + 2]); s4.w += __uint_as_float(v[4 * j + 3]);
                    accs[(2 * part + j) * kTT + e] = s4;
                }
                if (scell_pend) *scell_pend = 0;
            }
            tc_fence_before();
            warp_arrive(bar(B_STFREE + pb), lane);                 // the stage buffer (P) and recS of the tile may be overwritten
            pending = false;
        };
        for (int chunk = blockIdx.x; chunk < nchunks; chunk += gridDim.x) {
            const int cb = chunk / chunks_per_state, ci = chunk - cb * chunks_per_state;
            const int g0 = cb * n + ci * kCH, natoms = min(kCH, n - ci * kCH);
            if (BWD) {                                             // (y, mbar) rows of the chunk's own atoms
                for (int i = gt; i < kCH * 32; i += kGT) {
                    const int at = i >> 5;
                    uint4 v = make_uint4(0u, 0u, 0u, 0u);
                    if (at < natoms) v = *reinterpret_cast<const uint4*>(rows + (size_t)(g0 + at) * ROWB + (i & 31) * 16);
                    *reinterpret_cast<uint4*>(own + i * 16) = v;
                }
                if (gt < kCH) { fsum[4 * gt] = 0.f; fsum[4 * gt + 1] = 0.f; fsum[4 * gt + 2] = 0.f; }
            }
            accs[(2 * part) * kTT + e] = make_float4(0.f, 0.f, 0.f, 0.f);
            accs[(2 * part + 1) * kTT + e] = make_float4(0.f, 0.f, 0.f, 0.f);
            const int G = chunk_book(a, g0, natoms, gt, 2, gatom, pref);
            const int ntiles = (G + kGPT - 1) / kGPT;
            if (ntiles == 0) {                                     // no edges at all: empty sums
                uint16_t* out16 = BWD ? a.ybar16_out : a.m16_out;
                if (out16 && part == 0) for (int i = 0; i < natoms; ++i) out16[(size_t)(g0 + i) * kF + e] = 0;
                group_bar(2);
                continue;
            }
            for (int t = 0; t < ntiles; ++t) {
                const uint32_t sb = T & 1u, tA2 = kColA2 + 128u * sb;
                uint8_t* const stage = smem + L::oStage + sb * L::StageBytes;
                const float* const recS = reinterpret_cast<const float*>(smem + L::oRec + sb * L::RecBytes);
                TRACE(1);
                if (issuer) {
                    mbar_wait(bar(B_A2FULL + sb), (T >> 1) & 1u);  // the activation of this tile is complete
                    tc_fence_after();
                    issue_g2(0, tA2);
                    issue_g2(1, tA2);
                }
                TRACE(2);
                const int gl_t = t * kGPT + my_g;
                const int at = gl_t < G ? (int)gatom[gl_t] : -1;
                const uint8_t* const ownrow = own + (at >= 0 ? at : 0) * 512;
                f32x2 A2s = 0, B2s = 0;
#pragma unroll 1
                for (int o = 0; o < 4; ++o) {
                    const uint32_t nn = nq + (uint32_t)o, s = nn & 1u, k = nn >> 1;
                    mbar_wait(bar(B_STFULL + 4 * (int)sb + o), (T >> 1) & 1u);   // this quarter's pieces of the gathered rows have landed
                    mbar_wait(bar(B_D2FULL + s), k & 1u);
                    tc_fence_after();
                    TRACE(4);
                    const int c0 = 32 * o + 16 * part;             // first of this thread's 16 output channels in this quarter
                    uint32_t v[16], vp[16];
                    tmem_ld16(tl + kColD2 + 64 * s + 16 * part, v);
                    if (BWD) tmem_ld16(tl + kColD2 + 64 * s + 32 + 16 * part, vp);
                    tmem_wait_ld();
                    tc_fence_before();
                    warp_arrive(bar(B_D2FREE + s), lane);          // the slot is read: the contraction of quarter o + 2 may overwrite it
                    if (o == 3) warp_arrive(bar(B_A2FREE + sb), lane);   // every contraction that reads this A2 buffer is complete
                    if (issuer && o + 2 < 4) issue_g2(o + 2, tA2);
                    if (BWD) {
                        // P = bf16(lin) . mbar_j (in place), A += sum_f c_f lin'_f, B += sum_f c_f lin_f, c = mbar_a y_j + mbar_j y_a (bf16 pairs)
#pragma unroll
                        for (int q8 = 0; q8 < 2; ++q8) {           // 8 channels = two stage cells -> one P cell
                            const int slab = (c0 >> 2) + 2 * q8;
                            const uint4 s0v = *reinterpret_cast<const uint4*>(stage + slab * kSlab + e * 16);
                            const uint4 s1v = *reinterpret_cast<const uint4*>(stage + (slab + 1) * kSlab + e * 16);
                            const uint4 o0v = *reinterpret_cast<const uint4*>(ownrow + slab * 16);
                            const uint4 o1v = *reinterpret_cast<const uint4*>(ownrow + (slab + 1) * 16);
                            const uint32_t yj[4] = {s0v.x, s0v.z, s1v.x, s1v.z}, mj[4] = {s0v.y, s0v.w, s1v.y, s1v.w};
                            const uint32_t ya[4] = {o0v.x, o0v.z, o1v.x, o1v.z}, ma[4] = {o0v.y, o0v.w, o1v.y, o1v.w};
                            uint32_t pw[4];
#pragma unroll
                            for (int i = 0; i < 4; ++i) {
                                const int c = 8 * q8 + 2 * i;
                                const f32x2 cf = bf2_to_f2(bfma2(ma[i], yj[i], bmul2(mj[i], ya[i])));
                                A2s = fma2(cf, pk2u(vp[c], vp[c + 1]), A2s);
                                B2s = fma2(cf, pk2u(v[c], v[c + 1]), B2s);
                                pw[i] = bmul2(pack_bf16(__uint_as_float(v[c]), __uint_as_float(v[c + 1])), mj[i]);
                            }
                            if (need_sum) *reinterpret_cast<uint4*>(stage + slab * kSlab + e * 16) = make_uint4(pw[0], pw[1], pw[2], pw[3]);
                        }
                    } else {
                        // P = bf16(lin) . y_j, in place (8 channels = one 16-byte cell)
#pragma unroll
                        for (int q8 = 0; q8 < 2; ++q8) {
                            uint8_t* cell = stage + ((c0 >> 3) + q8) * kSlab + e * 16;
                            const uint4 y = *reinterpret_cast<const uint4*>(cell);
                            uint4 p;
                            p.x = bmul2(pack_bf16(__uint_as_float(v[8 * q8]), __uint_as_float(v[8 * q8 + 1])), y.x);
                            p.y = bmul2(pack_bf16(__uint_as_float(v[8 * q8 + 2]), __uint_as_float(v[8 * q8 + 3])), y.y);
                            p.z = bmul2(pack_bf16(__uint_as_float(v[8 * q8 + 4]), __uint_as_float(v[8 * q8 + 5])), y.z);
                            p.w = bmul2(pack_bf16(__uint_as_float(v[8 * q8 + 6]), __uint_as_float(v[8 * q8 + 7])), y.w);
                            *reinterpret_cast<uint4*>(cell) = p;
                        }
                    }
                    TRACE(5);
                }
                TRACE(6);
                const float fc = recS[e];
                if (BWD) {
                    // ---- force term of the edge, this part's channels: g = fc sum_f c_f lin'_f + fc' sum_f c_f lin_f, times the unit vector,
                    //      summed over the 16 edges of the group (shuffles); the two parts and the groups of an atom are added in list order below
                    float Al, Ah, Bl, Bh;
                    un2(A2s, Al, Ah); un2(B2s, Bl, Bh);
                    const float g = fc * (Al + Ah) + recS[kTT + e] * (Bl + Bh);
                    float fx = g * recS[2 * kTT + e], fy = g * recS[3 * kTT + e], fz = g * recS[4 * kTT + e];
#pragma unroll
                    for (int o = 8; o > 0; o >>= 1) {
                        fx += __shfl_xor_sync(0xffffffffu, fx, o); fy += __shfl_xor_sync(0xffffffffu, fy, o); fz += __shfl_xor_sync(0xffffffffu, fz, o);
                    }
                    if (my_s == 0) { float* gp = gpart + ((sb * 2 + part) * kGPT + my_g) * 4; gp[0] = fx; gp[1] = fy; gp[2] = fz; }
                }
                uint16_t* const scell = reinterpret_cast<uint16_t*>(ST + ((at >= 0 ? at : 0) >> 3) * 2048 + (e >> 3) * 128 + ((at >= 0 ? at : 0) & 7) * 16 + (e & 7) * 2);
                if (need_sum && part == 0 && at >= 0) {            // S^T[e][at] = fc (the cutoff rides on the segment matrix)
                    const __nv_bfloat16 fb = __float2bfloat16_rn(fc);
                    *scell = *reinterpret_cast<const uint16_t*>(&fb);
                }
                if (need_sum) fence_async_smem();
                tc_fence_before();
                warp_arrive(bar(B_PREADY), lane);
                TRACE(7);
                if (issuer) {
                    mbar_wait(bar(B_PREADY), T & 1u);              // P, S and the group force sums of every warp are published
                    if (need_sum) {                                // D3 = P^T S into the first 16 columns of the D2 slots (every warp has read its last quarter;
                                                                   // the next tile's second contractions are issued behind consume_d3)
                        tc_fence_after();
                        if (elect_one()) {
                            const uint64_t dP = make_desc(smem_u32(stage), 128, BWD ? 2 * kSlab : kSlab);
#pragma unroll
                            for (int k16 = 0; k16 < kTT / 16; ++k16) umma(tmem + kColD2, dP + (uint64_t)(k16 * 16), dS + (uint64_t)(k16 * 16), id3, k16 > 0);
                            umma_commit(bar(B_D3FULL));
                        }
                        __syncwarp();
                    }
                    if (BWD && lane < kCH) {                       // atom `lane`: its groups inside this tile in list order, part 0 then part 1
                        const int lo = max(pref[lane], t * kGPT), hi = min(pref[lane + 1], t * kGPT + kGPT);
                        if (lo < hi) {
                            float fax = fsum[4 * lane], fay = fsum[4 * lane + 1], faz = fsum[4 * lane + 2];
                            for (int g = lo; g < hi; ++g) {
                                const float* g0p = gpart + ((sb * 2) * kGPT + (g - t * kGPT)) * 4;
                                const float* g1p = g0p + kGPT * 4;
                                fax += g0p[0]; fay += g0p[1]; faz += g0p[2];
                                fax += g1p[0]; fay += g1p[1]; faz += g1p[2];
                            }
                            fsum[4 * lane] = fax; fsum[4 * lane + 1] = fay; fsum[4 * lane + 2] = faz;
                        }
                    }
                    __syncwarp();
                }
                scell_pend = (need_sum && part == 0 && at >= 0) ? scell : nullptr;
                pendT = T; pending = true;
                TRACE(8);
                consume_d3();                                      // (waiting here keeps the ACT group two tiles ahead; deferring it couples the groups)
                TRACE(9);
                nq += 4; ++T;
            }
            // ---- the chunk's sums -> bf16 rows (thread = channel e, atoms [8 part, 8 part + 8)) and its forces
            {
                uint16_t* out16 = BWD ? a.ybar16_out : a.m16_out;
                if (out16) {
                    float acc[8];
#pragma unroll
                    for (int j = 0; j < 2; ++j) {
                        const float4 s4 = accs[(2 * part + j) * kTT + e];
                        acc[4 * j] = s4.x; acc[4 * j + 1] = s4.y; acc[4 * j + 2] = s4.z; acc[4 * j + 3] = s4.w;
                    }
#pragma unroll
                    for (int i = 0; i < 8; ++i) {
                        const int at = part * 8 + i;
                        if (at < natoms) {
                            const __nv_bfloat16 pb = __float2bfloat16_rn(acc[i]);
                            out16[(size_t)(g0 + at) * kF + e] = *reinterpret_cast<const uint16_t*>(&pb);
                        }
                    }
                }
                if (BWD && issuer && lane < natoms) {              // the issuing warp holds the force sums (lane = atom)
                    const int i = ci * kCH + lane;
                    double* Fb = a.Fout + (size_t)cb * 3 * n;
                    Fb[i] += (double)fsum[4 * lane]; Fb[n + i] += (double)fsum[4 * lane + 1]; Fb[2 * n + i] += (double)fsum[4 * lane + 2];
                }
            }
            group_bar(2);                                          // book-keeping, own rows and sums are rewritten by the next chunk
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base_s), "n"(512));
}

int device_sm_count()
{
    int dev = 0, sms = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    return sms > 0 ? sms : 148;
}

template <bool BWD> void launch_pipe(Launcher L, const EdgeArgs& a)
{
    cudaFuncSetAttribute(k_edge_pipe<BWD>, cudaFuncAttributeMaxDynamicSharedMemorySize, Lay<BWD>::Smem);
    const int cps = (a.n + kCH - 1) / kCH;
    const int nchunks = cps * (a.total / a.n);
    const int grid = std::max(1, std::min(device_sm_count(), nchunks));
#ifdef LSD_EDGE_TRACE_BUILD
    static int trace_launch[2] = {0, 0};
    if (getenv("LSD_EDGE_TRACE") && ++trace_launch[BWD] == 8) {    // debug: time stamps of block 0, printed once per direction
        unsigned long long* dbuf = nullptr;
        cudaMalloc(&dbuf, 2048 * 8); cudaMemsetAsync(dbuf, 0, 2048 * 8, L.s);
        EdgeArgs at = a; at.trace = dbuf;
        k_edge_pipe<BWD><<<grid, kThreads, Lay<BWD>::Smem, L.s>>>(at, cps, nchunks);
        cudaStreamSynchronize(L.s);
        std::vector<unsigned long long> h(2048);
        cudaMemcpy(h.data(), dbuf, 2048 * 8, cudaMemcpyDeviceToHost); cudaFree(dbuf);
        for (int g = 0; g < 2; ++g) {
            fprintf(stderr, "[pipe trace] %s %s:", BWD ? "bwd" : "fwd", g ? "EPI" : "ACT");
            unsigned long long t0 = h[g * 1024] & 0xFFFFFFFFFFFFull, prev = t0;
            for (int i = 0; i < 160 && h[g * 1024 + i]; ++i) {
                const unsigned long long c = h[g * 1024 + i] & 0xFFFFFFFFFFFFull; const int tag = (int)(h[g * 1024 + i] >> 48);
                if (tag == 1) fprintf(stderr, "\n   tile @%llu:", c - t0);
                fprintf(stderr, " %d:+%llu", tag, c - prev); prev = c;
            }
            fprintf(stderr, "\n");
        }
        LSD_COUNT(L);
        return;
    }
#endif
    k_edge_pipe<BWD><<<grid, kThreads, Lay<BWD>::Smem, L.s>>>(a, cps, nchunks);
    note_edge_launch(BWD, 5, kCH, kThreads, grid, kF);
    LSD_COUNT(L);
}

}  // namespace

// a.ym16 (backward) must be in the pair layout: per channel pair (f, f+1) the words (y_f | y_f+1 << 16), (mbar_f | mbar_f+1 << 16)
void launch_edge_pipe(Launcher L, const EdgeArgs& a, bool backward)
{
    if (backward) launch_pipe<true>(L, a); else launch_pipe<false>(L, a);
}
