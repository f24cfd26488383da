// bf16 tcgen05 filter path for width F = 128 (the target networks of cfg4 / cfg5): continuous-filter convolution forward
// and its adjoint (M5, M9) with both per-edge filter contractions on the tensor cores, fp32 accumulation in TMEM.
//
// Same tile algebra as mlip_tc.cu ("channels are rows": TMEM lane = channel = thread, TMEM column = edge; the per-atom
// sums over edges are serial sums inside one thread, in the order of the atom's sorted neighbour row), re-organised
// around the instruction-issue limit the round-1 profile showed (profiles/r1_edge_tc128_fwd_cfg5.md):
//   * one persistent CTA per SM, 4 teams of 128 threads; every team owns 128 TMEM columns (D1, D2) and its own operand
//     buffers; the only team-wide barrier per tile publishes the asynchronous copies.  "Operand ready" is an mbarrier
//     every thread arrives on without waiting; only the issuing thread waits for it.
//   * every warp gathers the 32-channel segment of the neighbour rows that its own lanes consume (cp.async, 8 lanes x
//     16 B = one 128-byte run per row: conflict-free in shared memory, full sectors in L2).  The backward pass gathers
//     one interleaved row (y_j, mbar_j) per edge (one 32-bit shared-memory load per channel and edge).
//   * epilogue and activation arithmetic on packed fp32x2 instructions (FFMA2 / FMUL2), two edges per instruction.
//   * ssp(x) = max(x, 0) - ln(1 + tanh(|x| / 2)): one MUFU (tanh) per value; ln(1 + a) on [0, 1] is a cubic on the FMA
//     pipe (|error| < 4e-5, below the bf16 rounding of the operand it feeds), so the special-function unit is not the
//     bound.  logistic(x) = (1 + tanh(x / 2)) / 2 re-uses the same tanh.
#include <algorithm>
#include "lsd_internal.h"
#include "tc_ptx.cuh"

namespace {
using namespace tcp;

constexpr int kF = 128;
constexpr int kR = LSD_NRBF;
constexpr int kTeams = 4;
constexpr int kTT = 128;                // threads per team = accumulator rows
constexpr int kThreads = kTeams * kTT + kTeams * 32;   // + one MMA-issuing warp per team
constexpr int kCH = 64;                 // atoms per chunk
constexpr int kGE = 16;                 // edge slots per group
constexpr int kMaxGroups = kCH * (512 / kGE);
constexpr int kRecBufs = 4;             // tiles of record groups in flight
constexpr int kBars = 4 + kRecBufs;     // mbarriers per team

template <bool BWD> struct Cfg {
    static constexpr int NT = BWD ? 32 : 64;                // edges per tile
    static constexpr int GPT = NT / kGE;                    // groups per tile
    static constexpr int NCOLS = 64;                        // MMA N: value [+ tangent] columns
    static constexpr int SEG = BWD ? 128 : 64;              // bytes of a gathered row that one warp (32 channels) consumes
    static constexpr int W1Bytes = kF * kR * 2, W2Bytes = kF * kF * 2;
    static constexpr int B2Bytes = NCOLS * kF * 2, B1Bytes = NCOLS * kR * 2;
    static constexpr int StageBytes = 4 * NT * SEG;
    static constexpr int OwnBytes = BWD ? 4 * GPT * 128 : 0;
    static constexpr int RecFloats = NT * 8;
    static constexpr int RecBytes = kRecBufs * RecFloats * 4;
    static constexpr int PrefBytes = 272, CntBytes = kCH * 4;
    static constexpr int FpartBytes = BWD ? kCH * 4 * 3 * 4 : 0;
    static constexpr int TeamBytes = B2Bytes + B1Bytes + StageBytes + OwnBytes + RecBytes + PrefBytes + CntBytes + kMaxGroups + FpartBytes;
    static constexpr int Smem = W1Bytes + W2Bytes + kTeams * TeamBytes;
    static_assert(Smem + 512 <= 227 * 1024, "shared memory budget");
    static_assert(TeamBytes % 16 == 0, "regions stay 16-byte aligned");
};

constexpr float kLog2e = 1.44269504088896340736f;
// -ln(1 + a) / (2 a) on [0, 1] (weighted minimax fit of a P(a), |error| < 3.6e-5)
constexpr float kP0 = -0.49872449040412903f, kP1 = 0.2356506735086441f, kP2 = -0.11284290254116058f, kP3 = 0.02937859483063221f;

__device__ __forceinline__ void team_bar(int team) { asm volatile("bar.sync %0, %1;" ::"r"(team + 1), "n"(kTT) : "memory"); }

template <bool BWD, int CH>
__global__ void __launch_bounds__(kThreads, 1)
k_edge_tc128(EdgeArgs a, int chunks_per_state, int nchunks)
{
    static_assert(CH <= kCH, "buffers are sized for chunks of kCH atoms");
    using C = Cfg<BWD>;
    constexpr int GPT = C::GPT, NT = C::NT, NCOLS = C::NCOLS, SEG = C::SEG, RECF = C::RecFloats;
    constexpr int KPT = BWD ? 8 : 16;                  // radial basis functions per staging thread
    extern __shared__ __align__(128) uint8_t smem[];
    __shared__ __align__(8) uint64_t mbar[kBars * kTeams];
    __shared__ uint32_t tmem_base_s;
    __shared__ int next_chunk, s_chunk[kTeams];
    __shared__ volatile int s_done[kTeams];
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31, team = tid >> 7, tt = tid & (kTT - 1), wq = warp & 3;

    {   // resident A operand images (canonical K-major layout); every other operand buffer starts as zeros
        const uint4* s1 = reinterpret_cast<const uint4*>(a.Wf1_tc);
        const uint4* s2 = reinterpret_cast<const uint4*>(a.Wf2_tc);
        uint4* d1 = reinterpret_cast<uint4*>(smem);
        uint4* d2 = reinterpret_cast<uint4*>(smem + C::W1Bytes);
        for (int i = tid; i < C::W1Bytes / 16; i += kThreads) d1[i] = s1[i];
        for (int i = tid; i < C::W2Bytes / 16; i += kThreads) d2[i] = s2[i];
        uint4* z = reinterpret_cast<uint4*>(smem + C::W1Bytes + C::W2Bytes);
        for (int i = tid; i < kTeams * C::TeamBytes / 16; i += kThreads) z[i] = make_uint4(0u, 0u, 0u, 0u);
    }
    if (tid == 0) {
        for (int t = 0; t < kTeams; ++t) {
            mbar_init(smem_u32(&mbar[kBars * t]), 1); mbar_init(smem_u32(&mbar[kBars * t + 1]), 1);           // MMA1 / MMA2 complete
            mbar_init(smem_u32(&mbar[kBars * t + 2]), kTT / 32); mbar_init(smem_u32(&mbar[kBars * t + 3]), kTT / 32);   // B1 / B2 written by every warp
            for (int r = 0; r < kRecBufs; ++r) mbar_init(smem_u32(&mbar[kBars * t + 4 + r]), 1);              // record copies landed (byte count)
        }
        asm volatile("fence.mbarrier_init.release.cluster;");
        next_chunk = 0;
        for (int t = 0; t < kTeams; ++t) s_done[t] = 0;
    }
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&tmem_base_s)), "n"(512));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
    }
    fence_async_smem();
    tc_fence_before();
    __syncthreads();
    tc_fence_after();

    if (warp >= kTeams * 4) {
        // ---- MMA warps: warp 16 + k issues the contractions of team k.  A team's requests strictly alternate
        // (D1 = W_f1 B1, D2 = W_f2 B2, D1, ...); "done" arrives as a D1 request with the team's flag set.
        if (lane == 0) {
            const int tm = warp - kTeams * 4;
            const uint32_t sW1 = smem_u32(smem), sW2 = smem_u32(smem + C::W1Bytes);
            const uint32_t sB2 = smem_u32(smem + C::W1Bytes + C::W2Bytes + tm * C::TeamBytes), sB1 = sB2 + C::B2Bytes;
            const uint32_t bar1 = smem_u32(&mbar[kBars * tm]), bar2 = bar1 + 8, rdy1 = bar1 + 16, rdy2 = bar1 + 24;
            const uint32_t tmem1 = tmem_base_s + (uint32_t)(tm * 128), tmem2 = tmem1 + 64;
            const uint32_t idesc1 = make_idesc(128, NCOLS, 0), idesc2 = make_idesc(128, NCOLS, 1);
            uint32_t ph = 0;
            for (;;) {
                mbar_wait(rdy1, ph);
                if (s_done[tm]) break;
                tc_fence_after();
#pragma unroll
                for (int k16 = 0; k16 < kR / 16; ++k16)
                    umma(tmem1, make_desc(sW1 + k16 * 256, 128, 512), make_desc(sB1 + k16 * 256, 128, 512), idesc1, k16 > 0);
                umma_commit(bar1);
                mbar_wait(rdy2, ph);
                tc_fence_after();
#pragma unroll
                for (int k16 = 0; k16 < kF / 16; ++k16)
                    umma(tmem2, make_desc(sW2 + k16 * 256, 128, 2048), make_desc(sB2 + k16 * 256, 128, 2048), idesc2, k16 > 0);
                umma_commit(bar2);
                ph ^= 1u;
            }
        }
    } else {
    uint8_t* const tb = smem + C::W1Bytes + C::W2Bytes + team * C::TeamBytes;
    uint8_t* const B2 = tb;                                            // [NCOLS][128 k] MN-major
    uint8_t* const B1 = B2 + C::B2Bytes;                               // [NCOLS][32 k] K-major
    uint8_t* const stage = B1 + C::B1Bytes;                            // [4 warps][NT edges][SEG]
    uint8_t* const own = stage + C::StageBytes;                        // [4 warps][GPT groups][128]  (y_a, mbar_a) of the groups' atoms
    float* const recs = reinterpret_cast<float*>(own + C::OwnBytes);   // [kRecBufs][GPT groups][8 fields][16 slots]
    int* const pref = reinterpret_cast<int*>(reinterpret_cast<uint8_t*>(recs) + C::RecBytes);   // first group of every atom of the chunk
    int* const cnts = reinterpret_cast<int*>(reinterpret_cast<uint8_t*>(pref) + C::PrefBytes);
    uint8_t* const gatom = reinterpret_cast<uint8_t*>(cnts) + C::CntBytes;                      // group -> atom of the chunk
    float* const fpart = reinterpret_cast<float*>(gatom + kMaxGroups);
    uint8_t* const stage_w = stage + wq * (NT * SEG);
    uint8_t* const own_w = own + wq * (GPT * 128);
    const uint32_t bar1 = smem_u32(&mbar[kBars * team]), bar2 = bar1 + 8, rdy1 = bar1 + 16, rdy2 = bar1 + 24, recf = bar1 + 32;
    const uint32_t sStageW = smem_u32(stage_w), sOwnW = smem_u32(own_w), sRecs = smem_u32(recs);
    const uint32_t tmem1 = tmem_base_s + (uint32_t)(team * 128), tmem2 = tmem1 + 64;             // D1, D2 accumulators
    const uint32_t lane_sel = (uint32_t)(wq * 32) << 16;
    const uint32_t tl1 = tmem1 + lane_sel, tl2 = tmem2 + lane_sel;
    uint32_t phase1 = 0, phase2 = 0;
    uint32_t gt0 = 0;                                  // tiles this team has processed (record buffers and their mbarrier phases follow it)
    const int n = a.n;
    // staging role: edge sn of the tile, basis functions k0 .. k0 + KPT - 1; the 8 lanes of a quarter warp own 8 consecutive edges
    const int sn = BWD ? 8 * wq + (lane & 7) : 16 * wq + (lane & 7) + 8 * ((lane >> 3) & 1);
    const int k0 = BWD ? 8 * (lane >> 3) : 16 * (lane >> 4);
    const int srec = (sn >> 4) * LSD_REC_GROUP_FLOATS + (sn & 15);
    const float c2 = -0.5f * kLog2e * a.inv_delta2;
    const uint8_t* const rows16 = reinterpret_cast<const uint8_t*>(BWD ? (const void*)a.ym16 : (const void*)a.y16) + wq * SEG;
    constexpr int ROWB = BWD ? 4 * kF : 2 * kF;        // bytes of a gathered feature row

    for (;;) {
        if (tt == 0) s_chunk[team] = atomicAdd(&next_chunk, 1);
        team_bar(team);
        const int chunk = blockIdx.x + s_chunk[team] * gridDim.x;
        if (chunk >= nchunks) { if (tt == 0) s_done[team] = 1; team_bar(team); warp_arrive(rdy1, lane); break; }
        const int b = chunk / chunks_per_state, ci = chunk - b * chunks_per_state;
        const int g0 = b * n + ci * CH;                                // first feature row of the chunk
        const int natoms = min(CH, n - ci * CH);
        if (tt < CH) { const int c = tt < natoms ? a.count[g0 + tt] : 0; cnts[tt] = c; pref[tt + 1] = (c + kGE - 1) / kGE; }
        team_bar(team);
        if (tt == 0) { int s = 0; pref[0] = 0; for (int i = 1; i <= CH; ++i) { s += pref[i]; pref[i] = s; } }
        team_bar(team);
        if (tt < CH) for (int g = pref[tt]; g < pref[tt + 1]; ++g) gatom[g] = (uint8_t)tt;
        {   // atoms without neighbours: their sums are empty
            float* out = BWD ? a.ybar : a.m_out;
            uint16_t* out16 = BWD ? a.ybar16_out : a.m16_out;
            if (out16) { for (int i = 0; i < natoms; ++i) if (cnts[i] == 0) out16[(size_t)(g0 + i) * kF + tt] = 0; }
            else if (out) for (int i = 0; i < natoms; ++i) if (cnts[i] == 0) out[(size_t)(g0 + i) * kF + tt] = 0.f;
        }
        team_bar(team);
        const int G = pref[CH];                                        // groups of the chunk
        const int ntiles = (G + GPT - 1) / GPT;

        // bulk asynchronous copy of the record groups (512 bytes each) of tile t into buffer (gt0 + t) % kRecBufs, issued by one
        // thread (a zero group for groups behind the chunk's end); the buffer's mbarrier completes on the byte count
        auto fetch_records = [&](int t) {
            if (tt == 0) {
                const uint32_t buf = (gt0 + (uint32_t)t) & (kRecBufs - 1);
                mbar_expect_tx(recf + buf * 8, GPT * LSD_REC_GROUP_FLOATS * 4);
#pragma unroll
                for (int gs = 0; gs < GPT; ++gs) {
                    const int gl = t * GPT + gs;
                    const float* src = a.rec_zero;
                    if (gl < G) {
                        const int at = gatom[gl];
                        src = a.recs + lsd_rec_index((size_t)(g0 + at), a.cap, (gl - pref[at]) * kGE, 0);
                    }
                    bulk_g2s(sRecs + (uint32_t)((buf * RECF + gs * LSD_REC_GROUP_FLOATS) * 4), src, LSD_REC_GROUP_FLOATS * 4, recf + buf * 8);
                }
            }
        };
        auto wait_records = [&](int t) {                               // records of tile t are in shared memory
            const uint32_t g = gt0 + (uint32_t)t;
            mbar_wait(recf + (g & (kRecBufs - 1)) * 8, (g / kRecBufs) & 1u);
        };
        // radial basis (M1) of tile t -> B1, K-major: (n, k) at (n/8)*512 + (k/8)*128 + (n%8)*16 + (k%8)*2
        auto stage_basis = [&](int t) {
            const float r = recs[((gt0 + t) & (kRecBufs - 1)) * RECF + srec + LSD_REC_R * 16];
            uint32_t gv[KPT / 2], gt[KPT / 2];
            const f32x2 c22 = pk2(c2, c2), nid = pk2(-a.inv_delta2, -a.inv_delta2);
#pragma unroll
            for (int k = 0; k < KPT; k += 2) {
                const float x0 = r - (float)(k0 + k) * a.delta, x1 = x0 - a.delta;
                const f32x2 x2 = pk2(x0, x1);
                float e0, e1;
                un2(mul2(mul2(x2, x2), c22), e0, e1);
                const float v0 = ex2f(e0), v1 = ex2f(e1);
                gv[k >> 1] = pack_bf16(v0, v1);
                if (BWD) gt[k >> 1] = pack_bf16(mul2(mul2(pk2(v0, v1), x2), nid));
            }
            uint8_t* dst = B1 + (sn >> 3) * 512 + (sn & 7) * 16 + (k0 >> 3) * 128;
#pragma unroll
            for (int kc = 0; kc < KPT / 8; ++kc) *reinterpret_cast<uint4*>(dst + kc * 128) = make_uint4(gv[4 * kc], gv[4 * kc + 1], gv[4 * kc + 2], gv[4 * kc + 3]);
            if (BWD) {
                uint8_t* dt = B1 + ((NT + sn) >> 3) * 512 + (sn & 7) * 16 + (k0 >> 3) * 128;
#pragma unroll
                for (int kc = 0; kc < KPT / 8; ++kc) *reinterpret_cast<uint4*>(dt + kc * 128) = make_uint4(gt[4 * kc], gt[4 * kc + 1], gt[4 * kc + 2], gt[4 * kc + 3]);
            }
        };
        // everybody: "my part of B1 is written and I am done reading D1"; the MMA warp waits for all and issues D1 = W_f1 B1
        auto publish_b1_and_mma1 = [&]() {
            tc_fence_before();
            fence_async_smem();
            warp_arrive(rdy1, lane);
        };
        // this warp's 32-channel segment of the bf16 feature rows of tile t (and of the groups' own rows) -> gather stage
        auto issue_gathers = [&](int t) {
            const float* rj = recs + ((gt0 + t) & (kRecBufs - 1)) * RECF + LSD_REC_JROW * 16;
            if (BWD) {
#pragma unroll
                for (int i = 0; i < NT / 4; ++i) {
                    const int e = 4 * i + (lane >> 3), ch = lane & 7;
                    const int jrow = __float_as_int(rj[(e >> 4) * LSD_REC_GROUP_FLOATS + (e & 15)]);
                    cp_async16(sStageW + (uint32_t)(e * SEG + ch * 16), rows16 + (size_t)jrow * ROWB + ch * 16, 16);
                }
                if (lane < GPT * 8) {                                  // the groups' own rows (y_a, mbar_a)
                    const int g = lane >> 3, ch = lane & 7;
                    const size_t arow = (size_t)(g0 + (G > 0 ? gatom[min(t * GPT + g, G - 1)] : 0));
                    cp_async16(sOwnW + (uint32_t)(g * 128 + ch * 16), rows16 + arow * ROWB + ch * 16, 16);
                }
            } else {
#pragma unroll
                for (int i = 0; i < NT / 8; ++i) {
                    const int e = 8 * i + (lane >> 2), ch = lane & 3;
                    const int jrow = __float_as_int(rj[(e >> 4) * LSD_REC_GROUP_FLOATS + (e & 15)]);
                    cp_async16(sStageW + (uint32_t)(e * SEG + ch * 16), rows16 + (size_t)jrow * ROWB + ch * 16, 16);
                }
            }
        };

        int cur = -1;
        f32x2 part2 = 0, fx2 = 0, fy2 = 0, fz2 = 0, ya2 = 0, mba2 = 0;
        auto flush = [&]() {                                           // warp-uniform
            if (cur < 0) return;
            float lo, hi;
            un2(part2, lo, hi);
            const float part = lo + hi;
            const __nv_bfloat16 pb = __float2bfloat16_rn(part);
            if (!BWD) {
                if (a.m16_out) a.m16_out[(size_t)(g0 + cur) * kF + tt] = *reinterpret_cast<const uint16_t*>(&pb);
                else a.m_out[(size_t)(g0 + cur) * kF + tt] = part;
            } else {
                if (a.ybar16_out) a.ybar16_out[(size_t)(g0 + cur) * kF + tt] = *reinterpret_cast<const uint16_t*>(&pb);
                else if (a.ybar) a.ybar[(size_t)(g0 + cur) * kF + tt] = part;
                float fx, fy, fz;
                un2(fx2, lo, hi); fx = lo + hi; un2(fy2, lo, hi); fy = lo + hi; un2(fz2, lo, hi); fz = lo + hi;
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) {
                    fx += __shfl_xor_sync(0xffffffffu, fx, o); fy += __shfl_xor_sync(0xffffffffu, fy, o); fz += __shfl_xor_sync(0xffffffffu, fz, o);
                }
                if (lane == 0) { float* fp = fpart + (cur * 4 + wq) * 3; fp[0] = fx; fp[1] = fy; fp[2] = fz; }
            }
        };

        // ---- prologue: records of tiles 0 and 1, radial basis and MMA1 of tile 0
        if (ntiles > 0) fetch_records(0);
        if (ntiles > 1) fetch_records(1);
        cp_async_commit();
        if (ntiles > 0) { wait_records(0); stage_basis(0); publish_b1_and_mma1(); }

        for (int t = 0; t < ntiles; ++t) {
            const int ng = min(GPT, G - t * GPT);                      // groups of this tile
            // This warp is done with the epilogue of tile t-1, so its gather stage is free.  Record buffer (t+2) % 4 was last
            // read by the epilogue of tile t-2, which every warp of the team finished before it signalled B2(t-1) ready, i.e.
            // before MMA2(t-1) completed, which this warp has waited for.
            wait_records(t);
            issue_gathers(t);                                          // land under the activation, MMA2(t) and the staging of tile t+1
            cp_async_commit();
            if (t + 2 < ntiles) fetch_records(t + 2);
            cp_async_commit();                                         // (possibly empty) most recent group: not waited for below
            // ---- activation (M3) of tile t: D1 -> B2, MN-major: (n, k) at (n/8)*2048 + (k/8)*128 + (k%8)*16 + (n%8)*2, k = this thread's row
            mbar_wait(bar1, phase1); phase1 ^= 1u;
            tc_fence_after();
            for (int gq = 0; gq < ng; ++gq) {
                const int c0 = gq * kGE;
                uint32_t v[16], vp[16];
                tmem_ld16(tl1 + c0, v);
                if (BWD) tmem_ld16(tl1 + NT + c0, vp);
                tmem_wait_ld();
                uint32_t pa[8], pt[8];
                const f32x2 half2 = pk2(0.5f, 0.5f), p3 = pk2(kP3, kP3), p2 = pk2(kP2, kP2), p1 = pk2(kP1, kP1), p0 = pk2(kP0, kP0);
#pragma unroll
                for (int c = 0; c < 16; c += 2) {
                    // W_f1 is packed as W_f1 / 2 and W_f2 as 2 W_f2 (exact in bf16): the accumulator holds x / 2 and the
                    // operand written here is ssp(x) / 2 = max(x/2, 0) + a P(a), a = tanh(|x| / 2)  (and logistic(x) x' / 2)
                    const float h0 = __uint_as_float(v[c]), h1 = __uint_as_float(v[c + 1]);
                    float t0, t1, a0, a1;
                    if (BWD) { t0 = tanhf_approx(h0); t1 = tanhf_approx(h1); a0 = fabsf(t0); a1 = fabsf(t1); }
                    else { a0 = tanhf_approx(fabsf(h0)); a1 = tanhf_approx(fabsf(h1)); }
                    const f32x2 a2 = pk2(a0, a1);
                    f32x2 r2 = fma2(p3, a2, p2);
                    r2 = fma2(r2, a2, p1);
                    r2 = fma2(r2, a2, p0);
                    pa[c >> 1] = pack_bf16(fma2(r2, a2, pk2(fmaxf(h0, 0.f), fmaxf(h1, 0.f))));
                    if (BWD) pt[c >> 1] = pack_bf16(mul2(fma2(pk2(t0, t1), half2, half2), pk2u(vp[c], vp[c + 1])));
                }
                uint8_t* d0 = B2 + (c0 >> 3) * 2048 + tt * 16;
                *reinterpret_cast<uint4*>(d0) = make_uint4(pa[0], pa[1], pa[2], pa[3]);
                *reinterpret_cast<uint4*>(d0 + 2048) = make_uint4(pa[4], pa[5], pa[6], pa[7]);
                if (BWD) {
                    uint8_t* d1 = B2 + ((NT + c0) >> 3) * 2048 + tt * 16;
                    *reinterpret_cast<uint4*>(d1) = make_uint4(pt[0], pt[1], pt[2], pt[3]);
                    *reinterpret_cast<uint4*>(d1 + 2048) = make_uint4(pt[4], pt[5], pt[6], pt[7]);
                }
            }
            tc_fence_before();
            fence_async_smem();
            warp_arrive(rdy2, lane);                                   // my rows of B2 are written, I am done with D1 (and, earlier, with D2 of tile t-1)
            // ---- radial basis and MMA1 of tile t+1 (its records arrived an iteration ago) while MMA2(t) runs
            if (t + 1 < ntiles) { wait_records(t + 1); stage_basis(t + 1); publish_b1_and_mma1(); }
            // ---- epilogue of tile t: cutoff, cfconv products and their adjoints; per-atom sums stay in this thread's registers
            asm volatile("cp.async.wait_group 1;" ::: "memory");        // this thread's gathers of tile t have landed
            __syncwarp();                                              // ... and the rest of the warp's (a warp gathers only what it reads)
            mbar_wait(bar2, phase2); phase2 ^= 1u;
            tc_fence_after();
            const float* rt = recs + ((gt0 + t) & (kRecBufs - 1)) * RECF;
            for (int gq = 0; gq < ng; ++gq) {
                const int c0 = gq * kGE;
                const int at = gatom[t * GPT + gq];
                uint32_t v[16], vp[16];
                tmem_ld16(tl2 + c0, v);
                if (BWD) tmem_ld16(tl2 + NT + c0, vp);
                if (at != cur) {
                    flush(); cur = at; part2 = 0;
                    if (BWD) {
                        fx2 = fy2 = fz2 = 0;
                        const uint32_t wd = *reinterpret_cast<const uint32_t*>(own_w + gq * 128 + lane * 4);
                        ya2 = pk2u(wd << 16, wd << 16); mba2 = pk2u(wd & 0xFFFF0000u, wd & 0xFFFF0000u);
                    }
                }
                tmem_wait_ld();
                const float* rg = rt + gq * LSD_REC_GROUP_FLOATS;      // fields x 16 slots of this group
#pragma unroll
                for (int c4 = 0; c4 < 16; c4 += 4) {
                    const float4 fc4 = *reinterpret_cast<const float4*>(rg + LSD_REC_FC * 16 + c4);
                    if (!BWD) {
                        const uint8_t* sy = stage_w + (c0 + c4) * SEG + lane * 2;
#pragma unroll
                        for (int h = 0; h < 4; h += 2) {
                            const uint32_t y0 = *reinterpret_cast<const uint16_t*>(sy + h * SEG), y1 = *reinterpret_cast<const uint16_t*>(sy + (h + 1) * SEG);
                            const f32x2 fc2 = h ? pk2(fc4.z, fc4.w) : pk2(fc4.x, fc4.y);
                            part2 = fma2(pk2u(y0 << 16, y1 << 16), mul2(pk2u(v[c4 + h], v[c4 + h + 1]), fc2), part2);
                        }
                    } else {
                        const float4 fp4 = *reinterpret_cast<const float4*>(rg + LSD_REC_FCP * 16 + c4);
                        const float4 ux4 = *reinterpret_cast<const float4*>(rg + LSD_REC_UX * 16 + c4);
                        const float4 uy4 = *reinterpret_cast<const float4*>(rg + LSD_REC_UY * 16 + c4);
                        const float4 uz4 = *reinterpret_cast<const float4*>(rg + LSD_REC_UZ * 16 + c4);
                        const uint8_t* sy = stage_w + (c0 + c4) * SEG + lane * 4;
#pragma unroll
                        for (int h = 0; h < 4; h += 2) {
                            const uint32_t w0 = *reinterpret_cast<const uint32_t*>(sy + h * SEG), w1 = *reinterpret_cast<const uint32_t*>(sy + (h + 1) * SEG);
                            const f32x2 yj2 = pk2u(w0 << 16, w1 << 16), mbj2 = pk2u(w0 & 0xFFFF0000u, w1 & 0xFFFF0000u);
                            const f32x2 lin2 = pk2u(v[c4 + h], v[c4 + h + 1]), linp2 = pk2u(vp[c4 + h], vp[c4 + h + 1]);
                            const f32x2 fc2 = h ? pk2(fc4.z, fc4.w) : pk2(fc4.x, fc4.y), fp2 = h ? pk2(fp4.z, fp4.w) : pk2(fp4.x, fp4.y);
                            const f32x2 ux2 = h ? pk2(ux4.z, ux4.w) : pk2(ux4.x, ux4.y), uy2 = h ? pk2(uy4.z, uy4.w) : pk2(uy4.x, uy4.y);
                            const f32x2 uz2 = h ? pk2(uz4.z, uz4.w) : pk2(uz4.x, uz4.y);
                            const f32x2 w2 = mul2(lin2, fc2), wp2 = fma2(linp2, fc2, mul2(lin2, fp2));
                            part2 = fma2(mbj2, w2, part2);
                            const f32x2 g2 = mul2(fma2(mba2, yj2, mul2(mbj2, ya2)), wp2);
                            fx2 = fma2(g2, ux2, fx2); fy2 = fma2(g2, uy2, fy2); fz2 = fma2(g2, uz2, fz2);
                        }
                    }
                }
            }
            tc_fence_before();
        }
        flush();
        gt0 += (uint32_t)ntiles;
        if (BWD) {
            team_bar(team);
            if (tt < natoms && cnts[tt] > 0) {
                const int i = ci * CH + tt;
                const float* fp = fpart + tt * 4 * 3;
                double sx = 0.0, sy = 0.0, sz = 0.0;
#pragma unroll
                for (int w = 0; w < 4; ++w) { sx += (double)fp[3 * w]; sy += (double)fp[3 * w + 1]; sz += (double)fp[3 * w + 2]; }
                double* Fb = a.Fout + (size_t)b * 3 * n;
                Fb[i] += sx; Fb[n + i] += sy; Fb[2 * n + i] += sz;
            }
        }
    }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base_s), "n"(512));
}

int sm_count() { return lsd_sm_count(); }

}  // namespace

template <int CH> static void launch_edge_tc128_ch(Launcher L, const EdgeArgs& a, bool backward)
{
    static bool configured_dev[64] = {};
    bool& configured = configured_dev[lsd_current_device()];
    if (!configured) {
        cudaFuncSetAttribute(k_edge_tc128<false, CH>, cudaFuncAttributeMaxDynamicSharedMemorySize, Cfg<false>::Smem);
        cudaFuncSetAttribute(k_edge_tc128<true, CH>, cudaFuncAttributeMaxDynamicSharedMemorySize, Cfg<true>::Smem);
        configured = true;
    }
    const int cps = (a.n + CH - 1) / CH;
    const int nchunks = cps * (a.total / a.n);
    const int grid = std::max(1, std::min(sm_count(), nchunks));
    if (backward) k_edge_tc128<true, CH><<<grid, kThreads, Cfg<true>::Smem, L.s>>>(a, cps, nchunks);
    else k_edge_tc128<false, CH><<<grid, kThreads, Cfg<false>::Smem, L.s>>>(a, cps, nchunks);
    note_edge_launch(backward, 2, CH, kThreads, grid, kF);
    LSD_COUNT(L);
}

// small batches (one state of a few thousand atoms) are spread over all teams with chunks of 16 atoms; the sums do not depend
// on the chunking (thread-serial in row order)
void launch_edge_tc128(Launcher L, const EdgeArgs& a, bool backward)
{
    const long chunks64 = (long)((a.n + kCH - 1) / kCH) * (a.total / a.n);
    if (chunks64 < 2L * sm_count() * kTeams) launch_edge_tc128_ch<16>(L, a, backward);
    else launch_edge_tc128_ch<kCH>(L, a, backward);
}
