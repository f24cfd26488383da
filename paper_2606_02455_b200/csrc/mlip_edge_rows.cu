// bf16 tcgen05 filter path for width F = 128, second generation of the "edges are rows" schedule (M5, M9, section 4.1):
// continuous-filter convolution forward  m_i = sum_j y_j . w_ij  and its adjoint (ybar_a = sum_j mbar_j . w_aj and the force
// term sum_j [sum_f (mbar_a y_j + mbar_j y_a)_f w'_aj,f] rhat_aj) with the filter w = (W_f2 ssp(W_f1 g(r))) fc(r) and its
// r-derivative evaluated per edge on the tensor cores.
//
// A tile is 128 edge slots (8 record groups of 16 slots, every group belongs to one atom of a 16-atom chunk); a thread owns ONE
// edge (TMEM lane = edge) and walks along the channels, so everything that is per edge (distance, cutoff, unit vector, the
// sum over channels of the force term) lives in that thread's registers.  What is new against mlip_er128.cu / mlip_tc128.cu:
//   * the activations never touch shared memory: the thread writes ssp(x) (and logistic(x) x') as packed bf16 pairs straight
//     into tensor memory (tcgen05.st) and the second contraction takes its A operand from there (tcgen05.mma with [a_tmem]);
//     so does the radial basis.  Shared-memory bandwidth, the binding unit of the first generation, is left to the gathers,
//     the weight images (B operands) and the segment-sum operand P.
//   * neighbour rows are gathered by coalesced 16-byte cp.async (8 lanes = 128 contiguous bytes of one row) into a
//     slab layout [16-byte piece][edge] (slab stride 2064 B: conflict-free for the copies and for the 16-byte reads of the
//     edge's thread), instead of per-thread row loads that cost one L1 wavefront per 16 bytes.  A warp gathers exactly the
//     pieces its own lanes consume, so a cp.async.wait_group + __syncwarp is all the synchronisation the gather needs.
//   * the segment-sum operand P (bf16(lin) . y_j, or . mbar_j in the adjoint) overwrites, in place, the 16-byte cells of the
//     gather stage the same thread has just consumed: P is the stage, re-read by the third contraction D3 = P^T S with
//     S^T[e][a] = fc_e where edge e belongs to atom a (the cutoff rides on the 0/1 segment matrix).
//   * backward: value and tangent of a channel half share one round trip (D = [Dv | Dt], 64 + 64 columns), the contractions
//     run as N = 64 halves so that one team needs 256 TMEM columns (2 teams per SM); the force term is reduced over the
//     channels inside the thread (fp32), over the 16 edges of a group by shuffles, over an atom's groups in list order.
//   * 2 threads per edge (SPLIT = 2): a team is 8 warps, 16 compute warps per SM.
// Determinism / batch invariance: every sum has a fixed order that depends only on the atom's own sorted neighbour row and
// on the chunking of its state (16 consecutive atoms), never on the batch or on the grid.
#include <cuda.h>
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
constexpr int kTeams = 2;
constexpr int kTT = 128;                               // edge slots of a tile
constexpr int kCH = 16;                                // atoms per chunk = columns of D3
constexpr int kGE = 16;                                // edge slots per record group
constexpr int kGPT = kTT / kGE;                        // groups per tile
constexpr int kMaxGroups = kCH * (512 / kGE);
constexpr int kW1Bytes = kF * kR * 2, kW2Bytes = kF * kF * 2;
constexpr int kSlab = 2048 + 16;                       // bytes between slabs of the gather stage (16 B x 128 edges + shift by one bank group)
constexpr int kSTBytes = kCH * kTT * 2;

// TMA (backward only): the stage is four 1024-byte aligned regions [128 edges][128 B] with the 128-byte swizzle (region s =
// bytes 128 s .. 128 s + 127 of the gathered rows), written by cp.async.bulk.tensor gather4 instead of per-lane cp.async
template <bool BWD, bool TMA = false> struct Lay {
    static constexpr int NSLAB = BWD ? 32 : 16;        // 16-byte pieces of a gathered row (bwd: 4 channels x (y, y, mbar, mbar); fwd: 8 channels)
    static constexpr int StageBytes = TMA ? kTT * 512 : ((NSLAB * kSlab + 127) / 128) * 128;
    static constexpr int OwnBytes = BWD ? kCH * 512 : 0;
    static constexpr int AccBytes = BWD ? kTT * kCH * 4 : 0;    // bwd: per (channel, atom) sums over the chunk's tiles (D3 is per tile there)
    static constexpr int MiscBytes = kMaxGroups + 128 /*pref*/ + 128 /*gpart*/ + 1024 /*gx*/ + AccBytes + 5 * kTT * 4 /*recS*/ + 256 /*fsum*/ + (TMA ? 512 : 0);
    static constexpr int TeamBytes = StageBytes + OwnBytes + kSTBytes + MiscBytes;
    static constexpr int Smem = kW1Bytes + kW2Bytes + kTeams * TeamBytes + (TMA ? 1024 : 0);
    static_assert(!TMA || (TeamBytes % 1024 == 0 && (kW1Bytes + kW2Bytes) % 1024 == 0), "swizzled regions stay 1024-byte aligned");
    static_assert(Smem + 1024 <= 227 * 1024, "shared memory budget");
    static_assert(TeamBytes % 16 == 0, "regions stay 16-byte aligned");
};

constexpr float kLog2e = 1.44269504088896340736f;
// -ln(1 + a) / (2 a) on [0, 1] (weighted minimax fit of a P(a), |error| < 3.6e-5)
constexpr float kP0 = -0.49872449040412903f, kP1 = 0.2356506735086441f, kP2 = -0.11284290254116058f, kP3 = 0.02937859483063221f;

// TMEM columns of a team (256 per team)
// bwd: D = [Dv 0..63 | Dt 64..127], A2v 128..191, A2t 192..255; G aliases A2v's second half (160..175), G' A2t's (224..239):
//      they are dead when the activation of the second channel half overwrites them.  D3 of a tile lands in D (0..15).
// fwd: D 0..127, A2 128..191, G 192..207, D3 208..223 (accumulated over the tiles of a chunk)
constexpr uint32_t kColA2v = 128, kColA2t = 192, kColGb = 160, kColGtb = 224, kColGf = 192, kColD3f = 208;

template <int TT> __device__ __forceinline__ void team_bar(int team) { asm volatile("bar.sync %0, %1;" ::"r"(team + 1), "n"(TT) : "memory"); }

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

template <bool BWD, int SPLIT, bool TMA = false>
__global__ void __launch_bounds__(kTeams * kTT * SPLIT, 1)
k_edge_rows(EdgeArgs a, int chunks_per_state, int nchunks)
{
    static_assert(!TMA || (BWD && SPLIT == 2), "the TMA gather is implemented for the two-part backward");
    using L = Lay<BWD, TMA>;
    constexpr int TT = kTT * SPLIT;                    // threads of a team
    constexpr int TW = TT / 32;                        // warps of a team
    constexpr int kThreads = kTeams * TT;
    constexpr int NSLAB = L::NSLAB;
    extern __shared__ __align__(128) uint8_t smem_raw[];
    __shared__ __align__(8) uint64_t mbar[2 * kTeams];
    __shared__ __align__(8) uint64_t gbar_s[kTeams];    // TMA: "the tile's gathered rows have landed" (transaction count)
    __shared__ uint32_t tmem_base_s;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    uint8_t* const smem = TMA ? smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u) : smem_raw;

    {   // resident B operand images (K-major): W_f1 / 2 [128 x 32], 2 W_f2 [128 x 128]; every other buffer starts as zeros
        const uint4* s1 = reinterpret_cast<const uint4*>(a.Wf1_tc);
        const uint4* s2 = reinterpret_cast<const uint4*>(a.Wf2_tc);
        uint4* d1 = reinterpret_cast<uint4*>(smem);
        uint4* d2 = reinterpret_cast<uint4*>(smem + kW1Bytes);
        for (int i = tid; i < kW1Bytes / 16; i += kThreads) d1[i] = s1[i];
        for (int i = tid; i < kW2Bytes / 16; i += kThreads) d2[i] = s2[i];
        uint4* z = reinterpret_cast<uint4*>(smem + kW1Bytes + kW2Bytes);
        for (int i = tid; i < kTeams * L::TeamBytes / 16; i += kThreads) z[i] = make_uint4(0u, 0u, 0u, 0u);
    }
    if (tid == 0) {
        for (int t = 0; t < kTeams; ++t) {
            mbar_init(smem_u32(&mbar[2 * t]), TW);     // "operand published / accumulator consumed": one arrival per warp of the team
            mbar_init(smem_u32(&mbar[2 * t + 1]), 1);  // "contractions of the round complete" (tcgen05.commit)
            if (TMA) mbar_init(smem_u32(&gbar_s[t]), 1);
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

    const int team = __shfl_sync(0xffffffffu, warp, 0) / TW;     // warp-uniform (kept in uniform registers)
    uint8_t* const tbuf = smem + kW1Bytes + kW2Bytes + team * L::TeamBytes;
    const uint32_t sW1 = smem_u32(smem), sW2 = sW1 + kW1Bytes;
    const uint32_t sStage = smem_u32(tbuf), sST = sStage + L::StageBytes + L::OwnBytes;
    const uint32_t rdy = smem_u32(&mbar[2 * team]), done = rdy + 8;
    const uint32_t tb = tmem_base_s + (uint32_t)(team * 256);
    const bool need_sum = BWD ? (a.ybar16_out != nullptr) : true;     // the adjoint of the first block needs the forces only

    {
        const int tt = tid - team * TT;                            // thread of the team
        const int e = tt & (kTT - 1), part = tt >> 7, wq = warp & 3;   // edge slot, channel part, TMEM lane quarter (warp % 4)
        uint8_t* const stage = tbuf;
        uint8_t* const own = stage + L::StageBytes;                // bwd: [16 atoms][512 B] (y, mbar) rows of the chunk's atoms
        uint8_t* const ST = own + L::OwnBytes;
        uint8_t* const gatom = ST + kSTBytes;                      // group -> atom of the chunk
        int* const pref = reinterpret_cast<int*>(gatom + kMaxGroups);             // first group of every atom (17 entries)
        float* const gx = reinterpret_cast<float*>(gatom + kMaxGroups + 128) + 32;
        float* const gpart = gx;                                   // bwd: [2 tile parities][SPLIT parts][8 groups][4] force sums of the tile's groups
        float4* const accs = reinterpret_cast<float4*>(gx + 256);  // bwd: [4][128] float4: sums of channel e for atoms 4 j .. 4 j + 3
        float* const fsum = reinterpret_cast<float*>(tbuf + L::TeamBytes - 256);      // bwd: [16 atoms][4] force sums of the chunk
        float* const recS = reinterpret_cast<float*>(tbuf + L::TeamBytes - 256 - 5 * kTT * 4);   // [5 fields][128]: fc, fc', ux, uy, uz of the tile's slots
        const uint32_t lsel = (uint32_t)(wq * 32) << 16;
        const uint32_t tl = tb + lsel;
        const int n = a.n;
        const float c2 = -0.5f * kLog2e * a.inv_delta2;
        const int my_g = e >> 4, my_s = e & 15;
        // ---- round protocol.  Every warp publishes what it wrote / signals that it is done reading the accumulator (one arrival
        // per warp on `rdy`); the team's last warp (highest warp id: it wins the issue arbitration) waits for all arrivals and one
        // elected lane of it issues the contractions of the round and commits them to `done`; then every warp waits for `done`.
        // No dedicated MMA warps: 16 warps per SM leave 128 registers per thread (a spilled register costs an L2 round trip here,
        // the L1 cache is what the 200 KB of shared memory leave over).
        uint32_t ph = 0, phr = 0, gph = 0;
        const uint32_t gbar = smem_u32(&gbar_s[team]);
        const bool issuer = (warp % TW) == TW - 1;
        const uint32_t id64 = make_idesc(128, 64, 0), id128 = make_idesc(128, 128, 0), id3 = make_idesc(128, kCH, 0) | (1u << 15);
        const uint64_t dW1 = make_desc(sW1, 128, 512), dW2 = make_desc(sW2, 128, 2048);
        // P^T (MN-major): slab layout, or (TMA) two 128-byte swizzled atoms of 64 channel slots [region 0 | region 1]
        const uint64_t dP = TMA ? make_desc_sw128(sStage, kTT * 128, 1024) : make_desc(sStage, 128, BWD ? 2 * kSlab : kSlab);
        const uint64_t dS = make_desc(sST, 128, 2048);
        constexpr uint32_t kPStep = TMA ? 128 : 16;                // descriptor units (16 B) per 16 edges of K
        enum { R_G1H0 = 0, R_G1H1 = 1, R_G2O0 = 2, R_G2O1 = 3, R_G3 = 4, R_F1 = 5, R_F2 = 6, R_F3NEW = 7, R_F3ACC = 8, R_SYNC = 9 };
        int tile_in_chunk = 0;
        auto publish = [&](int kind) {
            tc_fence_before();
            warp_arrive(rdy, lane);
            if (issuer) {
                mbar_wait(rdy, phr); phr ^= 1u;
                tc_fence_after();
                if (kind != R_SYNC && elect_one()) {
                    if (kind == R_G1H0 || kind == R_G1H1) {        // x, x' of channel half h
                        const int h = kind - R_G1H0;
#pragma unroll
                        for (int k16 = 0; k16 < kR / 16; ++k16) {
                            const uint64_t db = dW1 + (uint64_t)((h * 4096 + k16 * 256) >> 4);
                            umma_ts(tb, tb + kColGb + 8 * k16, db, id64, k16 > 0);
                            umma_ts(tb + 64, tb + kColGtb + 8 * k16, db, id64, k16 > 0);
                        }
                    } else if (kind == R_G2O0 || kind == R_G2O1) { // lin, lin' of output channel half o
                        const int o = kind - R_G2O0;
#pragma unroll
                        for (int k16 = 0; k16 < kF / 16; ++k16) {
                            const uint64_t db = dW2 + (uint64_t)((o * 16384 + k16 * 256) >> 4);
                            umma_ts(tb, tb + kColA2v + 8 * k16, db, id64, k16 > 0);
                            umma_ts(tb + 64, tb + kColA2t + 8 * k16, db, id64, k16 > 0);
                        }
                    } else if (kind == R_G3) {                     // D3 (this tile) = P^T S
#pragma unroll
                        for (int k16 = 0; k16 < kTT / 16; ++k16) umma(tb, dP + (uint64_t)(k16 * kPStep), dS + (uint64_t)(k16 * 16), id3, k16 > 0);
                    } else if (kind == R_F1) {
#pragma unroll
                        for (int k16 = 0; k16 < kR / 16; ++k16) umma_ts(tb, tb + kColGf + 8 * k16, dW1 + (uint64_t)(k16 * 16), id128, k16 > 0);
                    } else if (kind == R_F2) {
#pragma unroll
                        for (int k16 = 0; k16 < kF / 16; ++k16) umma_ts(tb, tb + kColA2v + 8 * k16, dW2 + (uint64_t)(k16 * 16), id128, k16 > 0);
                    } else {                                       // D3 (+)= P^T S, accumulated over the tiles of the chunk
#pragma unroll
                        for (int k16 = 0; k16 < kTT / 16; ++k16)
                            umma(tb + kColD3f, dP + (uint64_t)(k16 * 16), dS + (uint64_t)(k16 * 16), id3, (kind == R_F3ACC || k16 > 0) ? 1u : 0u);
                    }
                    umma_commit(done);
                }
                __syncwarp();
                if (BWD && (kind == R_G3 || kind == R_SYNC) && lane < kCH) {
                    // every warp has published the force sums of its groups: atom `lane` adds those of its groups inside this tile,
                    // in list order, part 0 then part 1
                    const int t = tile_in_chunk;
                    const int lo = max(pref[lane], t * kGPT), hi = min(pref[lane + 1], t * kGPT + kGPT);
                    if (lo < hi) {
                        float fax = fsum[4 * lane], fay = fsum[4 * lane + 1], faz = fsum[4 * lane + 2];
                        for (int g = lo; g < hi; ++g) {
#pragma unroll
                            for (int pp = 0; pp < SPLIT; ++pp) {
                                const float* gp = gpart + ((((t & 1) * SPLIT + pp) * kGPT) + (g - t * kGPT)) * 4;
                                fax += gp[0]; fay += gp[1]; faz += gp[2];
                            }
                        }
                        fsum[4 * lane] = fax; fsum[4 * lane + 1] = fay; fsum[4 * lane + 2] = faz;
                    }
                }
                __syncwarp();
            }
        };
        auto await = [&]() { mbar_wait(done, ph); ph ^= 1u; tc_fence_after(); };
        int tr_n = 0;                                                  // debug trace: stamps of the second chunk of block 0, thread 0 of the team
        bool tr_on = false;
#ifdef LSD_EDGE_TRACE_BUILD
#define TRACE(tag) do { if (tr_on && tr_n < 500) { a.trace[team * 1024 + tr_n++] = ((unsigned long long)(tag) << 48) | (clock64() & 0xFFFFFFFFFFFFull); } } while (0)
#else
#define TRACE(tag) do { (void)tr_on; (void)tr_n; } while (0)
#endif
        const uint8_t* const rows = reinterpret_cast<const uint8_t*>(BWD ? (const void*)a.ym16 : (const void*)a.y16);
        constexpr int ROWB = BWD ? 512 : 256;

        for (int chunk = blockIdx.x * kTeams + team; chunk < nchunks; chunk += gridDim.x * kTeams) {
            const int b = chunk / chunks_per_state, ci = chunk - b * chunks_per_state;
            const int g0 = b * n + ci * kCH;                       // first feature row of the chunk
#ifdef LSD_EDGE_TRACE_BUILD
            tr_on = a.trace != nullptr && blockIdx.x == 0 && tt == 0 && chunk == blockIdx.x * kTeams + team + 3 * (int)gridDim.x * kTeams;
#endif
            const int natoms = min(kCH, n - ci * kCH);
            if (tt < 32) {                                         // groups per atom, exclusive scan over the 16 atoms
                const int c = tt < natoms ? a.count[g0 + tt] : 0;
                int v = (c + kGE - 1) / kGE;
#pragma unroll
                for (int o = 1; o < 16; o <<= 1) { const int u = __shfl_up_sync(0xffffffffu, v, o); if (tt >= o) v += u; }
                if (tt < kCH) pref[tt + 1] = v;
                if (tt == 0) pref[0] = 0;
            }
            if (BWD) {                                             // (y, mbar) rows of the chunk's own atoms
                for (int i = tt; i < kCH * 32; i += TT) {
                    const int at = i >> 5;
                    uint4 v = make_uint4(0u, 0u, 0u, 0u);
                    if (at < natoms) v = *reinterpret_cast<const uint4*>(rows + (size_t)(g0 + at) * ROWB + (i & 31) * 16);
                    *reinterpret_cast<uint4*>(own + i * 16) = v;
                }
            }
            team_bar<TT>(team);
            const int G0 = pref[kCH];
#define G (pref[kCH])
            if (tt < kCH) for (int g = pref[tt]; g < pref[tt + 1]; ++g) gatom[g] = (uint8_t)tt;
            const int ntiles = (G0 + kGPT - 1) / kGPT;
            if (ntiles == 0) {                                     // no edges at all: empty sums
                uint16_t* out16 = BWD ? a.ybar16_out : a.m16_out;
                if (out16 && part == 0) for (int i = 0; i < natoms; ++i) out16[(size_t)(g0 + i) * kF + e] = 0;
                team_bar<TT>(team);
                continue;
            }
            team_bar<TT>(team);

            // record of this thread's edge slot in tile t (the zero group behind the chunk's last group): distance, gathered row and
            // atom are fetched one tile ahead; cutoff, slope and unit vector are loaded at the start of their own tile and used at its end
            float r_n; int jrow_n, at_n; const float* rp_n;
            auto load_record = [&](int t) {
                const int gl = t * kGPT + my_g;
                at_n = -1; rp_n = a.rec_zero + my_s;
                if (gl < G) {
                    at_n = gatom[gl];
                    rp_n = a.recs + lsd_rec_index((size_t)(g0 + at_n), a.cap, (gl - pref[at_n]) * kGE + my_s, 0);
                }
                r_n = rp_n[LSD_REC_R * 16];
                jrow_n = at_n >= 0 ? __float_as_int(rp_n[LSD_REC_JROW * 16]) : g0;
            };
            // this warp's pieces of the neighbour rows of its 32 edges -> slabs (8 lanes = 128 contiguous bytes of one row)
            constexpr int NGRP = NSLAB / 8 / SPLIT;                // groups of 8 slabs this part consumes
            auto issue_gathers = [&](int jrow, int g_begin, int g_end) {
#pragma unroll
                for (int gq = 0; gq < NGRP; ++gq) {
                    if (gq < g_begin || gq >= g_end) continue;
                    // bwd: output half o = gq covers slabs 16 o + (16 / SPLIT) part ...; fwd: part owns channels [64 part, +64)
                    const int s0 = BWD ? (SPLIT == 2 ? 16 * gq + 8 * part : 8 * gq) : (SPLIT == 2 ? 8 * part : 8 * gq);
#pragma unroll
                    for (int i = 0; i < 8; ++i) {
                        const int el = 4 * i + (lane >> 3), s = s0 + (lane & 7);
                        const int jr = __shfl_sync(0xffffffffu, jrow, el);
#ifndef LSD_EXP_NOGATHER
                        // .ca: through L1, where the 8 lanes of a row coalesce to 4 sectors (with .cg every 16-byte piece fetched its
                        // own 32-byte sector from L2: twice the traffic, 1.4 x the kernel time)
                        cp_async16_ca(sStage + (uint32_t)(s * kSlab + (32 * wq + el) * 16), rows + (size_t)jr * ROWB + s * 16);
#endif
                    }
                }
            };
            // radial basis (M1) of the thread's edge (and its r-derivative) -> TMEM, packed bf16 pairs along k
            auto stage_basis = [&](float r) {
                constexpr int KH = kR / SPLIT;
                uint32_t gv[KH / 2], gt[KH / 2];
                const f32x2 c22 = pk2(c2, c2), nid = pk2(-a.inv_delta2, -a.inv_delta2);
                const float rh = r - (float)(part * KH) * a.delta;
#pragma unroll
                for (int k = 0; k < KH; k += 2) {
                    const float x0 = rh - (float)k * a.delta, x1 = x0 - a.delta;
                    const f32x2 x2 = pk2(x0, x1);
                    float e0, e1;
                    un2(mul2(mul2(x2, x2), c22), e0, e1);
                    const float v0 = ex2f(e0), v1 = ex2f(e1);
                    gv[k >> 1] = pack_bf16(v0, v1);
                    if (BWD) gt[k >> 1] = pack_bf16(mul2(mul2(pk2(v0, v1), x2), nid));
                }
                const uint32_t cg = (BWD ? kColGb : kColGf) + part * (KH / 2);
                if constexpr (KH == 16) { tmem_st8(tl + cg, gv); if (BWD) tmem_st8(tl + kColGtb + part * (KH / 2), gt); }
                else { tmem_st16(tl + cg, gv); if (BWD) tmem_st16(tl + kColGtb, gt); }
                tmem_wait_st();
            };

            if (BWD) {                                             // sums over edges of channel e for the atoms of this thread's part
#pragma unroll
                for (int j = 0; j < 4 / SPLIT; ++j) accs[(part * (4 / SPLIT) + j) * kTT + e] = make_float4(0.f, 0.f, 0.f, 0.f);
            }
            if (BWD && tt < kCH) { fsum[4 * tt] = 0.f; fsum[4 * tt + 1] = 0.f; fsum[4 * tt + 2] = 0.f; }   // force sum of atom tt
            load_record(0);
            for (int t = 0; t < ntiles; ++t) {
                TRACE(1);
                // TMA: the tile's 128 rows of 512 B by 128 gather4 copies (4 edges x 128 B each): the thread of every fourth edge
                // issues the two segments its part consumes (part p: segments p and 2 + p = channel halves o = 0, 1); a gather4
                // costs its issuing warp ~90 cycles, so they too are issued under the first two round trips
                [[maybe_unused]] const int j1 = TMA ? __shfl_down_sync(0xffffffffu, jrow_n, 1) : 0, j2 = TMA ? __shfl_down_sync(0xffffffffu, jrow_n, 2) : 0,
                                           j3 = TMA ? __shfl_down_sync(0xffffffffu, jrow_n, 3) : 0;
                auto tma_half = [&](int o) {
                    if ((e & 3) == 0) tma_gather4(sStage + (uint32_t)((2 * o + part) * (kTT * 128) + e * 128), a.ym_tmap, (2 * o + part) * 64, jrow_n, j1, j2, j3, gbar);
                };
                if constexpr (TMA) { if (tt == 0) mbar_expect_tx(gbar, (uint32_t)(kTT * 512)); }
                // first contraction first: its round trip runs under the issue of this tile's gathers
                stage_basis(r_n);
                TRACE(2);
                publish(BWD ? R_G1H0 : R_F1);
                TRACE(3);
                if constexpr (TMA) tma_half(0);
                else issue_gathers(jrow_n, 0, BWD ? NGRP / 2 : NGRP);   // bwd: the rows' first channel half (the second: under the next round trip)
                if (part == 0) {                                   // cutoff (slope, unit vector) of the slot: asynchronous 4-byte copies, read at the tile's end
                    const uint32_t d = smem_u32(recS) + (uint32_t)e * 4;
                    cp_async4(d, rp_n + LSD_REC_FC * 16);
                    if (BWD) {
                        cp_async4(d + kTT * 4, rp_n + LSD_REC_FCP * 16); cp_async4(d + 2 * kTT * 4, rp_n + LSD_REC_UX * 16);
                        cp_async4(d + 3 * kTT * 4, rp_n + LSD_REC_UY * 16); cp_async4(d + 4 * kTT * 4, rp_n + LSD_REC_UZ * 16);
                    }
                }
                cp_async_commit();

                if (BWD) {
                    constexpr int NC = 64 / SPLIT;                 // channels of a half this thread handles
                    // ---- activation (M3) of channel half h: [Dv | Dt] -> A2v, A2t
#pragma unroll 1
                    for (int h = 0; h < 2; ++h) {
                        TRACE(4);
                        await();
                        TRACE(5);
                        const uint32_t dcol = (uint32_t)(part * NC);
                        uint32_t pv[NC / 2], pt[NC / 2];
#pragma unroll
                        for (int c0 = 0; c0 < NC; c0 += 16) {
                            uint32_t v[16], vp[16];
                            tmem_ld16(tl + dcol + c0, v);
                            tmem_ld16(tl + 64 + dcol + c0, vp);
                            tmem_wait_ld();
#pragma unroll
                            for (int c = 0; c < 16; c += 2) act_pair<true>(v[c], v[c + 1], vp[c], vp[c + 1], pv[(c0 + c) >> 1], pt[(c0 + c) >> 1]);
                        }
                        const uint32_t acol = (uint32_t)(32 * h + part * (NC / 2));
                        if constexpr (NC == 32) { tmem_st16(tl + kColA2v + acol, pv); tmem_st16(tl + kColA2t + acol, pt); }
                        else {
                            uint32_t lo[16], hi[16];
#pragma unroll
                            for (int i = 0; i < 16; ++i) { lo[i] = pv[i]; hi[i] = pv[16 + i]; }
                            tmem_st16(tl + kColA2v + acol, lo); tmem_st16(tl + kColA2v + acol + 16, hi);
#pragma unroll
                            for (int i = 0; i < 16; ++i) { lo[i] = pt[i]; hi[i] = pt[16 + i]; }
                            tmem_st16(tl + kColA2t + acol, lo); tmem_st16(tl + kColA2t + acol + 16, hi);
                        }
                        tmem_wait_st();
                        TRACE(6);
                        publish(h == 0 ? R_G1H1 : R_G2O0);
                        if (h == 0) { if constexpr (TMA) tma_half(1); else { issue_gathers(jrow_n, NGRP / 2, NGRP); cp_async_commit(); } }
                    }
                    TRACE(7);
                    // ---- epilogue of output half o: P = bf16(lin) . mbar_j (in place), A = sum_f c_f lin'_f, B = sum_f c_f lin_f,
                    //      c = mbar_a y_j + mbar_j y_a (bf16 pairs)
                    asm volatile("cp.async.wait_group 0;" ::: "memory");
                    __syncwarp();
                    if constexpr (TMA) { mbar_wait(gbar, gph); gph ^= 1u; }
                    f32x2 A2 = 0, B2 = 0;
                    const int gl_t = t * kGPT + my_g;
                    const int at = gl_t < G ? (int)gatom[gl_t] : -1;
                    const uint8_t* const ownrow = own + (at >= 0 ? at : 0) * 512;
#pragma unroll 1
                    TRACE(8);
                    for (int o = 0; o < 2; ++o) {
                        await();
                        TRACE(9);
                        const uint32_t dcol = (uint32_t)(part * NC);
                        const int ch0 = 64 * o + part * NC;        // first channel of this thread in this round
#pragma unroll 1
                        for (int c0 = 0; c0 < NC; c0 += 16) {
                            uint32_t v[16], vp[16];
                            tmem_ld16(tl + dcol + c0, v);
                            tmem_ld16(tl + 64 + dcol + c0, vp);
                            tmem_wait_ld();
#pragma unroll
                            for (int q8 = 0; q8 < 2; ++q8) {       // 8 channels = two stage cells -> one P cell
                                const int slab = (ch0 + c0 + 8 * q8) >> 2;
                                // TMA: row e of segment 2 o + part, 16-byte chunks s and s + 1 (swizzled by the row)
                                const int sseg = (c0 + 8 * q8) >> 2;
                                const uint8_t* const srow = stage + (2 * o + part) * (kTT * 128) + e * 128;
                                const uint4 s0v = *reinterpret_cast<const uint4*>(TMA ? srow + ((sseg ^ (e & 7)) << 4) : stage + slab * kSlab + e * 16);
                                const uint4 s1v = *reinterpret_cast<const uint4*>(TMA ? srow + (((sseg + 1) ^ (e & 7)) << 4) : stage + (slab + 1) * kSlab + e * 16);
                                const uint4 o0v = *reinterpret_cast<const uint4*>(ownrow + slab * 16);
                                const uint4 o1v = *reinterpret_cast<const uint4*>(ownrow + (slab + 1) * 16);
                                const uint32_t yj[4] = {s0v.x, s0v.z, s1v.x, s1v.z}, mj[4] = {s0v.y, s0v.w, s1v.y, s1v.w};
                                const uint32_t ya[4] = {o0v.x, o0v.z, o1v.x, o1v.z}, ma[4] = {o0v.y, o0v.w, o1v.y, o1v.w};
                                uint32_t pw[4];
#pragma unroll
                                for (int i = 0; i < 4; ++i) {
                                    const int c = 8 * q8 + 2 * i;
                                    const f32x2 cf = bf2_to_f2(bfma2(ma[i], yj[i], bmul2(mj[i], ya[i])));
                                    A2 = fma2(cf, pk2u(vp[c], vp[c + 1]), A2);
                                    B2 = fma2(cf, pk2u(v[c], v[c + 1]), B2);
                                    pw[i] = bmul2(pack_bf16(__uint_as_float(v[c]), __uint_as_float(v[c + 1])), mj[i]);
                                }
                                // P cell of these 8 channels: in place (TMA: chunk 4 o + .. of the part's atom = region `part`, whose
                                // chunks this thread has consumed already: o = 0 reads region `part` itself, ahead of the writes)
                                uint8_t* const pcell = TMA ? stage + part * (kTT * 128) + e * 128 + (((4 * o + ((c0 + 8 * q8) >> 3)) ^ (e & 7)) << 4)
                                                           : stage + slab * kSlab + e * 16;
                                if (need_sum) *reinterpret_cast<uint4*>(pcell) = make_uint4(pw[0], pw[1], pw[2], pw[3]);
                            }
                        }
                        TRACE(10);
                        if (o == 0) publish(R_G2O1);                   // (P becomes visible to the contraction by the fence before G3)
                    }
                    // ---- force term of the edge, summed over the 16 edges of its group
                    float Al, Ah, Bl, Bh;
                    un2(A2, Al, Ah); un2(B2, Bl, Bh);
                    const float As = Al + Ah, Bs = Bl + Bh;        // this part's channels
                    const float fc = recS[e];
                    {
                        const float g = fc * As + recS[kTT + e] * Bs;
                        float fx = g * recS[2 * kTT + e], fy = g * recS[3 * kTT + e], fz = g * recS[4 * kTT + e];
#pragma unroll
                        for (int o = 8; o > 0; o >>= 1) {
                            fx += __shfl_xor_sync(0xffffffffu, fx, o); fy += __shfl_xor_sync(0xffffffffu, fy, o); fz += __shfl_xor_sync(0xffffffffu, fz, o);
                        }
                        if (my_s == 0) { float* gp = gpart + ((((t & 1) * SPLIT + part) * kGPT) + my_g) * 4; gp[0] = fx; gp[1] = fy; gp[2] = fz; }
                        if (need_sum && part == 0 && at >= 0) {    // S^T[e][at] = fc
                            const __nv_bfloat16 fb = __float2bfloat16_rn(fc);
                            *reinterpret_cast<uint16_t*>(ST + (at >> 3) * 2048 + (e >> 3) * 128 + (at & 7) * 16 + (e & 7) * 2) = *reinterpret_cast<const uint16_t*>(&fb);
                        }
                    }
                    TRACE(11);
                    if (t + 1 < ntiles) load_record(t + 1);        // lands under the last round trip
                    tile_in_chunk = t;
                    if (!need_sum) publish(R_SYNC);                // the issuing warp adds the groups' force sums
                    if (need_sum) {
                        fence_async_smem();
                        publish(R_G3);                             // -> D3 = P^T S
                        await();
                        TRACE(12);
                        constexpr int NA = kCH / SPLIT;
                        uint32_t v[NA];
                        if constexpr (NA == 8) tmem_ld8(tl + part * 8, v); else tmem_ld16(tl, v);
                        tmem_wait_ld();
#pragma unroll
                        for (int j = 0; j < NA / 4; ++j) {
                            float4 s4 = accs[(part * (NA / 4) + j) * kTT + e];
                            s4.x += __uint_as_float(v[4 * j]); s4.y += __uint_as_float(v[4 * j + 1]); s4.z += __uint_as_float(v[4 * j + 2]); s4.w += __uint_as_float(v[4 * j + 3]);
                            accs[(part * (NA / 4) + j) * kTT + e] = s4;
                        }
                        if (part == 0 && at >= 0) *reinterpret_cast<uint16_t*>(ST + (at >> 3) * 2048 + (e >> 3) * 128 + (at & 7) * 16 + (e & 7) * 2) = 0;
                    }
                    TRACE(13);
                } else {
                    constexpr int NC = kF / SPLIT;                 // channels this thread handles: [NC part, NC part + NC)
                    // ---- activation (M3): D -> A2
                    await();
#pragma unroll
                    for (int c0 = 0; c0 < NC; c0 += 32) {
                        uint32_t pv[16], dummy;
#pragma unroll
                        for (int c1 = 0; c1 < 32; c1 += 16) {
                            uint32_t v[16];
                            tmem_ld16(tl + part * NC + c0 + c1, v);
                            tmem_wait_ld();
#pragma unroll
                            for (int c = 0; c < 16; c += 2) act_pair<false>(v[c], v[c + 1], 0u, 0u, pv[(c1 + c) >> 1], dummy);
                        }
                        tmem_st16(tl + kColA2v + (part * NC + c0) / 2, pv);
                    }
                    tmem_wait_st();
                    publish(R_F2);
                    // ---- epilogue: P = bf16(lin) . y_j, in place (8 channels = one 16-byte cell)
                    asm volatile("cp.async.wait_group 0;" ::: "memory");
                    __syncwarp();
                    await();
#pragma unroll
                    for (int c0 = 0; c0 < NC; c0 += 16) {
                        uint32_t v[16];
                        tmem_ld16(tl + part * NC + c0, v);
                        tmem_wait_ld();
#pragma unroll
                        for (int q8 = 0; q8 < 2; ++q8) {
                            uint8_t* cell = stage + ((part * NC + c0 + 8 * q8) >> 3) * kSlab + e * 16;
                            const uint4 y = *reinterpret_cast<const uint4*>(cell);
                            uint4 p;
                            p.x = bmul2(pack_bf16(__uint_as_float(v[8 * q8]), __uint_as_float(v[8 * q8 + 1])), y.x);
                            p.y = bmul2(pack_bf16(__uint_as_float(v[8 * q8 + 2]), __uint_as_float(v[8 * q8 + 3])), y.y);
                            p.z = bmul2(pack_bf16(__uint_as_float(v[8 * q8 + 4]), __uint_as_float(v[8 * q8 + 5])), y.z);
                            p.w = bmul2(pack_bf16(__uint_as_float(v[8 * q8 + 6]), __uint_as_float(v[8 * q8 + 7])), y.w);
                            *reinterpret_cast<uint4*>(cell) = p;
                        }
                    }
                    const int gl_t = t * kGPT + my_g;
                    const int at = gl_t < G ? (int)gatom[gl_t] : -1;
                    if (part == 0 && at >= 0) {                    // S^T[e][at] = fc
                        const __nv_bfloat16 fb = __float2bfloat16_rn(recS[e]);
                        *reinterpret_cast<uint16_t*>(ST + (at >> 3) * 2048 + (e >> 3) * 128 + (at & 7) * 16 + (e & 7) * 2) = *reinterpret_cast<const uint16_t*>(&fb);
                    }
                    if (t + 1 < ntiles) load_record(t + 1);        // lands under the last round trip
                    fence_async_smem();
                    publish(t > 0 ? R_F3ACC : R_F3NEW);            // -> D3 += P^T S
                    await();                                       // the stage (P) and S are free again
                    if (part == 0 && at >= 0) *reinterpret_cast<uint16_t*>(ST + (at >> 3) * 2048 + (e >> 3) * 128 + (at & 7) * 16 + (e & 7) * 2) = 0;
                }
            }
            // ---- sums of the chunk -> bf16 rows (thread = channel e, atoms [part NA, part NA + NA))
            {
                constexpr int NA = kCH / SPLIT;
                uint16_t* out16 = BWD ? a.ybar16_out : a.m16_out;
                float acc[NA];
                if (!BWD) {
                    uint32_t v[NA];
                    if constexpr (NA == 8) tmem_ld8(tl + kColD3f + part * 8, v); else tmem_ld16(tl + kColD3f, v);
                    tmem_wait_ld();
#pragma unroll
                    for (int i = 0; i < NA; ++i) acc[i] = __uint_as_float(v[i]);
                } else {
#pragma unroll
                    for (int j = 0; j < NA / 4; ++j) {
                        const float4 s4 = accs[(part * (NA / 4) + j) * kTT + e];
                        acc[4 * j] = s4.x; acc[4 * j + 1] = s4.y; acc[4 * j + 2] = s4.z; acc[4 * j + 3] = s4.w;
                    }
                }
                const int b2 = chunk / chunks_per_state, ci2 = chunk - b2 * chunks_per_state;   // recomputed: nothing chunk-level stays in registers over the tiles
                const int g02 = b2 * n + ci2 * kCH, natoms2 = min(kCH, n - ci2 * kCH);
                if (out16) {
#pragma unroll
                    for (int i = 0; i < NA; ++i) {
                        const int at = part * NA + i;
                        if (at < natoms2) {
                            const __nv_bfloat16 pb = __float2bfloat16_rn(acc[i]);
                            // TMA: contraction row e = 64 part + 8 chunk + i holds channel 64 (chunk >> 2) + 32 part + 8 (chunk & 3) + i
                            const int ch = TMA ? 64 * ((e >> 5) & 1) + 32 * (e >> 6) + (e & 31) : e;
                            out16[(size_t)(g02 + at) * kF + ch] = *reinterpret_cast<const uint16_t*>(&pb);
                        }
                    }
                }
                if (BWD && issuer && lane < natoms2) {           // the issuing warp holds the force sums (lane = atom)
                    const int i = ci2 * kCH + lane;
                    double* Fb = a.Fout + (size_t)b2 * 3 * n;
                    Fb[i] += (double)fsum[4 * lane]; Fb[n + i] += (double)fsum[4 * lane + 1]; Fb[2 * n + i] += (double)fsum[4 * lane + 2];
                }
            }
#undef G
            tc_fence_before();
            team_bar<TT>(team);                                    // pref / gatom / own rows are rewritten by the next chunk
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base_s), "n"(512));
}

}  // namespace

// TMA tensor map over rows of `row_bytes` bytes of 16-bit elements: boxes of 64 elements (128 B) x 1 row (what tile::gather4
// takes), 128-byte swizzle.  The driver entry point is looked up through the runtime (no link against libcuda).
bool lsd_encode_row_tmap(void* host_map_128B, const void* base, size_t rows, int row_bytes)
{
    typedef CUresult (*EncodeFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*, const cuuint32_t*,
                                 const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
    static_assert(sizeof(CUtensorMap) == 128, "tensor map size");
    EncodeFn enc = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", (void**)&enc, cudaEnableDefault, &q) != cudaSuccess || enc == nullptr) { cudaGetLastError(); return false; }
    const cuuint64_t dims[2] = {(cuuint64_t)(row_bytes / 2), (cuuint64_t)rows}, strides[1] = {(cuuint64_t)row_bytes};
    const cuuint32_t box[2] = {64, 1}, es[2] = {1, 1};
    return enc(reinterpret_cast<CUtensorMap*>(host_map_128B), CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void*>(base), dims, strides, box, es,
               CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

namespace {
int device_sm_count()
{
    int dev = 0, sms = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    return sms > 0 ? sms : 148;
}

template <bool BWD, int SPLIT, bool TMA = false> void launch_rows(Launcher L, const EdgeArgs& a)
{
    constexpr int threads = kTeams * kTT * SPLIT;
    cudaFuncSetAttribute(k_edge_rows<BWD, SPLIT, TMA>, cudaFuncAttributeMaxDynamicSharedMemorySize, Lay<BWD, TMA>::Smem);
    const int cps = (a.n + kCH - 1) / kCH;
    const int nchunks = cps * (a.total / a.n);
    const int grid = std::max(1, std::min(device_sm_count(), (nchunks + kTeams - 1) / kTeams));
#ifdef LSD_EDGE_TRACE_BUILD                                         // debug builds only: this block allocates and synchronises inside a launch
    static const bool trace_on = [] { const char* v = getenv("LSD_EDGE_TRACE"); return v && v[0] == '1'; }();
    static int trace_launch[2] = {0, 0};
    if (trace_on && ++trace_launch[BWD] == 8) {                    // debug: time stamps of one chunk, printed once per direction
        unsigned long long* dbuf = nullptr;
        cudaMalloc(&dbuf, 2048 * 8); cudaMemsetAsync(dbuf, 0, 2048 * 8, L.s);
        EdgeArgs at = a; at.trace = dbuf;
        k_edge_rows<BWD, SPLIT, TMA><<<grid, threads, Lay<BWD, TMA>::Smem, L.s>>>(at, cps, nchunks);
        cudaStreamSynchronize(L.s);
        std::vector<unsigned long long> h(2048);
        cudaMemcpy(h.data(), dbuf, 2048 * 8, cudaMemcpyDeviceToHost); cudaFree(dbuf);
        for (int tm = 0; tm < kTeams; ++tm) {
            fprintf(stderr, "[edge trace] %s team %d:", BWD ? "bwd" : "fwd", tm);
            unsigned long long t0 = h[tm * 1024] & 0xFFFFFFFFFFFFull, prev = t0;
            for (int i = 0; i < 500 && h[tm * 1024 + i]; ++i) {
                const unsigned long long c = h[tm * 1024 + i] & 0xFFFFFFFFFFFFull; const int tag = (int)(h[tm * 1024 + i] >> 48);
                if (tag == 1) fprintf(stderr, "\n   tile @%llu:", c - t0);
                fprintf(stderr, " %d:+%llu", tag, c - prev); prev = c;
            }
            fprintf(stderr, "\n");
        }
        LSD_COUNT(L);
        return;
    }
#endif
    k_edge_rows<BWD, SPLIT, TMA><<<grid, threads, Lay<BWD, TMA>::Smem, L.s>>>(a, cps, nchunks);
    note_edge_launch(BWD, TMA ? 9 : 4, kCH, threads, grid, kF);
    LSD_COUNT(L);
}

}  // namespace

// a.ym16 (backward) must be in the pair layout: per channel pair (f, f+1) the words (y_f | y_f+1 << 16), (mbar_f | mbar_f+1 << 16)
void launch_edge_rows(Launcher L, const EdgeArgs& a, bool backward)
{
    // LSD_EDGE_TMA: the backward gathers its rows with TMA gather4 (needs the tensor map of alloc_work)
    static const bool tma = [] { const char* v = getenv("LSD_EDGE_TMA"); return v != nullptr && v[0] != '0'; }();
    if (backward && tma && a.ym_tmap) { launch_rows<true, 2, true>(L, a); return; }
    if (backward) launch_rows<true, 2>(L, a); else launch_rows<false, 2>(L, a);
}
