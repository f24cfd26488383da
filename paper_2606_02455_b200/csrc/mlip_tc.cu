// bf16 tcgen05 filter path (LSD_BF16_TC): the continuous-filter convolution of the SchNet-style MLIP (M5, M9)
// with the two per-edge filter contractions on the 5th-generation tensor cores (sm_100a), fp32 accumulation in TMEM.
//
// Orientation ("channels are rows"): for one tile of edges
//     D1[F x N] = W_f1[F x R] * G^T[R x N]          G   = radial basis rows (and, backward, their r-derivatives)
//     D2[F x N] = W_f2[F x F] * A^T[F x N]          A   = ssp(D1) (and, backward, logistic(D1) . D1')
// so TMEM lane = channel f = thread, TMEM column = edge.  The per-atom sums over edges (m_a, ybar_a, F_a) are then
// serial sums inside one thread in the order of the atom's sorted neighbour row (deterministic, independent of the
// batch and of the tiling), and every per-channel operand of the epilogue is read from shared memory.
//
// Widths below 128 fill the 128 accumulator rows with Q = 128 / F independent edge sets: row q F + f is channel f of
// set q.  The A operand of set q is a 128-row window into [128-F zero rows ; W ; 128-F zero rows] that puts W at rows
// q F.., so one MMA per set and K-slice accumulates D[q F + f, n] = sum_k W[f, k] B_q[k, n] and adds exact zeros
// elsewhere (all operand buffers are zero-initialised and only ever hold finite values).
//
// One persistent CTA per SM, 4 teams of 128 threads.  The weights (K-major canonical no-swizzle layout, packed on the
// host) are resident in shared memory and shared by the teams; each team owns 64 TMEM columns, one B-operand buffer
// and one gather stage, and walks chunks of 64 consecutive atoms of one state (set q owns atoms q 64/Q ..).  An
// atom's row is cut into groups of 16 edge slots (the last one padded with zero records), so a group never straddles
// two atoms; a tile is GPT groups per set.  Per tile and team:
//     cp.async: edge records of the NEXT tile, bf16 feature rows y_j (mbar_j) of THIS tile  -> smem (lands under the MMAs)
//     radial basis -> smem (B1, K-major)                 | MMA1 -> TMEM
//     TMEM -> activation -> smem (B2, MN-major, bf16)    | MMA2 -> TMEM (same columns)
//     TMEM -> cutoff, cfconv products and adjoints, per-atom accumulation in registers.
// The phases of different teams overlap (MUFU-bound activation of one team with the FMA/LSU-bound epilogue of another,
// both with the tensor pipe).  Edge geometry comes from the records k_compact wrote once per batched evaluation.
#include <cuda_bf16.h>
#include <algorithm>
#include "lsd_internal.h"

namespace {

constexpr int kR = LSD_NRBF;            // 32 = K of the first contraction (per set)
constexpr int kTeams = 4;
constexpr int kTT = 128;                // threads per team = accumulator rows
constexpr int kThreadsTC = kTeams * kTT;
constexpr int kCH = 64;                 // atoms per chunk (buffers are sized for it; small batches use chunks of 16, see launch_edge_tc_f)
constexpr int kGE = 16;                 // edge slots per group
constexpr int kMaxGroups = kCH * (512 / kGE);   // rows hold at most 512 slots (neighbor.cu)

template <int F, bool BWD> struct TcCfg {
    static constexpr int Q = 128 / F;                                   // edge sets
    static constexpr int GPT = F == 128 ? (BWD ? 2 : 4) : (BWD ? 1 : 2);   // groups per tile and set
    static constexpr int NT = GPT * kGE;                                // edges per tile and set
    static constexpr int NCOLS = NT * (BWD ? 2 : 1);                    // MMA N (value [+ tangent] columns)
    static constexpr int ET = Q * NT;                                   // edges per tile
    static constexpr int ZROWS = 256 - F;                               // rows of the padded weight images
    static constexpr int W1Bytes = ZROWS * kR * 2;
    static constexpr int W2Bytes = ZROWS * F * 2;
    static constexpr int B2Bytes = NCOLS * 128 * 2;
    static constexpr int B1Bytes = NCOLS * Q * kR * 2;
    static constexpr int StageBytes = ET * F * 2 * (BWD ? 2 : 1);
    static constexpr int OwnBytes = BWD ? Q * GPT * 2 * F * 2 : 0;
    static constexpr int RecBytes = 3 * ET * 32;                        // three tiles of record groups in flight
    static constexpr int PrefBytes = 272, CntBytes = kCH * 4;
    static constexpr int FpartBytes = BWD ? kCH * (F / 32) * 3 * 4 : 0;
    static constexpr int TeamBytes = B2Bytes + B1Bytes + StageBytes + OwnBytes + RecBytes + PrefBytes + CntBytes + kMaxGroups + FpartBytes;
    static constexpr int Smem = W1Bytes + W2Bytes + kTeams * TeamBytes;
    static_assert(Smem + 256 <= 227 * 1024, "shared memory budget");
    static_assert(TeamBytes % 16 == 0 && W1Bytes % 16 == 0 && W2Bytes % 16 == 0, "regions stay 16-byte aligned");
    static_assert(NCOLS <= 64 && NCOLS % 16 == 0, "TMEM columns per team and accumulator");
};

constexpr float kLn2 = 0.69314718055994530942f;
constexpr float kLog2e = 1.44269504088896340736f;

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ float ex2f(float x) { float y; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float lg2f(float x) { float y; asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float tanhf_approx(float x) { float y; asm("tanh.approx.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ uint32_t pack_bf16(float lo, float hi)
{
    __nv_bfloat162 v = __floats2bfloat162_rn(lo, hi);
    return *reinterpret_cast<uint32_t*>(&v);
}
__device__ __forceinline__ float bf16_ld(const uint8_t* p) { return __uint_as_float((uint32_t)(*reinterpret_cast<const uint16_t*>(p)) << 16); }

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
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2, %3;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(ok) : "r"(bar), "r"(parity), "r"(20000u) : "memory");       // suspend-time hint: sleep instead of spinning
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
__device__ __forceinline__ void tmem_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
// 16-byte asynchronous copy global -> shared, L2 only; src_bytes = 0 writes zeros (padding slots)
__device__ __forceinline__ void cp_async16(uint32_t dst, const void* src, uint32_t src_bytes)
{
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(dst), "l"(src), "r"(src_bytes) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

template <int F, bool BWD, int CH>
__global__ void __launch_bounds__(kThreadsTC, 1)
k_edge_tc(EdgeArgs a, int chunks_per_state, int nchunks)
{
    static_assert(CH <= kCH && CH % (128 / F) == 0, "chunk size");
    using C = TcCfg<F, BWD>;
    constexpr int Q = C::Q, GPT = C::GPT, NT = C::NT, NCOLS = C::NCOLS, ET = C::ET;
    constexpr int AQ = CH / Q;                         // atoms per set and chunk
    constexpr int TPE = kTT / ET;                      // threads per edge in the staging phase
    constexpr int KPT = kR / TPE;                      // radial basis functions per staging thread
    constexpr int RCH = F / 8;                         // 16-byte chunks per bf16 feature row
    constexpr int NSW = F >= 64 ? 8 : 4;               // stage swizzle period
    constexpr int RECF = ET * 8;                       // floats per tile of record groups
    static_assert(TPE >= 1 && TPE * ET == kTT, "staging roles");
    extern __shared__ __align__(128) uint8_t smem[];
    __shared__ __align__(8) uint64_t mbar[2 * kTeams];
    __shared__ uint32_t tmem_base_s;
    __shared__ int next_chunk, s_chunk[kTeams];
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31, team = tid >> 7, tt = tid & (kTT - 1);
    const int q = tt / F, f = tt % F;                  // this thread's accumulator row: set q, channel f

    {   // resident A operand images (canonical K-major layout); every other operand buffer starts as zeros
        const uint4* s1 = reinterpret_cast<const uint4*>(a.Wf1_tc);
        const uint4* s2 = reinterpret_cast<const uint4*>(a.Wf2_tc);
        uint4* d1 = reinterpret_cast<uint4*>(smem);
        uint4* d2 = reinterpret_cast<uint4*>(smem + C::W1Bytes);
        for (int i = tid; i < C::W1Bytes / 16; i += kThreadsTC) d1[i] = s1[i];
        for (int i = tid; i < C::W2Bytes / 16; i += kThreadsTC) d2[i] = s2[i];
        uint4* z = reinterpret_cast<uint4*>(smem + C::W1Bytes + C::W2Bytes);
        for (int i = tid; i < kTeams * C::TeamBytes / 16; i += kThreadsTC) z[i] = make_uint4(0u, 0u, 0u, 0u);
    }
    if (tid == 0) {
        for (int t = 0; t < 2 * kTeams; ++t) asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(smem_u32(&mbar[t])));
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

    uint8_t* const tb = smem + C::W1Bytes + C::W2Bytes + team * C::TeamBytes;
    uint8_t* const B2 = tb;                                            // [NCOLS][128 k] MN-major
    uint8_t* const B1 = B2 + C::B2Bytes;                               // [NCOLS][Q*32 k] K-major
    uint8_t* const stage = B1 + C::B1Bytes;
    uint8_t* const own = stage + C::StageBytes;
    float* const recs = reinterpret_cast<float*>(own + C::OwnBytes);   // [3][ET/16 groups][8 fields][16 slots]
    int* const pref = reinterpret_cast<int*>(reinterpret_cast<uint8_t*>(recs) + C::RecBytes);   // first group of every atom of the chunk
    int* const cnts = reinterpret_cast<int*>(reinterpret_cast<uint8_t*>(pref) + C::PrefBytes);
    uint8_t* const gatom = reinterpret_cast<uint8_t*>(cnts) + C::CntBytes;                      // group -> atom of the chunk
    float* const fpart = reinterpret_cast<float*>(gatom + kMaxGroups);
    const uint32_t sW1 = smem_u32(smem), sW2 = smem_u32(smem + C::W1Bytes), sB1 = smem_u32(B1), sB2 = smem_u32(B2);
    const uint32_t bar1 = smem_u32(&mbar[2 * team]), bar2 = smem_u32(&mbar[2 * team + 1]);
    const uint32_t sStage = smem_u32(stage), sOwn = smem_u32(own), sRecs = smem_u32(recs);
    const uint32_t tmem1 = tmem_base_s + (uint32_t)(team * 128), tmem2 = tmem1 + 64;             // D1, D2 accumulators
    const uint32_t lane_sel = (uint32_t)((warp & 3) * 32) << 16;
    const uint32_t tl1 = tmem1 + lane_sel, tl2 = tmem2 + lane_sel;
    const uint32_t idesc1 = make_idesc(128, NCOLS, 0), idesc2 = make_idesc(128, NCOLS, 1);
    uint32_t phase1 = 0, phase2 = 0;
    const int n = a.n;
    const int se = tt / TPE, sp = tt % TPE;            // staging role: edge of the tile (set sq, column sn), part of its row
    const int sq = se / NT, sn = se % NT;
    const int srec = (sq * GPT + sn / kGE) * LSD_REC_GROUP_FLOATS + (sn & (kGE - 1));   // this edge inside a tile of record groups
    const float c2 = -0.5f * kLog2e * a.inv_delta2;
    // gather stage rows are F/8 chunks of 16 B, chunk c of row e stored at c ^ swz(e) (conflict-free cp.async writes);
    // this thread's channel sits in chunk f/8: byte offset inside a row for each value of swz(e)
    int soff[NSW];
#pragma unroll
    for (int k = 0; k < NSW; ++k) soff[k] = (((f >> 3) ^ k) << 4) + (f & 7) * 2;
    auto swz = [](int e) { return F >= 64 ? (e & 7) : ((e >> 1) & 3); };

    for (;;) {
        if (tt == 0) s_chunk[team] = atomicAdd(&next_chunk, 1);
        team_bar(team);
        const int chunk = blockIdx.x + s_chunk[team] * gridDim.x;
        if (chunk >= nchunks) break;
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
            if (out && tt < F) for (int i = 0; i < natoms; ++i) if (cnts[i] == 0) out[(size_t)(g0 + i) * F + tt] = 0.f;
        }
        team_bar(team);
        int gmax = 0;
#pragma unroll
        for (int k = 0; k < Q; ++k) gmax = max(gmax, pref[(k + 1) * AQ] - pref[k * AQ]);
        const int ntiles = (gmax + GPT - 1) / GPT;
        const int gbase = pref[q * AQ], Gq = pref[(q + 1) * AQ] - gbase;      // this thread's set: first group, group count

        // asynchronous copy of the record groups of tile t into buffer t % 3 (zeros for groups behind a set's end)
        auto fetch_records = [&](int t) {
            for (int idx = tt; idx < ET * 2; idx += kTT) {
                const int gs = idx >> 5, chunk16 = idx & 31;           // gs = set * GPT + group of the tile
                const int eq = gs / GPT, gl = t * GPT + gs % GPT;
                const int gb = pref[eq * AQ];
                const float* src = a.recs;
                uint32_t bytes = 0;
                if (gl < pref[(eq + 1) * AQ] - gb) {
                    const int at = gatom[gb + gl];
                    src = a.recs + lsd_rec_index((size_t)(g0 + at), a.cap, (gb + gl - pref[at]) * kGE, 0);
                    bytes = 16;
                }
                cp_async16(sRecs + (uint32_t)(((t % 3) * RECF + gs * LSD_REC_GROUP_FLOATS) * 4 + chunk16 * 16),
                           reinterpret_cast<const uint8_t*>(src) + chunk16 * 16, bytes);
            }
        };
        // radial basis (M1) of tile t -> B1, K-major: (n, k) at (n/8)*Q*512 + (k/8)*128 + (n%8)*16 + (k%8)*2, k = sq*32 + basis index
        auto stage_basis = [&](int t) {
            const float r = recs[(t % 3) * RECF + srec + LSD_REC_R * 16];
            uint32_t gv[KPT / 2], gt[KPT / 2];
#pragma unroll
            for (int k = 0; k < KPT; k += 2) {
                const float x0 = r - (float)(sp * KPT + k) * a.delta, x1 = x0 - a.delta;
                const float v0 = ex2f(c2 * x0 * x0), v1 = ex2f(c2 * x1 * x1);
                gv[k >> 1] = pack_bf16(v0, v1);
                if (BWD) gt[k >> 1] = pack_bf16(-v0 * x0 * a.inv_delta2, -v1 * x1 * a.inv_delta2);
            }
            uint8_t* dst = B1 + (sn >> 3) * (Q * 512) + (sn & 7) * 16 + (sq * 4 + sp * (KPT / 8)) * 128;
#pragma unroll
            for (int kc = 0; kc < KPT / 8; ++kc) *reinterpret_cast<uint4*>(dst + kc * 128) = make_uint4(gv[4 * kc], gv[4 * kc + 1], gv[4 * kc + 2], gv[4 * kc + 3]);
            if (BWD) {
                uint8_t* dt = B1 + ((NT + sn) >> 3) * (Q * 512) + (sn & 7) * 16 + (sq * 4 + sp * (KPT / 8)) * 128;
#pragma unroll
                for (int kc = 0; kc < KPT / 8; ++kc) *reinterpret_cast<uint4*>(dt + kc * 128) = make_uint4(gt[4 * kc], gt[4 * kc + 1], gt[4 * kc + 2], gt[4 * kc + 3]);
            }
        };
        auto issue_mma1 = [&]() {                                      // one thread: D1 = sum over sets of window(W_f1) * B1
            tc_fence_after();
#pragma unroll
            for (int k = 0; k < Q; ++k)
#pragma unroll
                for (int k16 = 0; k16 < kR / 16; ++k16)
                    umma(tmem1, make_desc(sW1 + ((128 - F - k * F) / 8) * 512 + k16 * 256, 128, 512),
                         make_desc(sB1 + (k * 4 + k16 * 2) * 128, 128, Q * 512), idesc1, (k | k16) > 0);
            umma_commit(bar1);
        };
        // bf16 feature rows of tile t (y_j, mbar_j and the groups' own rows) -> gather stage
        auto issue_gathers = [&](int t) {
            const int jrow = __float_as_int(recs[(t % 3) * RECF + srec + LSD_REC_JROW * 16]);
            const uint8_t* sy = reinterpret_cast<const uint8_t*>(a.y16) + (size_t)jrow * (F * 2);
#pragma unroll
            for (int i = 0; i < RCH / TPE; ++i)
                cp_async16(sStage + (uint32_t)(se * (2 * F) + (((TPE * i + sp) ^ swz(se)) << 4)), sy + (TPE * i + sp) * 16, 16);
            if (BWD) {
                const uint8_t* sm = reinterpret_cast<const uint8_t*>(a.mbar16) + (size_t)jrow * (F * 2);
#pragma unroll
                for (int i = 0; i < RCH / TPE; ++i)
                    cp_async16(sStage + (uint32_t)((ET + se) * (2 * F) + (((TPE * i + sp) ^ swz(se)) << 4)), sm + (TPE * i + sp) * 16, 16);
                if (tt < Q * GPT * 2 * RCH) {                          // the groups' own rows (y_a, mbar_a)
                    const int ch = tt % RCH, arr = (tt / RCH) & 1, gs = tt / (2 * RCH);     // gs = set * GPT + group
                    const int oq = gs / GPT, gl = t * GPT + gs % GPT;
                    const int gb = pref[oq * AQ], gq_n = pref[(oq + 1) * AQ] - gb;
                    const size_t arow = (size_t)(g0 + (gq_n > 0 ? gatom[gb + min(gl, gq_n - 1)] : 0));
                    const uint8_t* so = reinterpret_cast<const uint8_t*>(arr ? a.mbar16 : a.y16) + arow * (F * 2) + ch * 16;
                    cp_async16(sOwn + (uint32_t)((gs * 2 + arr) * (2 * F) + ch * 16), so, 16);
                }
            }
        };

        int cur = -1;
        float part = 0.f, ya = 0.f, mba = 0.f, fx = 0.f, fy = 0.f, fz = 0.f;
        auto flush = [&]() {                                           // warp-uniform (a warp belongs to one set)
            if (cur < 0) return;
            if (!BWD) a.m_out[(size_t)(g0 + cur) * F + f] = part;
            else {
                if (a.ybar) a.ybar[(size_t)(g0 + cur) * F + f] = part;
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) {
                    fx += __shfl_xor_sync(0xffffffffu, fx, o); fy += __shfl_xor_sync(0xffffffffu, fy, o); fz += __shfl_xor_sync(0xffffffffu, fz, o);
                }
                if (lane == 0) { float* fp = fpart + (cur * (F / 32) + (f >> 5)) * 3; fp[0] = fx; fp[1] = fy; fp[2] = fz; }
            }
        };

        // ---- prologue: records of tiles 0 and 1, radial basis and MMA1 of tile 0
        if (ntiles > 0) fetch_records(0);
        if (ntiles > 1) fetch_records(1);
        cp_async_commit();
        cp_async_wait_all();
        team_bar(team);
        if (ntiles > 0) {
            stage_basis(0);
            fence_async_smem();
            team_bar(team);
            if (tt == 0) issue_mma1();
        }

        for (int t = 0; t < ntiles; ++t) {
            const int ng = max(0, min(GPT, Gq - t * GPT));             // groups of this tile in this thread's set
            const float* rt = recs + (t % 3) * RECF + (q * GPT) * LSD_REC_GROUP_FLOATS;   // this set's record groups of the tile
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
#pragma unroll
                for (int c = 0; c < 16; c += 2) {
                    float s[2], d[2];
#pragma unroll
                    for (int h = 0; h < 2; ++h) {
                        // W_f1 is packed as W_f1 / 2 and W_f2 as 2 W_f2 (exact in bf16): the accumulator holds x / 2 and the
                        // operand written here is ssp(x) / 2 (and logistic(x) x' / 2)
                        const float hx = __uint_as_float(v[c + h]);
                        const float th = tanhf_approx(hx);                             // logistic(x) = (1 + tanh(x/2)) / 2
                        s[h] = fmaf(-0.5f * kLn2, lg2f(1.f + fabsf(th)), fmaxf(hx, 0.f));   // ssp(x) = max(x,0) - ln(1 + |tanh(x/2)|)
                        if (BWD) d[h] = fmaf(0.5f, th, 0.5f) * __uint_as_float(vp[c + h]);
                    }
                    pa[c >> 1] = pack_bf16(s[0], s[1]);
                    if (BWD) pt[c >> 1] = pack_bf16(d[0], d[1]);
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
            team_bar(team);                                            // B2 complete; everybody is done with tile t-1's stage, D2 and records
            if (tt == 0) {
                tc_fence_after();
#pragma unroll
                for (int k = 0; k < Q; ++k)
#pragma unroll
                    for (int k16 = 0; k16 < F / 16; ++k16)
                        umma(tmem2, make_desc(sW2 + ((128 - F - k * F) / 8) * (F / 8) * 128 + k16 * 256, 128, (F / 8) * 128),
                             make_desc(sB2 + (k * (F / 16) + k16) * 256, 128, 2048), idesc2, (k | k16) > 0);
                umma_commit(bar2);
            }
            issue_gathers(t);                                          // land under MMA2(t) and the staging of tile t+1
            if (t + 2 < ntiles) fetch_records(t + 2);
            cp_async_commit();
            // ---- radial basis and MMA1 of tile t+1 (its records arrived an iteration ago) while MMA2(t) runs
            if (t + 1 < ntiles) {
                stage_basis(t + 1);
                fence_async_smem();
                team_bar(team);
                if (tt == 0) issue_mma1();
            }
            // ---- epilogue of tile t: cutoff, cfconv products and their adjoints; per-atom sums stay in this thread's registers
            cp_async_wait_all();                                       // this thread's gathers (and tile t+2's records) have landed
            mbar_wait(bar2, phase2); phase2 ^= 1u;
            tc_fence_after();
            team_bar(team);                                            // everybody's gathers are visible
            for (int gq = 0; gq < ng; ++gq) {
                const int c0 = gq * kGE;
                const int at = gatom[gbase + t * GPT + gq];
                uint32_t v[16], vp[16];
                tmem_ld16(tl2 + c0, v);
                if (BWD) tmem_ld16(tl2 + NT + c0, vp);
                if (at != cur) {
                    flush(); cur = at; part = 0.f;
                    if (BWD) {
                        fx = fy = fz = 0.f;
                        ya = bf16_ld(own + ((q * GPT + gq) * 2) * (2 * F) + f * 2); mba = bf16_ld(own + ((q * GPT + gq) * 2 + 1) * (2 * F) + f * 2);
                    }
                }
                tmem_wait_ld();
                const float* rg = rt + gq * LSD_REC_GROUP_FLOATS;      // fields x 16 slots of this group
                const uint8_t* sy = stage + (q * NT + c0) * (2 * F);
#pragma unroll
                for (int c4 = 0; c4 < 16; c4 += 4) {
                    const float4 fc4 = *reinterpret_cast<const float4*>(rg + LSD_REC_FC * 16 + c4);
                    const float fcs[4] = {fc4.x, fc4.y, fc4.z, fc4.w};
                    if (!BWD) {
#pragma unroll
                        for (int c = 0; c < 4; ++c) {
                            const float yj = bf16_ld(sy + (c4 + c) * (2 * F) + soff[swz(c4 + c)]);
                            part = fmaf(yj, __uint_as_float(v[c4 + c]) * fcs[c], part);
                        }
                    } else {
                        const float4 fp4 = *reinterpret_cast<const float4*>(rg + LSD_REC_FCP * 16 + c4);
                        const float4 ux4 = *reinterpret_cast<const float4*>(rg + LSD_REC_UX * 16 + c4);
                        const float4 uy4 = *reinterpret_cast<const float4*>(rg + LSD_REC_UY * 16 + c4);
                        const float4 uz4 = *reinterpret_cast<const float4*>(rg + LSD_REC_UZ * 16 + c4);
                        const float fps[4] = {fp4.x, fp4.y, fp4.z, fp4.w}, uxs[4] = {ux4.x, ux4.y, ux4.z, ux4.w};
                        const float uys[4] = {uy4.x, uy4.y, uy4.z, uy4.w}, uzs[4] = {uz4.x, uz4.y, uz4.z, uz4.w};
#pragma unroll
                        for (int c = 0; c < 4; ++c) {
                            const float yj = bf16_ld(sy + (c4 + c) * (2 * F) + soff[swz(c4 + c)]);
                            const float mbj = bf16_ld(sy + (ET + c4 + c) * (2 * F) + soff[swz(c4 + c)]);
                            const float lin = __uint_as_float(v[c4 + c]), linp = __uint_as_float(vp[c4 + c]);
                            const float w = lin * fcs[c], wp = fmaf(linp, fcs[c], lin * fps[c]);
                            part = fmaf(mbj, w, part);
                            const float gq_ = fmaf(mba, yj, mbj * ya) * wp;
                            fx = fmaf(gq_, uxs[c], fx); fy = fmaf(gq_, uys[c], fy); fz = fmaf(gq_, uzs[c], fz);
                        }
                    }
                }
            }
            tc_fence_before();
        }
        flush();
        if (BWD) {
            team_bar(team);
            if (tt < natoms && cnts[tt] > 0) {
                const int i = ci * CH + tt;
                const float* fp = fpart + tt * (F / 32) * 3;
                double sx = 0.0, sy = 0.0, sz = 0.0;
#pragma unroll
                for (int w = 0; w < F / 32; ++w) { sx += (double)fp[3 * w]; sy += (double)fp[3 * w + 1]; sz += (double)fp[3 * w + 2]; }
                double* Fb = a.Fout + (size_t)b * 3 * n;
                Fb[i] += sx; Fb[n + i] += sy; Fb[2 * n + i] += sz;
            }
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base_s), "n"(512));
}

int tc_num_sms() { return lsd_sm_count(); }

uint16_t bf16_rne(double x)
{
    float f = (float)x;
    uint32_t u; memcpy(&u, &f, 4);
    if ((u & 0x7F800000u) == 0x7F800000u) return (uint16_t)(u >> 16);
    u += 0x7FFFu + ((u >> 16) & 1u);
    return (uint16_t)(u >> 16);
}

template <int F, int CH>
void launch_edge_tc_ch(Launcher L, const EdgeArgs& a, bool backward)
{
    static bool configured_dev[64] = {};
    bool& configured = configured_dev[lsd_current_device()];
    if (!configured) {
        cudaFuncSetAttribute(k_edge_tc<F, false, CH>, cudaFuncAttributeMaxDynamicSharedMemorySize, TcCfg<F, false>::Smem);
        cudaFuncSetAttribute(k_edge_tc<F, true, CH>, cudaFuncAttributeMaxDynamicSharedMemorySize, TcCfg<F, true>::Smem);
        configured = true;
    }
    const int cps = (a.n + CH - 1) / CH;
    const int nchunks = cps * (a.total / a.n);
    const int grid = std::max(1, std::min(tc_num_sms(), nchunks));
    if (backward) k_edge_tc<F, true, CH><<<grid, kThreadsTC, TcCfg<F, true>::Smem, L.s>>>(a, cps, nchunks);
    else k_edge_tc<F, false, CH><<<grid, kThreadsTC, TcCfg<F, false>::Smem, L.s>>>(a, cps, nchunks);
    note_edge_launch(backward, 1, CH, kThreadsTC, grid, F);
    LSD_COUNT(L);
}

// A team works through a chunk serially (tile after tile), so a small batch (a draft step of a few thousand atoms) is spread
// over all teams of the device with chunks of 16 atoms; the per-atom sums do not depend on the chunking (thread-serial in row
// order), so both variants return identical bits.
template <int F>
void launch_edge_tc_f(Launcher L, const EdgeArgs& a, bool backward)
{
    const long B = a.total / a.n, teams = (long)tc_num_sms() * kTeams;
    const long chunks64 = (long)((a.n + kCH - 1) / kCH) * B, chunks16 = (long)((a.n + 15) / 16) * B;
    if (chunks16 < teams) launch_edge_tc_ch<F, 8>(L, a, backward);            // (a draft step of a few thousand atoms)
    else if (chunks64 < 2 * teams) launch_edge_tc_ch<F, 16>(L, a, backward);
    else launch_edge_tc_ch<F, kCH>(L, a, backward);
}

}  // namespace

bool mlip_tc_supported(const MlipDev& net) { return (net.F == 32 || net.F == 64 || net.F == 128) && net.R == kR; }

// A operand images: [128-F zero rows ; W/2 or 2W ; 128-F zero rows], (m, k) at byte (m/8)*SBO + (k/8)*128 + (m%8)*16 + (k%8)*2,
// SBO = (K/8)*128.  W_f1 is stored halved and W_f2 doubled (both exact in bf16), see the activation phase of k_edge_tc.
void tc_pack_weights(const double* Wf1, const double* Wf2, int F, int R, std::vector<uint16_t>& out1, std::vector<uint16_t>& out2)
{
    const int zrows = 256 - F, pad = 128 - F;
    out1.assign((size_t)zrows * R, 0); out2.assign((size_t)zrows * F, 0);
    for (int r = 0; r < F; ++r) {
        const int m = pad + r;
        for (int k = 0; k < R; ++k)
            out1[((size_t)(m / 8) * (R / 8) * 128 + (k / 8) * 128 + (m % 8) * 16 + (k % 8) * 2) / 2] = bf16_rne(0.5 * Wf1[(size_t)r * R + k]);
        for (int k = 0; k < F; ++k)
            out2[((size_t)(m / 8) * (F / 8) * 128 + (k / 8) * 128 + (m % 8) * 16 + (k % 8) * 2) / 2] = bf16_rne(2.0 * Wf2[(size_t)r * F + k]);
    }
}

void launch_edge_tc(Launcher L, const EdgeArgs& a, int F, bool backward)
{
    switch (F) {
        case 32: launch_edge_tc_f<32>(L, a, backward); break;
        case 64: launch_edge_tc_f<64>(L, a, backward); break;
        case 128: launch_edge_tc_f<128>(L, a, backward); break;
        default: break;
    }
}
