// C ABI of liblsd_b200.so (include/lsd.h): context, window slots, call sequencing.  No torch types, no CPU fallback.
#include <algorithm>
#include <chrono>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <map>
#include <new>

#include "lsd_internal.h"

namespace {

thread_local std::string g_init_error;

// A launch sequence that is identical from window to window (same slot, same K) is captured once into a CUDA graph and
// replayed: the small configurations are launch-bound (cfg2: ~200 launches per window of 22 atoms).
struct GraphEntry { cudaGraphExec_t exec = nullptr; int64_t launches = 0; int uses = 0; };

struct WindowSlot {
    int K = 0;
    int drafted = 0, verified = 0;
    uint64_t n0 = 0;                                         // step index of the window's start state ...
    uint64_t* n0_dev = nullptr;                              // ... and its device copy, read by the Philox-keyed kernels
    double* dF = nullptr;                                    // [3][n] EC cache as it stood when this window was drafted (Alg. 3)
    std::map<int, GraphEntry> g_roll, g_verify, g_transport, g_plain; // by K (g_plain: by 2 K + which)
    double *qstart = nullptr, *pstart = nullptr;             // [3][n]
    double *qhalf = nullptr, *Ft = nullptr, *yq = nullptr, *yp = nullptr;   // [kmax][3][n]
    double* Fprior = nullptr;                                // [kmax][3][n] prior part of the draft forces (kept when the target has the same prior)
    int prior_valid = 0;
    int* img = nullptr;                                      // [n] images of the reference (start) state
    VerletList vl_mlip, vl_pair;
    int* flags = nullptr;
    cudaEvent_t ev_drafted = nullptr;
};

}  // namespace

struct lsd_ctx {
    lsd_config cfg{};
    SysDev sys;
    PotDev pot[2];
    std::vector<void*> allocs;
    std::vector<void*> list_allocs;                          // neighbour-list rows: freed and re-made by setup_lists (lsd_set_skin)
    bool alloc_lists = false;                                // dalloc files under list_allocs
    double slack = 0.0;                                      // force slack eps_F of App. H (0 = off: exact)
    bool tiny_draft_lists_stale = true;                      // tiny contexts: no lsd_eval_forces(LSD_DRAFT) since the last one-kernel rollout (its rows stay on chip)
    double cap_growth = 1.0;                                 // extra head room of the rows after an overflow (x 1.5 per retry)
    double c1 = 0, b = 0, hdt = 0, kT = 0;
    double *q = nullptr, *p = nullptr;
    int64_t step = 0;
    WindowSlot slot[LSD_MAX_SLOTS];                          // ring of window slots: [verify_idx, verify_idx + pending) are drafted and unverified
    int nslots = 2;                                          // slots in use (lsd_set_window_slots)
    int verify_idx = 0, pending = 0, last_slot = -1, last_K = 0, last_l = 0, last_nc = 0, transported = 0;
    MlipWork work[2];
    CompactList cl_mlip[2], cl_pair[2];
    bool pair_is_mlip[2] = {false, false};                   // every pair term has the network's cutoff: the network's per-state list serves the prior too
    const int* cl_img[2] = {nullptr, nullptr};
    int bmax[2] = {1, 1};
    CellGrid grid;
    double rc_mlip_max = 0, rc_pair_max = 0;
    int cap_mlip = 0, cap_pair = 0;
    double* pair_rcs2 = nullptr;                             // [ns][ns] (largest pair cutoff of draft / target + skin)^2, 0 = the species pair has no pair term
    double* Fg = nullptr;
    double* obabo_p = nullptr;                               // scratch of lsd_get_window_obabo
    double *partial = nullptr, *S1 = nullptr, *S2 = nullptr, *ell = nullptr, *lnu = nullptr, *xi_dbg = nullptr;
    int* reject = nullptr;
    int nblk = 1;
    TransportResult* result = nullptr;
    TransportResult* result_host = nullptr;
    // lsd_eval_forces scratch
    double *q_eval = nullptr, *F_eval = nullptr, *e_eval = nullptr;
    int* img_eval = nullptr; int* flags_eval = nullptr;
    VerletList vl_eval_mlip, vl_eval_pair;
    cudaStream_t side = nullptr;
    int64_t launches = 0;
    int adaptive_k = 0;                                      // window length lsd_run's adaptive mode settled on last
    int ec = 0;                                              // speculative error correction (Alg. 3) on / off
    double* dF = nullptr;                                    // [3][n] EC cache: F - F~(bare) of the last committed step
    bool use_graphs = true;                                  // LSD_GRAPHS=0 disables graph replay
    bool same_prior = false;                                 // draft and target share the classical prior: the verification re-uses the rollout's prior forces
    bool tiny = false;                                       // draft rollout as one kernel launch (tiny_rollout.cu; LSD_TINY=0 disables)
    double* state_host = nullptr;                            // pinned [2][3][n] staging of lsd_set_state / lsd_get_state (small systems: one copy each way, no wait on upload)
    cudaEvent_t ev_state = nullptr;                          // the staged upload has reached q, p
    bool state_in_flight = false;
    std::vector<cudaStream_t> busy;                          // caller streams that may still hold work of this context (lsd_get_state / lsd_set_state wait for these only)
    Prof prof;
    lsd_stats stats{};
    std::string err;
};

namespace {

#define CK(expr)                                                                                             \
    do {                                                                                                     \
        cudaError_t e__ = (expr);                                                                            \
        if (e__ != cudaSuccess) {                                                                            \
            char buf__[512];                                                                                 \
            snprintf(buf__, sizeof buf__, "%s failed: %s (%s:%d)", #expr, cudaGetErrorString(e__), __FILE__, __LINE__); \
            ctx->err = buf__;                                                                                \
            return e__ == cudaErrorMemoryAllocation ? LSD_ERR_OOM : LSD_ERR_CUDA;                            \
        }                                                                                                    \
    } while (0)

lsd_status fail(lsd_ctx* ctx, lsd_status s, const char* msg) { if (ctx) ctx->err = msg; else g_init_error = msg; return s; }

template <typename T> lsd_status dalloc(lsd_ctx* ctx, T** p, size_t count)
{
    void* v = nullptr;
    CK(cudaMalloc(&v, std::max<size_t>(count, 1) * sizeof(T)));
    (ctx->alloc_lists ? ctx->list_allocs : ctx->allocs).push_back(v);
    *p = (T*)v;
    return LSD_OK;
}
template <typename T> lsd_status upload(lsd_ctx* ctx, T** p, const T* host, size_t count)
{
    lsd_status s = dalloc(ctx, p, count);
    if (s) return s;
    if (count) CK(cudaMemcpy(*p, host, count * sizeof(T), cudaMemcpyHostToDevice));
    return LSD_OK;
}
#define TRY(expr) do { lsd_status s__ = (expr); if (s__ != LSD_OK) return s__; } while (0)

Launcher mk(lsd_ctx* ctx, void* stream) { return Launcher{(cudaStream_t)stream, &ctx->launches, &ctx->prof}; }

void note_stream(lsd_ctx* ctx, cudaStream_t st) { if (std::find(ctx->busy.begin(), ctx->busy.end(), st) == ctx->busy.end()) ctx->busy.push_back(st); }
void stream_idle(lsd_ctx* ctx, cudaStream_t st) { ctx->busy.erase(std::remove(ctx->busy.begin(), ctx->busy.end(), st), ctx->busy.end()); }
// wait for the work this context has enqueued (not for the whole device: a state read-back between windows costs one
// stream synchronisation, cfg1's end-to-end window is ~0.1 ms)
lsd_status sync_pending(lsd_ctx* ctx)
{
    for (cudaStream_t st : ctx->busy) CK(cudaStreamSynchronize(st));
    ctx->busy.clear();
    ctx->state_in_flight = false;
    return LSD_OK;
}

void drop_graphs(lsd_ctx* ctx)
{
    for (int s = 0; s < LSD_MAX_SLOTS; ++s)
        for (auto* m : {&ctx->slot[s].g_roll, &ctx->slot[s].g_verify, &ctx->slot[s].g_transport, &ctx->slot[s].g_plain}) {
            for (auto& kv : *m) if (kv.second.exec) cudaGraphExecDestroy(kv.second.exec);
            m->clear();
        }
}

// Runs `body` (stream-ordered launches on `st` only) directly the first time (allocations, function attributes), captures
// it the second time and replays the graph from then on.  Never on the legacy default stream, never while profiling.
template <class Body> lsd_status run_graphed(lsd_ctx* ctx, cudaStream_t st, GraphEntry& g, Body body)
{
    if (!ctx->use_graphs || st == nullptr || ctx->prof.on) return body();
    if (g.uses++ == 0) return body();
    if (!g.exec) {
        const int64_t before = ctx->launches;
        CK(cudaStreamBeginCapture(st, cudaStreamCaptureModeThreadLocal));
        const lsd_status bs = body();
        cudaGraph_t graph = nullptr;
        const cudaError_t ce = cudaStreamEndCapture(st, &graph);
        if (bs != LSD_OK || ce != cudaSuccess || graph == nullptr) {          // not capturable here: fall back to direct launches for good
            if (graph) cudaGraphDestroy(graph);
            cudaGetLastError();
            ctx->use_graphs = false;
            ctx->launches = before;
            return body();
        }
        g.launches = ctx->launches - before;
        ctx->launches = before;
        const cudaError_t ie = cudaGraphInstantiate(&g.exec, graph, 0);
        cudaGraphDestroy(graph);
        if (ie != cudaSuccess) { g.exec = nullptr; cudaGetLastError(); ctx->use_graphs = false; return body(); }
    }
    CK(cudaGraphLaunch(g.exec, st));
    ctx->launches += g.launches;
    return LSD_OK;
}

lsd_status upload_mlip(lsd_ctx* ctx, const lsd_mlip& m, MlipDev& d)
{
    d.F = m.width; d.T = m.n_blocks; d.R = m.n_rbf; d.ns = m.n_species; d.rc = (float)m.cutoff; d.alpha = (float)m.energy_scale;
    const int F = d.F, R = d.R, T = d.T;
    const double* w = m.weights;
    std::vector<float> buf;
    auto up = [&](const double* src, int rows, int cols, bool transpose, float** out) -> lsd_status {
        buf.resize((size_t)rows * cols);
        if (!transpose) for (size_t i = 0; i < buf.size(); ++i) buf[i] = (float)src[i];
        else for (int r = 0; r < rows; ++r) for (int c = 0; c < cols; ++c) buf[(size_t)c * rows + r] = (float)src[(size_t)r * cols + c];
        return upload(ctx, out, buf.data(), buf.size());
    };
    TRY(up(w, m.n_species, F, false, &d.emb));
    const double* blk = w + (size_t)m.n_species * F;
    {   // y table of the first block (fp64 on the host, rounded once)
        std::vector<float> yt((size_t)m.n_species * F);
        const double* Win0 = blk;
        for (int sp = 0; sp < m.n_species; ++sp)
            for (int c = 0; c < F; ++c) {
                double acc = 0.0;
                for (int k = 0; k < F; ++k) acc += Win0[(size_t)c * F + k] * w[(size_t)sp * F + k];
                yt[(size_t)sp * F + c] = (float)acc;
            }
        TRY(upload(ctx, &d.ytab0, yt.data(), yt.size()));
    }
    const size_t per_block = (size_t)4 * F * F + (size_t)F * R;
    d.WinT.resize(T); d.Win.resize(T); d.Wf1T.resize(T); d.Wf2T.resize(T); d.Wo1T.resize(T); d.Wo1.resize(T); d.Wo2T.resize(T); d.Wo2.resize(T);
    for (int t = 0; t < T; ++t) {
        const double* Win = blk + t * per_block; const double* Wf1 = Win + (size_t)F * F; const double* Wf2 = Wf1 + (size_t)F * R;
        const double* Wo1 = Wf2 + (size_t)F * F; const double* Wo2 = Wo1 + (size_t)F * F;
        TRY(up(Win, F, F, true, &d.WinT[t])); TRY(up(Win, F, F, false, &d.Win[t]));
        TRY(up(Wf1, F, R, true, &d.Wf1T[t])); TRY(up(Wf2, F, F, true, &d.Wf2T[t]));
        TRY(up(Wo1, F, F, true, &d.Wo1T[t])); TRY(up(Wo1, F, F, false, &d.Wo1[t]));
        TRY(up(Wo2, F, F, true, &d.Wo2T[t])); TRY(up(Wo2, F, F, false, &d.Wo2[t]));
    }
    if (ctx->cfg.precision == LSD_BF16_TC && mlip_tc_supported(d)) {     // bf16 operands of the tcgen05 filter path
        d.Wf1_bf16.resize(T); d.Wf2_bf16.resize(T);
        std::vector<uint16_t> p1, p2;
        for (int t = 0; t < T; ++t) {
            const double* Wf1 = blk + t * per_block + (size_t)F * F; const double* Wf2 = Wf1 + (size_t)F * R;
            tc_pack_weights(Wf1, Wf2, F, R, p1, p2);
            uint16_t *a = nullptr, *b2 = nullptr;
            TRY(upload(ctx, &a, p1.data(), p1.size())); TRY(upload(ctx, &b2, p2.data(), p2.size()));
            d.Wf1_bf16[t] = a; d.Wf2_bf16[t] = b2;
        }
        if (F == 128) {                                                  // atom-wise layers on the tensor cores
            d.Win_tc.resize(T); d.WinT_tc.resize(T); d.Wo1_tc.resize(T); d.Wo1T_tc.resize(T); d.Wo2_tc.resize(T); d.Wo2T_tc.resize(T);
            auto upk = [&](const double* W, bool tr, void** out) -> lsd_status {
                tc_pack_square128(W, tr, p1);
                uint16_t* dev = nullptr;
                TRY(upload(ctx, &dev, p1.data(), p1.size()));
                *out = dev;
                return LSD_OK;
            };
            for (int t = 0; t < T; ++t) {
                const double* Win = blk + t * per_block; const double* Wo1 = Win + (size_t)2 * F * F + (size_t)F * R; const double* Wo2 = Wo1 + (size_t)F * F;
                TRY(upk(Win, false, &d.Win_tc[t])); TRY(upk(Win, true, &d.WinT_tc[t]));
                TRY(upk(Wo1, false, &d.Wo1_tc[t])); TRY(upk(Wo1, true, &d.Wo1T_tc[t]));
                TRY(upk(Wo2, false, &d.Wo2_tc[t])); TRY(upk(Wo2, true, &d.Wo2T_tc[t]));
            }
            const double* Wr1d = blk + (size_t)T * per_block;
            for (int tr = 0; tr < 2; ++tr) {
                tc_pack_rect128(Wr1d, F / 2, F, tr == 1, p1);
                uint16_t* dev = nullptr;
                TRY(upload(ctx, &dev, p1.data(), p1.size()));
                (tr ? d.Wr1T_tc : d.Wr1_tc) = dev;
            }
        }
    }
    const double* Wr1 = blk + (size_t)T * per_block;
    TRY(up(Wr1, F / 2, F, false, &d.Wr1));
    TRY(up(Wr1 + (size_t)(F / 2) * F, 1, F / 2, false, &d.wr2));
    return LSD_OK;
}

lsd_status upload_potential(lsd_ctx* ctx, const lsd_potential& p, PotDev& d)
{
    d.ns = p.n_species; d.use_bonded = p.use_bonded;
    const int ns = p.n_species;
    TRY(upload(ctx, &d.pair, p.pair, (size_t)ns * ns * LSD_PAIR_COLS));
    std::vector<double> rc2((size_t)ns * ns, 0.0), tether(ns, 0.0);
    d.pair_rcmax = 0.0; d.has_tether = 0;
    for (int a = 0; a < ns * ns; ++a) {
        const double* pp = p.pair + (size_t)a * LSD_PAIR_COLS;
        double rc = 0.0;
        if (pp[0] != 0.0) rc = std::max(rc, pp[2]);
        if (pp[3] != 0.0) rc = std::max(rc, pp[6]);
        rc2[a] = rc * rc;
        d.pair_rcmax = std::max(d.pair_rcmax, rc);
    }
    for (int s = 0; s < ns; ++s) { tether[s] = p.pair[((size_t)s * ns + s) * LSD_PAIR_COLS + 7]; if (tether[s] != 0.0) d.has_tether = 1; }
    TRY(upload(ctx, &d.pair_rc2, rc2.data(), rc2.size()));
    d.pair_rc2_host = rc2;
    TRY(upload(ctx, &d.tether, tether.data(), tether.size()));
    if (p.mlip.width > 0) TRY(upload_mlip(ctx, p.mlip, d.mlip));
    return LSD_OK;
}

lsd_status alloc_verlet(lsd_ctx* ctx, VerletList& vl, int cap, double rc)
{
    vl.cap = cap; vl.rc = rc;
    TRY(dalloc(ctx, &vl.count, ctx->sys.n));
    TRY(dalloc(ctx, &vl.keys, (size_t)ctx->sys.n * cap));
    return LSD_OK;
}
lsd_status alloc_compact(lsd_ctx* ctx, CompactList& cl, int cap, int bmax, bool records)
{
    cl.cap = cap; cl.bmax = bmax;
    TRY(dalloc(ctx, &cl.count, (size_t)ctx->sys.n * bmax));
    TRY(dalloc(ctx, &cl.keys, (size_t)ctx->sys.n * bmax * cap));
    if (records) {                                                     // + one zero group behind the last row (padding tiles of the tcgen05 kernels)
        const size_t nrec = (size_t)ctx->sys.n * bmax * cap * 8;
        TRY(dalloc(ctx, &cl.recs, nrec + LSD_REC_GROUP_FLOATS));
        CK(cudaMemset(cl.recs + nrec, 0, LSD_REC_GROUP_FLOATS * sizeof(float)));
        cl.rec_zero = cl.recs + nrec;
    }
    return LSD_OK;
}
lsd_status alloc_work(lsd_ctx* ctx, const MlipDev& net, MlipWork& w, int bmax)
{
    const size_t rows = (size_t)ctx->sys.n * bmax, e = rows * net.F;
    w.bmax = bmax;
    TRY(dalloc(ctx, &w.x, e)); TRY(dalloc(ctx, &w.m, e)); TRY(dalloc(ctx, &w.mbar, e)); TRY(dalloc(ctx, &w.xbar, e)); TRY(dalloc(ctx, &w.ybar, e));
    w.y.resize(net.T); w.h.resize(net.T);
    for (int t = 0; t < net.T; ++t) { TRY(dalloc(ctx, &w.y[t], e)); TRY(dalloc(ctx, &w.h[t], e)); }
    TRY(dalloc(ctx, &w.e_atom, rows));
    if (ctx->cfg.precision == LSD_BF16_TC && mlip_tc_supported(net)) {
        w.y16.resize(net.T);
        for (int t = 0; t < net.T; ++t) TRY(dalloc(ctx, &w.y16[t], e));
        TRY(dalloc(ctx, &w.mbar16, e));
        TRY(dalloc(ctx, &w.ym16, e));
        if (net.F == 128) {                                            // TMA tensor map over the pair rows (gather4 of the backward edge kernel)
            alignas(64) unsigned char hm[128];
            if (lsd_encode_row_tmap(hm, w.ym16, rows, 512)) {
                unsigned char* dm = nullptr;
                TRY(dalloc(ctx, &dm, (size_t)128));
                CK(cudaMemcpy(dm, hm, 128, cudaMemcpyHostToDevice));
                w.ym_tmap = dm;
            }
        }
    }
    return LSD_OK;
}

// Probe the neighbour-row capacity on the current base state (synchronises).
lsd_status probe_capacity(lsd_ctx* ctx, double rc_skin, int* cap_out)
{
    const int n = ctx->sys.n;
    VerletList tmp; tmp.cap = 512; tmp.rc = rc_skin;
    int *count = nullptr, *img = nullptr, *flags = nullptr; uint32_t* keys = nullptr;
    CK(cudaMalloc(&count, sizeof(int) * n)); CK(cudaMalloc(&keys, sizeof(uint32_t) * (size_t)n * tmp.cap));
    CK(cudaMalloc(&img, sizeof(int) * n)); CK(cudaMalloc(&flags, sizeof(int)));
    CK(cudaMemset(flags, 0, sizeof(int)));
    tmp.count = count; tmp.keys = keys;
    Launcher L = mk(ctx, nullptr);
    cellgrid_setup(ctx->grid, ctx->sys, rc_skin);
    launch_pack_ref(L, ctx->sys, ctx->q, img);
    launch_build_verlet(L, ctx->sys, ctx->grid, ctx->q, img, rc_skin, tmp, flags);
    CK(cudaDeviceSynchronize());
    std::vector<int> h(n);
    CK(cudaMemcpy(h.data(), count, sizeof(int) * n, cudaMemcpyDeviceToHost));
    int hf = 0; CK(cudaMemcpy(&hf, flags, sizeof(int), cudaMemcpyDeviceToHost));
    cudaFree(count); cudaFree(keys); cudaFree(img); cudaFree(flags);
    if (hf & LSD_FLAG_OVERFLOW) return fail(ctx, LSD_ERR_NBR_OVERFLOW, "neighbour row exceeds 512 entries (cutoff + skin too large for this density)");
    int mx = 0; for (int v : h) mx = std::max(mx, v);
    int cap = (int)(mx * 1.25 * ctx->cap_growth) + 8;
    cap = (cap + 15) / 16 * 16;
    *cap_out = std::min(cap, 512);
    return LSD_OK;
}

lsd_status setup_lists_impl(lsd_ctx* ctx);
lsd_status setup_lists(lsd_ctx* ctx)
{
    for (void* p : ctx->list_allocs) cudaFree(p);            // the superseded rows (the caller has synchronised the device)
    ctx->list_allocs.clear();
    ctx->alloc_lists = true;
    const lsd_status s = setup_lists_impl(ctx);
    ctx->alloc_lists = false;
    return s;
}
lsd_status setup_lists_impl(lsd_ctx* ctx)
{
    const double skin = ctx->cfg.skin;
    ctx->rc_mlip_max = std::max((double)ctx->pot[0].mlip.rc, (double)ctx->pot[1].mlip.rc);
    ctx->rc_pair_max = std::max(ctx->pot[0].pair_rcmax, ctx->pot[1].pair_rcmax);
    const double rmax = std::max(ctx->rc_mlip_max, ctx->rc_pair_max) + skin;
    if (ctx->sys.periodic) for (int c = 0; c < 3; ++c)
        if (ctx->sys.box[c] < 2.0 * rmax) return fail(ctx, LSD_ERR_INVALID_ARG, "periodic box must be >= 2 (r_c + skin) in every dimension (single minimum image, R10)");
    ctx->cap_mlip = ctx->cap_pair = 0;
    if (ctx->rc_mlip_max > 0) TRY(probe_capacity(ctx, ctx->rc_mlip_max + skin, &ctx->cap_mlip));
    if (ctx->rc_pair_max > 0) TRY(probe_capacity(ctx, ctx->rc_pair_max + skin, &ctx->cap_pair));
    {   // pair-prior list: only the species pairs that interact, each with its own cutoff (cfg3: O-O only, a ninth of the candidates)
        const int ns = ctx->sys.ns;
        std::vector<double> t((size_t)ns * ns, 0.0);
        for (int w = 0; w < 2; ++w) {
            if (!ctx->pot[w].pair_rc2_host.size()) continue;
            for (int a = 0; a < ns * ns; ++a) {
                const double rc2 = ctx->pot[w].pair_rc2_host[a];
                if (rc2 > 0.0) { const double r = std::sqrt(rc2) + skin; t[a] = std::max(t[a], r * r); }
            }
        }
        ctx->pair_rcs2 = nullptr;
        if (ctx->rc_pair_max > 0) TRY(upload(ctx, &ctx->pair_rcs2, t.data(), t.size()));
    }
    // equal cutoffs (cfg5: Morse and network both 6 A): one Verlet list serves both, build_lists builds it once
    const bool shared = ctx->cap_mlip && ctx->cap_pair && ctx->rc_mlip_max == ctx->rc_pair_max;
    for (int s = 0; s < ctx->nslots; ++s) {
        if (ctx->cap_mlip) TRY(alloc_verlet(ctx, ctx->slot[s].vl_mlip, ctx->cap_mlip, ctx->rc_mlip_max));
        if (shared) ctx->slot[s].vl_pair = ctx->slot[s].vl_mlip;
        else if (ctx->cap_pair) TRY(alloc_verlet(ctx, ctx->slot[s].vl_pair, ctx->cap_pair, ctx->rc_pair_max));
    }
    if (ctx->cap_mlip) TRY(alloc_verlet(ctx, ctx->vl_eval_mlip, ctx->cap_mlip, ctx->rc_mlip_max));
    if (shared) ctx->vl_eval_pair = ctx->vl_eval_mlip;
    else if (ctx->cap_pair) TRY(alloc_verlet(ctx, ctx->vl_eval_pair, ctx->cap_pair, ctx->rc_pair_max));
    for (int w = 0; w < 2; ++w) {
        if (ctx->pot[w].mlip.F > 0) TRY(alloc_compact(ctx, ctx->cl_mlip[w], ctx->cap_mlip, ctx->bmax[w], true));
        {   // the same directed edge set for the prior and the network: every species pair has a pair term, all with the network's cutoff
            const PotDev& pd = ctx->pot[w];
            bool same = pd.mlip.F > 0 && pd.pair_rcmax > 0;
            const double rc2 = (double)pd.mlip.rc * (double)pd.mlip.rc;
            for (double v : pd.pair_rc2_host) same = same && v == rc2;
            ctx->pair_is_mlip[w] = same;
        }
        if (ctx->pot[w].pair_rcmax > 0 && !ctx->pair_is_mlip[w]) TRY(alloc_compact(ctx, ctx->cl_pair[w], ctx->cap_pair, ctx->bmax[w], false));
    }
    return LSD_OK;
}

// state, window rows and event of ring slot s (its neighbour lists are made by setup_lists)
lsd_status alloc_slot(lsd_ctx* ctx, int s)
{
    const size_t n3 = (size_t)3 * ctx->sys.n;
    const int kmax = ctx->cfg.k_max;
    WindowSlot& w = ctx->slot[s];
    if (w.qstart) return LSD_OK;
    TRY(dalloc(ctx, &w.qstart, n3)); TRY(dalloc(ctx, &w.pstart, n3));
    TRY(dalloc(ctx, &w.qhalf, n3 * kmax)); TRY(dalloc(ctx, &w.Ft, n3 * kmax)); TRY(dalloc(ctx, &w.yq, n3 * kmax)); TRY(dalloc(ctx, &w.yp, n3 * kmax));
    if (ctx->same_prior) TRY(dalloc(ctx, &w.Fprior, n3 * kmax));
    TRY(dalloc(ctx, &w.img, ctx->sys.n)); TRY(dalloc(ctx, &w.flags, 1)); TRY(dalloc(ctx, &w.n0_dev, 1));
    TRY(dalloc(ctx, &w.dF, n3)); CK(cudaMemset(w.dF, 0, n3 * sizeof(double)));
    CK(cudaEventCreateWithFlags(&w.ev_drafted, cudaEventDisableTiming));
    return LSD_OK;
}
void reset_slots(lsd_ctx* ctx)                               // nothing drafted, nothing verified
{
    ctx->pending = 0; ctx->transported = 0;
    for (int s = 0; s < LSD_MAX_SLOTS; ++s) { ctx->slot[s].drafted = 0; ctx->slot[s].verified = 0; }
}

// Window-shared lists from the reference state qref (a1).
void build_lists(lsd_ctx* ctx, Launcher L, const double* qref, int* img, VerletList& vm, VerletList& vp, int* flags)
{
    launch_pack_ref(L, ctx->sys, qref, img);
    if (ctx->cap_mlip) {
        cellgrid_setup(ctx->grid, ctx->sys, ctx->rc_mlip_max + ctx->cfg.skin);
        launch_build_verlet(L, ctx->sys, ctx->grid, qref, img, ctx->rc_mlip_max + ctx->cfg.skin, vm, flags);
    }
    if (ctx->cap_pair && vp.keys != vm.keys) {                   // (shared list when the cutoffs are equal, setup_lists)
        cellgrid_setup(ctx->grid, ctx->sys, ctx->rc_pair_max + ctx->cfg.skin);
        launch_build_verlet(L, ctx->sys, ctx->grid, qref, img, ctx->rc_pair_max + ctx->cfg.skin, vp, flags, ctx->pair_rcs2);
    }
}

// One batched force evaluation of potential `which` on B <= bmax[which] states (a0 / a2).
// prior_out: also keep the prior part of the forces; prior_in: the prior part is known (same positions, same prior, computed by the
// same batch-invariant kernel: identical bits), only the network is evaluated
void eval_forces(lsd_ctx* ctx, Launcher L, int which, int B, const double* q, const int* img, const VerletList& vm,
                 const VerletList& vp, double* F, int* flags, double* e_atom, double* prior_out = nullptr, const double* prior_in = nullptr)
{
    PotDev& pot = ctx->pot[which];
    L.draft = which == LSD_DRAFT;
    ctx->cl_img[which] = img;
    CompactList* pl = nullptr;
    const bool one_list = ctx->pair_is_mlip[which];              // cfg5: Morse and network both 6 A: one per-state list, one launch less
    const size_t fbytes = (size_t)B * 3 * ctx->sys.n * sizeof(double);
    bool mlip_list_done = false;
    if (prior_in) cudaMemcpyAsync(F, prior_in, fbytes, cudaMemcpyDeviceToDevice, L.s);
    else {
        if (pot.mlip.F > 0 && one_list) {
            const double rc = (double)pot.mlip.rc;
            launch_compact(L, ctx->sys, B, q, img, vm, rc * rc, nullptr, ctx->cl_mlip[which], flags, pot.mlip.rc);
            pl = &ctx->cl_mlip[which];
            mlip_list_done = true;
        } else if (pot.pair_rcmax > 0) {
            launch_compact(L, ctx->sys, B, q, img, vp, 0.0, pot.pair_rc2, ctx->cl_pair[which], flags);
            pl = &ctx->cl_pair[which];
        }
        launch_prior_forces(L, ctx->sys, pot, B, q, img, pl, F);
        if (prior_out) cudaMemcpyAsync(prior_out, F, fbytes, cudaMemcpyDeviceToDevice, L.s);
    }
    if (pot.mlip.F > 0) {
        const double rc = (double)pot.mlip.rc;
        if (!mlip_list_done) launch_compact(L, ctx->sys, B, q, img, vm, rc * rc, nullptr, ctx->cl_mlip[which], flags, pot.mlip.rc);
        if (ctx->cfg.precision == LSD_BF16_TC && mlip_tc_supported(pot.mlip))
            mlip_forward_backward_bf16tc(L, ctx->sys, pot.mlip, ctx->work[which], B, q, img, ctx->cl_mlip[which], F, e_atom);
        else
            mlip_forward_backward_fp32(L, ctx->sys, pot.mlip, ctx->work[which], B, q, img, ctx->cl_mlip[which], F, e_atom);
    }
}

lsd_status flags_to_status(lsd_ctx* ctx, int flags)
{
    if (flags & LSD_FLAG_NONFINITE) return fail(ctx, LSD_ERR_NONFINITE, "non-finite positions or forces in the window");
    if (flags & LSD_FLAG_OVERFLOW) return fail(ctx, LSD_ERR_NBR_OVERFLOW, "neighbour row capacity exceeded (call lsd_set_skin to re-size the lists)");
    if (flags & LSD_FLAG_SKIN) return fail(ctx, LSD_ERR_SKIN_VIOLATED, "an atom moved more than skin/2 from the list's reference state");
    return LSD_OK;
}

lsd_status copy_out(lsd_ctx* ctx, void* dst, const void* src_dev, size_t bytes, int where)
{
    CK(cudaMemcpy(dst, src_dev, bytes, where == LSD_HOST ? cudaMemcpyDeviceToHost : cudaMemcpyDeviceToDevice));
    return LSD_OK;
}

// K serial ABOBA steps (PAPER.md:584-593 DRAFT_STEP; Eq. 2, Eq. 7) with the forces of potential `which` from the slot's start
// state: window-shared lists, then per step A(1/2), forces, B O B + A(1/2).  Stream-ordered launches only (capturable).
lsd_status rollout_body(lsd_ctx* ctx, WindowSlot& w, int K, int which, void* stream, bool ec)
{
    cudaStream_t st = (cudaStream_t)stream;
    const int n = ctx->sys.n;
    const size_t n3 = (size_t)3 * n;
    Launcher Lg = mk(ctx, stream);
    CK(cudaMemsetAsync(w.flags, 0, sizeof(int), st));
    build_lists(ctx, Lg, w.qstart, w.img, w.vl_mlip, w.vl_pair, w.flags);
    const double sh = 0.5 * ctx->cfg.skin, sh2 = sh * sh;
    if (ctx->tiny && which == LSD_DRAFT) {                                    // one launch for the K steps (the lists above serve the verification)
        Lg.draft = 1;
        launch_tiny_rollout(Lg, ctx->sys, ctx->pot[LSD_DRAFT], K, ctx->cfg.seed, w.n0_dev, ctx->c1, ctx->b, ctx->hdt, sh2, w.qstart, w.pstart,
                            ec ? w.dF : nullptr, w.qhalf, w.Ft, w.yq, w.yp, w.flags);
        return LSD_OK;
    }
    for (int j = 1; j <= K; ++j) {                                            // serial in j
        const double* pp = j == 1 ? w.pstart : w.yp + n3 * (j - 2);
        double* qh = w.qhalf + n3 * (j - 1);
        if (j == 1) launch_half_a(Lg, n, w.qstart, w.pstart, ctx->sys.mass, ctx->hdt, qh, w.qstart, sh2, w.flags);
        eval_forces(ctx, Lg, which, 1, qh, w.img, w.vl_mlip, w.vl_pair, w.Ft + n3 * (j - 1), w.flags, nullptr,
                    (ctx->same_prior && which == LSD_DRAFT) ? w.Fprior + n3 * (j - 1) : nullptr);
        launch_bob_a(Lg, n, ctx->cfg.seed, w.n0_dev, (uint64_t)j, pp, w.Ft + n3 * (j - 1), qh, ctx->sys.mass, ctx->sys.sigma,
                     ctx->c1, ctx->b, ctx->hdt, w.yq + n3 * (j - 1), w.yp + n3 * (j - 1), ec ? w.dF : nullptr,
                     j < K ? w.qhalf + n3 * j : nullptr, w.qstart, sh2, w.flags);       // + the first A(1/2) of step j + 1
    }
    return LSD_OK;
}

}  // namespace

extern "C" {

const char* lsd_version(void) { return "lsd-b200 0.1 (sm_100a)"; }

const char* lsd_last_error(const lsd_ctx* ctx) { return ctx ? ctx->err.c_str() : g_init_error.c_str(); }

int64_t lsd_launch_count(const lsd_ctx* ctx) { return ctx ? ctx->launches : 0; }

lsd_status lsd_get_edge_launch_info(int32_t pass, int32_t* out)
{
    if (!out || pass < 0 || pass > 1) return LSD_ERR_INVALID_ARG;
    const EdgeLaunchInfo& e = g_edge_last[pass];
    out[0] = e.kernel; out[1] = e.atoms_per_chunk; out[2] = e.threads; out[3] = e.grid; out[4] = e.width;
    return LSD_OK;
}

int32_t lsd_tc_enabled(const lsd_ctx* ctx)
{
    return ctx && ctx->cfg.precision == LSD_BF16_TC && ctx->pot[LSD_TARGET].mlip.F > 0 && mlip_tc_supported(ctx->pot[LSD_TARGET].mlip) ? 1 : 0;
}

int32_t lsd_tiny_rollout_enabled(const lsd_ctx* ctx) { return ctx && ctx->tiny ? 1 : 0; }

void lsd_destroy(lsd_ctx* ctx)
{
    if (!ctx) return;
    cudaDeviceSynchronize();
    drop_graphs(ctx);
    for (void* p : ctx->allocs) cudaFree(p);
    for (void* p : ctx->list_allocs) cudaFree(p);
    cudaFree(ctx->grid.cell_count); cudaFree(ctx->grid.cell_start); cudaFree(ctx->grid.cell_cursor);
    cudaFree(ctx->grid.cell_atoms); cudaFree(ctx->grid.atom_cell);
    for (int s = 0; s < LSD_MAX_SLOTS; ++s) if (ctx->slot[s].ev_drafted) cudaEventDestroy(ctx->slot[s].ev_drafted);
    for (cudaEvent_t e : ctx->prof.ev) cudaEventDestroy(e);
    if (ctx->side) cudaStreamDestroy(ctx->side);
    if (ctx->result_host) cudaFreeHost(ctx->result_host);
    if (ctx->state_host) cudaFreeHost(ctx->state_host);
    if (ctx->ev_state) cudaEventDestroy(ctx->ev_state);
    delete ctx;
}

static lsd_status init_impl(lsd_ctx* ctx, const lsd_config* cfg, const lsd_system* sys, const lsd_potential* draft,
                            const lsd_potential* target, const double* q0, const double* p0)
{
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) return fail(ctx, LSD_ERR_CUDA, "no CUDA device: liblsd_b200 has no CPU fallback");
    ctx->cfg = *cfg;
    const int n = sys->n_atoms, kmax = cfg->k_max;
    if (n < 1 || sys->n_species < 1 || !q0) return fail(ctx, LSD_ERR_INVALID_ARG, "n_atoms, n_species must be >= 1 and q0 non-null");
    if (kmax < 1 || kmax > LSD_MAX_K) return fail(ctx, LSD_ERR_INVALID_ARG, "k_max must be in 1..64");
    if (cfg->scheme != LSD_SCHEME_ABOBA) return fail(ctx, LSD_ERR_UNSUPPORTED, "only LSD_SCHEME_ABOBA is implemented (DESIGN.md R1)");
    if (cfg->precision != LSD_FP32 && cfg->precision != LSD_BF16_TC) return fail(ctx, LSD_ERR_INVALID_ARG, "precision must be LSD_FP32 or LSD_BF16_TC");
    if (!(cfg->dt_fs > 0) || !(cfg->friction_per_fs > 0) || !(cfg->temperature_K > 0) || !(cfg->skin > 0)) return fail(ctx, LSD_ERR_INVALID_ARG, "dt, friction, temperature and skin must be positive");
    for (const lsd_potential* p : {draft, target}) {
        if (p->n_species != sys->n_species) return fail(ctx, LSD_ERR_INVALID_ARG, "potential and system disagree on n_species");
        const int F = p->mlip.width;
        if (F != 0) {
            if (F != 32 && F != 64 && F != 128) return fail(ctx, LSD_ERR_UNSUPPORTED, "MLIP width must be 32, 64 or 128");
            if (p->mlip.n_rbf != LSD_NRBF) return fail(ctx, LSD_ERR_UNSUPPORTED, "MLIP n_rbf must be 32");
            if (p->mlip.n_blocks < 1 || p->mlip.n_species != sys->n_species || !(p->mlip.cutoff > 0) || !p->mlip.weights) return fail(ctx, LSD_ERR_INVALID_ARG, "bad MLIP description");
        }
    }
    for (int i = 0; i < n; ++i) if (sys->species[i] < 0 || sys->species[i] >= sys->n_species) return fail(ctx, LSD_ERR_INVALID_ARG, "species index out of range");

    SysDev& S = ctx->sys;
    S.n = n; S.ns = sys->n_species; S.periodic = sys->periodic;
    for (int c = 0; c < 3; ++c) S.box[c] = sys->box[c];
    ctx->kT = LSD_KB_EV * cfg->temperature_K;
    ctx->c1 = std::exp(-cfg->friction_per_fs * cfg->dt_fs);
    ctx->b = (1.0 + ctx->c1) * cfg->dt_fs / 2.0;
    ctx->hdt = cfg->dt_fs / 2.0;
    std::vector<double> mass(n), sigma(n);
    for (int i = 0; i < n; ++i) {
        mass[i] = sys->mass_amu[i] * LSD_AMU_EV;
        sigma[i] = std::sqrt(sys->mass_amu[i] * LSD_AMU_EV * LSD_KB_EV * cfg->temperature_K * (1.0 - ctx->c1 * ctx->c1));   // Eq. 7 covariance
    }
    TRY(upload(ctx, &S.species, sys->species, n));
    TRY(upload(ctx, &S.mass, mass.data(), n));
    TRY(upload(ctx, &S.sigma, sigma.data(), n));
    S.n_bonds = sys->n_bonds; S.n_angles = sys->n_angles;
    if (S.n_bonds) { TRY(upload(ctx, &S.bonds, sys->bonds, (size_t)2 * S.n_bonds)); TRY(upload(ctx, &S.bond_k, sys->bond_k, S.n_bonds)); TRY(upload(ctx, &S.bond_r0, sys->bond_r0, S.n_bonds)); }
    if (S.n_angles) { TRY(upload(ctx, &S.angles, sys->angles, (size_t)3 * S.n_angles)); TRY(upload(ctx, &S.angle_k, sys->angle_k, S.n_angles)); TRY(upload(ctx, &S.angle_t0, sys->angle_theta0, S.n_angles)); }
    {   // per-atom bonded-term lists (gather form; bonds first, then angles, in input order)
        std::vector<std::vector<int>> per(n);
        for (int t = 0; t < S.n_bonds; ++t) for (int k = 0; k < 2; ++k) {
            const int a = sys->bonds[2 * t + k];
            if (a < 0 || a >= n) return fail(ctx, LSD_ERR_INVALID_ARG, "bond atom index out of range");
            per[a].push_back(t);
        }
        for (int t = 0; t < S.n_angles; ++t) for (int k = 0; k < 3; ++k) {
            const int a = sys->angles[3 * t + k];
            if (a < 0 || a >= n) return fail(ctx, LSD_ERR_INVALID_ARG, "angle atom index out of range");
            per[a].push_back(S.n_bonds + t);
        }
        std::vector<int> start(n + 1, 0), term;
        for (int i = 0; i < n; ++i) { start[i + 1] = start[i] + (int)per[i].size(); term.insert(term.end(), per[i].begin(), per[i].end()); }
        TRY(upload(ctx, &S.bt_start, start.data(), start.size()));
        TRY(upload(ctx, &S.bt_term, term.data(), term.size()));
    }
    TRY(upload_potential(ctx, *draft, ctx->pot[LSD_DRAFT]));
    TRY(upload_potential(ctx, *target, ctx->pot[LSD_TARGET]));
    {   // Tiny systems: the draft rollout is one kernel (tiny_rollout.cu).  Its sums run in another order than the batched kernels,
        // so it is used only where the draft is a different potential: draft == target must reproduce the target bitwise (R8).
        auto n_weights = [&](const lsd_mlip& m) { const size_t F = m.width, R = m.n_rbf; return (size_t)m.n_species * F + (size_t)m.n_blocks * (4 * F * F + F * R) + (F / 2) * F + F / 2; };
        bool same = draft->use_bonded == target->use_bonded && draft->mlip.width == target->mlip.width &&
                    std::memcmp(draft->pair, target->pair, sizeof(double) * (size_t)sys->n_species * sys->n_species * LSD_PAIR_COLS) == 0;
        if (same && draft->mlip.width > 0)
            same = draft->mlip.n_blocks == target->mlip.n_blocks && draft->mlip.cutoff == target->mlip.cutoff && draft->mlip.energy_scale == target->mlip.energy_scale &&
                   std::memcmp(draft->mlip.weights, target->mlip.weights, sizeof(double) * n_weights(draft->mlip)) == 0;
        const char* pv = getenv("LSD_PRIOR_REUSE");
        ctx->same_prior = !same && !(pv && pv[0] == '0') && draft->use_bonded == target->use_bonded &&
                          std::memcmp(draft->pair, target->pair, sizeof(double) * (size_t)sys->n_species * sys->n_species * LSD_PAIR_COLS) == 0;
        const char* tv = getenv("LSD_TINY");
        ctx->tiny = !same && !(tv && tv[0] == '0') && tiny_rollout_supported(ctx->sys, ctx->pot[LSD_DRAFT]);
    }
    ctx->bmax[LSD_DRAFT] = 1; ctx->bmax[LSD_TARGET] = kmax;

    const size_t n3 = (size_t)3 * n;
    TRY(dalloc(ctx, &ctx->q, 2 * n3));                       // q and p are one allocation: a state moves with one copy
    ctx->p = ctx->q + n3;
    CK(cudaMemcpy(ctx->q, q0, n3 * sizeof(double), cudaMemcpyHostToDevice));
    if (n3 * 2 * sizeof(double) <= (size_t)512 * 1024) {
        CK(cudaMallocHost(&ctx->state_host, 2 * n3 * sizeof(double)));
        CK(cudaEventCreateWithFlags(&ctx->ev_state, cudaEventDisableTiming));
    }
    if (p0) CK(cudaMemcpy(ctx->p, p0, n3 * sizeof(double), cudaMemcpyHostToDevice));
    else launch_initial_momenta(mk(ctx, nullptr), n, cfg->seed, S.mass, ctx->kT, ctx->p);
    TRY(setup_lists(ctx));
    for (int s = 0; s < ctx->nslots; ++s) TRY(alloc_slot(ctx, s));
    for (int w = 0; w < 2; ++w) if (ctx->pot[w].mlip.F > 0) TRY(alloc_work(ctx, ctx->pot[w].mlip, ctx->work[w], ctx->bmax[w]));
    TRY(dalloc(ctx, &ctx->Fg, n3 * kmax));
    TRY(dalloc(ctx, &ctx->dF, n3)); CK(cudaMemset(ctx->dF, 0, n3 * sizeof(double)));
    ctx->nblk = transport_blocks(n);
    TRY(dalloc(ctx, &ctx->partial, (size_t)2 * ctx->nblk * kmax));
    TRY(dalloc(ctx, &ctx->S1, kmax)); TRY(dalloc(ctx, &ctx->S2, kmax)); TRY(dalloc(ctx, &ctx->ell, kmax)); TRY(dalloc(ctx, &ctx->lnu, kmax));
    TRY(dalloc(ctx, &ctx->reject, kmax)); TRY(dalloc(ctx, &ctx->result, 1));
    TRY(dalloc(ctx, &ctx->q_eval, n3 * kmax)); TRY(dalloc(ctx, &ctx->F_eval, n3 * kmax)); TRY(dalloc(ctx, &ctx->e_eval, (size_t)n * kmax));
    TRY(dalloc(ctx, &ctx->img_eval, n)); TRY(dalloc(ctx, &ctx->flags_eval, 1));
    CK(cudaMallocHost(&ctx->result_host, sizeof(TransportResult)));
    CK(cudaStreamCreateWithFlags(&ctx->side, cudaStreamNonBlocking));
    { const char* g = getenv("LSD_GRAPHS"); ctx->use_graphs = !(g && g[0] == '0'); }
    CK(cudaDeviceSynchronize());
    CK(cudaGetLastError());
    return LSD_OK;
}

lsd_status lsd_init(const lsd_config* cfg, const lsd_system* sys, const lsd_potential* draft, const lsd_potential* target,
                    const double* q0, const double* p0, lsd_ctx** out)
{
    if (!cfg || !sys || !draft || !target || !out) return fail(nullptr, LSD_ERR_INVALID_ARG, "null argument");
    *out = nullptr;
    lsd_ctx* ctx = new (std::nothrow) lsd_ctx();
    if (!ctx) return fail(nullptr, LSD_ERR_OOM, "host allocation failed");
    lsd_status s = init_impl(ctx, cfg, sys, draft, target, q0, p0);
    if (s != LSD_OK) { g_init_error = ctx->err; lsd_destroy(ctx); return s; }
    *out = ctx;
    return LSD_OK;
}

lsd_status lsd_set_skin(lsd_ctx* ctx, double skin)
{
    if (!ctx || !(skin > 0)) return LSD_ERR_INVALID_ARG;
    CK(cudaDeviceSynchronize());
    ctx->cfg.skin = skin;
    drop_graphs(ctx);                                        // captured pointers and the skin value change
    reset_slots(ctx);
    return setup_lists(ctx);      // frees the superseded rows
}

lsd_status lsd_set_window_slots(lsd_ctx* ctx, int32_t n_slots)
{
    if (!ctx || n_slots < 2 || n_slots > LSD_MAX_SLOTS) return LSD_ERR_INVALID_ARG;
    CK(cudaDeviceSynchronize());
    drop_graphs(ctx);
    reset_slots(ctx);
    ctx->verify_idx = 0; ctx->last_slot = -1;
    ctx->nslots = n_slots;
    for (int s = 0; s < n_slots; ++s) TRY(alloc_slot(ctx, s));
    return setup_lists(ctx);                                 // every slot owns its window-shared Verlet lists
}

lsd_status lsd_draft_rollout(lsd_ctx* ctx, int32_t K, void* stream)
{
    if (!ctx) return LSD_ERR_INVALID_ARG;
    if (K < 1 || K > ctx->cfg.k_max) return fail(ctx, LSD_ERR_INVALID_ARG, "K must be in 1..k_max");
    if (ctx->pending >= ctx->nslots) return fail(ctx, LSD_ERR_STATE, "every window slot holds an unverified window (lsd_set_window_slots)");
    const int n = ctx->sys.n;
    const size_t n3 = (size_t)3 * n;
    const int si = (ctx->verify_idx + ctx->pending) % ctx->nslots;
    WindowSlot& w = ctx->slot[si];
    cudaStream_t st = (cudaStream_t)stream;
    Launcher L = mk(ctx, stream);
    note_stream(ctx, st);
    if (ctx->state_in_flight) CK(cudaStreamWaitEvent(st, ctx->ev_state, 0));  // a staged lsd_set_state upload
    if (w.ev_drafted) CK(cudaStreamWaitEvent(st, w.ev_drafted, 0));          // a discarded rollout into this slot may still run
    if (ctx->pending == 0) {
        // flushed speculative rollouts may still run on another stream: they share the draft's work buffers
        for (int s = 0; s < ctx->nslots; ++s) if (s != si && ctx->slot[s].ev_drafted) CK(cudaStreamWaitEvent(st, ctx->slot[s].ev_drafted, 0));
        CK(cudaMemcpyAsync(w.qstart, ctx->q, n3 * sizeof(double), cudaMemcpyDeviceToDevice, st));
        CK(cudaMemcpyAsync(w.pstart, ctx->p, n3 * sizeof(double), cudaMemcpyDeviceToDevice, st));
        if (ctx->ec) CK(cudaMemcpyAsync(w.dF, ctx->dF, n3 * sizeof(double), cudaMemcpyDeviceToDevice, st));
        w.n0 = (uint64_t)ctx->step;
    } else {                                                                  // speculative: continue from y_K of the unverified window
        WindowSlot& pv = ctx->slot[(si + ctx->nslots - 1) % ctx->nslots];
        CK(cudaStreamWaitEvent(st, pv.ev_drafted, 0));
        CK(cudaMemcpyAsync(w.qstart, pv.yq + n3 * (pv.K - 1), n3 * sizeof(double), cudaMemcpyDeviceToDevice, st));
        CK(cudaMemcpyAsync(w.pstart, pv.yp + n3 * (pv.K - 1), n3 * sizeof(double), cudaMemcpyDeviceToDevice, st));
        if (ctx->ec) CK(cudaMemcpyAsync(w.dF, pv.dF, n3 * sizeof(double), cudaMemcpyDeviceToDevice, st));   // the cache has not seen the unverified window
        w.n0 = pv.n0 + (uint64_t)pv.K;
    }
    launch_set_u64(L, w.n0_dev, w.n0);
    TRY(run_graphed(ctx, st, w.g_roll[K], [&]() -> lsd_status { return rollout_body(ctx, w, K, LSD_DRAFT, stream, ctx->ec != 0); }));
    ctx->cl_img[LSD_DRAFT] = w.img;                                           // (set by eval_forces only when the body runs)
    CK(cudaEventRecord(w.ev_drafted, st));
    w.K = K; w.drafted = 1; w.verified = 0;
    w.prior_valid = ctx->same_prior && !ctx->tiny;               // (the one-kernel rollout keeps its prior forces on chip)
    if (ctx->tiny) ctx->tiny_draft_lists_stale = true;            // ... and its neighbour rows: the per-state draft lists no longer belong to the last evaluation
    ctx->pending++;
    CK(cudaGetLastError());
    return LSD_OK;
}

lsd_status lsd_verify_window(lsd_ctx* ctx, int32_t K, void* stream)
{
    if (!ctx) return LSD_ERR_INVALID_ARG;
    WindowSlot& w = ctx->slot[ctx->verify_idx];
    if (ctx->pending < 1 || !w.drafted) return fail(ctx, LSD_ERR_STATE, "no drafted window to verify");
    if (K != w.K) return fail(ctx, LSD_ERR_INVALID_ARG, "K differs from the drafted window length");
    cudaStream_t st = (cudaStream_t)stream;
    note_stream(ctx, st);
    CK(cudaStreamWaitEvent(st, w.ev_drafted, 0));
    TRY(run_graphed(ctx, st, w.g_verify[K], [&]() -> lsd_status {
        eval_forces(ctx, mk(ctx, stream), LSD_TARGET, K, w.qhalf, w.img, w.vl_mlip, w.vl_pair, ctx->Fg, w.flags, nullptr, nullptr,
                    (ctx->same_prior && w.prior_valid) ? w.Fprior : nullptr);
        return LSD_OK;
    }));
    ctx->cl_img[LSD_TARGET] = w.img;
    w.verified = 1;
    CK(cudaGetLastError());
    return LSD_OK;
}

lsd_status lsd_transport_accept(lsd_ctx* ctx, int32_t K, void* stream, int32_t* first_reject, int32_t* n_commit)
{
    if (!ctx || !first_reject || !n_commit) return LSD_ERR_INVALID_ARG;
    WindowSlot& w = ctx->slot[ctx->verify_idx];
    if (ctx->pending < 1 || !w.verified) return fail(ctx, LSD_ERR_STATE, "lsd_verify_window has not run on this window");
    if (K != w.K) return fail(ctx, LSD_ERR_INVALID_ARG, "K differs from the drafted window length");
    cudaStream_t st = (cudaStream_t)stream;
    Launcher L = mk(ctx, stream);
    const int n = ctx->sys.n;
    TRY(run_graphed(ctx, st, w.g_transport[K], [&]() -> lsd_status {
        Launcher Lg = mk(ctx, stream);
        launch_transport(Lg, n, K, ctx->cfg.seed, w.n0_dev, w.Ft, ctx->Fg, ctx->sys.sigma, ctx->b, ctx->partial, ctx->nblk, ctx->S1, ctx->S2,
                         ctx->ell, ctx->lnu, ctx->reject, w.flags, ctx->result, ctx->xi_dbg, ctx->ec ? w.dF : nullptr, ctx->slack);
        launch_commit(Lg, n, K, ctx->cfg.seed, w.n0_dev, ctx->result, ctx->S1, ctx->S2, w.Ft, ctx->Fg, w.qhalf, w.pstart, w.yq, w.yp,
                      ctx->sys.mass, ctx->sys.sigma, ctx->c1, ctx->b, ctx->hdt, ctx->q, ctx->p, ctx->ec ? w.dF : nullptr, ctx->ec ? ctx->dF : nullptr, ctx->slack);
        return LSD_OK;
    }));
    CK(cudaMemcpyAsync(ctx->result_host, ctx->result, sizeof(TransportResult), cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    stream_idle(ctx, st);
    CK(cudaGetLastError());
    const TransportResult r = *ctx->result_host;
    ctx->last_slot = ctx->verify_idx; ctx->last_K = K;
    if (r.flags) {                                             // nothing committed: drop every drafted window
        reset_slots(ctx);
        return flags_to_status(ctx, r.flags);
    }
    ctx->last_l = r.first_reject; ctx->last_nc = r.n_commit; ctx->transported = 1;
    ctx->stats.beta_sum += r.beta_sum;
    *first_reject = r.first_reject; *n_commit = r.n_commit;
    return LSD_OK;
}

lsd_status lsd_rollback(lsd_ctx* ctx, int32_t first_reject)
{
    if (!ctx) return LSD_ERR_INVALID_ARG;
    if (!ctx->transported) return fail(ctx, LSD_ERR_STATE, "lsd_transport_accept has not run on this window");
    if (first_reject != ctx->last_l) return fail(ctx, LSD_ERR_INVALID_ARG, "first_reject differs from the value lsd_transport_accept returned");
    WindowSlot& w = ctx->slot[ctx->verify_idx];
    ctx->step += ctx->last_nc;
    ctx->stats.windows++; ctx->stats.committed_steps += ctx->last_nc; ctx->stats.rejections += first_reject ? 1 : 0; ctx->stats.step = ctx->step;
    w.drafted = 0; w.verified = 0;
    ctx->verify_idx = (ctx->verify_idx + 1) % ctx->nslots; ctx->pending--;
    if (first_reject != 0 && ctx->pending > 0) {              // flush every speculative window
        for (int s = 0; s < LSD_MAX_SLOTS; ++s) ctx->slot[s].drafted = 0;
        ctx->pending = 0;
    }
    ctx->transported = 0;
    return LSD_OK;
}

lsd_status lsd_run(lsd_ctx* ctx, int64_t n_steps, int32_t K, int32_t overlap, void* stream)
{
    if (!ctx) return LSD_ERR_INVALID_ARG;
    if (K < 0 || K > ctx->cfg.k_max || n_steps < 0) return fail(ctx, LSD_ERR_INVALID_ARG, "bad K or n_steps");
    // K == 0: adaptive lookahead (the paper's lookahead L is a free parameter).
    // Hill climbing over K in {1, 2, 4, ..., k_max} on the MEASURED committed steps per second of whole windows (host clock
    // around windows that end in a synchronising read anyway): 8 windows per visit, a move to the better neighbour, an
    // unexplored neighbour is visited once, the neighbours are re-measured every 64 windows.  On one GPU the batched target
    // call costs ~K target evaluations once the batch fills the device, so large systems with low acceptance settle at K = 1;
    // small latency-bound systems settle where the verified run length saturates.
    const bool adaptive = K == 0;
    constexpr int kVisit = 8, kRefresh = 64;
    double a_nc[8] = {0}, a_t[8] = {0};                      // per log2(K): committed steps and seconds (decayed)
    int a_idx = 0, a_in_visit = 0, a_since_refresh = 0, a_home = 0;
    int kmax_idx = 0;
    while ((2 << kmax_idx) <= ctx->cfg.k_max && kmax_idx < 7) ++kmax_idx;
    if (adaptive) {
        a_idx = ctx->adaptive_k > 0 ? (int)std::lround(std::log2((double)ctx->adaptive_k)) : kmax_idx;
        a_idx = std::min(std::max(a_idx, 0), kmax_idx);
        a_home = a_idx;
        K = 1 << a_idx;
    }
    auto rate = [&](int i) { return a_t[i] > 0 ? a_nc[i] / a_t[i] : -1.0; };
    std::chrono::steady_clock::time_point t_win = std::chrono::steady_clock::now();
    int64_t remaining = n_steps;
    const int depth = std::min(std::max((int)overlap, 0), ctx->nslots - 1);   // speculative windows kept in flight
    constexpr int kMaxListRetries = 6;                        // per call: a window that still fails returns its error
    int list_retries = 0;
    while (remaining > 0) {
        if (ctx->pending == 0) TRY(lsd_draft_rollout(ctx, (int32_t)std::min<int64_t>(K, remaining), stream));
        const int k = ctx->slot[ctx->verify_idx].K;
        TRY(lsd_verify_window(ctx, k, stream));
        if (depth > 0) {
            // Alg. 2 semantics on one device: the drafter does not wait for the verdict of the window being
            // verified; up to `depth` speculative windows stay drafted ahead on the second stream, each continuing from y_K of the
            // one before it, all flushed by a rejection (:611-612)
            int64_t ahead = 0;
            for (int i = 0; i < ctx->pending; ++i) ahead += ctx->slot[(ctx->verify_idx + i) % ctx->nslots].K;
            while (ctx->pending < 1 + depth && remaining - ahead > 0) {
                const int kw = (int)std::min<int64_t>(K, remaining - ahead);
                TRY(lsd_draft_rollout(ctx, kw, ctx->side));
                ahead += kw;
            }
        }
        int32_t l = 0, nc = 0;
        lsd_status ts = lsd_transport_accept(ctx, k, stream, &l, &nc);
        if ((ts == LSD_ERR_SKIN_VIOLATED || ts == LSD_ERR_NBR_OVERFLOW) && list_retries < kMaxListRetries) {
            // answered by a rebuild, never by an incomplete list: twice the skin, or rows with 1.5 x the head room
            ++list_retries;
            CK(cudaStreamSynchronize(ctx->side));
            if (ts == LSD_ERR_NBR_OVERFLOW) ctx->cap_growth *= 1.5;
            TRY(lsd_set_skin(ctx, ts == LSD_ERR_SKIN_VIOLATED ? 2.0 * ctx->cfg.skin : ctx->cfg.skin));
            continue;
        }
        TRY(ts);
        TRY(lsd_rollback(ctx, l));
        remaining -= nc;
        if (adaptive) {
            const auto now = std::chrono::steady_clock::now();
            const double dt = std::chrono::duration<double>(now - t_win).count();
            t_win = now;
            if (k == (1 << a_idx)) { a_nc[a_idx] = 0.9 * a_nc[a_idx] + nc; a_t[a_idx] = 0.9 * a_t[a_idx] + dt; }   // (shortened last windows do not count)
            ++a_since_refresh;
            if (++a_in_visit >= kVisit) {
                a_in_visit = 0;
                if (a_idx != a_home) {                       // back from a visit: stay if it was better
                    if (rate(a_idx) > rate(a_home)) a_home = a_idx;
                    a_idx = a_home;
                } else {
                    const int lo = a_home - 1, hi = a_home + 1;
                    if (a_since_refresh >= kRefresh) { a_since_refresh = 0; if (lo >= 0) a_t[lo] = 0; if (hi <= kmax_idx) a_t[hi] = 0; }
                    if (lo >= 0 && rate(lo) < 0) a_idx = lo;                 // unexplored (or due for a refresh)
                    else if (hi <= kmax_idx && rate(hi) < 0) a_idx = hi;
                    else {
                        if (lo >= 0 && rate(lo) > rate(a_home)) a_home = lo;
                        else if (hi <= kmax_idx && rate(hi) > rate(a_home)) a_home = hi;
                        a_idx = a_home;
                    }
                }
                const int newK = 1 << a_idx;
                K = newK;                                    // a speculative window already in flight keeps its own length (slot.K)
                ctx->adaptive_k = 1 << a_home;
            }
        }
        if (ctx->pending >= 1 && ctx->slot[ctx->verify_idx].K > remaining) {   // cannot happen with the K choice above; defensive
            CK(cudaStreamSynchronize(ctx->side));
            reset_slots(ctx);
        }
    }
    if (ctx->pending) { CK(cudaStreamSynchronize(ctx->side)); reset_slots(ctx); }
    return LSD_OK;
}

int32_t lsd_get_adaptive_k(const lsd_ctx* ctx) { return ctx ? ctx->adaptive_k : 0; }

lsd_status lsd_plain_langevin(lsd_ctx* ctx, int32_t which, int64_t n_steps, void* stream)
{
    if (!ctx || (which != LSD_DRAFT && which != LSD_TARGET) || n_steps < 0) return LSD_ERR_INVALID_ARG;
    if (ctx->pending) return fail(ctx, LSD_ERR_STATE, "a drafted window is pending");
    cudaStream_t st = (cudaStream_t)stream;
    note_stream(ctx, st);
    if (ctx->state_in_flight) CK(cudaStreamWaitEvent(st, ctx->ev_state, 0));
    const size_t n3 = (size_t)3 * ctx->sys.n;
    WindowSlot& w = ctx->slot[ctx->verify_idx];
    // flushed speculative rollouts of ANY slot (after a rejection, or after an error return of lsd_run) may still run on another
    // stream; they share the draft's work buffers, the per-state lists and the cell grid with this rollout (as in lsd_draft_rollout)
    for (int s = 0; s < ctx->nslots; ++s) if (ctx->slot[s].ev_drafted) CK(cudaStreamWaitEvent(st, ctx->slot[s].ev_drafted, 0));
    int list_retries = 0;
    int64_t remaining = n_steps;
    while (remaining > 0) {
        const int K = (int)std::min<int64_t>(ctx->cfg.k_max, remaining);
        CK(cudaMemcpyAsync(w.qstart, ctx->q, n3 * sizeof(double), cudaMemcpyDeviceToDevice, st));
        CK(cudaMemcpyAsync(w.pstart, ctx->p, n3 * sizeof(double), cudaMemcpyDeviceToDevice, st));
        w.n0 = (uint64_t)ctx->step;
        launch_set_u64(mk(ctx, stream), w.n0_dev, w.n0);
        TRY(run_graphed(ctx, st, w.g_plain[2 * K + which], [&]() -> lsd_status { return rollout_body(ctx, w, K, which, stream, false); }));
        int flags = 0;
        CK(cudaMemcpyAsync(&flags, w.flags, sizeof(int), cudaMemcpyDeviceToHost, st));
        CK(cudaStreamSynchronize(st));
        if ((flags & (LSD_FLAG_SKIN | LSD_FLAG_OVERFLOW)) && list_retries < 6) {   // as in lsd_run: answered by a rebuild; the base state is untouched
            if (flags & LSD_FLAG_NONFINITE) return flags_to_status(ctx, flags);
            ++list_retries;
            if (flags & LSD_FLAG_OVERFLOW) ctx->cap_growth *= 1.5;
            TRY(lsd_set_skin(ctx, (flags & LSD_FLAG_SKIN) ? 2.0 * ctx->cfg.skin : ctx->cfg.skin));
            continue;
        }
        if (flags) return flags_to_status(ctx, flags);
        CK(cudaMemcpyAsync(ctx->q, w.yq + n3 * (K - 1), n3 * sizeof(double), cudaMemcpyDeviceToDevice, st));
        CK(cudaMemcpyAsync(ctx->p, w.yp + n3 * (K - 1), n3 * sizeof(double), cudaMemcpyDeviceToDevice, st));
        ctx->step += K; ctx->stats.step = ctx->step;
        remaining -= K;
    }
    w.drafted = 0; w.verified = 0;
    CK(cudaStreamSynchronize(st));            // the last chunk's copy into the base state
    stream_idle(ctx, st);                     // the caller may destroy `stream` now: the context keeps no handle of it
    if (ctx->tiny && which == LSD_DRAFT) ctx->tiny_draft_lists_stale = true;
    return LSD_OK;
}

lsd_status lsd_get_state(lsd_ctx* ctx, double* q, double* p, int64_t* step, int32_t where)
{
    if (!ctx) return LSD_ERR_INVALID_ARG;
    TRY(sync_pending(ctx));
    // caller-owned DEVICE buffers: the copies below run on the internal non-blocking stream, which is not ordered against the
    // caller's streams (nor torch's default stream), so kernels of the caller that still read q / p must have finished first
    if (where == LSD_DEVICE) CK(cudaDeviceSynchronize());
    const size_t bytes = (size_t)3 * ctx->sys.n * sizeof(double);
    if (where == LSD_HOST && ctx->state_host && q && p) {     // small system: one device-to-host copy of (q, p) through the pinned staging
        CK(cudaMemcpyAsync(ctx->state_host, ctx->q, 2 * bytes, cudaMemcpyDeviceToHost, ctx->side));
        CK(cudaStreamSynchronize(ctx->side));
        std::memcpy(q, ctx->state_host, bytes);
        std::memcpy(p, ctx->state_host + 3 * ctx->sys.n, bytes);
        if (step) *step = ctx->step;
        return LSD_OK;
    }
    const cudaMemcpyKind kind = where == LSD_HOST ? cudaMemcpyDeviceToHost : cudaMemcpyDeviceToDevice;
    if (q) CK(cudaMemcpyAsync(q, ctx->q, bytes, kind, ctx->side));
    if (p) CK(cudaMemcpyAsync(p, ctx->p, bytes, kind, ctx->side));
    if (q || p) CK(cudaStreamSynchronize(ctx->side));
    if (step) *step = ctx->step;
    return LSD_OK;
}

lsd_status lsd_set_state(lsd_ctx* ctx, const double* q, const double* p, int64_t step, int32_t where)
{
    if (!ctx || !q || !p) return LSD_ERR_INVALID_ARG;
    TRY(sync_pending(ctx));
    // caller-owned DEVICE buffers: whatever kernel of the caller produces q / p (on any stream) must have finished before the
    // internal non-blocking stream reads them
    if (where == LSD_DEVICE) CK(cudaDeviceSynchronize());
    const size_t bytes = (size_t)3 * ctx->sys.n * sizeof(double);
    if (where == LSD_HOST && ctx->state_host) {
        // small system: the caller's buffers are copied into the pinned staging (they are free again on return), ONE upload is
        // enqueued on the internal stream and the call does not wait for it: whatever reads q, p next waits for ev_state
        std::memcpy(ctx->state_host, q, bytes);
        std::memcpy(ctx->state_host + 3 * ctx->sys.n, p, bytes);
        CK(cudaMemcpyAsync(ctx->q, ctx->state_host, 2 * bytes, cudaMemcpyHostToDevice, ctx->side));
        if (ctx->ec) CK(cudaMemsetAsync(ctx->dF, 0, bytes, ctx->side));
        CK(cudaEventRecord(ctx->ev_state, ctx->side));
        note_stream(ctx, ctx->side);
        ctx->state_in_flight = true;
        ctx->step = step; ctx->stats.step = step;
        reset_slots(ctx);
        return LSD_OK;
    }
    const cudaMemcpyKind kind = where == LSD_HOST ? cudaMemcpyHostToDevice : cudaMemcpyDeviceToDevice;
    CK(cudaMemcpyAsync(ctx->q, q, bytes, kind, ctx->side));
    CK(cudaMemcpyAsync(ctx->p, p, bytes, kind, ctx->side));
    ctx->step = step; ctx->stats.step = step;
    if (ctx->ec) CK(cudaMemsetAsync(ctx->dF, 0, bytes, ctx->side));   // a new trajectory starts with an empty EC cache; it is all zeros while EC is off
    CK(cudaStreamSynchronize(ctx->side));
    reset_slots(ctx);
    return LSD_OK;
}

lsd_status lsd_set_error_correction(lsd_ctx* ctx, int32_t enable)
{
    if (!ctx) return LSD_ERR_INVALID_ARG;
    CK(cudaDeviceSynchronize());
    ctx->ec = enable ? 1 : 0;
    CK(cudaMemset(ctx->dF, 0, (size_t)3 * ctx->sys.n * sizeof(double)));
    drop_graphs(ctx);                                        // the captured kernels take the cache pointer (or null) by value
    reset_slots(ctx);
    return LSD_OK;
}

lsd_status lsd_set_force_slack(lsd_ctx* ctx, double eps_F)
{
    if (!ctx || !(eps_F >= 0.0)) return LSD_ERR_INVALID_ARG;
    CK(cudaDeviceSynchronize());
    ctx->slack = eps_F;
    drop_graphs(ctx);                                        // the captured kernels take the value by value
    return LSD_OK;
}

lsd_status lsd_get_ec_cache(lsd_ctx* ctx, double* dF, int32_t where)
{
    if (!ctx || !dF) return LSD_ERR_INVALID_ARG;
    CK(cudaDeviceSynchronize());
    return copy_out(ctx, dF, ctx->dF, (size_t)3 * ctx->sys.n * sizeof(double), where);
}

lsd_status lsd_set_ec_cache(lsd_ctx* ctx, const double* dF, int32_t where)
{
    if (!ctx || !dF) return LSD_ERR_INVALID_ARG;
    if (!ctx->ec) return fail(ctx, LSD_ERR_STATE, "error correction is off (lsd_set_error_correction)");
    CK(cudaDeviceSynchronize());
    CK(cudaMemcpy(ctx->dF, dF, (size_t)3 * ctx->sys.n * sizeof(double), where == LSD_HOST ? cudaMemcpyHostToDevice : cudaMemcpyDeviceToDevice));
    reset_slots(ctx);
    return LSD_OK;
}

lsd_status lsd_get_stats(const lsd_ctx* ctx, lsd_stats* out)
{
    if (!ctx || !out) return LSD_ERR_INVALID_ARG;
    *out = ctx->stats; out->step = ctx->step;
    return LSD_OK;
}

lsd_status lsd_get_window_obabo(lsd_ctx* ctx, int32_t j, double* q, double* p, int32_t where)
{
    if (!ctx) return LSD_ERR_INVALID_ARG;
    if (ctx->last_slot < 0) return fail(ctx, LSD_ERR_STATE, "no window has been transported yet");
    if (j < 1 || j > ctx->last_nc) return fail(ctx, LSD_ERR_INVALID_ARG, "j must be in 1..n_commit");
    // Eq. 30 rebuilds p_mid from the kick the step was committed with; with force slack that kick used F_(eps), not the F kept in Fg
    if (ctx->slack > 0.0) return fail(ctx, LSD_ERR_STATE, "OBABO outputs are not available while force slack is on (lsd_set_force_slack(0) first)");
    CK(cudaDeviceSynchronize());
    const WindowSlot& w = ctx->slot[ctx->last_slot];
    const int n = ctx->sys.n;
    const size_t n3 = (size_t)3 * n;
    if (q) TRY(copy_out(ctx, q, w.qhalf + n3 * (j - 1), n3 * sizeof(double), where));      // the (B O B) block leaves positions fixed (:753)
    if (p) {
        if (!ctx->obabo_p) TRY(dalloc(ctx, &ctx->obabo_p, n3));
        launch_obabo(mk(ctx, nullptr), n, ctx->cfg.seed, w.n0_dev, (uint64_t)j, j == 1 ? w.pstart : w.yp + n3 * (j - 2), w.yp + n3 * (j - 1),
                     ctx->Fg + n3 * (j - 1), ctx->sys.mass, ctx->kT, ctx->c1, std::exp(-0.5 * ctx->cfg.friction_per_fs * ctx->cfg.dt_fs), ctx->hdt,
                     ctx->obabo_p);
        CK(cudaDeviceSynchronize());
        TRY(copy_out(ctx, p, ctx->obabo_p, n3 * sizeof(double), where));
    }
    return LSD_OK;
}

lsd_status lsd_get_window_state(lsd_ctx* ctx, int32_t j, double* q, double* p, int32_t where)
{
    if (!ctx) return LSD_ERR_INVALID_ARG;
    if (ctx->last_slot < 0) return fail(ctx, LSD_ERR_STATE, "no window has been transported yet");
    if (j < 1 || j > ctx->last_nc) return fail(ctx, LSD_ERR_INVALID_ARG, "j must be in 1..n_commit");
    // Eq. 30 rebuilds p_mid from the kick the step was committed with; with force slack that kick used F_(eps), not the F kept in Fg
    if (ctx->slack > 0.0) return fail(ctx, LSD_ERR_STATE, "OBABO outputs are not available while force slack is on (lsd_set_force_slack(0) first)");
    CK(cudaDeviceSynchronize());
    const WindowSlot& w = ctx->slot[ctx->last_slot];
    const size_t n3 = (size_t)3 * ctx->sys.n;
    if (q) TRY(copy_out(ctx, q, w.yq + n3 * (j - 1), n3 * sizeof(double), where));
    if (p) TRY(copy_out(ctx, p, w.yp + n3 * (j - 1), n3 * sizeof(double), where));
    return LSD_OK;
}

lsd_status lsd_get_window_debug(lsd_ctx* ctx, int32_t what, void* out, int32_t where)
{
    if (!ctx || !out) return LSD_ERR_INVALID_ARG;
    if (ctx->last_slot < 0) return fail(ctx, LSD_ERR_STATE, "no window has been transported yet");
    CK(cudaDeviceSynchronize());
    const WindowSlot& w = ctx->slot[ctx->last_slot];
    const int K = ctx->last_K;
    const size_t big = (size_t)3 * ctx->sys.n * K * sizeof(double), small = (size_t)K * sizeof(double);
    switch (what) {
        case LSD_DBG_QHALF:   return copy_out(ctx, out, w.qhalf, big, where);
        case LSD_DBG_FDRAFT:  return copy_out(ctx, out, w.Ft, big, where);
        case LSD_DBG_FTARGET: return copy_out(ctx, out, ctx->Fg, big, where);
        case LSD_DBG_YP:      return copy_out(ctx, out, w.yp, big, where);
        case LSD_DBG_YQ:      return copy_out(ctx, out, w.yq, big, where);
        case LSD_DBG_S1:      return copy_out(ctx, out, ctx->S1, small, where);
        case LSD_DBG_S2:      return copy_out(ctx, out, ctx->S2, small, where);
        case LSD_DBG_ELL:     return copy_out(ctx, out, ctx->ell, small, where);
        case LSD_DBG_LNU:     return copy_out(ctx, out, ctx->lnu, small, where);
        case LSD_DBG_REJECT:  return copy_out(ctx, out, ctx->reject, (size_t)K * sizeof(int), where);
        case LSD_DBG_XI: {
            if (!ctx->xi_dbg) TRY(dalloc(ctx, &ctx->xi_dbg, (size_t)3 * ctx->sys.n * ctx->cfg.k_max));
            launch_transport(mk(ctx, nullptr), ctx->sys.n, K, ctx->cfg.seed, w.n0_dev, w.Ft, ctx->Fg, ctx->sys.sigma, ctx->b, ctx->partial, ctx->nblk,
                             ctx->S1, ctx->S2, ctx->ell, ctx->lnu, ctx->reject, w.flags, ctx->result, ctx->xi_dbg, ctx->ec ? w.dF : nullptr, ctx->slack);
            CK(cudaDeviceSynchronize());
            return copy_out(ctx, out, ctx->xi_dbg, big, where);
        }
        default: return fail(ctx, LSD_ERR_INVALID_ARG, "unknown debug row");
    }
}

lsd_status lsd_eval_forces(lsd_ctx* ctx, int32_t which, int32_t n_states, const double* q, double* F, double* energy_nn,
                           int32_t where, void* stream)
{
    if (!ctx || !q || !F || (which != LSD_DRAFT && which != LSD_TARGET)) return LSD_ERR_INVALID_ARG;
    if (n_states < 1 || n_states > ctx->cfg.k_max) return fail(ctx, LSD_ERR_INVALID_ARG, "n_states must be in 1..k_max");
    cudaStream_t st = (cudaStream_t)stream;
    Launcher L = mk(ctx, stream);
    const int n = ctx->sys.n;
    const size_t n3 = (size_t)3 * n;
    const cudaMemcpyKind in_kind = where == LSD_HOST ? cudaMemcpyHostToDevice : cudaMemcpyDeviceToDevice;
    const cudaMemcpyKind out_kind = where == LSD_HOST ? cudaMemcpyDeviceToHost : cudaMemcpyDeviceToDevice;
    CK(cudaMemcpyAsync(ctx->q_eval, q, n3 * n_states * sizeof(double), in_kind, st));
    CK(cudaMemsetAsync(ctx->flags_eval, 0, sizeof(int), st));
    build_lists(ctx, L, ctx->q_eval, ctx->img_eval, ctx->vl_eval_mlip, ctx->vl_eval_pair, ctx->flags_eval);
    const double sh = 0.5 * ctx->cfg.skin;
    launch_check_skin(L, n, n_states, ctx->q_eval, ctx->q_eval, sh * sh, ctx->flags_eval);
    const int bm = ctx->bmax[which];
    for (int b0 = 0; b0 < n_states; b0 += bm) {
        const int B = std::min(bm, n_states - b0);
        eval_forces(ctx, L, which, B, ctx->q_eval + n3 * b0, ctx->img_eval, ctx->vl_eval_mlip, ctx->vl_eval_pair, ctx->F_eval + n3 * b0,
                    ctx->flags_eval, ctx->pot[which].mlip.F > 0 ? ctx->work[which].e_atom : nullptr);
        if (energy_nn && ctx->pot[which].mlip.F > 0)
            CK(cudaMemcpyAsync(ctx->e_eval + (size_t)n * b0, ctx->work[which].e_atom, (size_t)n * B * sizeof(double), cudaMemcpyDeviceToDevice, st));
    }
    CK(cudaMemcpyAsync(F, ctx->F_eval, n3 * n_states * sizeof(double), out_kind, st));
    if (energy_nn) {
        if (ctx->pot[which].mlip.F > 0) CK(cudaMemcpyAsync(energy_nn, ctx->e_eval, (size_t)n * n_states * sizeof(double), out_kind, st));
        else if (where == LSD_HOST) std::memset(energy_nn, 0, (size_t)n * n_states * sizeof(double));
        else CK(cudaMemsetAsync(energy_nn, 0, (size_t)n * n_states * sizeof(double), st));
    }
    int hf = 0;
    CK(cudaMemcpyAsync(&hf, ctx->flags_eval, sizeof(int), cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    CK(cudaGetLastError());
    if (which == LSD_DRAFT) ctx->tiny_draft_lists_stale = false;             // the per-state draft lists are this evaluation's
    return flags_to_status(ctx, hf);
}

lsd_status lsd_get_edge_count(lsd_ctx* ctx, int32_t which, int32_t kind, int32_t n_states, int64_t* total)
{
    if (!ctx || !total || (which != 0 && which != 1) || (kind != 0 && kind != 1)) return LSD_ERR_INVALID_ARG;
    const CompactList& cl = (kind == 0 || ctx->pair_is_mlip[which]) ? ctx->cl_mlip[which] : ctx->cl_pair[which];
    *total = 0;
    if (!cl.count) return LSD_OK;
    if (n_states < 1 || n_states > cl.bmax) return fail(ctx, LSD_ERR_INVALID_ARG, "n_states out of range");
    CK(cudaDeviceSynchronize());
    std::vector<int> count((size_t)ctx->sys.n * n_states);
    CK(cudaMemcpy(count.data(), cl.count, sizeof(int) * count.size(), cudaMemcpyDeviceToHost));
    int64_t t = 0; for (int v : count) t += v;
    *total = t;
    return LSD_OK;
}

lsd_status lsd_profile(lsd_ctx* ctx, int32_t enable)
{
    if (!ctx) return LSD_ERR_INVALID_ARG;
    CK(cudaDeviceSynchronize());
    Prof& p = ctx->prof;
    if (enable && p.ev.empty()) {
        p.ev.resize(2 * 16384); p.cls.resize(16384);
        for (auto& e : p.ev) CK(cudaEventCreate(&e));
    }
    p.on = enable != 0; p.used = 0;
    for (int c = 0; c < PROF_NCLASS; ++c) { p.ms[c] = 0; p.cnt[c] = 0; }
    return LSD_OK;
}

lsd_status lsd_get_profile(lsd_ctx* ctx, double* ms, int64_t* count)
{
    if (!ctx || !ms || !count) return LSD_ERR_INVALID_ARG;
    CK(cudaDeviceSynchronize());
    Prof& p = ctx->prof;
    for (int i = 0; i < p.used; ++i) {
        float t = 0.f;
        CK(cudaEventElapsedTime(&t, p.ev[2 * i], p.ev[2 * i + 1]));
        p.ms[p.cls[i]] += t; p.cnt[p.cls[i]]++;
    }
    p.used = 0;
    for (int c = 0; c < PROF_NCLASS; ++c) { ms[c] = p.ms[c]; count[c] = p.cnt[c]; }
    return LSD_OK;
}

lsd_status lsd_get_neighbors(lsd_ctx* ctx, int32_t which, int32_t kind, int32_t b, int64_t cap, int64_t* start, int32_t* idx,
                             int8_t* shifts, int64_t* n_edges)
{
    if (!ctx || !start || !n_edges || (which != 0 && which != 1) || (kind != 0 && kind != 1)) return LSD_ERR_INVALID_ARG;
    const CompactList& cl = (kind == 0 || ctx->pair_is_mlip[which]) ? ctx->cl_mlip[which] : ctx->cl_pair[which];
    if (!cl.count || !ctx->cl_img[which]) return fail(ctx, LSD_ERR_STATE, "this potential has no such list (or no evaluation has run yet)");
    if (ctx->tiny && which == LSD_DRAFT && ctx->tiny_draft_lists_stale)
        return fail(ctx, LSD_ERR_STATE, "the one-kernel draft rollout of a tiny system keeps its neighbour rows on chip (call lsd_eval_forces(LSD_DRAFT) for a list)");
    if (b < 0 || b >= cl.bmax) return fail(ctx, LSD_ERR_INVALID_ARG, "state index out of range");
    CK(cudaDeviceSynchronize());
    const int n = ctx->sys.n;
    std::vector<int> count(n), img(n);
    std::vector<uint32_t> keys((size_t)n * cl.cap);
    CK(cudaMemcpy(count.data(), cl.count + (size_t)b * n, sizeof(int) * n, cudaMemcpyDeviceToHost));
    CK(cudaMemcpy(keys.data(), cl.keys + (size_t)b * n * cl.cap, sizeof(uint32_t) * keys.size(), cudaMemcpyDeviceToHost));
    CK(cudaMemcpy(img.data(), ctx->cl_img[which], sizeof(int) * n, cudaMemcpyDeviceToHost));
    auto unpack = [](int v, int* o) { o[0] = (v & 1023) - 512; o[1] = ((v >> 10) & 1023) - 512; o[2] = ((v >> 20) & 1023) - 512; };
    int64_t e = 0;
    for (int i = 0; i < n; ++i) {
        start[i] = e;
        int ii[3]; unpack(img[i], ii);
        for (int k = 0; k < count[i]; ++k, ++e) {
            if (e >= cap || !idx || !shifts) continue;
            const uint32_t key = keys[(size_t)i * cl.cap + k];
            const int j = (int)(key >> 5), code = (int)(key & 31u);
            int jj[3]; unpack(img[j], jj);
            idx[e] = j;
            shifts[3 * e + 0] = (int8_t)(code / 9 - 1 + ii[0] - jj[0]);
            shifts[3 * e + 1] = (int8_t)((code / 3) % 3 - 1 + ii[1] - jj[1]);
            shifts[3 * e + 2] = (int8_t)(code % 3 - 1 + ii[2] - jj[2]);
        }
    }
    start[n] = e; *n_edges = e;
    return LSD_OK;
}

}  // extern "C"
