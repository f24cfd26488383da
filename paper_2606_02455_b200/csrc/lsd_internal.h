// Internal declarations shared by the translation units of liblsd_b200.so (sm_100a only).
// Nothing here is shared with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdlib.h>
#include <string>
#include <vector>

#include "lsd.h"

#define LSD_KB_EV   8.617333262e-5   // eV / K
#define LSD_AMU_EV  103.642696       // eV fs^2 / A^2 per amu
#define LSD_NRBF    32               // R (M1)
#define LSD_MAX_K   64
#define LSD_MAX_SLOTS 8             // window slots of a context (lsd_set_window_slots)
#define LSD_TINY_MAX_ATOMS 64      // systems up to this size roll their draft out in one kernel launch (tiny_rollout.cu)
#define LSD_TINY_CLUSTER 8         // ... on one thread-block cluster of this many CTAs

// flags raised on the device during a window
#define LSD_FLAG_SKIN      1
#define LSD_FLAG_OVERFLOW  2
#define LSD_FLAG_NONFINITE 4

struct SysDev {
    int n = 0, ns = 0, periodic = 0;
    double box[3] = {0, 0, 0};
    int* species = nullptr;          // [n]
    double* mass = nullptr;          // [n] internal units (amu * LSD_AMU_EV)
    double* sigma = nullptr;         // [n] sqrt(m kT (1 - c1^2))
    // bonded terms, gather form: per atom list of (term, role)
    int n_bonds = 0, n_angles = 0;
    int* bonds = nullptr; double* bond_k = nullptr; double* bond_r0 = nullptr;
    int* angles = nullptr; double* angle_k = nullptr; double* angle_t0 = nullptr;
    int* bt_start = nullptr;         // [n+1]
    int* bt_term = nullptr;          // term id: bonds 0..nb-1, angles nb..nb+na-1 ; role packed in high bits
};

struct MlipDev {
    int F = 0, T = 0, R = LSD_NRBF, ns = 0;
    float rc = 0.f, alpha = 0.f;
    float* emb = nullptr;                       // [ns][F]
    float* ytab0 = nullptr;                     // [ns][F]  W_in(0) Emb[s]: y of the first block depends on the species only
    // per block, fp32, all stored k-major [K][N] for  C[rows][N] = A[rows][K] * W[K][N]
    std::vector<float*> WinT, Win, Wf1T, Wf2T, Wo1T, Wo1, Wo2T, Wo2;
    float* Wr1 = nullptr;                       // [F/2][F]
    float* wr2 = nullptr;                       // [F/2]
    // bf16 copies for the tcgen05 path (K-major operands), filled when precision == LSD_BF16_TC
    std::vector<void*> Wf1_bf16, Wf2_bf16;
    // width 128: bf16 A operand images of the atom-wise layers and their transposes (mlip_atom_tc128.cu)
    std::vector<void*> Win_tc, WinT_tc, Wo1_tc, Wo1T_tc, Wo2_tc, Wo2T_tc;
    void *Wr1_tc = nullptr, *Wr1T_tc = nullptr;   // readout W_r1 [F/2][F] and its transpose, zero padded to 128 x 128
};

struct PotDev {
    int ns = 0, use_bonded = 0;
    double* pair = nullptr;          // [ns*ns*8]
    double* pair_rc2 = nullptr;      // [ns*ns] squared cutoff of the pair term (0 = none)
    std::vector<double> pair_rc2_host;
    double* tether = nullptr;        // [ns]
    double pair_rcmax = 0.0;
    int has_tether = 0;
    MlipDev mlip;
};

struct VerletList {                  // window-shared candidate list (r < rc + skin at the reference state)
    int cap = 0;
    double rc = 0.0;                 // largest cutoff served
    int* count = nullptr;            // [n]
    uint32_t* keys = nullptr;        // [n][cap]  key = (j << 5) | shiftcode, sorted ascending
};

// Geometry of the directed edges i <- j of one state, written once per batched evaluation by k_compact and read by every
// block's forward and backward edge kernel.  A row (state b, atom i) holds cap/16 groups of 16 slots; a group is a
// 512-byte block of 8 fields x 16 slots (structure of arrays, so a kernel copies it verbatim and reads float4 runs):
//   r = |q_j - q_i + s L|, fc, fc' (cosine cutoff M2 and its slope), ux, uy, uz (unit vector), jrow = b*n + j (row of the
//   gathered features, as int bits), pad.  Slots behind the row's count inside its last group are zero records
//   (fc = fc' = 0, jrow = own row).
#define LSD_REC_R 0
#define LSD_REC_FC 1
#define LSD_REC_FCP 2
#define LSD_REC_UX 3
#define LSD_REC_UY 4
#define LSD_REC_UZ 5
#define LSD_REC_JROW 6
#define LSD_REC_GROUP_FLOATS 128
__host__ __device__ inline size_t lsd_rec_index(size_t row, int cap, int slot, int field)
{
    return row * (size_t)cap * 8 + (size_t)(slot >> 4) * LSD_REC_GROUP_FLOATS + field * 16 + (slot & 15);
}

struct CompactList {                 // per-state exact list (r < rc), rows padded with 0xFFFFFFFF
    int cap = 0, bmax = 0;
    int* count = nullptr;            // [bmax*n]
    uint32_t* keys = nullptr;        // [bmax*n][cap]
    float* recs = nullptr;           // [bmax*n][cap/16][8][16], MLIP lists only (cap is a multiple of 16)
    const float* rec_zero = nullptr; // one zero group behind the records
};

struct CellGrid {
    int nc[3] = {1, 1, 1};
    int ncell = 1;
    int* cell_count = nullptr;       // [ncell]
    int* cell_start = nullptr;       // [ncell+1]
    int* cell_cursor = nullptr;      // [ncell]
    int* cell_atoms = nullptr;       // [n]
    int* atom_cell = nullptr;        // [n]
    int cap_cells = 0;
};

struct MlipWork {                    // activations of one batched evaluation (kept for the analytic backward, M9)
    int bmax = 0;
    float *x = nullptr, *m = nullptr, *mbar = nullptr, *xbar = nullptr, *ybar = nullptr;
    std::vector<float*> y, h;        // [T] each [bmax*n][F]
    std::vector<uint16_t*> y16;      // [T] bf16 copies of y gathered by the tcgen05 edge kernels (LSD_BF16_TC only)
    uint16_t* mbar16 = nullptr;      // bf16 copy of mbar
    uint32_t* ym16 = nullptr;        // width 128 only: rows of (y, mbar) bf16 pairs gathered by the backward tcgen05 kernel
    void* ym_tmap = nullptr;         // device copy of the TMA tensor map over ym16 (rows of 512 B, boxes of 128 B x 1 row, 128-byte swizzle)
    double* e_atom = nullptr;        // [bmax*n]
    int y0_rows = 0;                 // one-block networks: rows of y[0] / y16[0] (species-only) already written
};

// optional per-kernel-class timing with CUDA events on the launching stream (bench.py's roofline numbers)
enum ProfClass { PROF_NBR = 0, PROF_PRIOR = 1, PROF_DENSE = 2, PROF_EDGE_FWD = 3, PROF_EDGE_BWD = 4, PROF_INTEG = 5, PROF_TRANSPORT = 6, PROF_DRAFT_MLIP = 7, PROF_NCLASS = 8 };
struct Prof {
    bool on = false;
    std::vector<cudaEvent_t> ev;     // pairs
    std::vector<int> cls;
    int used = 0;
    double ms[PROF_NCLASS] = {0};
    int64_t cnt[PROF_NCLASS] = {0};
};
struct Launcher {                    // stream + launch counter (+ profiler)
    cudaStream_t s;
    int64_t* counter;
    Prof* prof = nullptr;
    int draft = 0;                   // 1: kernels of the draft potential (their MLIP launches are timed as one class)
};
#define LSD_COUNT(L) (++(*(L).counter))

// Programmatic dependent launch (PDL): the small kernels of a window form one long dependency chain (a draft step is ~10
// kernels of a few microseconds), so each kernel is launched with the programmatic-stream-serialization attribute and begins
// with pdl_sync(): wait until the kernels before it have completed and flushed, then let the next kernel's CTAs be scheduled
// (they block in their own wait until this grid has completed), which takes the launch latency off the critical path.
// pdl_sync() must be the first statement of the kernel, before any early return (completion is transitive only if every
// CTA waits).  A kernel without the attribute, or behind a kernel without pdl_sync(), simply keeps the full dependency.
#ifdef __CUDACC__
__device__ __forceinline__ void pdl_sync()
{
    asm volatile("griddepcontrol.wait;" ::: "memory");
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
}
inline bool lsd_pdl_enabled()
{
    static const bool on = [] { const char* v = getenv("LSD_PDL"); return !(v && v[0] == '0'); }();
    return on;
}
template <typename... KA, typename... A>
inline void launch_pdl(const Launcher& L, void (*kernel)(KA...), dim3 grid, dim3 block, size_t smem, A&&... args)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = L.s;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = lsd_pdl_enabled() ? 1 : 0;
    cudaLaunchKernelEx(&cfg, kernel, static_cast<KA>(args)...);
}
#endif
inline int prof_begin(const Launcher& L, int cls)
{
    Prof* p = L.prof;
    if (!p || !p->on || (size_t)(2 * p->used + 2) > p->ev.size()) return -1;
    const int id = p->used++;
    if (L.draft && (cls == PROF_DENSE || cls == PROF_EDGE_FWD || cls == PROF_EDGE_BWD)) cls = PROF_DRAFT_MLIP;
    p->cls[id] = cls;
    cudaEventRecord(p->ev[2 * id], L.s);
    return id;
}
inline void prof_end(const Launcher& L, int id) { if (id >= 0) cudaEventRecord(L.prof->ev[2 * id + 1], L.s); }

// ---- integrator.cu
void launch_half_a(Launcher L, int n, const double* q, const double* p, const double* mass, double hdt,
                   double* qhalf, const double* qref, double skin_half2, int* flags);
void launch_set_u64(Launcher L, uint64_t* dst, uint64_t v);
void launch_bob_a(Launcher L, int n, uint64_t seed, const uint64_t* n0_dev, uint64_t j, const double* p_prev, const double* Ft,
                  const double* qhalf, const double* mass, const double* sigma, double c1, double b, double hdt,
                  double* q_new, double* p_new, const double* dF /*EC cache or null*/,
                  double* qhalf_next = nullptr /*also write the next step's q_half and check the skin against qref*/,
                  const double* qref = nullptr, double skin_half2 = 0.0, int* flags = nullptr);
void launch_initial_momenta(Launcher L, int n, uint64_t seed, const double* mass, double kT, double* p);
struct TransportResult { int first_reject, n_commit, flags, pad; double beta_sum; };
void launch_transport(Launcher L, int n, int K, uint64_t seed, const uint64_t* n0_dev, const double* Ft, const double* Fg,
                      const double* sigma, double b, double* partial, int nblk, double* S1, double* S2, double* ell,
                      double* lnu, int* reject, const int* flags, TransportResult* result, double* xi_dbg, const double* dF, double slack = 0.0);
void launch_commit(Launcher L, int n, int K, uint64_t seed, const uint64_t* n0_dev, const TransportResult* result,
                   const double* S1, const double* S2, const double* Ft, const double* Fg, const double* qhalf,
                   const double* pstart, double* yq, double* yp, const double* mass, const double* sigma,
                   double c1, double b, double hdt, double* q_base, double* p_base, const double* dF, double* dF_out, double slack = 0.0);
int transport_blocks(int n);
void launch_obabo(Launcher L, int n, uint64_t seed, const uint64_t* n0_dev, uint64_t j, const double* p_prev, const double* p_new,
                  const double* F, const double* mass, double kT, double c1, double ch, double hdt, double* p_mid);

// ---- tiny_rollout.cu: the K draft steps of a window of a tiny system as one kernel launch
bool tiny_rollout_supported(const SysDev& sys, const PotDev& pot);
void launch_tiny_rollout(Launcher L, const SysDev& sys, const PotDev& pot, int K, uint64_t seed, const uint64_t* n0_dev,
                         double c1, double b, double hdt, double skin_half2, const double* qstart, const double* pstart,
                         const double* dF /*EC cache or null*/, double* qhalf, double* Ft, double* yq, double* yp, int* flags);

// ---- neighbor.cu
void cellgrid_setup(CellGrid& g, const SysDev& sys, double rc_skin);
void launch_pack_ref(Launcher L, const SysDev& sys, const double* qref, int* img);
void launch_build_verlet(Launcher L, const SysDev& sys, CellGrid& g, const double* qref, const int* img,
                         double rc_skin, VerletList& vl, int* flags,
                         const double* pair_rcs2 = nullptr /*[ns][ns] per-species-pair (cutoff + skin)^2 of a pair-prior list, 0 = pair does not interact*/);
void launch_compact(Launcher L, const SysDev& sys, int B, const double* q /*[B][3][n]*/, const int* img,
                    const VerletList& vl, double rc2_single, const double* pair_rc2 /*or null*/, CompactList& cl, int* flags,
                    float rc_records = 0.f /* > 0: also write cl.recs with the cutoff function of this radius */);
void launch_check_skin(Launcher L, int n, int B, const double* q, const double* qref, double skin_half2, int* flags);

// ---- prior.cu
void launch_prior_forces(Launcher L, const SysDev& sys, const PotDev& pot, int B, const double* q, const int* img,
                         const CompactList* pairlist, double* F /*[B][3][n], overwritten*/);

// arguments of the continuous-filter convolution kernels (fp32 and tcgen05 variants)
struct EdgeArgs {
    int total, n, cap;
    const int* count; const uint32_t* keys; const float* recs;
    const float* rec_zero = nullptr;  // one all-zero record group (512 bytes) behind the records
    float rc, inv_rc, delta, inv_delta2;
    const float *Wf1, *Wf2;           // [R][F], [F][F] (k-major), fp32 path
    const void *Wf1_tc = nullptr, *Wf2_tc = nullptr;   // bf16, UMMA canonical K-major layouts (mlip_tc.cu)
    const float* y;                   // [total][F]
    const uint16_t *y16 = nullptr, *mbar16 = nullptr;   // bf16 rows gathered by the tcgen05 kernels
    const uint32_t* ym16 = nullptr;   // [total][F] (y | mbar << 16) bf16 pairs, width-128 backward kernel
    const void* ym_tmap = nullptr;    // TMA tensor map over ym16 (global memory); null: cp.async gathers
    float* m_out;                     // FWD: m
    uint16_t* m16_out = nullptr;      // FWD, width 128: m as bf16 rows instead of m_out
    uint16_t* ybar16_out = nullptr;   // BWD, width 128: ybar as bf16 rows instead of ybar
    const float* mbar; float* ybar;   // BWD
    double* Fout;                     // BWD: [B][3][n], accumulated
#ifdef LSD_EDGE_TRACE_BUILD
    unsigned long long* trace = nullptr;   // debug builds (LSD_NVCC_FLAGS=-DLSD_EDGE_TRACE_BUILD, then LSD_EDGE_TRACE=1): clock64 stamps of one chunk of block 0
#endif
};

// per-device one-time state (function attributes, SM count): indexed by the current device, not per process
inline int lsd_current_device() { int d = 0; cudaGetDevice(&d); return (d < 0 || d >= 64) ? 0 : d; }
inline int lsd_sm_count()
{
    static int sms[64] = {};
    int& v = sms[lsd_current_device()];
    if (!v) { int dev = 0; cudaGetDevice(&dev); cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, dev); if (v <= 0) v = 148; }
    return v;
}

// which tcgen05 edge kernel the last forward / backward launch of this process used (parity tests assert that the timed
// instantiation is the one they compared with the oracle): kernel 4 = k_edge_rows (width 128), 7 = k_edge_rows (narrow widths),
// 8 = k_edge_fwd4, 9 = k_edge_rows with TMA gathers (1, 2, 3, 5 were round-1 / opt-in kernels, removed in round 3)
struct EdgeLaunchInfo { int kernel = 0, atoms_per_chunk = 0, threads = 0, grid = 0, width = 0; };
inline EdgeLaunchInfo g_edge_last[2];
inline void note_edge_launch(bool backward, int kernel, int atoms_per_chunk, int threads, int grid, int width)
{
    g_edge_last[backward ? 1 : 0] = EdgeLaunchInfo{kernel, atoms_per_chunk, threads, grid, width};
}

// ---- mlip_simt.cu
void mlip_forward_backward_fp32(Launcher L, const SysDev& sys, const MlipDev& net, MlipWork& w, int B, const double* q,
                                const int* img, const CompactList& cl, double* F /*accumulated*/, double* e_atom);
size_t mlip_work_bytes(const MlipDev& net, int n, int bmax);

// ---- bf16 tcgen05 filter path (mlip_tc.cu: host-side packing; the kernels are in mlip_edge_*.cu)
bool mlip_tc_supported(const MlipDev& net);
void launch_edge_rows(Launcher L, const EdgeArgs& a, bool backward);       // mlip_edge_rows.cu: width 128, edges-as-rows, activations in TMEM
bool lsd_encode_row_tmap(void* host_map_128B, const void* base, size_t rows, int row_bytes);   // mlip_edge_rows.cu: false if the driver lacks the entry point
void launch_edge_fwd4(Launcher L, const EdgeArgs& a);                      // mlip_edge_fwd4.cu: width 128, forward, four tiles in flight per SM
void launch_edge_rows_narrow(Launcher L, const EdgeArgs& a, int F, bool backward);   // mlip_edge_rows_narrow.cu: the same kernel, width-generic, for widths 32 / 64 (fp32 rows out)
// host: pack W_f1 [F][R] / W_f2 [F][F] (row-major fp64) as bf16 in the no-swizzle K-major UMMA layout
void tc_pack_weights(const double* Wf1, const double* Wf2, int F, int R, std::vector<uint16_t>& out1, std::vector<uint16_t>& out2);
void mlip_forward_backward_bf16tc(Launcher L, const SysDev& sys, const MlipDev& net, MlipWork& w, int B, const double* q,
                                  const int* img, const CompactList& cl, double* F, double* e_atom);

// ---- mlip_atom_tc128.cu (width 128: atom-wise layers on the tensor cores, whole bf16 network driver)
void tc_pack_square128(const double* W, bool transpose, std::vector<uint16_t>& out);
void tc_pack_rect128(const double* W, int rows, int cols, bool transpose, std::vector<uint16_t>& out);
void mlip_forward_backward_tc128(Launcher L, const SysDev& sys, const MlipDev& net, MlipWork& w, int B, const double* q,
                                 const int* img, const CompactList& cl, double* F, double* e_atom);
