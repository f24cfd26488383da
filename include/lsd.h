/*
 * lsd.h -- C ABI of liblsd_b200.so: the window-verification hot path of Langevin Speculative
 * Dynamics (LSD, arxiv/paper_2606_02455) on one NVIDIA B200 (sm_100a).
 *
 * Citations are /root/reference/PAPER.md:<line> plus section / equation / algorithm; readings of
 * points where the paper is silent are numbered R1..R16 / M1..M9 in DESIGN.md.
 *
 * The problem statement fixes the arguments (PAPER.md:41 positions q, momenta p, diagonal mass
 * matrix M; :45-50, :66 temperature T, friction gamma, time step dt; :76 a draft and a target
 * force field; :572 initial state x_0).  "BAOAB" in the task metadata is implemented as the paper's
 * ABOBA splitting (Eq. 2; Alg. 2 :568); R1.
 *
 * Conventions
 *   - plain C, no exceptions; every call returns an lsd_status (0 = LSD_OK, negative = error) and
 *     leaves a message retrievable with lsd_last_error().
 *   - units: Angstrom, fs, eV, K; masses in amu at the boundary (1 amu A^2/fs^2 = 103.642696 eV).
 *   - vectors over atoms are component-major ("SoA"): q[c * n_atoms + i], c = 0,1,2.  Batches of
 *     states are state-major: q[(k * 3 + c) * n_atoms + i].
 *   - pointers inside lsd_system / lsd_potential and q0/p0 of lsd_init are HOST pointers; they are
 *     copied during lsd_init and need not outlive it.
 *   - `where` arguments say whether a bulk pointer is host (LSD_HOST) or device (LSD_DEVICE)
 *     memory.  Device buffers are owned by the caller (e.g. torch tensors).
 *   - `stream` is a cudaStream_t passed as void* (NULL = default stream).  Calls enqueue work on it
 *     and return immediately, except where a host-visible result is produced (stated below).
 *   - the context owns all internal device memory; one context must not be used from two host
 *     threads at once.
 *   - there is no CPU fallback: without a CUDA device lsd_init fails with LSD_ERR_CUDA.
 */
#ifndef LSD_H
#define LSD_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef int32_t lsd_status;
#define LSD_OK                  0
#define LSD_ERR_INVALID_ARG    (-1)
#define LSD_ERR_CUDA           (-2)
#define LSD_ERR_OOM            (-3)
#define LSD_ERR_STATE          (-4)   /* call order violated                                        */
#define LSD_ERR_UNSUPPORTED    (-5)
#define LSD_ERR_NBR_OVERFLOW   (-6)   /* a neighbour row exceeded its capacity                      */
#define LSD_ERR_SKIN_VIOLATED  (-7)   /* an atom moved > skin/2 from the list's reference state     */
#define LSD_ERR_NONFINITE      (-8)

#define LSD_HOST    0
#define LSD_DEVICE  1

#define LSD_SCHEME_ABOBA 0            /* A(1/2) B(1/2) O B(1/2) A(1/2), Eq. 2        */

/* arithmetic of the MLIP (state, priors, transport reductions are always fp64)                     */
#define LSD_FP32     1                /* fp32 FMA pipes                                              */
#define LSD_BF16_TC  2                /* bf16 tcgen05 filter contractions, fp32 accumulation         */

/* which potential */
#define LSD_DRAFT   0
#define LSD_TARGET  1

/* pair-parameter table columns, per ordered species pair (zero = term off) */
#define LSD_PAIR_COLS 8               /* lj_eps, lj_sigma, lj_rc, morse_D, morse_a, morse_r0, morse_rc, tether_k */

typedef struct lsd_ctx lsd_ctx;

typedef struct {
    int32_t n_atoms, n_species;
    int32_t periodic;                 /* 1: orthorhombic periodic box (box >= 2 (r_c + skin) required); 0: vacuum */
    double  box[3];
    const int32_t* species;           /* [n_atoms], 0 <= s < n_species                               */
    const double*  mass_amu;          /* [n_atoms] diagonal of M                       */
    int32_t n_bonds;  const int32_t* bonds;  /* [n_bonds][2]                                        */
    const double*  bond_k;  const double* bond_r0;          /* U = k/2 (r - r0)^2                   */
    int32_t n_angles; const int32_t* angles; /* [n_angles][3] (end, apex, end)                      */
    const double*  angle_k; const double* angle_theta0;     /* U = k/2 (theta - theta0)^2, radians  */
} lsd_system;

/* SchNet-style network, M1-M8.  weights: flat fp64, emb[ns][F]; per block W_in[F][F],
 * W_f1[F][R], W_f2[F][F], W_o1[F][F], W_o2[F][F] (row-major [out][in]); W_r1[F/2][F]; w_r2[F/2]. */
typedef struct {
    int32_t width;                    /* F in {32, 64, 128}; 0 = no network                          */
    int32_t n_blocks;                 /* T >= 1                                                      */
    int32_t n_rbf;                    /* R = 32                                                      */
    int32_t n_species;
    double  cutoff;                   /* r_c (A)                                                     */
    double  energy_scale;             /* alpha                                                       */
    const double* weights;
} lsd_mlip;

typedef struct {
    int32_t n_species;
    int32_t use_bonded;               /* include the system's bonds and angles                        */
    const double* pair;               /* [n_species][n_species][LSD_PAIR_COLS]                       */
    lsd_mlip mlip;
} lsd_potential;

typedef struct {
    double   temperature_K, friction_per_fs, dt_fs;
    uint64_t seed;                    /* Philox4x32-10 key (R5)                                      */
    int32_t  scheme;                  /* LSD_SCHEME_ABOBA                                            */
    int32_t  precision;               /* LSD_FP32 | LSD_BF16_TC                                      */
    int32_t  k_max;                   /* largest window length K that will be requested (<= 64)      */
    double   skin;                    /* Verlet skin (A) of the window-shared neighbour lists        */
} lsd_config;

typedef struct {
    int64_t windows, committed_steps, rejections;
    double  beta_sum;                 /* sum over committed steps of erf(sqrt(S2)/sqrt 8), Eq. 9     */
    int64_t step;                     /* committed step index n of the base state                    */
} lsd_stats;

/* Create a context.  q0: [3][n_atoms].  p0: [3][n_atoms] or NULL -> Maxwell-Boltzmann momenta
 * p_i = sqrt(m_i k_B T) xi from Philox stream tag 2 (R12).  Builds the first neighbour lists to size
 * the rows (synchronises).  Errors: INVALID_ARG (sizes, widths, box < 2 (r_c + skin)), CUDA, OOM. */
lsd_status lsd_init(const lsd_config* cfg, const lsd_system* sys, const lsd_potential* draft,
                    const lsd_potential* target, const double* q0, const double* p0, lsd_ctx** out);
void        lsd_destroy(lsd_ctx* ctx);
const char* lsd_last_error(const lsd_ctx* ctx);   /* ctx may be NULL: error of the last failed lsd_init */

/* a0 (PAPER.md:584-593 DRAFT_STEP; Eq. 2, Eq. 7): draft K ABOBA steps from the current draft head
 * (the base state, or y_K of the previous, still unverified window), storing per step q_half_j,
 * draft forces F~_j and y_j in the next window slot.  Builds the window-shared Verlet lists from the
 * head state first.  Noise xi_j = Philox(seed; step index n + j, atom) (R5).  Asynchronous.
 * Errors: INVALID_ARG (K < 1 or > k_max), STATE (every window slot already holds an unverified window). */
lsd_status lsd_draft_rollout(lsd_ctx* ctx, int32_t K, void* stream);

/* a1 + a2 (PAPER.md:598-599 VERIFY_STEP): one batched target force evaluation F_j = F(q_half_j) for
 * all K draft states of the oldest unverified window (waits on the rollout's event).  Asynchronous. */
lsd_status lsd_verify_window(lsd_ctx* ctx, int32_t K, void* stream);

/* a3 + a4 + a5 (PAPER.md:108-111 Eq. 8 REFLECTIONVERIFY; :424 l = min{j : x_j != y_j}; :602 map g):
 * per step d = (b/sigma)(F~ - F), S1 = xi.d, S2 = d.d, ell = -S1 - S2/2, u_j ~ U(0,1);
 * reject_j = S2 > 0 and ln u_j > min(0, ell).  The first rejected step l is overridden with
 * p* = c1 p_{l-1} + b F_l + sigma (xi_l - 2 (S1/S2) d_l), q* = q_half_l + (dt/2) p* / m and becomes the
 * new base state; with no rejection y_K does.  SYNCHRONISES on `stream` and returns
 * *first_reject (0 = none, else 1..K) and *n_commit (l, or K).  Errors: STATE, SKIN_VIOLATED /
 * NBR_OVERFLOW (nothing is committed; enlarge with lsd_set_skin and redo the window), NONFINITE. */
lsd_status lsd_transport_accept(lsd_ctx* ctx, int32_t K, void* stream, int32_t* first_reject, int32_t* n_commit);

/* a6 (PAPER.md:78 "flush them and restart drafting from the just overridden state"; :612 y <- x'):
 * book-keeping after lsd_transport_accept.  first_reject == 0: the K drafted states are committed,
 * a speculative next window (if drafted) stays valid.  first_reject == l > 0: l states are committed,
 * any speculative window is discarded and the draft head returns to the base state (also for l == K). */
lsd_status lsd_rollback(lsd_ctx* ctx, int32_t first_reject);

/* Convenience driver: repeat {rollout, verify, transport, rollback} until n_steps more steps are committed (the last
 * window is shortened).  overlap = d > 0: Alg. 2's asynchronous drafting on one device (Eq. 22 against the
 * synchronous Eq. 21, :555-566): while a window is verified, up to d speculative windows -- each continuing from y_K of the
 * one before it -- are kept drafted ahead on a second internal stream, so the drafter never waits for the 8-byte verdict; a
 * rejection flushes all of them (:611-612).  d is capped at (window slots - 1); the committed trajectory does not depend
 * on d (R5).  Synchronous. */
lsd_status lsd_run(lsd_ctx* ctx, int64_t n_steps, int32_t K, int32_t overlap, void* stream);
/* Number of window slots of the context (2 after lsd_init, at most 8): lsd_draft_rollout may hold that many drafted,
 * unverified windows (Alg. 2's buffers of drafted steps); every slot owns its window rows and its
 * window-shared neighbour lists.  Synchronises, drops drafted windows.  Errors: INVALID_ARG, OOM. */
lsd_status lsd_set_window_slots(lsd_ctx* ctx, int32_t n_slots);
/* lsd_run with K = 0: adaptive lookahead (the window length is the paper's free parameter L): K moves
 * over {1, 2, 4, ..., k_max} by hill climbing on the measured committed steps per second.  With error correction off the
 * committed trajectory does not depend on the K sequence (R5).  lsd_get_adaptive_k: the length it last settled on (0: never). */
int32_t lsd_get_adaptive_k(const lsd_ctx* ctx);

/* Plain Langevin dynamics (no speculation): n_steps ABOBA steps (Eq. 2) with the forces of potential `which`
 * (LSD_TARGET: the serial baseline in the paper's definition of speed-up; LSD_DRAFT: the draft alone) from
 * the base state, same kernels and same noise keying as the draft rollout (R5), committed in chunks of k_max steps that
 * share one neighbour list; synchronises once per chunk and before it returns (`stream` may be destroyed afterwards).  With `which` = LSD_TARGET the trajectory equals LSD with
 * draft = target.  A skin violation or row overflow inside a chunk is answered like in lsd_run (lists rebuilt with a larger
 * skin, chunk repeated).  Errors: STATE (a drafted window is pending), NONFINITE (the base state is the last good one). */
lsd_status lsd_plain_langevin(lsd_ctx* ctx, int32_t which, int64_t n_steps, void* stream);

/* Base state x_n: q, p [3][n_atoms] (either may be NULL), *step = n.
 * where = LSD_DEVICE (caller-owned device buffers): both calls synchronise the WHOLE device first, so the copy is ordered after
 * every kernel of the caller that produces (set) or still reads (get) the buffers, whatever stream it runs on, and is complete
 * on return.  where = LSD_HOST: lsd_get_state waits for this context's own work and returns with q, p filled.  lsd_set_state
 * copies the caller's arrays before it returns (they may be re-used at once); for small systems the upload itself is only
 * enqueued, and every later call of this context that reads the state waits for it. */
lsd_status lsd_get_state(lsd_ctx* ctx, double* q, double* p, int64_t* step, int32_t where);
lsd_status lsd_set_state(lsd_ctx* ctx, const double* q, const double* p, int64_t step, int32_t where);
lsd_status lsd_get_stats(const lsd_ctx* ctx, lsd_stats* out);

/* Committed state j (1..n_commit) of the window most recently passed to lsd_transport_accept. */
lsd_status lsd_get_window_state(lsd_ctx* ctx, int32_t j, double* q, double* p, int32_t where);

/* (OBABO) output of committed step j (1 <= j <= n_commit) of the window lsd_transport_accept handled last, recovered by time
 * staggering (App. F :632-753): q = q_half_j (:753), p = p_mid of Eq. 30 from the committed
 * momenta before and after the step, the target force F_j already evaluated by the verification (no force call) and one
 * extra normal per component drawn from Philox stream tag 3 at step index n0 + j (R18).  Valid until the next
 * lsd_verify_window (it overwrites F).  q, p: [3][n_atoms] or NULL; `where` = LSD_HOST | LSD_DEVICE.  Synchronises.
 * Errors: STATE (no window transported yet; or force slack is on: the committed kicks then used F_(eps), which is not kept,
 * so Eq. 30 cannot be evaluated consistently -- switch slack off first), INVALID_ARG (j). */
lsd_status lsd_get_window_obabo(lsd_ctx* ctx, int32_t j, double* q, double* p, int32_t where);

/* Speculative error correction, EC (App. E :626-630; Alg. 3 :663-717), window form:
 * the draft kick uses F~ + dF, the transport map uses delta = (b/sigma)(F~ + dF - F), and after every window the cache
 * becomes dF = F - F~ (BARE draft output, :628) of the window's last committed step.  A window uses the cache as it stood
 * when it was drafted (a speculative next-window rollout inherits the cache of the window before it).  Target exactness
 * is unaffected (Thm. 3.1 holds for any draft law, :630); the committed trajectory is no longer independent of K.
 * lsd_set_error_correction: enable != 0 switches EC on; either way the cache is zeroed (:669) and drafted windows are
 * dropped.  lsd_get/set_ec_cache: dF is [3][n_atoms] fp64, `where` = LSD_HOST | LSD_DEVICE; set requires EC on (STATE).
 * lsd_set_state also zeroes the cache.  All three synchronise the device. */
lsd_status lsd_set_error_correction(lsd_ctx* ctx, int32_t enable);
lsd_status lsd_get_ec_cache(lsd_ctx* ctx, double* dF, int32_t where);
lsd_status lsd_set_ec_cache(lsd_ctx* ctx, const double* dF, int32_t where);

/* Force slack (App. H), OFF by default: with eps_F > 0 the verification replaces the target
 * force F by F_(eps) = F + clip(-eps_F; F~ - F; eps_F) component by component (F~: the force the draft was drawn around), in the
 * transport map and in the override.  This BREAKS target exactness (:781; the paper recommends against it, :787); eps_F = 0 restores
 * the exact method.  Units eV/A.  Synchronises; captured launch sequences are dropped.  Errors: INVALID_ARG (eps_F < 0 or NaN). */
lsd_status lsd_set_force_slack(lsd_ctx* ctx, double eps_F);

/* Debug rows of that window (parity tests).  `what`: */
#define LSD_DBG_QHALF    0   /* double [K][3][n]   positions after the first A half-step                */
#define LSD_DBG_FDRAFT   1   /* double [K][3][n]   F~_j                                                */
#define LSD_DBG_FTARGET  2   /* double [K][3][n]   F_j                                                 */
#define LSD_DBG_S1       3   /* double [K]                                                             */
#define LSD_DBG_S2       4   /* double [K]                                                             */
#define LSD_DBG_ELL      5   /* double [K]         log-ratio                                           */
#define LSD_DBG_LNU      6   /* double [K]         ln u_j                                              */
#define LSD_DBG_REJECT   7   /* int32  [K]                                                             */
#define LSD_DBG_XI       8   /* double [K][3][n]   the regenerated normals                             */
#define LSD_DBG_YP       9   /* double [K][3][n]   draft momenta p~_j                                  */
#define LSD_DBG_YQ      10   /* double [K][3][n]   draft positions q~_j                                */
lsd_status lsd_get_window_debug(lsd_ctx* ctx, int32_t what, void* out, int32_t where);

/* One batched force evaluation outside the LSD loop (parity, benchmarks): F[b] = F_which(q[b]) for
 * n_states states, q and F [n_states][3][n_atoms].  All states must lie within skin/2 of state 0
 * (they share one Verlet list) else SKIN_VIOLATED.  energy_nn (may be NULL): [n_states][n_atoms]
 * per-atom network energies alpha e_i (M6).  Synchronises. */
lsd_status lsd_eval_forces(lsd_ctx* ctx, int32_t which, int32_t n_states, const double* q, double* F,
                           double* energy_nn, int32_t where, void* stream);

/* Effective directed edge set of state b of the last lsd_eval_forces / lsd_verify_window call
 * (T1): kind 0 = network list (r < r_c), 1 = pair-prior list (r < r_c(s_i, s_j)).
 * Host outputs: start[n_atoms + 1], idx[cap], shifts[cap][3]; *n_edges = total (may exceed cap, then
 * only cap entries are written).  Rows are sorted by (j, shift).  Synchronises.  Errors: STATE (no evaluation yet; or
 * which = LSD_DRAFT in a context with the one-kernel tiny rollout and no lsd_eval_forces(LSD_DRAFT) since the last rollout:
 * that rollout keeps its neighbour rows on chip). */
lsd_status lsd_get_neighbors(lsd_ctx* ctx, int32_t which, int32_t kind, int32_t b, int64_t cap,
                             int64_t* start, int32_t* idx, int8_t* shifts, int64_t* n_edges);

/* Re-size the window-shared lists for a new skin (synchronises; drops drafted windows).  lsd_run calls it with
 * 2 x skin when a window reports SKIN_VIOLATED and redoes that window. */
lsd_status lsd_set_skin(lsd_ctx* ctx, double skin);

/* Total number of directed edges in the exact lists of the first n_states states of the last evaluation of
 * potential `which` (kind as in lsd_get_neighbors).  Synchronises. */
lsd_status lsd_get_edge_count(lsd_ctx* ctx, int32_t which, int32_t kind, int32_t n_states, int64_t* total);

/* Per-kernel-class device timing with CUDA events on the launching stream (used by bench.py for the roofline).
 * Classes: 0 neighbour lists, 1 priors, 2 MLIP atom-wise layers, 3 MLIP edge forward, 4 MLIP edge backward,
 * 5 integrator, 6 transport, 7 all MLIP kernels of the draft potential (classes 2-4 then hold the target's only).
 * lsd_profile(1) starts (and clears), lsd_profile(0) stops.  lsd_get_profile
 * synchronises and returns accumulated milliseconds and launch counts, ms[8], count[8]. */
lsd_status lsd_profile(lsd_ctx* ctx, int32_t enable);
lsd_status lsd_get_profile(lsd_ctx* ctx, double* ms, int64_t* count);

/* Measured plain-FMA peak of the current device in TFLOP/s, kind 0 = fp32, 1 = fp64 (16 independent FMA chains per thread on a
 * grid of resident warps, CUDA events on `stream`, best of three): the roofline denominators of the fp32 MLIP path and of the
 * fp64 path ("measured fp32-FMA peak", "measured fp64 peak").  Synchronises.  Errors: INVALID_ARG, CUDA. */
lsd_status lsd_measure_fma_peak(int32_t kind, void* stream, double* tflops);
/* Number of kernels this library has launched on behalf of ctx (bench.py's gpu_launches). */
int64_t     lsd_launch_count(const lsd_ctx* ctx);
const char* lsd_version(void);
/* Which tcgen05 edge kernel the last MLIP edge launch of this process used, pass 0 = forward (M5), 1 = backward (M9); parity
 * tests use it to assert that the instantiation they compared with the oracle is the one the benchmark times.
 * out[5] = {kernel (0: none yet; 4 k_edge_rows [width 128: the default backward; the forward with LSD_EDGE_FWD4=0], 7 k_edge_rows of
 * the narrow widths 32 / 64, 8 k_edge_fwd4 [width 128, the default forward], 9 k_edge_rows with TMA gathers [LSD_EDGE_TMA=1];
 * ids 1, 2, 3, 5 belonged to kernels removed in round 3), atoms per chunk, threads per block, grid size, network width}.
 * Errors: INVALID_ARG. */
lsd_status lsd_get_edge_launch_info(int32_t pass, int32_t* out);
/* 1 if the target network's filter contractions run on the bf16 tcgen05 path in this context, else 0. */
int32_t     lsd_tc_enabled(const lsd_ctx* ctx);
/* 1 if lsd_draft_rollout drafts a window with ONE kernel launch in this context (a0: the K serial
 * DRAFT_STEPs of a system of <= 64 atoms on one thread-block cluster), else 0 (one launch sequence
 * per step).  It is used when the draft is a different potential than the target and is a prior with at most a width-32,
 * one-block network; the environment variable LSD_TINY=0, read by lsd_init, turns it off (A/B measurements). */
int32_t     lsd_tiny_rollout_enabled(const lsd_ctx* ctx);

/* ---- The one entry point that allocates nothing ----------------------------------------------------------------------------
 * lsd_transport_window_noalloc: steps a3 + a4 (PAPER.md:108-111 Eq. 8 REFLECTIONVERIFY, :424 l = min{j : x_j != y_j}) for a window
 * whose draft and target forces the caller already holds in device memory.  No context, and no cudaMalloc / cudaFree / other
 * allocating call, ever.
 *
 * It exists for callers that are not allowed to allocate GPU memory: a host program (an MD engine, a PyTorch job) whose own
 * pool already owns almost all of the device, so that a cudaMalloc made by this library would fail or fragment the pool; and a
 * force / acceptance callback inside another program's step loop, where the device-wide synchronisation that cudaMalloc and
 * cudaFree imply would stall that program's other streams.  Every other call of this header needs an lsd_ctx, and lsd_init
 * allocates.
 *
 * The per-block partial sums of S1 and S2 go to a fixed array inside the library (151,552 bytes of device memory, held by every
 * GPU that has loaded liblsd_b200.so until the process exits).  Its size sets the limits: K <= LSD_NOALLOC_MAX_K and
 * n_atoms <= LSD_NOALLOC_MAX_ATOMS; anything larger is refused with LSD_ERR_INVALID_ARG and a message, nothing is launched.
 *
 *   inputs  (DEVICE, caller-owned): mass_amu [n_atoms]; F_draft, F_target [K][3][n_atoms] fp64 (F~_j and F_j at q_half_j, eV/A).
 *           seed and n0 key the noise exactly as in the context path: step j (1..K) uses xi = Philox(seed; n0 + j, atom) and
 *           u_j = Philox(seed; n0 + j) (R5), n0 = committed step index of the window's start state.
 *   outputs (DEVICE, caller-owned): stats [4][K] = S1 | S2 | ell | ln u;  reject [K] (1 = step rejected);
 *           verdict [3] = {first_reject l (0: none), n_commit (l, or K), 1 if S1 or S2 of a committed step is not finite}.
 *           The override of step l (a5) is not part of this call.
 *   The arithmetic, reduction order and block decomposition are those of lsd_transport_accept, so with the same forces, seed
 *   and n0 the numbers agree with lsd_get_window_debug(S1 / S2 / ELL / LNU / REJECT).
 *
 * Asynchronous on `stream`; nothing is synchronised.  The FIRST call on each device also looks up the device address of the
 * array (once per device, with that device current): make that first call before you begin any stream capture.
 * All calls on a device share the array, and it keeps what the last call wrote.  Nothing in it needs to start at zero (each
 * call overwrites every slot it later reads), so calls that follow each other on one stream, or are otherwise ordered, are safe;
 * two calls that may run on the GPU at the same time (different streams, different host threads, no ordering) race on it and
 * give wrong sums.  Serialise them.
 * Errors: INVALID_ARG (sizes beyond the limits, non-positive T / friction / dt, null or non-device pointers), CUDA (launch or
 * address look-up failed).  The message is returned by lsd_noalloc_last_error() (per host thread). */
#define LSD_NOALLOC_MAX_K      64
#define LSD_NOALLOC_MAX_ATOMS  (1 << 28)
lsd_status lsd_transport_window_noalloc(int32_t n_atoms, int32_t K, uint64_t seed, uint64_t n0, double temperature_K,
                                        double friction_per_fs, double dt_fs, const double* mass_amu, const double* F_draft,
                                        const double* F_target, double* stats, int32_t* reject, int32_t* verdict, void* stream);
const char* lsd_noalloc_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* LSD_H */
