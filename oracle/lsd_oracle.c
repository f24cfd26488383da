/*
 * lsd_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, fp64 CPU implementation of the hot path of Langevin Speculative
 * Dynamics (arxiv/paper_2606_02455), written from PAPER.md step by step.  It
 * shares no code with the CUDA path (paper_2606_02455_b200/): no common header,
 * helper, table or constant generator.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference leg may load it.
 *
 * Citations are PAPER.md:<line> (section / equation) or SURVEY.md 8(c) readings
 * (R1..R16, M1..M9, O-1..O-4), which DESIGN.md restates.
 *
 * Parity pins (tests/test_oracle_*.py, all -m "not gpu"):
 *   orc_philox4x32_10   : cuRAND host generator CURAND_RNG_PSEUDO_PHILOX4_32_10 (library)
 *   orc_normals/uniform : sample moments, KS
 *   priors              : zero force at LJ minimum 2^(1/6) sigma, U=-eps; Morse r0; FD; sum F = 0
 *   neighbours          : exact lattice shell counts (sc: 26, fcc: 78), symmetry, cell list == brute force
 *   MLIP energy/forces  : central finite differences, invariances, perfect fcc => F = 0
 *   ABOBA               : harmonic-oscillator closed forms <q^2> = kT/k, <p^2>/m = kT/(1-dt^2 k/4m)
 *   transport           : 1-D mirror image (Fig. 2), Householder invariants, Monte-Carlo vs erf (Eq. 9)
 *   window              : draft==target => acceptance 1 and trajectory == plain ABOBA; K-invariance
 *   window with EC      : dF = 0 == plain window; constant force error => S2 == 0 after one commit; target <q^2>
 * Functions with no independent pin: none ("parity unpinned" would be stated here).
 *
 * Layout: positions/momenta/forces are [N][3] doubles (AoS) inside the oracle.
 * Units: Angstrom, fs, eV, K; masses passed in amu and converted with AMU (O-1).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define ORC_KB  8.617333262e-5   /* eV/K            (O-1) */
#define ORC_AMU 103.642696       /* eV fs^2/A^2/amu (O-1) */
#define ORC_PI  3.14159265358979323846

/* ------------------------------------------------------------------------------------------
 * Data passed in from Python (ctypes mirrors these structs field by field).
 * ---------------------------------------------------------------------------------------- */
typedef struct {
    int32_t width, n_blocks, n_rbf, n_species;   /* F, T, R, species count; width==0 -> no MLIP */
    double cutoff, alpha;
    const double *w;                              /* flat weights, layout of lsd_inputs.mlip_weight_offsets */
} orc_mlip;

typedef struct {
    int32_t n_species, use_bonded;
    const double *pair;    /* [ns][ns][8]: lj_eps, lj_sigma, lj_rc, morse_D, morse_a, morse_r0, morse_rc, tether_k */
    orc_mlip mlip;
} orc_potential;

typedef struct {
    int32_t n, periodic;
    double box[3];
    const int32_t *species;
    const double *mass_amu;
    int32_t n_bonds;  const int32_t *bonds;  const double *bond_k, *bond_r0;
    int32_t n_angles; const int32_t *angles; const double *angle_k, *angle_t0;
} orc_system;

typedef struct {
    double temperature_K, friction_per_fs, dt_fs;
    uint64_t seed;
} orc_params;

/* ------------------------------------------------------------------------------------------
 * R5: Philox4x32-10 counter-based generator (Salmon et al. 2011, public algorithm).
 * ---------------------------------------------------------------------------------------- */
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        uint64_t p0 = (uint64_t)0xD2511F53u * c0;
        uint64_t p1 = (uint64_t)0xCD9E8D57u * c2;
        uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
        uint32_t n1 = (uint32_t)p1;
        uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        uint32_t n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

static void philox_block(uint64_t seed, uint64_t step, uint32_t atom, uint32_t tag, uint32_t w[4])
{
    uint32_t ctr[4] = { (uint32_t)step, (uint32_t)(step >> 32), atom, tag };
    uint32_t key[2] = { (uint32_t)seed, (uint32_t)(seed >> 32) };
    orc_philox4x32_10(ctr, key, w);
}

/* R5: three standard normals per (step, atom): xi_x, xi_y = Box-Muller(w0, w1) (cos, sin),
 * xi_z = cos branch of Box-Muller(w2, w3); uniforms (w + 1/2) 2^-32 in (0,1). */
static void normals3(uint64_t seed, uint64_t step, uint32_t atom, uint32_t tag, double xi[3])
{
    uint32_t w[4];
    philox_block(seed, step, atom, tag, w);
    const double s = 1.0 / 4294967296.0;
    double u0 = ((double)w[0] + 0.5) * s, u1 = ((double)w[1] + 0.5) * s;
    double u2 = ((double)w[2] + 0.5) * s, u3 = ((double)w[3] + 0.5) * s;
    double r0 = sqrt(-2.0 * log(u0)), r1 = sqrt(-2.0 * log(u2));
    xi[0] = r0 * cos(2.0 * ORC_PI * u1);
    xi[1] = r0 * sin(2.0 * ORC_PI * u1);
    xi[2] = r1 * cos(2.0 * ORC_PI * u3);
}

/* xi[n][3] for simulation step index `step` (tag 0 = integrator noise, 2 = initial momenta). */
void orc_normals(uint64_t seed, uint64_t step, int32_t n, uint32_t tag, double *xi)
{
    for (int32_t i = 0; i < n; ++i) normals3(seed, step, (uint32_t)i, tag, xi + 3 * i);
}

/* R5: u_j for step index `step`: tag 1, atom index 0xFFFFFFFF, 53-bit uniform in (0,1). */
double orc_uniform(uint64_t seed, uint64_t step)
{
    uint32_t w[4];
    philox_block(seed, step, 0xFFFFFFFFu, 1u, w);
    return ((double)(w[0] >> 5) * 67108864.0 + (double)(w[1] >> 6) + 0.5) * (1.0 / 9007199254740992.0);
}

/* R12: Maxwell-Boltzmann momenta p_i = sqrt(m_i kT) xi, stream tag 2, step 0. */
void orc_initial_momenta(const orc_system *sys, const orc_params *par, double *p)
{
    for (int32_t i = 0; i < sys->n; ++i) {
        double xi[3];
        normals3(par->seed, 0, (uint32_t)i, 2u, xi);
        double s = sqrt(sys->mass_amu[i] * ORC_AMU * ORC_KB * par->temperature_K);
        for (int c = 0; c < 3; ++c) p[3 * i + c] = s * xi[c];
    }
}

/* ------------------------------------------------------------------------------------------
 * R10: displacement j - i with single minimum image (orthorhombic box), fp64, no fma.
 * T1: d = q_j - q_i;  s = -rint(d / L);  d = d + s L   (s is the integer image shift).
 * ---------------------------------------------------------------------------------------- */
static inline void min_image(const orc_system *sys, const double *qi, const double *qj, double d[3], int shift[3])
{
    for (int c = 0; c < 3; ++c) {
        double x = qj[c] - qi[c];
        int s = 0;
        if (sys->periodic) {
            double k = rint(x / sys->box[c]);
            s = -(int)k;
            x = x - k * sys->box[c];
        }
        d[c] = x; shift[c] = s;
    }
}

static inline double norm2(const double d[3]) { return (d[0] * d[0] + d[1] * d[1]) + d[2] * d[2]; }

/* ------------------------------------------------------------------------------------------
 * Neighbour lists (T1): directed edge set {(i, j, shift): r_ij < r_c, j != i}, per atom sorted by j.
 * Brute force O(N^2).  Output CSR: start[n+1], idx[cap], shifts[cap][3] (int8).  Returns the
 * number of edges (also when it exceeds cap; then nothing beyond cap is written).
 * ---------------------------------------------------------------------------------------- */
int64_t orc_neighbors_brute(const orc_system *sys, const double *q, double rc, int64_t cap,
                            int64_t *start, int32_t *idx, int8_t *shifts)
{
    int64_t e = 0;
    const double rc2 = rc * rc;
    for (int32_t i = 0; i < sys->n; ++i) {
        start[i] = e;
        for (int32_t j = 0; j < sys->n; ++j) {
            if (j == i) continue;
            double d[3]; int s[3];
            min_image(sys, q + 3 * i, q + 3 * j, d, s);
            if (norm2(d) < rc2) {
                if (e < cap) { idx[e] = j; shifts[3 * e] = (int8_t)s[0]; shifts[3 * e + 1] = (int8_t)s[1]; shifts[3 * e + 2] = (int8_t)s[2]; }
                ++e;
            }
        }
    }
    start[sys->n] = e;
    return e;
}

/* Cell-list version (same edge set; pinned against the brute force).  Cells of side >= rc;
 * a dimension with fewer than 3 cells (or a non-periodic system) is searched in full (R10). */
static int cmp_i32(const void *a, const void *b) { int32_t x = *(const int32_t *)a, y = *(const int32_t *)b; return (x > y) - (x < y); }

int64_t orc_neighbors_cell(const orc_system *sys, const double *q, double rc, int64_t cap,
                           int64_t *start, int32_t *idx, int8_t *shifts)
{
    int nc[3];
    if (!sys->periodic) return orc_neighbors_brute(sys, q, rc, cap, start, idx, shifts);
    for (int c = 0; c < 3; ++c) { nc[c] = (int)floor(sys->box[c] / rc); if (nc[c] < 3) nc[c] = 1; }
    int64_t ncell = (int64_t)nc[0] * nc[1] * nc[2];
    int32_t *head = (int32_t *)malloc(sizeof(int32_t) * (size_t)ncell);
    int32_t *next = (int32_t *)malloc(sizeof(int32_t) * (size_t)sys->n);
    int32_t *cellof = (int32_t *)malloc(sizeof(int32_t) * 3 * (size_t)sys->n);
    for (int64_t c = 0; c < ncell; ++c) head[c] = -1;
    for (int32_t i = sys->n - 1; i >= 0; --i) {
        int cc[3];
        for (int c = 0; c < 3; ++c) {
            double f = q[3 * i + c] / sys->box[c];
            f -= floor(f);
            cc[c] = (int)(f * nc[c]); if (cc[c] >= nc[c]) cc[c] = nc[c] - 1;
            cellof[3 * i + c] = cc[c];
        }
        int64_t id = ((int64_t)cc[0] * nc[1] + cc[1]) * nc[2] + cc[2];
        next[i] = head[id]; head[id] = i;
    }
    const double rc2 = rc * rc;
    int32_t *tmp = (int32_t *)malloc(sizeof(int32_t) * (size_t)sys->n);
    int64_t e = 0;
    for (int32_t i = 0; i < sys->n; ++i) {
        start[i] = e;
        int cnt = 0;
        int lo[3], hi[3];
        for (int c = 0; c < 3; ++c) { if (nc[c] == 1) { lo[c] = 0; hi[c] = 0; } else { lo[c] = -1; hi[c] = 1; } }
        for (int dx = lo[0]; dx <= hi[0]; ++dx) for (int dy = lo[1]; dy <= hi[1]; ++dy) for (int dz = lo[2]; dz <= hi[2]; ++dz) {
            int cx = (cellof[3 * i] + dx + nc[0]) % nc[0], cy = (cellof[3 * i + 1] + dy + nc[1]) % nc[1], cz = (cellof[3 * i + 2] + dz + nc[2]) % nc[2];
            for (int32_t j = head[((int64_t)cx * nc[1] + cy) * nc[2] + cz]; j >= 0; j = next[j]) {
                if (j == i) continue;
                double d[3]; int s[3];
                min_image(sys, q + 3 * i, q + 3 * j, d, s);
                if (norm2(d) < rc2) tmp[cnt++] = j;
            }
        }
        qsort(tmp, (size_t)cnt, sizeof(int32_t), cmp_i32);
        for (int k = 0; k < cnt; ++k) {
            if (e < cap) {
                double d[3]; int s[3];
                min_image(sys, q + 3 * i, q + 3 * tmp[k], d, s);
                idx[e] = tmp[k]; shifts[3 * e] = (int8_t)s[0]; shifts[3 * e + 1] = (int8_t)s[1]; shifts[3 * e + 2] = (int8_t)s[2];
            }
            ++e;
        }
    }
    start[sys->n] = e;
    free(head); free(next); free(cellof); free(tmp);
    return e;
}

/* internal CSR holder */
typedef struct { int64_t *start; int32_t *idx; int8_t *shifts; } nbr_list;

static void nbr_build(const orc_system *sys, const double *q, double rc, nbr_list *nl)
{
    nl->start = (int64_t *)malloc(sizeof(int64_t) * ((size_t)sys->n + 1));
    int64_t cap = (int64_t)sys->n * 64 + 1024;
    for (;;) {
        nl->idx = (int32_t *)malloc(sizeof(int32_t) * (size_t)cap);
        nl->shifts = (int8_t *)malloc(3 * (size_t)cap);
        int64_t e = orc_neighbors_cell(sys, q, rc, cap, nl->start, nl->idx, nl->shifts);
        if (e <= cap) break;
        free(nl->idx); free(nl->shifts); cap = e;
    }
}
static void nbr_free(nbr_list *nl) { free(nl->start); free(nl->idx); free(nl->shifts); }

static inline void edge_vec(const orc_system *sys, const double *q, int32_t i, int32_t j, const int8_t *s, double d[3])
{
    for (int c = 0; c < 3; ++c) d[c] = (q[3 * j + c] - q[3 * i + c]) + (double)s[c] * sys->box[c];
}

/* ------------------------------------------------------------------------------------------
 * O-4 priors.  Pair terms: U_LJ = 4 eps [(s/r)^12 - (s/r)^6] - U_LJ(rc);
 * U_Morse = D[(1 - e^{-a(r-r0)})^2 - 1] - U_Morse(rc).  Energy counted 1/2 per directed edge.
 * F_i = -dU/dq_i = +U'(r) rhat_ij with rhat_ij = (q_j - q_i + shift)/r.
 * ---------------------------------------------------------------------------------------- */
static double lj_u(double eps, double sig, double r)  { double s6 = pow(sig / r, 6.0); return 4.0 * eps * (s6 * s6 - s6); }
static double lj_du(double eps, double sig, double r) { double s6 = pow(sig / r, 6.0); return -24.0 * eps / r * (2.0 * s6 * s6 - s6); }
static double morse_u(double D, double a, double r0, double r)  { double x = exp(-a * (r - r0)); return D * ((1.0 - x) * (1.0 - x) - 1.0); }
static double morse_du(double D, double a, double r0, double r) { double x = exp(-a * (r - r0)); return 2.0 * D * a * x * (1.0 - x); }

static double pair_forces(const orc_system *sys, const orc_potential *pot, const double *q, double *F)
{
    double rcmax = 0.0;
    const int ns = pot->n_species;
    for (int a = 0; a < ns * ns; ++a) {
        if (pot->pair[8 * a + 0] != 0.0 && pot->pair[8 * a + 2] > rcmax) rcmax = pot->pair[8 * a + 2];
        if (pot->pair[8 * a + 3] != 0.0 && pot->pair[8 * a + 6] > rcmax) rcmax = pot->pair[8 * a + 6];
    }
    if (rcmax == 0.0) return 0.0;
    nbr_list nl; nbr_build(sys, q, rcmax, &nl);
    double E = 0.0;
    for (int32_t i = 0; i < sys->n; ++i) {
        for (int64_t e = nl.start[i]; e < nl.start[i + 1]; ++e) {
            int32_t j = nl.idx[e];
            const double *pp = pot->pair + 8 * (sys->species[i] * ns + sys->species[j]);
            double d[3]; edge_vec(sys, q, i, j, nl.shifts + 3 * e, d);
            double r = sqrt(norm2(d)), u = 0.0, du = 0.0;
            if (pp[0] != 0.0 && r < pp[2]) { u += lj_u(pp[0], pp[1], r) - lj_u(pp[0], pp[1], pp[2]); du += lj_du(pp[0], pp[1], r); }
            if (pp[3] != 0.0 && r < pp[6]) { u += morse_u(pp[3], pp[4], pp[5], r) - morse_u(pp[3], pp[4], pp[5], pp[6]); du += morse_du(pp[3], pp[4], pp[5], r); }
            E += 0.5 * u;
            for (int c = 0; c < 3; ++c) F[3 * i + c] += du * d[c] / r;
        }
    }
    nbr_free(&nl);
    return E;
}

/* Harmonic well at the coordinate origin, U = k_s/2 |q_i|^2 with k_s = pair[s][s][7] (vacuum only):
 * 3N independent 1-D harmonic oscillators -- the system whose ABOBA statistics have closed forms. */
static double tether_forces(const orc_system *sys, const orc_potential *pot, const double *q, double *F)
{
    double E = 0.0;
    const int ns = pot->n_species;
    for (int32_t i = 0; i < sys->n; ++i) {
        double k = pot->pair[8 * (sys->species[i] * ns + sys->species[i]) + 7];
        if (k == 0.0) continue;
        for (int c = 0; c < 3; ++c) { E += 0.5 * k * q[3 * i + c] * q[3 * i + c]; F[3 * i + c] -= k * q[3 * i + c]; }
    }
    return E;
}

/* bonds U = k/2 (r - r0)^2; angles U = k/2 (theta - theta0)^2, theta at the apex (middle index). */
static double bonded_forces(const orc_system *sys, const double *q, double *F)
{
    double E = 0.0;
    for (int32_t b = 0; b < sys->n_bonds; ++b) {
        int32_t i = sys->bonds[2 * b], j = sys->bonds[2 * b + 1];
        double d[3]; int s[3];
        min_image(sys, q + 3 * i, q + 3 * j, d, s);
        double r = sqrt(norm2(d)), dr = r - sys->bond_r0[b];
        E += 0.5 * sys->bond_k[b] * dr * dr;
        for (int c = 0; c < 3; ++c) { double f = sys->bond_k[b] * dr * d[c] / r; F[3 * i + c] += f; F[3 * j + c] -= f; }
    }
    for (int32_t a = 0; a < sys->n_angles; ++a) {
        int32_t ia = sys->angles[3 * a], ib = sys->angles[3 * a + 1], ic = sys->angles[3 * a + 2];
        double u[3], v[3]; int s[3];
        min_image(sys, q + 3 * ib, q + 3 * ia, u, s);
        min_image(sys, q + 3 * ib, q + 3 * ic, v, s);
        double nu = sqrt(norm2(u)), nv = sqrt(norm2(v));
        double ct = (u[0] * v[0] + u[1] * v[1] + u[2] * v[2]) / (nu * nv);
        if (ct > 1.0) ct = 1.0; if (ct < -1.0) ct = -1.0;
        double th = acos(ct), st = fmax(sqrt(1.0 - ct * ct), 1e-12), dth = th - sys->angle_t0[a];   /* collinear arms: bounded, not 0/0 (R19) */
        E += 0.5 * sys->angle_k[a] * dth * dth;
        double dU = sys->angle_k[a] * dth;                         /* dU/dtheta */
        for (int c = 0; c < 3; ++c) {
            double uh = u[c] / nu, vh = v[c] / nv;
            double dth_da = -(vh - ct * uh) / (nu * st);           /* dtheta/dq_a */
            double dth_dc = -(uh - ct * vh) / (nv * st);           /* dtheta/dq_c */
            F[3 * ia + c] -= dU * dth_da;
            F[3 * ic + c] -= dU * dth_dc;
            F[3 * ib + c] += dU * (dth_da + dth_dc);
        }
    }
    return E;
}

/* ------------------------------------------------------------------------------------------
 * M1-M9: SchNet-style MLIP energy and hand-derived forces.
 * ---------------------------------------------------------------------------------------- */
static inline double ssp(double x)      { return fmax(x, 0.0) + log1p(exp(-fabs(x))) - 0.6931471805599453094; } /* M3 */
static inline double logistic(double x) { return x >= 0.0 ? 1.0 / (1.0 + exp(-x)) : exp(x) / (1.0 + exp(x)); }

typedef struct { int F, T, R, ns; double rc, alpha; const double *emb, *blk, *Wr1, *wr2; int per_block; } mlip_view;

static mlip_view mlip_open(const orc_mlip *m)
{
    mlip_view v; v.F = m->width; v.T = m->n_blocks; v.R = m->n_rbf; v.ns = m->n_species; v.rc = m->cutoff; v.alpha = m->alpha;
    v.emb = m->w; v.blk = m->w + (size_t)v.ns * v.F; v.per_block = 4 * v.F * v.F + v.F * v.R;
    v.Wr1 = v.blk + (size_t)v.T * v.per_block; v.wr2 = v.Wr1 + (size_t)(v.F / 2) * v.F;
    return v;
}
#define W_IN(v, t)  ((v).blk + (size_t)(t) * (v).per_block)
#define W_F1(v, t)  (W_IN(v, t) + (v).F * (v).F)
#define W_F2(v, t)  (W_F1(v, t) + (v).F * (v).R)
#define W_O1(v, t)  (W_F2(v, t) + (v).F * (v).F)
#define W_O2(v, t)  (W_O1(v, t) + (v).F * (v).F)

/* out[rows] = W[rows][cols] in[cols] */
static void matvec(const double *W, int rows, int cols, const double *in, double *out)
{ for (int r = 0; r < rows; ++r) { double s = 0.0; for (int c = 0; c < cols; ++c) s += W[(size_t)r * cols + c] * in[c]; out[r] = s; } }
/* out[cols] = W^T in[rows] */
static void matvec_t(const double *W, int rows, int cols, const double *in, double *out)
{ for (int c = 0; c < cols; ++c) out[c] = 0.0; for (int r = 0; r < rows; ++r) for (int c = 0; c < cols; ++c) out[c] += W[(size_t)r * cols + c] * in[r]; }

/* M1, M2, M5: filter value w(r) = (W_f2 ssp(W_f1 g(r))) f_c(r) and, if dw != NULL, its r-derivative
 * dw/dr = (W_f2 (logistic(W_f1 g) . (W_f1 g'))) f_c + (W_f2 a) f_c'   (M9 filter tangent). */
static void filter_eval(const mlip_view *v, int t, double r, double *w, double *dw, double *scratch)
{
    const int F = v->F, R = v->R;
    double *g = scratch, *gp = g + R, *pre = gp + R, *prep = pre + F, *a = prep + F, *ap = a + F, *lin = ap + F, *linp = lin + F;
    const double delta = v->rc / (R - 1);
    for (int k = 0; k < R; ++k) {
        double x = r - k * delta;
        g[k] = exp(-x * x / (2.0 * delta * delta));                       /* M1 */
        gp[k] = -g[k] * x / (delta * delta);
    }
    double fc = 0.0, fcp = 0.0;
    if (r < v->rc) { fc = 0.5 * (cos(ORC_PI * r / v->rc) + 1.0); fcp = -0.5 * ORC_PI / v->rc * sin(ORC_PI * r / v->rc); }  /* M2 */
    matvec(W_F1(*v, t), F, R, g, pre);
    for (int f = 0; f < F; ++f) a[f] = ssp(pre[f]);
    matvec(W_F2(*v, t), F, F, a, lin);
    for (int f = 0; f < F; ++f) w[f] = lin[f] * fc;
    if (dw) {
        matvec(W_F1(*v, t), F, R, gp, prep);
        for (int f = 0; f < F; ++f) ap[f] = logistic(pre[f]) * prep[f];
        matvec(W_F2(*v, t), F, F, ap, linp);
        for (int f = 0; f < F; ++f) dw[f] = linp[f] * fc + lin[f] * fcp;
    }
}

/* E_NN and (if F != NULL) F += -dE_NN/dq.  Gather form of M9: every loop over atoms writes
 * only that atom's rows, so `omp parallel for` does not change any summation order.
 *   ybar_a = sum_{j in N(a)} mbar_j . w_aj                       (w_ja = w_aj)
 *   F_a   += sum_{j in N(a)} [ sum_f (mbar_a y_j + mbar_j y_a)_f w'_aj,f ] rhat_aj
 * (the bracket is g_{a<-j} + g_{j<-a} of M9; rhat_aj = (q_j - q_a + shift)/r). */
static double mlip_energy_forces(const orc_system *sys, const orc_mlip *m, const double *q, double *Fout)
{
    mlip_view v = mlip_open(m);
    const int F = v.F, T = v.T, n = sys->n, H = F / 2;
    nbr_list nl; nbr_build(sys, q, v.rc, &nl);
    size_t NF = (size_t)n * F;
    double *x = (double *)malloc(sizeof(double) * NF);
    double *y = (double *)malloc(sizeof(double) * NF * T);     /* y^t = W_in x^{t-1}      (kept, M9) */
    double *h = (double *)malloc(sizeof(double) * NF * T);     /* h^t = W_o1 m^t          (kept, M9) */
    double *mm = (double *)malloc(sizeof(double) * NF);
    for (int i = 0; i < n; ++i) memcpy(x + (size_t)i * F, v.emb + (size_t)sys->species[i] * F, sizeof(double) * F);   /* M4 */
    for (int t = 0; t < T; ++t) {                                                                                     /* M5 */
        double *yt = y + NF * t, *ht = h + NF * t;
        #pragma omp parallel for schedule(static)
        for (int i = 0; i < n; ++i) matvec(W_IN(v, t), F, F, x + (size_t)i * F, yt + (size_t)i * F);
        #pragma omp parallel for schedule(dynamic, 8)
        for (int i = 0; i < n; ++i) {
            double *w = (double *)malloc(sizeof(double) * (F + 2 * v.R + 6 * F));
            double *mi = mm + (size_t)i * F;
            for (int f = 0; f < F; ++f) mi[f] = 0.0;
            for (int64_t e = nl.start[i]; e < nl.start[i + 1]; ++e) {
                int32_t j = nl.idx[e];
                double d[3]; edge_vec(sys, q, i, j, nl.shifts + 3 * e, d);
                filter_eval(&v, t, sqrt(norm2(d)), w, NULL, w + F);
                for (int f = 0; f < F; ++f) mi[f] += yt[(size_t)j * F + f] * w[f];
            }
            free(w);
        }
        #pragma omp parallel for schedule(static)
        for (int i = 0; i < n; ++i) {
            double a[512], vv[512];
            matvec(W_O1(v, t), F, F, mm + (size_t)i * F, ht + (size_t)i * F);
            for (int f = 0; f < F; ++f) a[f] = ssp(ht[(size_t)i * F + f]);
            matvec(W_O2(v, t), F, F, a, vv);
            for (int f = 0; f < F; ++f) x[(size_t)i * F + f] += vv[f];
        }
    }
    double E = 0.0;                                                                                                   /* M6 */
    double *xbar = (double *)malloc(sizeof(double) * NF);
    for (int i = 0; i < n; ++i) {
        double z[256], s[256];
        matvec(v.Wr1, H, F, x + (size_t)i * F, z);
        double ei = 0.0;
        for (int k = 0; k < H; ++k) { ei += v.wr2[k] * ssp(z[k]); s[k] = logistic(z[k]) * v.wr2[k]; }
        E += ei;
        matvec_t(v.Wr1, H, F, s, xbar + (size_t)i * F);
        for (int f = 0; f < F; ++f) xbar[(size_t)i * F + f] *= v.alpha;
    }
    E *= v.alpha;
    if (Fout) {                                                                                                       /* M9 */
        double *mbar = (double *)malloc(sizeof(double) * NF);
        double *ybar = (double *)malloc(sizeof(double) * NF);
        for (int t = T - 1; t >= 0; --t) {
            const double *yt = y + NF * t, *ht = h + NF * t;
            #pragma omp parallel for schedule(static)
            for (int i = 0; i < n; ++i) {
                double tmp[512], hb[512];
                matvec_t(W_O2(v, t), F, F, xbar + (size_t)i * F, tmp);
                for (int f = 0; f < F; ++f) hb[f] = logistic(ht[(size_t)i * F + f]) * tmp[f];
                matvec_t(W_O1(v, t), F, F, hb, mbar + (size_t)i * F);
            }
            #pragma omp parallel for schedule(dynamic, 8)
            for (int a = 0; a < n; ++a) {
                double *w = (double *)malloc(sizeof(double) * (2 * F + 2 * v.R + 6 * F));
                double *dw = w + F;
                double *yb = ybar + (size_t)a * F;
                for (int f = 0; f < F; ++f) yb[f] = 0.0;
                for (int64_t e = nl.start[a]; e < nl.start[a + 1]; ++e) {
                    int32_t j = nl.idx[e];
                    double d[3]; edge_vec(sys, q, a, j, nl.shifts + 3 * e, d);
                    double r = sqrt(norm2(d));
                    filter_eval(&v, t, r, w, dw, dw + F);
                    double gsym = 0.0;
                    for (int f = 0; f < F; ++f) {
                        gsym += (mbar[(size_t)a * F + f] * yt[(size_t)j * F + f] + mbar[(size_t)j * F + f] * yt[(size_t)a * F + f]) * dw[f];
                        yb[f] += mbar[(size_t)j * F + f] * w[f];
                    }
                    for (int c = 0; c < 3; ++c) Fout[3 * a + c] += gsym * d[c] / r;
                }
                free(w);
            }
            if (t > 0) {
                #pragma omp parallel for schedule(static)
                for (int i = 0; i < n; ++i) {
                    double tmp[512];
                    matvec_t(W_IN(v, t), F, F, ybar + (size_t)i * F, tmp);
                    for (int f = 0; f < F; ++f) xbar[(size_t)i * F + f] += tmp[f];
                }
            }
        }
        free(mbar); free(ybar);
    }
    free(x); free(y); free(h); free(mm); free(xbar); nbr_free(&nl);
    return E;
}

/* Total potential energy; F (may be NULL) receives forces F = -dE/dq, [n][3]. */
double orc_energy_forces(const orc_system *sys, const orc_potential *pot, const double *q, double *F)
{
    double E = 0.0;
    double *scratch = F;
    if (!F) scratch = (double *)malloc(sizeof(double) * 3 * (size_t)sys->n);
    for (int i = 0; i < 3 * sys->n; ++i) scratch[i] = 0.0;
    E += pair_forces(sys, pot, q, scratch);
    E += tether_forces(sys, pot, q, scratch);
    if (pot->use_bonded) E += bonded_forces(sys, q, scratch);
    if (pot->mlip.width > 0) E += mlip_energy_forces(sys, &pot->mlip, q, F ? scratch : NULL);
    if (!F) free(scratch);
    return E;
}

/* MLIP-only energy / forces (for pins that isolate the network). */
double orc_mlip_energy_forces(const orc_system *sys, const orc_mlip *m, const double *q, double *F)
{
    if (F) for (int i = 0; i < 3 * sys->n; ++i) F[i] = 0.0;
    return mlip_energy_forces(sys, m, q, F);
}

/* ------------------------------------------------------------------------------------------
 * O-2: one ABOBA step (PAPER.md:60-66 Eq. 2; :584-593 DRAFT_STEP) with forces `pot`.
 * c1 = e^{-gamma dt}; b = (1 + c1) dt / 2; sigma_i = sqrt(m_i kT (1 - c1^2)) (Eq. 7, :105).
 * Outputs: q_half (after the first A), Fh = F(q_half), xi (the draw), q, p updated in place.
 * ---------------------------------------------------------------------------------------- */
typedef struct { double c1, b, hdt; } aboba_consts;
static aboba_consts aboba_k(const orc_params *par)
{ aboba_consts k; k.c1 = exp(-par->friction_per_fs * par->dt_fs); k.b = (1.0 + k.c1) * par->dt_fs / 2.0; k.hdt = par->dt_fs / 2.0; return k; }
static inline double sigma_i(const orc_system *sys, const orc_params *par, double c1, int i)
{ return sqrt(sys->mass_amu[i] * ORC_AMU * ORC_KB * par->temperature_K * (1.0 - c1 * c1)); }

void orc_aboba_step(const orc_system *sys, const orc_params *par, const orc_potential *pot, uint64_t step,
                    double *q, double *p, double *q_half, double *Fh, double *xi)
{
    aboba_consts k = aboba_k(par);
    const int n = sys->n;
    for (int i = 0; i < n; ++i) for (int c = 0; c < 3; ++c)
        q_half[3 * i + c] = q[3 * i + c] + k.hdt * p[3 * i + c] / (sys->mass_amu[i] * ORC_AMU);       /* A(1/2) */
    orc_energy_forces(sys, pot, q_half, Fh);
    orc_normals(par->seed, step, n, 0u, xi);
    for (int i = 0; i < n; ++i) {
        double sg = sigma_i(sys, par, k.c1, i);
        for (int c = 0; c < 3; ++c) {
            p[3 * i + c] = k.c1 * p[3 * i + c] + k.b * Fh[3 * i + c] + sg * xi[3 * i + c];              /* B O B = Eq. 7 */
            q[3 * i + c] = q_half[3 * i + c] + k.hdt * p[3 * i + c] / (sys->mass_amu[i] * ORC_AMU);    /* A(1/2) */
        }
    }
}

/* ------------------------------------------------------------------------------------------
 * O-3 second half: transport map of ONE step (Eq. 8; R6, R7, R8, R13).
 * d = (b / sigma) (Ft - F)  (= delta);  S1 = xi . d;  S2 = d . d;  ell = -S1 - S2/2;
 * accept iff S2 == 0 or ln u <= min(0, ell).  On reject (returns 1) p_out, q_out receive
 * pstar = c1 p_prev + b F + sigma (xi - 2 (S1/S2) d),  qstar = q_half + (dt/2) pstar / m  (map g, :602).
 * ---------------------------------------------------------------------------------------- */
int32_t orc_transport_step(const orc_system *sys, const orc_params *par, const double *Ft, const double *F,
                           const double *xi, double u, const double *p_prev, const double *q_half,
                           double *S1, double *S2, double *ell, double *q_out, double *p_out)
{
    aboba_consts k = aboba_k(par);
    const int n = sys->n;
    double s1 = 0.0, s2 = 0.0;
    for (int i = 0; i < n; ++i) {
        double sg = sigma_i(sys, par, k.c1, i);
        for (int c = 0; c < 3; ++c) {
            double d = k.b / sg * (Ft[3 * i + c] - F[3 * i + c]);
            s1 += xi[3 * i + c] * d; s2 += d * d;
        }
    }
    *S1 = s1; *S2 = s2; *ell = -s1 - 0.5 * s2;
    if (s2 == 0.0) return 0;                                    /* R8 */
    if (log(u) <= fmin(0.0, *ell)) return 0;                    /* R7 */
    if (q_out && p_out) {
        for (int i = 0; i < n; ++i) {
            double sg = sigma_i(sys, par, k.c1, i);
            for (int c = 0; c < 3; ++c) {
                double d = k.b / sg * (Ft[3 * i + c] - F[3 * i + c]);
                double ps = k.c1 * p_prev[3 * i + c] + k.b * F[3 * i + c] + sg * (xi[3 * i + c] - 2.0 * (s1 / s2) * d);
                p_out[3 * i + c] = ps;
                q_out[3 * i + c] = q_half[3 * i + c] + k.hdt * ps / (sys->mass_amu[i] * ORC_AMU);
            }
        }
    }
    return 1;
}

/* Force slack (App. H): F_(eps) = F + clip(-eps_F; F~ - F; eps_F), component by component: the target force is
 * pushed towards the draft force inside an L-infinity ball of radius eps_F.  The verification then runs orc_transport_step with
 * F_(eps) in the place of F (breaks exactness, :781; eps_F = 0 leaves F unchanged).  Ft: the force the draft was drawn around
 * (F~, or F~ + dF with error correction).  Not on the hot path by default (optional). */
void orc_force_slack(int32_t n, const double *Ft, const double *F, double eps_F, double *F_out)
{
    for (int i = 0; i < 3 * n; ++i) {
        double x = Ft[i] - F[i];
        if (x > eps_F) x = eps_F;
        if (x < -eps_F) x = -eps_F;
        F_out[i] = F[i] + x;
    }
}

/* ------------------------------------------------------------------------------------------
 * O-3: one synchronous window (Alg. 1, L = K; R2, R3, R4).
 * In : base state (q, p) at committed step index n0.
 * Out: q, p <- new base; traj_q/traj_p [K][n][3] receive the committed states (first n_commit rows);
 *      per-step debug rows (all K steps): q_half, Ft, Ftgt, S1, S2, ell, lnu, reject flags.
 * Returns n_commit; *first_reject = 0 (none) or l in 1..K.
 * ---------------------------------------------------------------------------------------- */
int32_t orc_lsd_window(const orc_system *sys, const orc_params *par, const orc_potential *draft, const orc_potential *target,
                       uint64_t n0, int32_t K, double *q, double *p, int32_t *first_reject,
                       double *traj_q, double *traj_p,
                       double *dbg_qhalf, double *dbg_Ft, double *dbg_F, double *dbg_S1, double *dbg_S2,
                       double *dbg_ell, double *dbg_lnu, int32_t *dbg_reject)
{
    const size_t n3 = 3 * (size_t)sys->n;
    double *yq = (double *)malloc(sizeof(double) * n3 * (K + 1)), *yp = (double *)malloc(sizeof(double) * n3 * (K + 1));
    double *qh = (double *)malloc(sizeof(double) * n3 * K), *Ft = (double *)malloc(sizeof(double) * n3 * K);
    double *xi = (double *)malloc(sizeof(double) * n3 * K), *Fg = (double *)malloc(sizeof(double) * n3);
    double *xq = (double *)malloc(sizeof(double) * n3), *xp = (double *)malloc(sizeof(double) * n3);
    memcpy(yq, q, sizeof(double) * n3); memcpy(yp, p, sizeof(double) * n3);
    for (int j = 1; j <= K; ++j) {                                      /* serial draft rollout */
        memcpy(yq + n3 * j, yq + n3 * (j - 1), sizeof(double) * n3);
        memcpy(yp + n3 * j, yp + n3 * (j - 1), sizeof(double) * n3);
        orc_aboba_step(sys, par, draft, n0 + j, yq + n3 * j, yp + n3 * j, qh + n3 * (j - 1), Ft + n3 * (j - 1), xi + n3 * (j - 1));
    }
    int32_t l = 0;
    for (int j = 1; j <= K; ++j) {                                      /* "in parallel for": order irrelevant */
        double S1, S2, ell, u = orc_uniform(par->seed, n0 + j);
        orc_energy_forces(sys, target, qh + n3 * (j - 1), Fg);          /* :598-599 same q_half */
        int32_t rej = orc_transport_step(sys, par, Ft + n3 * (j - 1), Fg, xi + n3 * (j - 1), u, yp + n3 * (j - 1), qh + n3 * (j - 1),
                                         &S1, &S2, &ell, (l == 0) ? xq : NULL, (l == 0) ? xp : NULL);
        if (dbg_qhalf) memcpy(dbg_qhalf + n3 * (j - 1), qh + n3 * (j - 1), sizeof(double) * n3);
        if (dbg_Ft) memcpy(dbg_Ft + n3 * (j - 1), Ft + n3 * (j - 1), sizeof(double) * n3);
        if (dbg_F) memcpy(dbg_F + n3 * (j - 1), Fg, sizeof(double) * n3);
        if (dbg_S1) dbg_S1[j - 1] = S1; if (dbg_S2) dbg_S2[j - 1] = S2; if (dbg_ell) dbg_ell[j - 1] = ell;
        if (dbg_lnu) dbg_lnu[j - 1] = log(u); if (dbg_reject) dbg_reject[j - 1] = rej;
        if (rej && l == 0) l = j;                                       /* l = min{j : x_j != y_j}, :424 */
        if (l != 0 && !dbg_reject && !dbg_F) break;                     /* later results are discarded anyway (:78) */
    }
    int32_t n_commit = l ? l : K;                                        /* R3: no bonus step; R4: x_l counts */
    for (int j = 1; j <= n_commit; ++j) {
        const double *sq = (l && j == l) ? xq : yq + n3 * j, *sp = (l && j == l) ? xp : yp + n3 * j;
        if (traj_q) memcpy(traj_q + n3 * (j - 1), sq, sizeof(double) * n3);
        if (traj_p) memcpy(traj_p + n3 * (j - 1), sp, sizeof(double) * n3);
        if (j == n_commit) { memcpy(q, sq, sizeof(double) * n3); memcpy(p, sp, sizeof(double) * n3); }
    }
    *first_reject = l;
    free(yq); free(yp); free(qh); free(Ft); free(xi); free(Fg); free(xq); free(xp);
    return n_commit;
}

/* Run LSD until n_steps are committed (the last window is shortened so that exactly n_steps are kept).
 * traj_q/traj_p (may be NULL): [n_steps][n][3].  stats[0] = windows, [1] = rejections,
 * [2] = sum over evaluated first-reject-or-earlier steps of erf(sqrt(S2)/sqrt 8) (Eq. 9), [3] = steps so examined. */
int64_t orc_run_lsd(const orc_system *sys, const orc_params *par, const orc_potential *draft, const orc_potential *target,
                    int64_t n_steps, int32_t K, double *q, double *p, double *traj_q, double *traj_p, double *stats)
{
    const size_t n3 = 3 * (size_t)sys->n;
    int64_t n = 0, windows = 0, rejections = 0; double beta_sum = 0.0; int64_t examined = 0;
    double *tq = (double *)malloc(sizeof(double) * n3 * K), *tp = (double *)malloc(sizeof(double) * n3 * K);
    double *S2 = (double *)malloc(sizeof(double) * K); int32_t *rej = (int32_t *)malloc(sizeof(int32_t) * K);
    while (n < n_steps) {
        int32_t k = K; if (n + k > n_steps) k = (int32_t)(n_steps - n);
        int32_t l;
        int32_t nc = orc_lsd_window(sys, par, draft, target, (uint64_t)n, k, q, p, &l, tq, tp, NULL, NULL, NULL, NULL, S2, NULL, NULL, NULL);
        for (int j = 0; j < nc; ++j) { beta_sum += erf(sqrt(S2[j]) / sqrt(8.0)); ++examined; }
        if (l) ++rejections;
        if (traj_q) memcpy(traj_q + n3 * n, tq, sizeof(double) * n3 * nc);
        if (traj_p) memcpy(traj_p + n3 * n, tp, sizeof(double) * n3 * nc);
        n += nc; ++windows;
    }
    if (stats) { stats[0] = (double)windows; stats[1] = (double)rejections; stats[2] = beta_sum; stats[3] = (double)examined; }
    free(tq); free(tp); free(S2); free(rej);
    return n;
}

/* Plain target Langevin (no speculation): n_steps of ABOBA with `pot` under the same noise keying. */
void orc_run_aboba(const orc_system *sys, const orc_params *par, const orc_potential *pot, int64_t n_steps,
                   double *q, double *p, double *traj_q, double *traj_p)
{
    const size_t n3 = 3 * (size_t)sys->n;
    double *qh = (double *)malloc(sizeof(double) * n3), *Fh = (double *)malloc(sizeof(double) * n3), *xi = (double *)malloc(sizeof(double) * n3);
    for (int64_t s = 1; s <= n_steps; ++s) {
        orc_aboba_step(sys, par, pot, (uint64_t)s, q, p, qh, Fh, xi);
        if (traj_q) memcpy(traj_q + n3 * (s - 1), q, sizeof(double) * n3);
        if (traj_p) memcpy(traj_p + n3 * (s - 1), p, sizeof(double) * n3);
    }
    free(qh); free(Fh); free(xi);
}

/* Eq. 9: rejection probability of one step, beta = erf(||delta|| / sqrt 8). */
double orc_rejection_probability(double delta_norm) { return erf(delta_norm / sqrt(8.0)); }

/* ------------------------------------------------------------------------------------------
 * O-5: speculative error correction, EC ("Speculative error
 * correction"; App. E :626-630; Alg. 3 :663-717), written for the synchronous window of O-3.
 *   DRAFT_STEP(y, dF) (:675-684): F~ = DraftModel(q_half) is the BARE output and is what is stored;
 *       <p~> = [Eq. 7](F~ + dF), i.e. p' = c1 p + b (F~ + dF) + sigma xi.
 *   VERIFY_STEP (:686-700): <p~> = [Eq. 7](F~ + dF), <p> = [Eq. 7](F), so
 *       d = (b / sigma)((F~ + dF) - F);  dF' = F - F~ uses the EC-UNCORRECTED draft forces (:628, :694)
 *       "which avoids self-feedback instability".
 *   PROCESS_NEW_RETURNS (:710-713): the cache becomes the dF' "stored in this step" when the step
 *       is added to the verified queue V, i.e. committed.
 * [reading R17] In the window form every draft step of a window is proposed before any of its target
 * results exists, so the whole window uses the cache as it stands when the window is drafted (the
 * dF' of the last step committed by the previous window); after the window the cache is the dF' of
 * its LAST committed step c = l (the overridden step counts, R4) or K.
 * dF: in = cache used by this window, out = cache after it.  dbg_Ft receives the bare F~.
 * Pins (tests/test_oracle_ec.py): dF = 0 <=> orc_lsd_window bit for bit; draft = target + constant
 * force => after the first committed step every step has S2 == 0 and is accepted (closed form);
 * harmonic oscillator with a wrong draft keeps the target's <q^2> = kT/k (Thm. 3.1 holds for any
 * draft law, :630); rejection count vs sum of erf(sqrt(S2)/sqrt 8) (Eq. 9).
 * ---------------------------------------------------------------------------------------- */
int32_t orc_lsd_window_ec(const orc_system *sys, const orc_params *par, const orc_potential *draft, const orc_potential *target,
                          uint64_t n0, int32_t K, double *q, double *p, double *dF, int32_t *first_reject,
                          double *traj_q, double *traj_p,
                          double *dbg_qhalf, double *dbg_Ft, double *dbg_F, double *dbg_S1, double *dbg_S2,
                          double *dbg_ell, double *dbg_lnu, int32_t *dbg_reject)
{
    const size_t n3 = 3 * (size_t)sys->n;
    const int n = sys->n;
    aboba_consts k = aboba_k(par);
    double *yq = (double *)malloc(sizeof(double) * n3 * (K + 1)), *yp = (double *)malloc(sizeof(double) * n3 * (K + 1));
    double *qh = (double *)malloc(sizeof(double) * n3 * K), *Ft = (double *)malloc(sizeof(double) * n3 * K);
    double *xi = (double *)malloc(sizeof(double) * n3 * K), *Fg = (double *)malloc(sizeof(double) * n3);
    double *xq = (double *)malloc(sizeof(double) * n3), *xp = (double *)malloc(sizeof(double) * n3);
    double *Fe = (double *)malloc(sizeof(double) * n3), *Fc = (double *)malloc(sizeof(double) * n3);
    memcpy(yq, q, sizeof(double) * n3); memcpy(yp, p, sizeof(double) * n3);
    for (int j = 1; j <= K; ++j) {                                      /* DRAFT_STEP(y, dF), serial */
        const double *q0 = yq + n3 * (j - 1), *p0 = yp + n3 * (j - 1);
        double *q1 = yq + n3 * j, *p1 = yp + n3 * j, *qhj = qh + n3 * (j - 1), *Fb = Ft + n3 * (j - 1), *xj = xi + n3 * (j - 1);
        for (int i = 0; i < n; ++i) for (int c = 0; c < 3; ++c)
            qhj[3 * i + c] = q0[3 * i + c] + k.hdt * p0[3 * i + c] / (sys->mass_amu[i] * ORC_AMU);
        orc_energy_forces(sys, draft, qhj, Fb);                         /* bare F~ */
        orc_normals(par->seed, n0 + j, n, 0u, xj);
        for (int i = 0; i < n; ++i) {
            double sg = sigma_i(sys, par, k.c1, i);
            for (int c = 0; c < 3; ++c) {
                p1[3 * i + c] = k.c1 * p0[3 * i + c] + k.b * (Fb[3 * i + c] + dF[3 * i + c]) + sg * xj[3 * i + c];
                q1[3 * i + c] = qhj[3 * i + c] + k.hdt * p1[3 * i + c] / (sys->mass_amu[i] * ORC_AMU);
            }
        }
    }
    int32_t l = 0;
    for (int j = 1; j <= K; ++j) {                                      /* VERIFY_STEP for every j */
        double S1, S2, ell, u = orc_uniform(par->seed, n0 + j);
        orc_energy_forces(sys, target, qh + n3 * (j - 1), Fg);
        for (size_t a = 0; a < n3; ++a) Fe[a] = Ft[n3 * (j - 1) + a] + dF[a];      /* <p~> was drawn around F~ + dF */
        if (l == 0) memcpy(Fc, Fg, sizeof(double) * n3);                /* target forces of the last step that will be committed */
        int32_t rej = orc_transport_step(sys, par, Fe, Fg, xi + n3 * (j - 1), u, yp + n3 * (j - 1), qh + n3 * (j - 1),
                                         &S1, &S2, &ell, (l == 0) ? xq : NULL, (l == 0) ? xp : NULL);
        if (dbg_qhalf) memcpy(dbg_qhalf + n3 * (j - 1), qh + n3 * (j - 1), sizeof(double) * n3);
        if (dbg_Ft) memcpy(dbg_Ft + n3 * (j - 1), Ft + n3 * (j - 1), sizeof(double) * n3);
        if (dbg_F) memcpy(dbg_F + n3 * (j - 1), Fg, sizeof(double) * n3);
        if (dbg_S1) dbg_S1[j - 1] = S1; if (dbg_S2) dbg_S2[j - 1] = S2; if (dbg_ell) dbg_ell[j - 1] = ell;
        if (dbg_lnu) dbg_lnu[j - 1] = log(u); if (dbg_reject) dbg_reject[j - 1] = rej;
        if (rej && l == 0) l = j;
        if (l != 0 && !dbg_reject && !dbg_F) break;
    }
    int32_t n_commit = l ? l : K;
    for (int j = 1; j <= n_commit; ++j) {
        const double *sq = (l && j == l) ? xq : yq + n3 * j, *sp = (l && j == l) ? xp : yp + n3 * j;
        if (traj_q) memcpy(traj_q + n3 * (j - 1), sq, sizeof(double) * n3);
        if (traj_p) memcpy(traj_p + n3 * (j - 1), sp, sizeof(double) * n3);
        if (j == n_commit) { memcpy(q, sq, sizeof(double) * n3); memcpy(p, sp, sizeof(double) * n3); }
    }
    for (size_t a = 0; a < n3; ++a) dF[a] = Fc[a] - Ft[n3 * (n_commit - 1) + a];   /* dF' = F - F~(bare) of the last committed step */
    *first_reject = l;
    free(yq); free(yp); free(qh); free(Ft); free(xi); free(Fg); free(xq); free(xp); free(Fe); free(Fc);
    return n_commit;
}

/* orc_run_lsd with EC: the cache starts at zero (:669 "dF <- 0") and is carried from window to window. */
int64_t orc_run_lsd_ec(const orc_system *sys, const orc_params *par, const orc_potential *draft, const orc_potential *target,
                       int64_t n_steps, int32_t K, double *q, double *p, double *dF, double *traj_q, double *traj_p, double *stats)
{
    const size_t n3 = 3 * (size_t)sys->n;
    int64_t n = 0, windows = 0, rejections = 0; double beta_sum = 0.0; int64_t examined = 0;
    double *tq = (double *)malloc(sizeof(double) * n3 * K), *tp = (double *)malloc(sizeof(double) * n3 * K);
    double *S2 = (double *)malloc(sizeof(double) * K);
    while (n < n_steps) {
        int32_t k = K; if (n + k > n_steps) k = (int32_t)(n_steps - n);
        int32_t l;
        int32_t nc = orc_lsd_window_ec(sys, par, draft, target, (uint64_t)n, k, q, p, dF, &l, tq, tp, NULL, NULL, NULL, NULL, S2, NULL, NULL, NULL);
        for (int j = 0; j < nc; ++j) { beta_sum += erf(sqrt(S2[j]) / sqrt(8.0)); ++examined; }
        if (l) ++rejections;
        if (traj_q) memcpy(traj_q + n3 * n, tq, sizeof(double) * n3 * nc);
        if (traj_p) memcpy(traj_p + n3 * n, tp, sizeof(double) * n3 * nc);
        n += nc; ++windows;
    }
    if (stats) { stats[0] = (double)windows; stats[1] = (double)rejections; stats[2] = beta_sum; stats[3] = (double)examined; }
    free(tq); free(tp); free(S2);
    return n;
}

/* ------------------------------------------------------------------------------------------
 * O-6: (OBABO) output momentum of a committed step by time staggering
 * (App. F :632-753).  The ABOBA run already contains the staggered states: after the B O B
 * block of step n the state is ybar_n = (q_half_n, p_n), and A(dt) = A(1/2) A(1/2) leads to q_half_{n+1}
 * (Eq. 25 :652).  With F = F_target(q_half_n) (known from the verification, :735), p_prev = pbar_{n-1},
 * p_new = pbar_n:
 *   Sigma_half = M kT (1 - e^{-gamma dt})                                   (:648)
 *   w      = Sigma_half^{-1/2} (p_new - e^{-gamma dt} p_prev - (1 + e^{-gamma dt}) (dt/2) F)      Eq. 28
 *   xi1*   ~ N( e^{-gamma dt/2} / (1 + e^{-gamma dt}) w ,  1 / (1 + e^{-gamma dt}) I )             Eq. 29
 *   p_mid  = e^{-gamma dt/2} (p_prev + (dt/2) F) + Sigma_half^{1/2} xi1*                           Eq. 30
 * and the OBABO output position is q_half_n (:753).  [reading R18] The extra standard normal is drawn
 * from the same counter-based generator, stream tag 3, keyed by the step index like every other draw (R5).
 * Pins (tests/test_oracle_obabo.py): stationary covariance of (q, p_mid) on the harmonic oscillator vs the
 * discrete Lyapunov solution of the OBABO map Eq. 24 composed in numpy; the implied second half-step
 * noise xi2 = w - e^{-gamma dt/2} xi1* is standard normal and uncorrelated with xi1*.
 * ---------------------------------------------------------------------------------------- */
void orc_obabo_momentum(const orc_system *sys, const orc_params *par, uint64_t step, const double *p_prev,
                        const double *p_new, const double *F, double *p_mid)
{
    const int n = sys->n;
    const double c1 = exp(-par->friction_per_fs * par->dt_fs), ch = exp(-0.5 * par->friction_per_fs * par->dt_fs);
    const double hdt = 0.5 * par->dt_fs;
    double *zeta = (double *)malloc(sizeof(double) * 3 * (size_t)n);
    orc_normals(par->seed, step, n, 3u, zeta);
    for (int i = 0; i < n; ++i) {
        const double sh = sqrt(sys->mass_amu[i] * ORC_AMU * ORC_KB * par->temperature_K * (1.0 - c1));
        for (int c = 0; c < 3; ++c) {
            const int a = 3 * i + c;
            const double w = (p_new[a] - c1 * p_prev[a] - (1.0 + c1) * hdt * F[a]) / sh;
            const double xi1 = ch / (1.0 + c1) * w + sqrt(1.0 / (1.0 + c1)) * zeta[a];
            p_mid[a] = ch * (p_prev[a] + hdt * F[a]) + sh * xi1;
        }
    }
    free(zeta);
}
