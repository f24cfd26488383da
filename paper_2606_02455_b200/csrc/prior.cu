// Classical priors in fp64 (O-4): shifted Lennard-Jones and Morse pair terms, harmonic bonds and angles,
// harmonic well at the origin.  One warp per (state, atom), gather form: every atom sums its own terms in a fixed
// order (sorted neighbour row, then its bonded terms), so results are bit-reproducible and batch-invariant.
// F_i = -dU/dq_i = +U'(r) rhat_ij,  rhat_ij = (q_j - q_i + s L) / r.
#include "lsd_internal.h"

namespace {

__device__ __forceinline__ void img_unpack(int v, int& ix, int& iy, int& iz) { ix = (v & 1023) - 512; iy = ((v >> 10) & 1023) - 512; iz = ((v >> 20) & 1023) - 512; }

struct BoxC { double L[3]; int periodic; };

__device__ __forceinline__ void min_image(const BoxC& box, const double* __restrict__ q, int n, int i, int j, double d[3])
{
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        double x = q[c * n + j] - q[c * n + i];
        if (box.periodic) x -= rint(x / box.L[c]) * box.L[c];
        d[c] = x;
    }
}

__global__ void __launch_bounds__(256)
k_prior(int n, int B, BoxC box, const double* __restrict__ q, const int* __restrict__ img, const int* __restrict__ species, int ns,
        const double* __restrict__ pair, const double* __restrict__ tether, const int* __restrict__ pcount,
        const uint32_t* __restrict__ pkeys, int pcap, int use_bonded, const int* __restrict__ bt_start, const int* __restrict__ bt_term,
        int n_bonds, const int* __restrict__ bonds, const double* __restrict__ bond_k, const double* __restrict__ bond_r0,
        const int* __restrict__ angles, const double* __restrict__ angle_k, const double* __restrict__ angle_t0, double* __restrict__ F)
{
    pdl_sync();
    const int warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    if (warp >= n * B) return;
    const int b = warp / n, i = warp % n;
    const double* qb = q + (size_t)b * 3 * n;
    double f[3] = {0.0, 0.0, 0.0};
    if (pcount) {
        const int cnt = pcount[warp];
        const int si = species[i];
        int iix, iiy, iiz; img_unpack(img[i], iix, iiy, iiz);
        for (int e = lane; e < cnt; e += 32) {
            const uint32_t key = pkeys[(size_t)warp * pcap + e];
            const int j = (int)(key >> 5), code = (int)(key & 31u);
            int jx, jy, jz; img_unpack(img[j], jx, jy, jz);
            const int s[3] = {code / 9 - 1 + iix - jx, (code / 3) % 3 - 1 + iiy - jy, code % 3 - 1 + iiz - jz};
            double d[3];
#pragma unroll
            for (int c = 0; c < 3; ++c) d[c] = (qb[c * n + j] - qb[c * n + i]) + (double)s[c] * box.L[c];
            const double r = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
            const double* pp = pair + 8 * (si * ns + species[j]);
            double du = 0.0;
            if (pp[0] != 0.0 && r < pp[2]) { const double sr = pp[1] / r, s2 = sr * sr, s6 = s2 * s2 * s2; du += -24.0 * pp[0] / r * (2.0 * s6 * s6 - s6); }
            if (pp[3] != 0.0 && r < pp[6]) { const double x = exp(-pp[4] * (r - pp[5])); du += 2.0 * pp[3] * pp[4] * x * (1.0 - x); }
            const double g = du / r;
            f[0] += g * d[0]; f[1] += g * d[1]; f[2] += g * d[2];
        }
    }
    if (use_bonded) {
        for (int t = bt_start[i] + lane; t < bt_start[i + 1]; t += 32) {
            const int term = bt_term[t];
            if (term < n_bonds) {                                  // U = k/2 (r - r0)^2
                const int a0 = bonds[2 * term], a1 = bonds[2 * term + 1];
                const int other = (a0 == i) ? a1 : a0;
                double d[3]; min_image(box, qb, n, i, other, d);
                const double r = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
                const double g = bond_k[term] * (r - bond_r0[term]) / r;
                f[0] += g * d[0]; f[1] += g * d[1]; f[2] += g * d[2];
            } else {                                               // U = k/2 (theta - theta0)^2, apex = middle index
                const int a = term - n_bonds;
                const int ia = angles[3 * a], ib = angles[3 * a + 1], ic = angles[3 * a + 2];
                double u[3], v[3];
                min_image(box, qb, n, ib, ia, u); min_image(box, qb, n, ib, ic, v);
                const double nu = sqrt(u[0] * u[0] + u[1] * u[1] + u[2] * u[2]), nv = sqrt(v[0] * v[0] + v[1] * v[1] + v[2] * v[2]);
                double ct = (u[0] * v[0] + u[1] * v[1] + u[2] * v[2]) / (nu * nv);
                ct = fmin(1.0, fmax(-1.0, ct));
                const double th = acos(ct), st = fmax(sqrt(1.0 - ct * ct), 1e-12);   // collinear arms: bounded instead of 0/0 (R19)
                const double dU = angle_k[a] * (th - angle_t0[a]);
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    const double uh = u[c] / nu, vh = v[c] / nv;
                    const double da = -(vh - ct * uh) / (nu * st), dc = -(uh - ct * vh) / (nv * st);
                    double contrib;
                    if (i == ia) contrib = -dU * da; else if (i == ic) contrib = -dU * dc; else contrib = dU * (da + dc);
                    f[c] += contrib;
                }
            }
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        f[0] += __shfl_xor_sync(0xffffffffu, f[0], o);
        f[1] += __shfl_xor_sync(0xffffffffu, f[1], o);
        f[2] += __shfl_xor_sync(0xffffffffu, f[2], o);
    }
    if (lane == 0) {
        if (tether) { const double k = tether[species[i]]; f[0] -= k * qb[i]; f[1] -= k * qb[n + i]; f[2] -= k * qb[2 * n + i]; }
        F[((size_t)b * 3 + 0) * n + i] = f[0];
        F[((size_t)b * 3 + 1) * n + i] = f[1];
        F[((size_t)b * 3 + 2) * n + i] = f[2];
    }
}

}  // namespace

void launch_prior_forces(Launcher L, const SysDev& sys, const PotDev& pot, int B, const double* q, const int* img,
                         const CompactList* pl, double* F)
{
    BoxC box; for (int c = 0; c < 3; ++c) box.L[c] = sys.box[c]; box.periodic = sys.periodic;
    const size_t warps = (size_t)sys.n * B;
    const int blocks = (int)((warps * 32 + 255) / 256);
    const int pid = prof_begin(L, PROF_PRIOR);
    launch_pdl(L, k_prior, dim3(blocks), dim3(256), 0, sys.n, B, box, q, img, sys.species, sys.ns, pot.pair, pot.has_tether ? pot.tether : nullptr,
                                     pl ? pl->count : nullptr, pl ? pl->keys : nullptr, pl ? pl->cap : 0,
                                     pot.use_bonded && (sys.n_bonds + sys.n_angles) > 0, sys.bt_start, sys.bt_term, sys.n_bonds, sys.bonds,
                                     sys.bond_k, sys.bond_r0, sys.angles, sys.angle_k, sys.angle_t0, F);
    LSD_COUNT(L);
    prof_end(L, pid);
}
