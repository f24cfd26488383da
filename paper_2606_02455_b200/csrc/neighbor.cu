// Window-shared cell list -> Verlet (skin) list -> per-state exact lists.
// DESIGN.md T1: the compared object is the per-state directed edge set {(i, j, shift) : r < r_c}; the distance
// test is done in fp64 on the unwrapped positions with the oracle's operation order and no FMA contraction:
//   x = q_j - q_i;  x = x + s L  (s = -rint(x/L), the minimum-image shift);  r2 = (dx dx + dy dy) + dz dz.
// Shifts are stored relative to the images of the reference state: s = s_w + img_i - img_j, s_w in {-1,0,1}.
#include "lsd_internal.h"

namespace {

__host__ __device__ __forceinline__ int img_pack(int ix, int iy, int iz) { return (ix + 512) | ((iy + 512) << 10) | ((iz + 512) << 20); }
__device__ __forceinline__ void img_unpack(int v, int& ix, int& iy, int& iz) { ix = (v & 1023) - 512; iy = ((v >> 10) & 1023) - 512; iz = ((v >> 20) & 1023) - 512; }

struct BoxC { double L[3]; int periodic; };

// wrapped image index of every atom at the reference state: q = qw + img L, qw in [0, L)
__global__ void k_images(int n, BoxC box, const double* __restrict__ q, int* __restrict__ img)
{
    pdl_sync();
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    int im[3] = {0, 0, 0};
    if (box.periodic) {
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            int v = (int)floor(q[c * n + i] / box.L[c]);
            v = max(-511, min(511, v));
            im[c] = v;
        }
    }
    img[i] = img_pack(im[0], im[1], im[2]);
}

__device__ __forceinline__ int cell_of(const BoxC& box, const int nc[3], const double* q, int n, int i, int img)
{
    int ix, iy, iz; img_unpack(img, ix, iy, iz);
    const int im[3] = {ix, iy, iz};
    int cc[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        int v = 0;
        if (nc[c] > 1) {
            const double f = (q[c * n + i] - (double)im[c] * box.L[c]) / box.L[c];
            v = (int)(f * nc[c]);
            v = max(0, min(nc[c] - 1, v));
        }
        cc[c] = v;
    }
    return (cc[0] * nc[1] + cc[1]) * nc[2] + cc[2];
}

struct GridC { int nc[3]; };

__global__ void k_cell_count(int n, BoxC box, GridC g, const double* __restrict__ q, const int* __restrict__ img,
                             int* __restrict__ atom_cell, int* __restrict__ cell_count)
{
    pdl_sync();
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const int c = cell_of(box, g.nc, q, n, i, img[i]);
    atom_cell[i] = c;
    atomicAdd(&cell_count[c], 1);
}

__global__ void k_cell_scan(int ncell, const int* __restrict__ cell_count, int* __restrict__ cell_start, int* __restrict__ cell_cursor)
{
    pdl_sync();
    // single block exclusive scan (ncell is a few thousand)
    __shared__ int carry;
    __shared__ int buf[1024];
    if (threadIdx.x == 0) carry = 0;
    __syncthreads();
    for (int base = 0; base < ncell; base += 1024) {
        const int i = base + threadIdx.x;
        const int v = i < ncell ? cell_count[i] : 0;
        buf[threadIdx.x] = v;
        __syncthreads();
        for (int o = 1; o < 1024; o <<= 1) {
            const int t = threadIdx.x >= o ? buf[threadIdx.x - o] : 0;
            __syncthreads();
            buf[threadIdx.x] += t;
            __syncthreads();
        }
        const int excl = carry + buf[threadIdx.x] - v;
        if (i < ncell) { cell_start[i] = excl; cell_cursor[i] = excl; }
        __syncthreads();
        if (threadIdx.x == 1023) carry += buf[1023];
        __syncthreads();
    }
    if (threadIdx.x == 0) cell_start[ncell] = carry;
}

__global__ void k_cell_fill(int n, const int* __restrict__ atom_cell, int* __restrict__ cell_cursor, int* __restrict__ cell_atoms)
{
    pdl_sync();
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    cell_atoms[atomicAdd(&cell_cursor[atom_cell[i]], 1)] = i;     // order inside a cell is fixed later by the row sort
}

// fp64, FMA-free minimum-image displacement j - i; returns r2 and the wrapped-frame shift code
__device__ __forceinline__ double pair_r2(const BoxC& box, const double* __restrict__ q, int n, int i, int j, int& sx, int& sy, int& sz)
{
    double d[3]; int s[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        double x = __dsub_rn(q[c * n + j], q[c * n + i]);
        int k = 0;
        if (box.periodic) {
            const double kk = rint(__ddiv_rn(x, box.L[c]));
            k = (int)kk;
            x = __dsub_rn(x, __dmul_rn(kk, box.L[c]));
        }
        d[c] = x; s[c] = -k;
    }
    sx = s[0]; sy = s[1]; sz = s[2];
    return __dadd_rn(__dadd_rn(__dmul_rn(d[0], d[0]), __dmul_rn(d[1], d[1])), __dmul_rn(d[2], d[2]));
}

constexpr int kVlWarps = 8;
constexpr int kVlMaxRow = 512;

// One warp per atom: enumerate the (de-duplicated) 27-cell stencil, keep r < rc + skin, sort the row by key.
__global__ void __launch_bounds__(kVlWarps * 32)
k_build_verlet(int n, BoxC box, GridC g, const double* __restrict__ q, const int* __restrict__ img,
               const int* __restrict__ atom_cell, const int* __restrict__ cell_start, const int* __restrict__ cell_atoms,
               double rcs2, int cap, int* __restrict__ count, uint32_t* __restrict__ keys, int* flags,
               const int* __restrict__ species, int ns, const double* __restrict__ pair_rcs2 /*or null: [ns][ns] (r_c(s_i, s_j) + skin)^2, 0 = no pair term*/)
{
    pdl_sync();
    __shared__ uint32_t rows[kVlWarps][kVlMaxRow];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int i = blockIdx.x * kVlWarps + warp;
    if (i >= n) return;
    uint32_t* row = rows[warp];
    int cnt = 0;
    const int ci = atom_cell ? atom_cell[i] : 0;            // (no cell tables: the whole system is one cell, launch_build_verlet)
    const int cz = ci % g.nc[2], cy = (ci / g.nc[2]) % g.nc[1], cx = ci / (g.nc[2] * g.nc[1]);
    int iix, iiy, iiz; img_unpack(img[i], iix, iiy, iiz);
    const double* const lim_row = pair_rcs2 ? pair_rcs2 + species[i] * ns : nullptr;
    const int lox = g.nc[0] >= 3 ? -1 : 0, hix = g.nc[0] >= 3 ? 1 : g.nc[0] - 1;   // < 3 cells: visit each cell once (R10)
    const int loy = g.nc[1] >= 3 ? -1 : 0, hiy = g.nc[1] >= 3 ? 1 : g.nc[1] - 1;
    const int loz = g.nc[2] >= 3 ? -1 : 0, hiz = g.nc[2] >= 3 ? 1 : g.nc[2] - 1;
    for (int dx = lox; dx <= hix; ++dx) for (int dy = loy; dy <= hiy; ++dy) for (int dz = loz; dz <= hiz; ++dz) {
        const int ox = g.nc[0] >= 3 ? (cx + dx + g.nc[0]) % g.nc[0] : dx;
        const int oy = g.nc[1] >= 3 ? (cy + dy + g.nc[1]) % g.nc[1] : dy;
        const int oz = g.nc[2] >= 3 ? (cz + dz + g.nc[2]) % g.nc[2] : dz;
        const int c = (ox * g.nc[1] + oy) * g.nc[2] + oz;
        const int beg = cell_start ? cell_start[c] : 0, end = cell_start ? cell_start[c + 1] : n;
        for (int t0 = beg; t0 < end; t0 += 32) {
            const int t = t0 + lane;
            bool keep = false; uint32_t key = 0;
            if (t < end) {
                const int j = cell_atoms ? cell_atoms[t] : t;
                if (j != i) {
                    int sx, sy, sz;
                    const double r2 = pair_r2(box, q, n, i, j, sx, sy, sz);
                    if (r2 < (lim_row ? lim_row[species[j]] : rcs2)) {   // pair-prior list: candidates of the species pairs that interact only
                        int jx, jy, jz; img_unpack(img[j], jx, jy, jz);
                        const int wx = sx - iix + jx, wy = sy - iiy + jy, wz = sz - iiz + jz;   // s_w = s - img_i + img_j
                        keep = true;
                        key = ((uint32_t)j << 5) | (uint32_t)((wx + 1) * 9 + (wy + 1) * 3 + (wz + 1));
                        if (wx < -1 || wx > 1 || wy < -1 || wy > 1 || wz < -1 || wz > 1) { keep = false; atomicOr(flags, LSD_FLAG_OVERFLOW); }
                    }
                }
            }
            const unsigned m = __ballot_sync(0xffffffffu, keep);
            if (keep) { const int pos = cnt + __popc(m & ((1u << lane) - 1)); if (pos < kVlMaxRow) row[pos] = key; }
            cnt += __popc(m);
        }
    }
    __syncwarp();
    if (cnt > cap || cnt > kVlMaxRow) { if (lane == 0) atomicOr(flags, LSD_FLAG_OVERFLOW); cnt = min(cap, kVlMaxRow); }
    // rank sort (keys are unique): row is small
    for (int e = lane; e < cnt; e += 32) {
        const uint32_t k = row[e];
        int rank = 0;
        for (int f = 0; f < cnt; ++f) rank += row[f] < k;
        keys[(size_t)i * cap + rank] = k;
    }
    for (int e = cnt + lane; e < cap; e += 32) keys[(size_t)i * cap + e] = 0xFFFFFFFFu;
    if (lane == 0) count[i] = cnt;
}

// One warp per (state b, atom i): keep the Verlet candidates with r < rc in state b (order preserved).
__global__ void __launch_bounds__(256)
k_compact(int n, int B, BoxC box, const double* __restrict__ q, const int* __restrict__ img, const int* __restrict__ species, int ns,
          const int* __restrict__ vcount, const uint32_t* __restrict__ vkeys, int vcap, double rc2_single,
          const double* __restrict__ pair_rc2, int cap, int* __restrict__ count, uint32_t* __restrict__ keys, int* flags,
          float* __restrict__ recs, float inv_rc)
{
    pdl_sync();
    const int warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    if (warp >= n * B) return;
    const int b = warp / n, i = warp % n;
    const double* qb = q + (size_t)b * 3 * n;
    const int vc = vcount[i];
    int iix, iiy, iiz; img_unpack(img[i], iix, iiy, iiz);
    const int si = species[i];
    uint32_t* out = keys + (size_t)warp * cap;
    int cnt = 0;
    for (int e0 = 0; e0 < vc; e0 += 32) {
        const int e = e0 + lane;
        bool keep = false; uint32_t key = 0xFFFFFFFFu;
        double d[3] = {0.0, 0.0, 0.0}, r2 = 0.0;
        int j = 0;
        if (e < vc) {
            key = vkeys[(size_t)i * vcap + e];
            j = (int)(key >> 5);
            const int code = (int)(key & 31u);
            int jx, jy, jz; img_unpack(img[j], jx, jy, jz);
            const int s[3] = {code / 9 - 1 + iix - jx, (code / 3) % 3 - 1 + iiy - jy, code % 3 - 1 + iiz - jz};
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                const double x = __dsub_rn(qb[c * n + j], qb[c * n + i]);
                d[c] = __dadd_rn(x, __dmul_rn((double)s[c], box.L[c]));     // x - k L with k = -s (exact negation)
            }
            r2 = __dadd_rn(__dadd_rn(__dmul_rn(d[0], d[0]), __dmul_rn(d[1], d[1])), __dmul_rn(d[2], d[2]));
            const double lim = pair_rc2 ? pair_rc2[si * ns + species[j]] : rc2_single;
            keep = r2 < lim;
        }
        const unsigned m = __ballot_sync(0xffffffffu, keep);
        if (keep) {
            const int pos = cnt + __popc(m & ((1u << lane) - 1));
            if (pos < cap) {
                out[pos] = key;
                if (recs) {                                                 // fp64 geometry rounded once to fp32
                    const double rd = sqrt(r2);
                    const float rf = (float)rd;
                    float fc = 0.f, fcp = 0.f;
                    const float t = rf * inv_rc;
                    if (t < 1.f) {                                          // M2
                        float sn, cs; sincospif(t, &sn, &cs);
                        fc = 0.5f * (cs + 1.f); fcp = -0.5f * 3.14159265358979323846f * inv_rc * sn;
                    }
                    float* o = recs + lsd_rec_index((size_t)warp, cap, pos, 0);
                    o[LSD_REC_R * 16] = rf; o[LSD_REC_FC * 16] = fc; o[LSD_REC_FCP * 16] = fcp;
                    const double rinv = 1.0 / rd;                           // one fp64 division per edge; the unit vector is rounded to fp32
                    o[LSD_REC_UX * 16] = (float)(d[0] * rinv); o[LSD_REC_UY * 16] = (float)(d[1] * rinv); o[LSD_REC_UZ * 16] = (float)(d[2] * rinv);
                    o[LSD_REC_JROW * 16] = __int_as_float(b * n + j);
                }
            }
        }
        cnt += __popc(m);
    }
    if (cnt > cap) { if (lane == 0) atomicOr(flags, LSD_FLAG_OVERFLOW); cnt = cap; }
    for (int e = cnt + lane; e < cap; e += 32) out[e] = 0xFFFFFFFFu;
    if (recs) {                                                             // zero records behind the count, to the end of the last group
        const int e = cnt + lane;
        if (lane < 16 && e < ((cnt + 15) & ~15) && e < cap) {
            float* o = recs + lsd_rec_index((size_t)warp, cap, e, 0);
#pragma unroll
            for (int fld = 0; fld < 6; ++fld) o[fld * 16] = 0.f;
            o[LSD_REC_JROW * 16] = __int_as_float(warp);
        }
    }
    if (lane == 0) count[warp] = cnt;
}

__global__ void k_check_skin(int n, int B, const double* __restrict__ q, const double* __restrict__ qref, double skin_half2, int* flags)
{
    const size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= (size_t)n * B) return;
    const int b = (int)(t / n), i = (int)(t % n);
    double d2 = 0.0;
#pragma unroll
    for (int c = 0; c < 3; ++c) { const double d = q[((size_t)b * 3 + c) * n + i] - qref[c * n + i]; d2 += d * d; }
    if (d2 > skin_half2) atomicOr(flags, LSD_FLAG_SKIN);
    if (!isfinite(d2)) atomicOr(flags, LSD_FLAG_NONFINITE);
}

BoxC make_box(const SysDev& sys) { BoxC b; for (int c = 0; c < 3; ++c) b.L[c] = sys.box[c]; b.periodic = sys.periodic; return b; }

}  // namespace

void cellgrid_setup(CellGrid& g, const SysDev& sys, double rc_skin)
{
    int nc[3] = {1, 1, 1};
    if (sys.periodic) for (int c = 0; c < 3; ++c) { nc[c] = (int)floor(sys.box[c] / rc_skin); if (nc[c] < 3) nc[c] = 1; }
    const int ncell = nc[0] * nc[1] * nc[2];
    if (ncell > g.cap_cells) {
        cudaFree(g.cell_count); cudaFree(g.cell_start); cudaFree(g.cell_cursor);
        cudaMalloc(&g.cell_count, sizeof(int) * ncell); cudaMalloc(&g.cell_start, sizeof(int) * (ncell + 1));
        cudaMalloc(&g.cell_cursor, sizeof(int) * ncell);
        g.cap_cells = ncell;
    }
    if (!g.cell_atoms) { cudaMalloc(&g.cell_atoms, sizeof(int) * sys.n); cudaMalloc(&g.atom_cell, sizeof(int) * sys.n); }
    g.nc[0] = nc[0]; g.nc[1] = nc[1]; g.nc[2] = nc[2]; g.ncell = ncell;
}

void launch_pack_ref(Launcher L, const SysDev& sys, const double* qref, int* img)
{
    launch_pdl(L, k_images, dim3((sys.n + 255) / 256), dim3(256), 0, sys.n, make_box(sys), qref, img);
    LSD_COUNT(L);
}

void launch_build_verlet(Launcher L, const SysDev& sys, CellGrid& g, const double* qref, const int* img,
                         double rc_skin, VerletList& vl, int* flags, const double* pair_rcs2)
{
    const int n = sys.n;
    const int pid = prof_begin(L, PROF_NBR);
    GridC gc; gc.nc[0] = g.nc[0]; gc.nc[1] = g.nc[1]; gc.nc[2] = g.nc[2];
    const bool one_cell = g.ncell == 1;                      // small boxes / vacuum: every atom is a candidate, no binning (three launches less)
    if (!one_cell) {
        cudaMemsetAsync(g.cell_count, 0, sizeof(int) * g.ncell, L.s);
        launch_pdl(L, k_cell_count, dim3((n + 255) / 256), dim3(256), 0, n, make_box(sys), gc, qref, img, g.atom_cell, g.cell_count); LSD_COUNT(L);
        launch_pdl(L, k_cell_scan, dim3(1), dim3(1024), 0, g.ncell, g.cell_count, g.cell_start, g.cell_cursor); LSD_COUNT(L);
        launch_pdl(L, k_cell_fill, dim3((n + 255) / 256), dim3(256), 0, n, g.atom_cell, g.cell_cursor, g.cell_atoms); LSD_COUNT(L);
    }
    launch_pdl(L, k_build_verlet, dim3((n + kVlWarps - 1) / kVlWarps), dim3(kVlWarps * 32), 0, n, make_box(sys), gc, qref, img,
               one_cell ? (const int*)nullptr : (const int*)g.atom_cell, one_cell ? (const int*)nullptr : (const int*)g.cell_start,
               one_cell ? (const int*)nullptr : (const int*)g.cell_atoms, rc_skin * rc_skin, vl.cap, vl.count, vl.keys, flags, sys.species, sys.ns, pair_rcs2);
    LSD_COUNT(L);
    prof_end(L, pid);
}

void launch_compact(Launcher L, const SysDev& sys, int B, const double* q, const int* img, const VerletList& vl,
                    double rc2_single, const double* pair_rc2, CompactList& cl, int* flags, float rc_records)
{
    const size_t warps = (size_t)sys.n * B;
    const int blocks = (int)((warps * 32 + 255) / 256);
    const int pid = prof_begin(L, PROF_NBR);
    launch_pdl(L, k_compact, dim3(blocks), dim3(256), 0, sys.n, B, make_box(sys), q, img, sys.species, sys.ns, vl.count, vl.keys, vl.cap, rc2_single,
                                       pair_rc2, cl.cap, cl.count, cl.keys, flags, rc_records > 0.f ? cl.recs : nullptr,
                                       rc_records > 0.f ? 1.f / rc_records : 0.f);
    LSD_COUNT(L);
    prof_end(L, pid);
}

void launch_check_skin(Launcher L, int n, int B, const double* q, const double* qref, double skin_half2, int* flags)
{
    const size_t t = (size_t)n * B;
    k_check_skin<<<(int)((t + 255) / 256), 256, 0, L.s>>>(n, B, q, qref, skin_half2, flags);
    LSD_COUNT(L);
}
