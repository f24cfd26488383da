// bf16 tcgen05 filter path (LSD_BF16_TC), host side: which networks it serves, and the packing of the filter weights W_f1 / W_f2 as
// bf16 A-operand images in the no-swizzle K-major UMMA layout that the edge kernels (mlip_edge_rows.cu, mlip_edge_rows_narrow.cu,
// mlip_edge_fwd4.cu) keep resident in shared memory.  (The round-1 "channels are rows" kernel k_edge_tc that lived here, and the
// round-1 / opt-in width-128 kernels of mlip_tc128.cu, mlip_er128.cu and mlip_edge_pipe.cu, were removed in round 3: the default path
// never launched them; their measurements are in profiles/r1_*.md and profiles/r2_edge_rows_bwd_cfg5.md.)
#include <cstring>
#include "lsd_internal.h"

namespace {

constexpr int kR = LSD_NRBF;            // 32 = K of the first contraction

uint16_t bf16_rne(double x)
{
    float f = (float)x;
    uint32_t u; memcpy(&u, &f, 4);
    if ((u & 0x7F800000u) == 0x7F800000u) return (uint16_t)(u >> 16);
    u += 0x7FFFu + ((u >> 16) & 1u);
    return (uint16_t)(u >> 16);
}

}  // namespace

bool mlip_tc_supported(const MlipDev& net) { return (net.F == 32 || net.F == 64 || net.F == 128) && net.R == kR; }

// A operand images: [128-F zero rows ; W/2 or 2W ; 128-F zero rows], (m, k) at byte (m/8)*SBO + (k/8)*128 + (m%8)*16 + (k%8)*2,
// SBO = (K/8)*128.  W_f1 is stored halved and W_f2 doubled (both exact in bf16), the kernels' activation phase undoes the factors.
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
