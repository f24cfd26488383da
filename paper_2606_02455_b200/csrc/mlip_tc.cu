// bf16 tcgen05 filter path (LSD_BF16_TC).  Not enabled yet: mlip_tc_supported() returns false and the
// library runs the fp32 FMA-pipe kernels of mlip_simt.cu instead (still on the GPU).
#include "lsd_internal.h"

bool mlip_tc_supported(const MlipDev&) { return false; }

void mlip_forward_backward_bf16tc(Launcher L, const SysDev& sys, const MlipDev& net, MlipWork& w, int B, const double* q,
                                  const int* img, const CompactList& cl, double* F, double* e_atom)
{
    mlip_forward_backward_fp32(L, sys, net, w, B, q, img, cl, F, e_atom);
}
