// Counter-based noise of the integrator (R5): Philox4x32-10, the fp64 Box-Muller transform and the 53-bit uniform.
// Shared by integrator.cu and tiny_rollout.cu.  Nothing here is shared with oracle/.
#pragma once
#include <stdint.h>

namespace lsdrng {

constexpr double kTwoPowM32 = 1.0 / 4294967296.0;

// Philox4x32-10 (Salmon et al., SC'11).  Counter = (step lo, step hi, atom, tag), key = seed (R5).
__device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                              uint32_t k0, uint32_t k1, uint32_t out[4])
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
        const uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
        const uint32_t n0 = hi1 ^ c1 ^ k0, n2 = hi0 ^ c3 ^ k1;
        c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// three standard normals per (step, atom): Box-Muller in fp64 on (w + 1/2) 2^-32 (R5)
__device__ __forceinline__ void normals3(uint64_t seed, uint64_t step, uint32_t atom, uint32_t tag, double xi[3])
{
    uint32_t w[4];
    philox4x32_10((uint32_t)step, (uint32_t)(step >> 32), atom, tag, (uint32_t)seed, (uint32_t)(seed >> 32), w);
    const double u0 = ((double)w[0] + 0.5) * kTwoPowM32, u1 = ((double)w[1] + 0.5) * kTwoPowM32;
    const double u2 = ((double)w[2] + 0.5) * kTwoPowM32, u3 = ((double)w[3] + 0.5) * kTwoPowM32;
    const double r0 = sqrt(-2.0 * log(u0)), r1 = sqrt(-2.0 * log(u2));
    double s, c;
    sincospi(2.0 * u1, &s, &c);
    xi[0] = r0 * c; xi[1] = r0 * s;
    xi[2] = r1 * cospi(2.0 * u3);
}

__device__ __forceinline__ double uniform53(uint64_t seed, uint64_t step)
{
    uint32_t w[4];
    philox4x32_10((uint32_t)step, (uint32_t)(step >> 32), 0xFFFFFFFFu, 1u, (uint32_t)seed, (uint32_t)(seed >> 32), w);
    return ((double)(w[0] >> 5) * 67108864.0 + (double)(w[1] >> 6) + 0.5) * (1.0 / 9007199254740992.0);
}

}  // namespace lsdrng
