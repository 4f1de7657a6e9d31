// philox.cuh -- Philox4x32-10 (Salmon et al., SC'11) and the thermostat normal of the O step.
// Keying DESIGN R-10: key = (seed_lo, seed_hi); counter = (step_lo, step_hi, atom i, 4*k + alpha).
#pragma once
#include <stdint.h>

namespace pimd {

__device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0,
                                              uint32_t k1, uint32_t out[4]) {
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        if (r > 0) { k0 += 0x9E3779B9u; k1 += 0xBB67AE85u; }
        const uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
        const uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
        const uint32_t n0 = hi1 ^ c1 ^ k0, n2 = hi0 ^ c3 ^ k1;
        c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// eta = sqrt(-2 ln u1) cos(2 pi u2), u1 = (n1 + 1) 2^-53 in (0,1], u2 = n2 2^-53 in [0,1),
// n = (w_a >> 5) 2^26 + (w_b >> 6)  (Box-Muller, cosine branch; DESIGN R-10; Eq. D2's eta)
__device__ __forceinline__ double philox_normal(uint32_t seed_lo, uint32_t seed_hi, uint32_t step_lo,
                                                uint32_t step_hi, uint32_t atom, uint32_t kdim) {
    uint32_t w[4];
    philox4x32_10(step_lo, step_hi, atom, kdim, seed_lo, seed_hi, w);
    const uint64_t n1 = ((uint64_t)(w[0] >> 5) << 26) + (uint64_t)(w[1] >> 6);
    const uint64_t n2 = ((uint64_t)(w[2] >> 5) << 26) + (uint64_t)(w[3] >> 6);
    const double u1 = (double)n1 * 0x1p-53 + 0x1p-53;     // exact
    const double u2 = (double)n2 * 0x1p-53;
    return sqrt(-2.0 * log(u1)) * cospi(2.0 * u2);
}

}  // namespace pimd
