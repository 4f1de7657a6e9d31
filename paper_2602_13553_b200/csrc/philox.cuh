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

// 53-bit grid uniform ((wa >> 5) 2^26 + (wb >> 6) + add) 2^-53, exact: the two pieces are turned into doubles
// by the 2^52 exponent trick (no 64-bit integer conversion), both products and the sum are exact.
__device__ __forceinline__ double philox_u53(uint32_t wa, uint32_t wb, uint32_t add) {
    const double dh = __hiloint2double(0x43300000, (int)(wa >> 5)) - 4503599627370496.0;
    const double dl = __hiloint2double(0x43300000, (int)((wb >> 6) + add)) - 4503599627370496.0;
    return fma(dh, 0x1p-27, dl * 0x1p-53);
}

// Thermostat normals of the mode pair (2q, 2q+1) of atom `atom`, component alpha (DESIGN R-10; Eq. D2's eta,
// PAPER.md:L476): one draw, counter word 3 = 4q + alpha; u1 in (0,1], u2 in [0,1);
// r = sqrt(-2 ln u1); eta_even = r cos(2 pi u2), eta_odd = r sin(2 pi u2)  (Box-Muller, both branches).
__device__ __forceinline__ void philox_normal_pair(uint32_t seed_lo, uint32_t seed_hi, uint32_t step_lo,
                                                   uint32_t step_hi, uint32_t atom, uint32_t qdim, double* eta_even,
                                                   double* eta_odd) {
    uint32_t w[4];
    philox4x32_10(step_lo, step_hi, atom, qdim, seed_lo, seed_hi, w);
    const double u1 = philox_u53(w[0], w[1], 1u);
    const double u2 = philox_u53(w[2], w[3], 0u);
    const double r = sqrt(-2.0 * log(u1));
    double sn, cs;
    sincospi(2.0 * u2, &sn, &cs);
    *eta_even = r * cs;
    *eta_odd = r * sn;
}

}  // namespace pimd
