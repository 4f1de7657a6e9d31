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


// ---------------------------------------------------------------------------------------------------------------
// Four draws at once, branch-free.  The library routines behind philox_normal_pair (log, sqrt, sincospi) carry
// slow-path branches, so the compiler cannot interleave the draws of an unrolled loop and every draw runs as one long
// dependent chain (10 Philox rounds, a division, three polynomials); with two warps per scheduler that chain, not a
// pipe, bounds the O step.  Here the four chains are written side by side: same words, same u1 / u2, and log / sqrt /
// sincospi by the classical argument reductions and minimax kernels, without the last-ulp compensation terms of a libm
// (every step keeps <= 2e-16 on the ranges that occur: u1 in [2^-53, 1], 2 u2 in [0, 2)): the O step is bound by the
// FP64 pipe, so each dropped DFMA is time; eta agrees with the oracle's libm to ~1e-15 (test bound 1e-13).
// ---------------------------------------------------------------------------------------------------------------
namespace pn4 {
__device__ __forceinline__ double rcp_nr(double d) {            // 1/d, d normal and positive: MUFU seed + 2 Newton steps
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(d));
    double e = fma(-d, r, 1.0);
    r = fma(r, e, r);
    e = fma(-d, r, 1.0);
    return fma(r, e, r);
}
// 53-bit grid uniform of philox_u53 times 2^SH, still exact, in three FP64 operations: the 2^52 offsets of the exponent
// trick are taken off inside the fused multiply-adds (2^52 2^-27 = 2^25 from the high piece, 2^52 2^-53 = 1/2 from the low)
template <int SH>
__device__ __forceinline__ double u53_scaled(uint32_t wa, uint32_t wb, uint32_t add) {
    const double dh = __hiloint2double(0x43300000, (int)(wa >> 5));              // 2^52 + a
    const double dl = __hiloint2double(0x43300000, (int)((wb >> 6) + add));      // 2^52 + b
    constexpr double sc = (double)(1 << SH);
    const double hi = fma(dh, 0x1p-27 * sc, -0x1p25 * sc);                        // a 2^(SH-27), exact
    return fma(dl, 0x1p-53 * sc, hi - 0.5 * sc);                                  // + b 2^(SH-53), exact (53 bits)
}
__device__ __forceinline__ double neg2log_01(double x) {        // -2 ln x for normal x in (0, 1]
    int hx = __double2hiint(x);
    const int lx = __double2loint(x);
    int k = (hx >> 20) - 1023;
    hx &= 0x000fffff;
    const int i = (hx + 0x95f64) & 0x100000;                     // 1 + f in [sqrt(2)/2, sqrt(2))
    k += i >> 20;
    const double f = __hiloint2double(hx | (i ^ 0x3ff00000), lx) - 1.0;
    const double dk = __hiloint2double(0x43300000, k + 1024) - 4503599627371520.0;   // (double)k without a conversion: 2^52 + 1024
    const double d = 2.0 + f;
    const double r = rcp_nr(d);
    const double s = f * r;                                      // f / (2 + f) to ~1.5 ulp: it only multiplies the
                                                                 // O(f^2) tail below, so the log keeps < 1e-16 absolute
    // ln(1 + f) = f - f^2/2 + s (f^2/2 + R(z)), z = s^2, R = Lg1 z + .. + Lg7 z^7 (the classical minimax kernel).  Here
    // times -2 with the factor folded into the coefficients (R2 = 2 R), Horner in z, and one ln 2 constant: k <= 53, so
    // the rounding of k (2 ln 2) is <= 1e-16 of the result
    const double z = s * s;
    const double R2 = z * fma(z, fma(z, fma(z, fma(z, fma(z, fma(z, 2.959639721023317182e-01, 3.062767539841874664e-01),
                                                          3.636714432323610024e-01), 4.444439686429956792e-01),
                                            5.714285748732478298e-01), 7.999999999881883816e-01), 1.333333333333347026e+00);
    const double ff = f * f;
    const double t = fma(-s, ff + R2, ff);                       // f^2 - s (f^2 + 2 R)
    return fma(dk, -1.3862943611198906188, fma(-2.0, f, t));
}
__device__ __forceinline__ double sqrt_nr(double x) {           // sqrt x, x >= 0 (x = 0 -> 0)
    double r;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
    double g = x * r, h = 0.5 * r;
    const double e = fma(-h, g, 0.5);                            // seed 2^-22 -> one coupled step 2^-43 ..
    g = fma(g, e, g); h = fma(h, e, h);
    g = fma(fma(-g, g, x), h, g);                                // .. -> Newton step on the residual: below 1 ulp
    return x > 0.0 ? g : 0.0;
}
__device__ __forceinline__ void sincos_quarter(double v, double* sn, double* cs) {  // sin, cos of (pi/2) v, v in [0, 4)
    // n = rint(v) = 0 .. 4 and its integer value without FRND / F2I (64-bit conversions issue at a quarter of the DADD
    // rate): adding 1.5 2^52 rounds v to an integer (ties to even, like rint) and leaves it in the low word
    const double big = v + 6755399441055744.0;
    const int q = __double2loint(big) & 3;
    const double n = big - 6755399441055744.0;
    const double r = v - n;                                      // exact, in [-1/2, 1/2]
    // x = (pi/2) r rounded once: 1e-16 relative on an argument <= pi/4, i.e. <= 9e-17 absolute on sin / cos -- no
    // two-word argument, and both kernels (minimax on [-pi/4, pi/4]) in plain Horner form
    const double x = r * 1.570796326794896558;
    const double z = x * x;
    const double rs = fma(z, fma(z, fma(z, fma(z, fma(z, 1.58969099521155010221e-10, -2.50507602534068634195e-08), 2.75573137070700676789e-06),
                                        -1.98412698298579493134e-04), 8.33333333332248946124e-03), -1.66666666666666324348e-01);
    const double s0 = fma(z * x, rs, x);
    const double rc = fma(z, fma(z, fma(z, fma(z, fma(z, -1.13596475577881948265e-11, 2.08757232129817482790e-09), -2.75573143513906633035e-07),
                                        2.48015872894767294178e-05), -1.38888888888741095749e-03), 4.16666666666666019037e-02);
    const double c0 = fma(z, fma(z, rc, -0.5), 1.0);
    const double sv = (q & 1) ? c0 : s0, cv = (q & 1) ? s0 : c0;
    *sn = (q & 2) ? -sv : sv;
    *cs = ((q + 1) & 2) ? -cv : cv;
}
}  // namespace pn4

// the normals of W consecutive mode pairs (counter word 3 = qdim0, qdim0 + 4, ..): R-10 as philox_normal_pair
template <int W>
__device__ __forceinline__ void philox_normal_pairs(uint32_t seed_lo, uint32_t seed_hi, uint32_t step_lo, uint32_t step_hi,
                                                    uint32_t atom, uint32_t qdim0, double* ee, double* eo) {
    uint32_t c0[W], c1[W], c2[W], c3[W];
#pragma unroll
    for (int j = 0; j < W; ++j) { c0[j] = step_lo; c1[j] = step_hi; c2[j] = atom; c3[j] = qdim0 + 4u * j; }
    uint32_t k0 = seed_lo, k1 = seed_hi;
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        if (r > 0) { k0 += 0x9E3779B9u; k1 += 0xBB67AE85u; }
#pragma unroll
        for (int j = 0; j < W; ++j) {
            const uint32_t hi0 = __umulhi(0xD2511F53u, c0[j]), lo0 = 0xD2511F53u * c0[j];
            const uint32_t hi1 = __umulhi(0xCD9E8D57u, c2[j]), lo1 = 0xCD9E8D57u * c2[j];
            const uint32_t n0 = hi1 ^ c1[j] ^ k0, n2 = hi0 ^ c3[j] ^ k1;
            c0[j] = n0; c1[j] = lo1; c2[j] = n2; c3[j] = lo0;
        }
    }
    double rad[W];
#pragma unroll
    for (int j = 0; j < W; ++j) rad[j] = pn4::neg2log_01(pn4::u53_scaled<0>(c0[j], c1[j], 1u));
#pragma unroll
    for (int j = 0; j < W; ++j) rad[j] = pn4::sqrt_nr(rad[j]);
#pragma unroll
    for (int j = 0; j < W; ++j) {
        double sn, cs;
        pn4::sincos_quarter(pn4::u53_scaled<2>(c2[j], c3[j], 0u), &sn, &cs);       // angle 2 pi u2 = (pi/2) (4 u2)
        ee[j] = rad[j] * cs;
        eo[j] = rad[j] * sn;
    }
}

__device__ __forceinline__ void philox_normal_pairs4(uint32_t seed_lo, uint32_t seed_hi, uint32_t step_lo, uint32_t step_hi,
                                                     uint32_t atom, uint32_t qdim0, double* ee, double* eo) {
    philox_normal_pairs<4>(seed_lo, seed_hi, step_lo, step_hi, atom, qdim0, ee, eo);
}

}  // namespace pimd
