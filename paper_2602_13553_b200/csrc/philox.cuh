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
// sincospi by the classical argument reductions and minimax kernels (errors below 1 ulp each on the ranges that occur:
// u1 in [2^-53, 1], 2 u2 in [0, 2)), so eta agrees with the oracle's libm to ~1e-15.
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
__device__ __forceinline__ double log_01(double x) {            // ln x for normal x in (0, 1]
    int hx = __double2hiint(x);
    const int lx = __double2loint(x);
    int k = (hx >> 20) - 1023;
    hx &= 0x000fffff;
    const int i = (hx + 0x95f64) & 0x100000;                     // 1 + f in [sqrt(2)/2, sqrt(2))
    k += i >> 20;
    const double f = __hiloint2double(hx | (i ^ 0x3ff00000), lx) - 1.0;
    const double dk = (double)k;
    const double d = 2.0 + f;
    const double r = rcp_nr(d);
    double s = f * r;
    s = fma(r, fma(-s, d, f), s);                                // one correction: s = f / (2 + f) to < 1 ulp
    const double z = s * s, w = z * z;
    const double t1 = w * fma(w, fma(w, 1.531383769920937332e-01, 2.222219843214978396e-01), 3.999999999940941908e-01);
    const double t2 = z * fma(w, fma(w, fma(w, 1.479819860511658591e-01, 1.818357216161805012e-01), 2.857142874366239149e-01),
                              6.666666666666735130e-01);
    const double R = t2 + t1, hfsq = 0.5 * f * f;
    return dk * 6.93147180369123816490e-01 - ((hfsq - (s * (hfsq + R) + dk * 1.90821492927058770002e-10)) - f);
}
__device__ __forceinline__ double sqrt_nr(double x) {           // sqrt x, x >= 0 (x = 0 -> 0)
    double r;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
    double g = x * r, h = 0.5 * r;
    double e = fma(-h, g, 0.5);
    g = fma(g, e, g); h = fma(h, e, h);
    e = fma(-h, g, 0.5);
    g = fma(g, e, g); h = fma(h, e, h);
    g = fma(fma(-g, g, x), h, g);                                // final correction
    return x > 0.0 ? g : 0.0;
}
__device__ __forceinline__ void sincospi_02(double t, double* sn, double* cs) {     // sin, cos of pi t, t in [0, 2)
    const double n = rint(2.0 * t);                              // 0 .. 4
    const double r = fma(n, -0.5, t);                            // exact, in [-1/4, 1/4]
    const double xh = r * 3.141592653589793116;
    const double xl = fma(r, 3.141592653589793116, -xh) + r * 1.2246467991473532e-16;
    const double z = xh * xh;
    // kernels on [-pi/4, pi/4]
    const double rs = fma(z, fma(z, fma(z, fma(z, 1.58969099521155010221e-10, -2.50507602534068634195e-08), 2.75573137070700676789e-06),
                                 -1.98412698298579493134e-04), 8.33333333332248946124e-03);
    const double v = z * xh;
    const double s0 = xh - ((z * (0.5 * xl - v * rs) - xl) - v * -1.66666666666666324348e-01);
    const double rc = z * fma(z, fma(z, fma(z, fma(z, fma(z, -1.13596475577881948265e-11, 2.08757232129817482790e-09), -2.75573143513906633035e-07),
                                            2.48015872894767294178e-05), -1.38888888888741095749e-03), 4.16666666666666019037e-02);
    const double hz = 0.5 * z, w = 1.0 - hz;
    const double c0 = w + (((1.0 - w) - hz) + (z * rc - xh * xl));
    const int q = (int)n & 3;
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
    for (int j = 0; j < W; ++j) rad[j] = -2.0 * pn4::log_01(philox_u53(c0[j], c1[j], 1u));
#pragma unroll
    for (int j = 0; j < W; ++j) rad[j] = pn4::sqrt_nr(rad[j]);
#pragma unroll
    for (int j = 0; j < W; ++j) {
        double sn, cs;
        pn4::sincospi_02(2.0 * philox_u53(c2[j], c3[j], 0u), &sn, &cs);
        ee[j] = rad[j] * cs;
        eo[j] = rad[j] * sn;
    }
}

__device__ __forceinline__ void philox_normal_pairs4(uint32_t seed_lo, uint32_t seed_hi, uint32_t step_lo, uint32_t step_hi,
                                                     uint32_t atom, uint32_t qdim0, double* ee, double* eo) {
    philox_normal_pairs<4>(seed_lo, seed_hi, step_lo, step_hi, atom, qdim0, ee, eo);
}

}  // namespace pimd
