// integrator4.cu -- the fused FP64 BAOAB / PILE-L kernel I1 (SURVEY 8(a) rows I-a .. I-i) in north_star's layout: a
// GROUP OF FOUR LANES owns the P beads of one atom-dimension (P = 16, 32, 64; B = P/4 beads per lane), the three
// normal-mode transforms of PAPER.md:L192 / L208 are FFTs whose radix-4 stage runs across the lanes by warp shuffles
// and whose size-B stage runs in registers.  Against integrator.cu (one thread owns all P beads: 244 registers, 98 KB
// of shared-memory staging, 8 warps per SM) a lane here keeps 3 B doubles of state, needs no staging tile, and 16+
// warps per SM hide the Philox / log / sincospi chain of the O step behind the loads.
//
// Data flow of one transform (beads j = B q + m in lane q, W = exp(-2 pi i / P)):
//   X[4r + s] = sum_m W^{m s} u_s[m] W_B^{m r},   u_s[m] = sum_q (-i)^{q s} x[B q + m]
//   lanes after the two shuffle stages:  L0: u_0 (real)   L1: u_2 (real)   L2: Re u_1   L3: -Im u_1
//   every lane: y[m] = W^{m s_lane} * (its real sequence), s_lane = {0, 2, 1, 1};  Z = complex FFT_B(y)   (uniform code)
//   L0 owns modes 4r (Hermitian), L1 owns 4r + 2, L2 owns 4r + 1, L3 owns 4r + 3 (= conj of P - 4r' - 1): each lane
//   ends with B real normal-mode coefficients (B/2 pairs (Re, Im) = the NM indices (k, P - k) of Eq. B1, R-2); L2 and
//   L3 swap half of their spectra (X[4r+1] = A[r] - i B[r], A from L2's sequence, B from L3's).
// The O-step normals (R-10: one Philox draw per NM index pair (2m, 2m+1)): every lane generates B/2 draws, keeps one
// Box-Muller branch and hands the other to the lane that owns the partner index (a rotation inside the group).
// Same arithmetic per mode as integrator.cu.
//
// MEASURED (B200, 2^20 atoms x 32 beads): parity-green at P = 16, 32, 64, but 2.24 ms against 1.14 ms
// for integrator.cu (NVE: 1.77 against 0.75 ms).  The layout trades registers for FP64 work: uniform code across the
// four lanes means a COMPLEX size-B FFT per lane and transform (4 x ~170 flops against ~200 for the in-register real
// FFT of 32 points), and the FP64 pipe of sm_100a (64 lanes per clock and SM) then binds at ~1.8 ms.  The kernel is kept
// as the measured A/B partner and runs only on request (environment variable PIMD_INT4=1); integrator.cu is the path.
#include "common.cuh"
#include "philox.cuh"

namespace pimd {

namespace i4 {

constexpr int kThreads = 128;                  // 4 warps x 8 atom-dimensions x 4 lanes

// cos / sin of 2 pi q / 64, q = 0..63, from the first quadrant
__device__ constexpr double kC64[17] = {
    1.0, 0.99518472667219693, 0.98078528040323043, 0.95694033573220882, 0.92387953251128674,
    0.88192126434835505, 0.83146961230254524, 0.77301045336273699, 0.70710678118654757,
    0.63439328416364549, 0.55557023301960229, 0.47139673682599781, 0.38268343236508984,
    0.29028467725446233, 0.19509032201612833, 0.09801714032956077, 0.0};
__device__ constexpr double cos64(int q) { return q <= 16 ? kC64[q] : (q <= 32 ? -kC64[32 - q] : (q <= 48 ? -kC64[q - 32] : kC64[64 - q])); }
__device__ constexpr double sin64(int q) { return q <= 16 ? kC64[16 - q] : (q <= 32 ? kC64[q - 16] : (q <= 48 ? -kC64[48 - q] : -kC64[q - 48])); }

// complex FFT of size n by decimation in time, out[k] = sum_j in[j * stride] exp(SIGN 2 pi i j k / n); all indices are
// compile-time, everything stays in registers
template <int n, int stride, int SIGN>
struct CFFT {
    __device__ __forceinline__ static void run(const double* inr, const double* ini, double* outr, double* outi) {
        double er[n / 2], ei[n / 2], orr[n / 2], oi[n / 2];
        CFFT<n / 2, stride * 2, SIGN>::run(inr, ini, er, ei);
        CFFT<n / 2, stride * 2, SIGN>::run(inr + stride, ini + stride, orr, oi);
#pragma unroll
        for (int m = 0; m < n / 2; ++m) {
            const double wr = cos64(m * (64 / n)), wi = SIGN * sin64(m * (64 / n));
            double tr, ti;
            if (m == 0) { tr = orr[0]; ti = oi[0]; }
            else if (4 * m == n) { tr = -SIGN * oi[m]; ti = SIGN * orr[m]; }          // w = SIGN i
            else { tr = wr * orr[m] - wi * oi[m]; ti = wr * oi[m] + wi * orr[m]; }
            outr[m] = er[m] + tr; outi[m] = ei[m] + ti;
            outr[m + n / 2] = er[m] - tr; outi[m + n / 2] = ei[m] - ti;
        }
    }
};
template <int stride, int SIGN>
struct CFFT<1, stride, SIGN> {
    __device__ __forceinline__ static void run(const double* inr, const double* ini, double* outr, double* outi) {
        outr[0] = inr[0]; outi[0] = ini[0];
    }
};

__device__ __forceinline__ double shx(double v, int mask) { return __shfl_xor_sync(0xffffffffu, v, mask); }

// a[m] = bead B q + m  ->  a[2i], a[2i+1] = the lane's normal-mode coefficients (pair i; NM indices: nm_index below)
template <int P>
__device__ __forceinline__ void nm_forward4(double* a, const double2* tw, int sl, int q) {
    constexpr int B = P / 4;
#pragma unroll
    for (int m = 0; m < B; ++m) {
        const double o = shx(a[m], 2);
        a[m] = (q < 2) ? a[m] + o : o - a[m];
    }
#pragma unroll
    for (int m = 0; m < B; ++m) {
        const double o = shx(a[m], 1);
        a[m] = (q == 0) ? a[m] + o : (q == 1 ? o - a[m] : a[m]);
    }
    double yr[B], yi[B], zr[B], zi[B];
#pragma unroll
    for (int m = 0; m < B; ++m) { const double2 w = tw[m * sl]; yr[m] = w.x * a[m]; yi[m] = -w.y * a[m]; }   // W^{m s} = (cos, -sin)
    CFFT<B, 1, -1>::run(yr, yi, zr, zi);
    const double s0 = rsqrt((double)P), s1 = sqrt(2.0 / (double)P);
#pragma unroll
    for (int i = 0; i < B / 2; ++i) {
        // L2 sends A[B-1-i] (L3's pair i needs it), L3 sends B[i] (L2's pair i needs it)
        const double rr = shx(q == 2 ? zr[B - 1 - i] : zr[i], 1);
        const double ri = shx(q == 2 ? zi[B - 1 - i] : zi[i], 1);
        const double base_r = (q == 3) ? rr : zr[i];
        const double add_r = (q == 2) ? ri : (q == 3 ? zi[B - 1 - i] : 0.0);
        const double base_i = (q == 3) ? zr[B - 1 - i] : ((q == 0 && i == 0) ? zr[B / 2] : zi[i]);
        const double sub_i = (q == 2) ? rr : (q == 3 ? ri : 0.0);
        const double sc = (q == 0 && i == 0) ? s0 : s1;
        a[2 * i] = sc * (base_r + add_r);
        a[2 * i + 1] = sc * (base_i - sub_i);
    }
}

// the transpose: normal-mode coefficients of the lane -> beads B q + m
template <int P>
__device__ __forceinline__ void nm_inverse4(double* a, const double2* tw, int sl, int q) {
    constexpr int B = P / 4;
    const double s0 = rsqrt((double)P), s1 = sqrt(2.0 / (double)P), h = 0.5 * s1;
    double cr[B], ci[B], wr[B], wi[B];
#pragma unroll
    for (int r = 0; r < B; ++r) { cr[r] = 0.0; ci[r] = 0.0; }
    // spectrum of the lane's family: L0: C[4r] Hermitian; L1: C[4r+2], C[4(B-1-r)+2] = conj; L2: C[4r+1], r < B/2
    // (x 2: the conjugate family s = 3 is folded in); L3: C[4(B-1-i)+1] = conj of its mode 4i+3 (x 2)
#pragma unroll
    for (int i = 0; i < B / 2; ++i) {
        const double pr = a[2 * i], pi = a[2 * i + 1];
        if (i == 0) {
            cr[0] = (q == 0) ? s0 * pr : ((q == 1) ? h * pr : (q == 2 ? s1 * pr : 0.0));
            ci[0] = (q == 0) ? 0.0 : ((q == 1) ? h * pi : (q == 2 ? s1 * pi : 0.0));
            cr[B / 2] += (q == 0) ? s0 * pi : 0.0;
            cr[B - 1] += (q == 1) ? h * pr : (q == 3 ? s1 * pr : 0.0);
            ci[B - 1] += (q == 1) ? -h * pi : (q == 3 ? -s1 * pi : 0.0);
        } else {
            cr[i] += (q < 2) ? h * pr : (q == 2 ? s1 * pr : 0.0);
            ci[i] += (q < 2) ? h * pi : (q == 2 ? s1 * pi : 0.0);
            cr[B - i] += (q == 0) ? h * pr : 0.0;
            ci[B - i] += (q == 0) ? -h * pi : 0.0;
            cr[B - 1 - i] += (q == 1) ? h * pr : (q == 3 ? s1 * pr : 0.0);
            ci[B - 1 - i] += (q == 1) ? -h * pi : (q == 3 ? -s1 * pi : 0.0);
        }
    }
    CFFT<B, 1, +1>::run(cr, ci, wr, wi);
#pragma unroll
    for (int m = 0; m < B; ++m) {
        // times conj(W^{m s}) = (cos, +sin)
        const double2 w = tw[m * sl];
        const double gr = wr[m] * w.x - wi[m] * w.y;
        const double gi = wi[m] * w.x + wr[m] * w.y;
        // xor 1: L0 <-> L1 (w0, w2), L2 <-> L3 (Im g, Re h)
        const double o = shx(q == 2 ? gi : gr, 1);
        const double val = (q == 0) ? gr + o : (q == 1 ? o - gr : (q == 2 ? gr + o : gi + o));
        // xor 2: L0: p0 + E, L2: p0 - E, L1: p1 - F, L3: p1 + F
        const double o2 = shx(val, 2);
        a[m] = (q == 0) ? val + o2 : (q == 1 ? val - o2 : (q == 2 ? o2 - val : o2 + val));
    }
}

// NM index (row of Eq. B1) of slot t of lane q
template <int P>
__device__ __forceinline__ int nm_index(int q, int t) {
    const int i = t >> 1, o = (q == 0) ? 0 : (q == 1 ? 2 : (q == 2 ? 1 : 3));
    if (q == 0 && i == 0) return (t & 1) ? P / 2 : 0;
    return (t & 1) ? P - 4 * i - o : 4 * i + o;
}

template <int P>
__global__ void __launch_bounds__(kThreads, P == 64 ? 2 : 4)
integrator4_kernel(const __grid_constant__ IntegratorArgs a, const __grid_constant__ ModeConsts mc) {
    constexpr int B = P / 4;
    __shared__ double s_mc[6][P];
    __shared__ double red[3][kThreads / 32];
    __shared__ double2 s_tw[P];                            // (cos, sin)(2 pi n / P): twiddles W^{m s} = conj of entry m s
    __shared__ double s_eta[B][kThreads];                  // O-step normals of my B slots (thread-private column)
    for (int k = threadIdx.x; k < P; k += kThreads) {
        double sn, cs;
        sincospi(2.0 * (double)k / (double)P, &sn, &cs);
        s_tw[k] = make_double2(cs, sn);
    }
    for (int k = threadIdx.x; k < P; k += kThreads) {
        s_mc[0][k] = mc.cosA[k]; s_mc[1][k] = mc.sinA_w[k]; s_mc[2][k] = mc.msinA_w[k];
        s_mc[3][k] = mc.c1[k]; s_mc[4][k] = mc.c2[k]; s_mc[5][k] = mc.om2[k];
    }
    __syncthreads();
    const int lane = threadIdx.x & 31, q = lane & 3;
    const int e = (blockIdx.x * (kThreads / 32) + (threadIdx.x >> 5)) * 8 + (lane >> 2);
    const bool live = e < a.n_dof;
    const int ec = live ? e : a.n_dof - 1;
    const int iat = ec / 3, alpha = ec - 3 * iat;
    const size_t stride = (size_t)a.n_dof;
    const bool start = (a.flags & I_START) != 0;
    const bool thermo = start && a.thermostat;

    // ---- loads: f and x of my B beads, v~ of my B normal modes (independent: all in flight together) ----
    double ft[B], xt[B], vt[B];
#pragma unroll
    for (int m = 0; m < B; ++m) ft[m] = a.f[(size_t)(B * q + m) * stride + ec];
#pragma unroll
    for (int m = 0; m < B; ++m) xt[m] = a.x_in[(size_t)(B * q + m) * stride + ec];
#pragma unroll
    for (int t = 0; t < B; ++t) vt[t] = a.vt_in[(size_t)nm_index<P>(q, t) * stride + ec];

    const int sl = (q == 0) ? 0 : (q == 1 ? 2 : 1);        // twiddle family of the lane: W^{m s}, s = {0, 2, 1, 1}

    // ---- O-step normals while the loads are in flight (R-10) ----
    double* eta = &s_eta[0][threadIdx.x];
    if (thermo) {
        uint32_t step_lo = a.step_lo, step_hi = a.step_hi;
        if (a.ctl != nullptr) { const unsigned long long st = (unsigned long long)a.ctl[0]; step_lo = (uint32_t)st; step_hi = (uint32_t)(st >> 32); }
        double kept[B / 2], recv[B / 2];
        const int src = (lane & ~3) | ((q == 0) ? 3 : (q == 1 ? 2 : (q == 2 ? 0 : 1)));
#pragma unroll
        for (int g = 0; g < B / 2; ++g) {
            // draw index m = 2 i' (+1 for L1, L2), i' = g (L0, L1) or B/2 + g (L2, L3)
            const int ip = (q < 2) ? g : B / 2 + g;
            const int md = 2 * ip + ((q == 1 || q == 2) ? 1 : 0);
            double ee, eo;
            philox_normal_pair(a.seed_lo, a.seed_hi, step_lo, step_hi, (uint32_t)iat, (uint32_t)(4 * md + alpha), &ee, &eo);
            kept[g] = (q < 2) ? ee : eo;                    // L0, L1 own the even index of the pair, L2, L3 the odd one
            recv[g] = __shfl_sync(0xffffffffu, (q < 2) ? eo : ee, src);
        }
#pragma unroll
        for (int i = 0; i < B / 2; ++i) {
            // Re slots: own draws (L0, L1) or received (L2, L3), pair i <- g = i
            eta[(2 * i) * kThreads] = (q < 2) ? kept[i] : recv[i];
            // Im slots: pair i <- g = (B/2 - i) mod (B/2) for L0, B/2 - 1 - i otherwise
            const int g0 = (B / 2 - i) % (B / 2), g1 = B / 2 - 1 - i;
            const double from_recv = (q == 0) ? recv[g0] : recv[g1];
            eta[(2 * i + 1) * kThreads] = (q < 2) ? from_recv : kept[g1];
        }
    }

    const double m_at = a.mass[iat];
    const double kick = a.half_dt_mvv / m_at;
    const double sigma = sqrt(a.PkT_mvv / m_at);
    double xf = 0.0;
#pragma unroll
    for (int m = 0; m < B; ++m) xf += xt[m] * ft[m];
    nm_forward4<P>(ft, s_tw, sl, q);
    nm_forward4<P>(xt, s_tw, sl, q);
    if (q == 0) xf -= xt[0] * ft[0];                       // A9 in NM form: sum_j x_j f_j - x~_0 f~_0

    double accK = 0.0, accS = 0.0;
#pragma unroll
    for (int t = 0; t < B; ++t) {
        const int k = nm_index<P>(q, t);
        double v = vt[t];
        if (a.flags & I_BCLOSE) v += kick * ft[t];
        if (a.flags & I_EST) {
            accK += v * v;
            accS += s_mc[5][k] * xt[t] * xt[t];
        }
        if (start) {
            v += kick * ft[t];
            const double cA = s_mc[0][k], sA = s_mc[1][k], mA = s_mc[2][k];
            const double x = xt[t];
            const double xn = cA * x + sA * v;
            double vn = mA * x + cA * v;
            if (thermo) vn = s_mc[3][k] * vn + s_mc[4][k] * sigma * eta[t * kThreads];
            xt[t] = cA * xn + sA * vn;
            v = mA * xn + cA * vn;
        }
        if (live && (a.flags & (I_BCLOSE | I_START))) a.vt_out[(size_t)k * stride + ec] = v;
    }

    if (a.flags & I_EST) {
        double est_k = live ? 0.5 * m_at * accK * kMvv2e : 0.0;
        double est_s = live ? 0.5 * m_at * accS * kMvv2e : 0.0;
        double est_c = live ? xf : 0.0;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            est_k += __shfl_xor_sync(0xffffffffu, est_k, o);
            est_s += __shfl_xor_sync(0xffffffffu, est_s, o);
            est_c += __shfl_xor_sync(0xffffffffu, est_c, o);
        }
        const int w = threadIdx.x >> 5;
        if (lane == 0) { red[0][w] = est_k; red[1][w] = est_s; red[2][w] = est_c; }
        __syncthreads();
        double* est = a.est;
        if (a.ctl != nullptr) {
            const long long idx = a.ctl[0] - 1 - a.ctl[1];
            est = (idx >= 0 && idx < kEstCap) ? a.est_base + (size_t)idx * kEstWidth : a.est_scratch;
        }
        if (threadIdx.x < 3) {
            double tsum = 0.0;
#pragma unroll
            for (int w2 = 0; w2 < kThreads / 32; ++w2) tsum += red[threadIdx.x][w2];
            atomicAdd(est + threadIdx.x, tsum);
        }
        if (blockIdx.x == 0 && threadIdx.x == 3 && a.U != nullptr) {
            double u = 0.0;
            for (int k = 0; k < P; ++k) u += a.U[k];
            atomicAdd(est + 3, u);
        }
    }

    if (start) {
        nm_inverse4<P>(xt, s_tw, sl, q);
        if (live) {
#pragma unroll
            for (int m = 0; m < B; ++m) a.x_out[(size_t)(B * q + m) * stride + ec] = xt[m];
        }
    }
}

}  // namespace i4

// 1 if the launch was taken by the four-lane kernel: BAOAB in normal modes, P = 16 / 32 / 64, no fixcom, no barostat
int launch_integrator4(int P, const IntegratorArgs& a, const ModeConsts& mc, cudaStream_t s) {
    if (a.flags & (I_OBABO | I_COMACC | I_COMSUB | I_CART | I_NOISE_PER_MODE)) return 0;
    if (a.baro != nullptr) return 0;
    const int per_block = (i4::kThreads / 32) * 8;
    const int blocks = (a.n_dof + per_block - 1) / per_block;
    switch (P) {
        case 16: i4::integrator4_kernel<16><<<blocks, i4::kThreads, 0, s>>>(a, mc); return 1;
        case 32: i4::integrator4_kernel<32><<<blocks, i4::kThreads, 0, s>>>(a, mc); return 1;
        case 64: i4::integrator4_kernel<64><<<blocks, i4::kThreads, 0, s>>>(a, mc); return 1;
        default: return 0;
    }
}

}  // namespace pimd
