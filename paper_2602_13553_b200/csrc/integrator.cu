// integrator.cu -- fused FP64 BAOAB / PILE-L kernel I1 (SURVEY 8(a) rows I-a .. I-i).
//
// One THREAD owns all P beads of one atom-dimension (with the [P][N][3] layout a
// warp then reads 32 consecutive doubles of every bead row -> fully coalesced, and the three
// normal-mode transforms of PAPER.md:L192/L208 become in-register real FFTs with no shuffles).
//   closing B of step t (needs f~ = M f)
//   estimators K, S, sum x.f (Appendix A)  -> block reduction -> one atomicAdd per block
//   opening B, A(dt/2), O(dt), A(dt/2) of step t+1   L165, L190-192, Eq. D1-D2
//   x = M^T x~                                       Eq. B3
// reads x, v~, f once and writes x, v~ once: 40 B per bead-atom-dim.
#include "common.cuh"
#include <cstdlib>
#include <cuda_pipeline.h>
#include "philox.cuh"

namespace pimd {

// cos(2 pi q / 64), q = 0..16
__device__ constexpr double kCos64[17] = {
    1.0, 0.99518472667219693, 0.98078528040323043, 0.95694033573220882, 0.92387953251128674,
    0.88192126434835505, 0.83146961230254524, 0.77301045336273699, 0.70710678118654757,
    0.63439328416364549, 0.55557023301960229, 0.47139673682599781, 0.38268343236508984,
    0.29028467725446233, 0.19509032201612833, 0.09801714032956077, 0.0};

// Real-input FFT X_m = sum_j in[j*stride] exp(-2 pi i m j / n), m = 0..n/2, by decimation in time on
// the half-complex representation.  re[0..n/2], im[1..n/2-1] are written; im[0], im[n/2] are never
// written nor read (they are zero).  All indices are compile-time so everything stays in registers.
template <int n, int stride>
struct RFFT {
    __device__ __forceinline__ static void run(const double* in, double* re, double* im) {
        double er[n / 4 + 1], ei[n / 4 + 1], orr[n / 4 + 1], oi[n / 4 + 1];
        RFFT<n / 2, stride * 2>::run(in, er, ei);
        RFFT<n / 2, stride * 2>::run(in + stride, orr, oi);
        re[0] = er[0] + orr[0];
        re[n / 2] = er[0] - orr[0];
        re[n / 4] = er[n / 4];
        im[n / 4] = -orr[n / 4];
#pragma unroll
        for (int m = 1; m < n / 4; ++m) {
            const double wr = kCos64[m * (64 / n)];
            const double wi = -kCos64[16 - m * (64 / n)];
            const double tr = wr * orr[m] - wi * oi[m];
            const double ti = wr * oi[m] + wi * orr[m];
            re[m] = er[m] + tr;
            im[m] = ei[m] + ti;
            re[n / 2 - m] = er[m] - tr;
            im[n / 2 - m] = ti - ei[m];
        }
    }
};
template <int stride>
struct RFFT<2, stride> {
    __device__ __forceinline__ static void run(const double* in, double* re, double* im) {
        re[0] = in[0] + in[stride];
        re[1] = in[0] - in[stride];
    }
};
template <int stride>
struct RFFT<1, stride> {
    __device__ __forceinline__ static void run(const double* in, double* re, double* im) { re[0] = in[0]; }
};

// a~ = M a with M of Eq. B1 (reading DESIGN R-2), in place.
template <int P>
__device__ __forceinline__ void nm_forward(double* a) {
    if constexpr (P == 1) return;
    double re[P / 2 + 1], im[P / 2 + 1];
    RFFT<P, 1>::run(a, re, im);
    const double s0 = rsqrt((double)P), s1 = sqrt(2.0 / (double)P);
    a[0] = re[0] * s0;
    a[P / 2] = re[P / 2] * s0;
#pragma unroll
    for (int k = 1; k < P / 2; ++k) {
        a[k] = s1 * re[k];
        a[P - k] = s1 * im[k];
    }
}

// a = M^T a~ (Eq. B3), in place: the transposed real-DFT matrix equals a forward real FFT of the
// sequence z with z_k + z_{P-k} = sqrt(2/P) a~_k, z_k - z_{P-k} = sqrt(2/P) a~_{P-k}; x_j = Re Z_j + Im Z_j.
template <int P>
__device__ __forceinline__ void nm_inverse(double* a) {
    if constexpr (P == 1) return;
    double z[P];
    const double s0 = rsqrt((double)P), s2 = rsqrt(2.0 * (double)P);
    z[0] = a[0] * s0;
    z[P / 2] = a[P / 2] * s0;
#pragma unroll
    for (int k = 1; k < P / 2; ++k) {
        z[k] = (a[k] + a[P - k]) * s2;
        z[P - k] = (a[k] - a[P - k]) * s2;
    }
    double re[P / 2 + 1], im[P / 2 + 1];
    RFFT<P, 1>::run(z, re, im);
    a[0] = re[0];
    a[P / 2] = re[P / 2];
#pragma unroll
    for (int j = 1; j < P / 2; ++j) {
        a[j] = re[j] + im[j];
        a[P - j] = re[j] - im[j];
    }
}

constexpr int kIntThreads = 128;
#ifndef PIMD_NOISE_WIDE
#define PIMD_NOISE_WIDE 4
#endif
constexpr int kNoiseWide = PIMD_NOISE_WIDE;     // draws generated side by side (4: 0.874 ms at 2^20 x 32; 8: 0.927)

// step counters (Philox counter words 0, 1; R-10) and estimator slot of a launch: launch arguments, or -- under graph
// replay -- derived from the device-resident step counter
struct StepView { uint32_t step_lo, step_hi, cstep_lo, cstep_hi; double* est; };
__device__ __forceinline__ StepView resolve_step(const IntegratorArgs& a) {
    StepView v = {a.step_lo, a.step_hi, a.cstep_lo, a.cstep_hi, a.est};
    if (a.ctl != nullptr) {
        const unsigned long long st = (unsigned long long)a.ctl[0], cs = st - 1ull;
        v.step_lo = (uint32_t)st; v.step_hi = (uint32_t)(st >> 32);
        v.cstep_lo = (uint32_t)cs; v.cstep_hi = (uint32_t)(cs >> 32) | 0x80000000u;
        const long long idx = a.ctl[0] - 1 - a.ctl[1];
        v.est = (idx >= 0 && idx < kEstCap) ? a.est_base + (size_t)idx * kEstWidth : a.est_scratch;
    }
    return v;
}

template <int P, bool kObabo>
__global__ void __launch_bounds__(kIntThreads)
integrator_kernel(const __grid_constant__ IntegratorArgs a, const __grid_constant__ ModeConsts mc) {
    // dynamic smem: f, x and v~ tiles [P][kIntThreads], staged with cp.async in that order (all 3P loads of
    // a thread are in flight at once, independent of the register budget).  Every thread only ever touches
    // its own column, so no block-level synchronisation is needed and the thermostat normals can overlay
    // the f tile once f sits in registers.
    extern __shared__ double dyn_s[];
    double* fs = dyn_s + threadIdx.x;
    double* xs = fs + P * kIntThreads;
    double* vs = xs + P * kIntThreads;
    double* eta_s = fs;
    const int e = blockIdx.x * kIntThreads + threadIdx.x;
    const bool live = e < a.n_dof;
    const int ec = live ? e : a.n_dof - 1;             // dead threads shadow the last dof, never store
    const int i = ec / 3, alpha = ec - 3 * i;
    const bool start = (a.flags & I_START) != 0;
    const bool thermo = start && a.thermostat;
    const size_t stride = (size_t)a.n_dof;
    const StepView sv = resolve_step(a);

#pragma unroll
    for (int k = 0; k < P; ++k) __pipeline_memcpy_async(fs + k * kIntThreads, a.f + k * stride + ec, sizeof(double));
    __pipeline_commit();
#pragma unroll
    for (int k = 0; k < P; ++k) __pipeline_memcpy_async(xs + k * kIntThreads, a.x_in + k * stride + ec, sizeof(double));
    __pipeline_commit();
#pragma unroll
    for (int k = 0; k < P; ++k) __pipeline_memcpy_async(vs + k * kIntThreads, a.vt_in + k * stride + ec, sizeof(double));
    __pipeline_commit();

    // The block that will take this block's place on the SM (blockIdx.x + one wave) finds its inputs in L2: the ALU
    // phases of this kernel (O-step normals, transforms) and its memory phases do not overlap inside a block, and the
    // two blocks an SM holds drift into lockstep, so HBM would idle while both compute.  One prefetch per 128 B line.
    if ((threadIdx.x & 15) == 0) {
        const long long e2 = (long long)e + (long long)a.prefetch_ahead * kIntThreads;
        if (a.prefetch_ahead > 0 && e2 < (long long)a.n_dof) {
#pragma unroll 8
            for (int k = 0; k < P; ++k) {
                asm volatile("prefetch.global.L2 [%0];" ::"l"(a.f + k * stride + e2));
                asm volatile("prefetch.global.L2 [%0];" ::"l"(a.x_in + k * stride + e2));
                asm volatile("prefetch.global.L2 [%0];" ::"l"(a.vt_in + k * stride + e2));
            }
        }
    }

    const double m = a.mass[i];
    double xt[P], ft[P];
    __pipeline_wait_prior(2);
#pragma unroll
    for (int k = 0; k < P; ++k) ft[k] = fs[k * kIntThreads];

    // ---- O-step normals while x and v~ are still in flight: one draw per mode pair (R-10).  BAOAB: the O of
    //      the step this launch opens; OBABO: first the closing O(dt/2) of the previous step (its second half-step
    //      stream), the opening O's normals are generated between the two mode loops below ----
    auto gen_normals = [&](uint32_t s_lo, uint32_t s_hi) {
        if (a.flags & I_NOISE_PER_MODE) {
            // TIMING ONLY (pimd_time_kernel kind 1; DESIGN R-10's A/B number): the keying SURVEY C-7 first proposed,
            // one draw per mode, counter word 3 = 4k + alpha, sine branch discarded -- twice the Philox / log / sqrt /
            // sincospi work of the pair scheme the library (and the oracle) use.  Never reached by pimd_step.
#pragma unroll 4
            for (int k = 0; k < P; ++k) {
                double ee, eo;
                philox_normal_pair(a.seed_lo, a.seed_hi, s_lo, s_hi, (uint32_t)i, (uint32_t)(4 * k + alpha), &ee, &eo);
                eta_s[k * kIntThreads] = ee;
            }
            return;
        }
        if constexpr (P >= 8) {
            // W draws side by side (philox.cuh): the dependent chains of a draw interleave
            constexpr int W = kNoiseWide < P / 2 ? kNoiseWide : P / 2;
#pragma unroll 1
            for (int q = 0; q < P / 2; q += W) {
                double ee[W], eo[W];
                philox_normal_pairs<W>(a.seed_lo, a.seed_hi, s_lo, s_hi, (uint32_t)i, (uint32_t)(4 * q + alpha), ee, eo);
#pragma unroll
                for (int j = 0; j < W; ++j) {
                    eta_s[(2 * (q + j)) * kIntThreads] = ee[j];
                    eta_s[(2 * (q + j) + 1) * kIntThreads] = eo[j];
                }
            }
        } else {
#pragma unroll 4
            for (int q = 0; q < (P + 1) / 2; ++q) {
                double ee, eo;
                philox_normal_pair(a.seed_lo, a.seed_hi, s_lo, s_hi, (uint32_t)i, (uint32_t)(4 * q + alpha), &ee, &eo);
                eta_s[(2 * q) * kIntThreads] = ee;
                if (2 * q + 1 < P) eta_s[(2 * q + 1) * kIntThreads] = eo;
            }
        }
    };
    const bool thermo_close = kObabo && a.thermostat && (a.flags & I_BCLOSE);
    if (kObabo) {
        if (thermo_close) gen_normals(sv.cstep_lo, sv.cstep_hi);
    } else if (thermo) {
        gen_normals(sv.step_lo, sv.step_hi);
    }

    __pipeline_wait_prior(1);
    double xf = 0.0;
#pragma unroll
    for (int k = 0; k < P; ++k) xt[k] = xs[k * kIntThreads];
#pragma unroll
    for (int k = 0; k < P; ++k) xf += xt[k] * ft[k];
    nm_forward<P>(ft);                                  // f~ = M f      (L192, third transform)
    nm_forward<P>(xt);                                  // x~ = M x      (first transform)
    __pipeline_wait_prior(0);
    if (a.flags & I_COMSUB) vs[0] -= a.com[alpha] * a.inv_mtot;     // fixcom (L180, R-19): centroid COM velocity

    const double kick = a.half_dt_mvv / m;              // (dt/2)/(m mvv2e)
    const double sigma = sqrt(a.PkT_mvv / m);           // sqrt(P k_B T/(m mvv2e))  (Eq. D2)
    // A9 in normal-mode form: sum_k (r_k - r_c).F_k = sum_{k>=1} x~_k f~_k = sum_j x_j f_j - x~_0 f~_0
    const double cv_term = xf - xt[0] * ft[0];
    double accK = 0.0, accS = 0.0, v0c = 0.0;
    if constexpr (!kObabo) {
#pragma unroll
        for (int k = 0; k < P; ++k) {
            double v = vs[k * kIntThreads];
            if (a.flags & I_BCLOSE) v += kick * ft[k];      // closing B of the previous step
            if (k == 0) v0c = v;
            if (a.flags & I_EST) {
                accK += v * v;                               // A1: 1/2 m v~^2
                accS += mc.om2[k] * xt[k] * xt[k];           // A3: 1/2 m omega_k^2 x~^2
            }
            if (start) {
                v += kick * ft[k];                           // B(dt/2)
                const double x = xt[k];
                if (k == 0 && a.baro != nullptr) {
                    // BZP barostat (Eq. E4/E5, L507-512; R-21: centroid mode only): the two half drifts with the
                    // cell velocity before and after its own thermostat step (barostat.cu prepared the factors)
                    const double* bf = a.baro + BS_FAC + 6 * alpha;
                    const double xn = bf[0] * x + bf[1] * v;
                    double vn = bf[2] * v;
                    if (thermo) vn = mc.c1[k] * vn + mc.c2[k] * sigma * eta_s[k * kIntThreads];
                    xt[k] = bf[3] * xn + bf[4] * vn;
                    v = bf[5] * vn;
                } else {
                    const double xn = mc.cosA[k] * x + mc.sinA_w[k] * v;    // A(dt/2): exact rotation (R-5)
                    double vn = mc.msinA_w[k] * x + mc.cosA[k] * v;
                    if (thermo) vn = mc.c1[k] * vn + mc.c2[k] * sigma * eta_s[k * kIntThreads];   // O(dt)
                    xt[k] = mc.cosA[k] * xn + mc.sinA_w[k] * vn;            // A(dt/2)
                    v = mc.msinA_w[k] * xn + mc.cosA[k] * vn;
                }
            }
            if (live && (a.flags & (I_BCLOSE | I_START | I_COMSUB))) a.vt_out[k * stride + ec] = v;
        }
    } else {
        // OBABO: close the previous step with B(dt/2) O(dt/2), then estimators ...
#pragma unroll
        for (int k = 0; k < P; ++k) {
            double v = vs[k * kIntThreads];
            if (a.flags & I_BCLOSE) {
                v += kick * ft[k];
                if (thermo_close) v = mc.c1[k] * v + mc.c2[k] * sigma * eta_s[k * kIntThreads];
            }
            if (k == 0) v0c = v;
            if (a.flags & I_EST) {
                accK += v * v;
                accS += mc.om2[k] * xt[k] * xt[k];
            }
            vs[k * kIntThreads] = v;
        }
        // ... and open the next one with O(dt/2) B(dt/2) A(dt) (mc holds cos/sin for dt and c1, c2 for dt/2)
        if (thermo) gen_normals(sv.step_lo, sv.step_hi);
#pragma unroll
        for (int k = 0; k < P; ++k) {
            double v = vs[k * kIntThreads];
            if (start) {
                if (thermo) v = mc.c1[k] * v + mc.c2[k] * sigma * eta_s[k * kIntThreads];
                v += kick * ft[k];
                const double x = xt[k];
                if (k == 0 && a.baro != nullptr) {           // BZP barostat: Eq. E4/E5 over dt on the centroid mode
                    const double* bf = a.baro + BS_FAC + 6 * alpha;
                    xt[k] = bf[0] * x + bf[1] * v;
                    v = bf[2] * v;
                } else {
                    xt[k] = mc.cosA[k] * x + mc.sinA_w[k] * v;
                    v = mc.msinA_w[k] * x + mc.cosA[k] * v;
                }
            }
            if (live && (a.flags & (I_BCLOSE | I_START | I_COMSUB))) a.vt_out[k * stride + ec] = v;
        }
    }

    if (a.flags & I_COMACC) {                                // fixcom: sum_i m_i v~_0,i per component
        double c3[3];
#pragma unroll
        for (int c = 0; c < 3; ++c) c3[c] = (live && alpha == c) ? m * v0c : 0.0;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1)
#pragma unroll
            for (int c = 0; c < 3; ++c) c3[c] += __shfl_xor_sync(0xffffffffu, c3[c], o);
        if ((threadIdx.x & 31) == 0)
#pragma unroll
            for (int c = 0; c < 3; ++c) atomicAdd(a.com + c, c3[c]);
    }

    if (a.flags & I_EST) {
        double r0 = live ? 0.5 * m * accK * kMvv2e : 0.0;     // K_ring share
        double r1 = live ? 0.5 * m * accS * kMvv2e : 0.0;     // S_ring share
        double r2 = live ? cv_term : 0.0;
        __shared__ double red[3][kIntThreads / 32];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            r0 += __shfl_xor_sync(0xffffffffu, r0, o);
            r1 += __shfl_xor_sync(0xffffffffu, r1, o);
            r2 += __shfl_xor_sync(0xffffffffu, r2, o);
        }
        const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
        if (l == 0) { red[0][w] = r0; red[1][w] = r1; red[2][w] = r2; }
        __syncthreads();
        if (threadIdx.x < 3) {
            double t = 0.0;
#pragma unroll
            for (int q = 0; q < kIntThreads / 32; ++q) t += red[threadIdx.x][q];
            atomicAdd(sv.est + threadIdx.x, t);
        }
        if (blockIdx.x == 0 && threadIdx.x == 3 && a.U != nullptr) {
            double u = 0.0;
            for (int k = 0; k < P; ++k) u += a.U[k];
            atomicAdd(sv.est + 3, u);
        }
    }

    if (start) {
        nm_inverse<P>(xt);                              // x = M^T x~    (second transform)
        if (live) {
#pragma unroll
            for (int k = 0; k < P; ++k) a.x_out[k * stride + ec] = xt[k];
        }
    }
}

template <int P>
static void launch_int_t(const IntegratorArgs& a, const ModeConsts& mc, cudaStream_t s) {
    const int blocks = (a.n_dof + kIntThreads - 1) / kIntThreads;
    const size_t smem = (size_t)3 * P * kIntThreads * sizeof(double);
    ensure_dyn_smem(integrator_kernel<P, false>, (int)smem);
    ensure_dyn_smem(integrator_kernel<P, true>, (int)smem);
    if (a.flags & I_OBABO) integrator_kernel<P, true><<<blocks, kIntThreads, smem, s>>>(a, mc);
    else integrator_kernel<P, false><<<blocks, kIntThreads, smem, s>>>(a, mc);
}

// ---------------------------------------------------------------------------------------------
// `method pimd` (Eq. D3; DESIGN R-27): the same fused launch in Cartesian coordinates.
// No transforms: v is the Cartesian bead velocity, B kicks with the bead force plus the ring-spring force
// -m omega_n^2 (2 x_k - x_{k-1} - x_{k+1}) (Eq. 1), A is the drift x += h v, O is Eq. D3 with the same
// c1 = exp(-l 2 omega_n) on every bead (mc.c1[0], mc.c2[0]; mc.sinA_w[0] = the drift length).  Not the headline
// path: plain coalesced loads, the normals of all beads staged in shared memory.
// ---------------------------------------------------------------------------------------------
template <int P, bool kObabo>
__global__ void __launch_bounds__(kIntThreads)
integrator_cart_kernel(const __grid_constant__ IntegratorArgs a, const __grid_constant__ ModeConsts mc) {
    extern __shared__ double dyn_s[];
    double* eta_s = dyn_s + threadIdx.x;
    const int e = blockIdx.x * kIntThreads + threadIdx.x;
    const bool live = e < a.n_dof;
    const int ec = live ? e : a.n_dof - 1;
    const int i = ec / 3, alpha = ec - 3 * i;
    const bool start = (a.flags & I_START) != 0;
    const bool close = (a.flags & I_BCLOSE) != 0;
    const bool thermo = start && a.thermostat;
    const size_t stride = (size_t)a.n_dof;
    const StepView sv = resolve_step(a);
    const double m = a.mass[i];
    double x[P], v[P], g[P];             // g: total acceleration-kick h (f + f_spring)/(m mvv2e)
#pragma unroll
    for (int k = 0; k < P; ++k) { x[k] = a.x_in[k * stride + ec]; v[k] = a.vt_in[k * stride + ec]; g[k] = a.f[k * stride + ec]; }
    auto gen_normals = [&](uint32_t s_lo, uint32_t s_hi) {
#pragma unroll 4
        for (int q = 0; q < (P + 1) / 2; ++q) {
            double ee, eo;
            philox_normal_pair(a.seed_lo, a.seed_hi, s_lo, s_hi, (uint32_t)i, (uint32_t)(4 * q + alpha), &ee, &eo);
            eta_s[(2 * q) * kIntThreads] = ee;
            if (2 * q + 1 < P) eta_s[(2 * q + 1) * kIntThreads] = eo;
        }
    };
    const double kick = a.half_dt_mvv / m;
    const double hh = a.half_dt_mvv * kMvv2e;          // dt/2
    const double sigma = sqrt(a.PkT_mvv / m);
    double sx = 0.0, sf = 0.0, xf = 0.0, accS = 0.0;
#pragma unroll
    for (int k = 0; k < P; ++k) { sx += x[k]; sf += g[k]; xf += x[k] * g[k]; }
#pragma unroll
    for (int k = 0; k < P; ++k) {
        const double dr = x[k] - x[(k + 1) % P];
        accS += dr * dr;                                 // A3 in Cartesian form: 1/2 m omega_n^2 |r_k - r_{k+1}|^2
    }
#pragma unroll
    for (int k = 0; k < P; ++k) {
        const double lap = (P == 1) ? 0.0 : 2.0 * x[k] - x[(k + P - 1) % P] - x[(k + 1) % P];
        g[k] = kick * g[k] - hh * a.wP2 * lap;
    }
    const double cv_term = xf - (sx / (double)P) * sf;   // A9: sum_k (r_k - r_c).F_k
    if (a.flags & I_COMSUB) {                            // fixcom, "for each bead individually"
#pragma unroll
        for (int k = 0; k < P; ++k) v[k] -= a.com[3 * k + alpha] * a.inv_mtot;
    }
    if (close) {
#pragma unroll
        for (int k = 0; k < P; ++k) v[k] += g[k];        // closing B(dt/2)
        if (kObabo && a.thermostat) {                    // closing O(dt/2), second half-step stream
            gen_normals(sv.cstep_lo, sv.cstep_hi);
#pragma unroll
            for (int k = 0; k < P; ++k) v[k] = mc.c1[0] * v[k] + mc.c2[0] * sigma * eta_s[k * kIntThreads];
        }
    }
    if (a.flags & I_COMACC) {                            // sum_i m_i v_k,i per bead and component -> com[3k + alpha]
        __shared__ double s_com[3 * P];
        for (int q = threadIdx.x; q < 3 * P; q += kIntThreads) s_com[q] = 0.0;
        __syncthreads();
        if (live) {
#pragma unroll
            for (int k = 0; k < P; ++k) atomicAdd(&s_com[3 * k + alpha], m * v[k]);
        }
        __syncthreads();
        for (int q = threadIdx.x; q < 3 * P; q += kIntThreads) atomicAdd(a.com + q, s_com[q]);
    }
    double accK = 0.0;
#pragma unroll
    for (int k = 0; k < P; ++k) accK += v[k] * v[k];
    if (start) {
        const double hd = mc.sinA_w[0];                  // drift length: dt/2 (BAOAB), dt (OBABO)
        if (thermo) gen_normals(sv.step_lo, sv.step_hi);
        if (kObabo) {
#pragma unroll
            for (int k = 0; k < P; ++k) {
                if (thermo) v[k] = mc.c1[0] * v[k] + mc.c2[0] * sigma * eta_s[k * kIntThreads];
                v[k] += g[k];
                x[k] += hd * v[k];
            }
        } else {
#pragma unroll
            for (int k = 0; k < P; ++k) {
                v[k] += g[k];
                x[k] += hd * v[k];
                if (thermo) v[k] = mc.c1[0] * v[k] + mc.c2[0] * sigma * eta_s[k * kIntThreads];
                x[k] += hd * v[k];
            }
        }
    }
    if (live && (close || start || (a.flags & I_COMSUB))) {
#pragma unroll
        for (int k = 0; k < P; ++k) a.vt_out[k * stride + ec] = v[k];
    }
    if (live && start) {
#pragma unroll
        for (int k = 0; k < P; ++k) a.x_out[k * stride + ec] = x[k];
    }
    if (a.flags & I_EST) {
        double r0 = live ? 0.5 * m * accK * kMvv2e : 0.0;
        double r1 = live ? 0.5 * m * a.wP2 * accS * kMvv2e : 0.0;
        double r2 = live ? cv_term : 0.0;
        __shared__ double red[3][kIntThreads / 32];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            r0 += __shfl_xor_sync(0xffffffffu, r0, o);
            r1 += __shfl_xor_sync(0xffffffffu, r1, o);
            r2 += __shfl_xor_sync(0xffffffffu, r2, o);
        }
        const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
        if (l == 0) { red[0][w] = r0; red[1][w] = r1; red[2][w] = r2; }
        __syncthreads();
        if (threadIdx.x < 3) {
            double t = 0.0;
#pragma unroll
            for (int q = 0; q < kIntThreads / 32; ++q) t += red[threadIdx.x][q];
            atomicAdd(sv.est + threadIdx.x, t);
        }
        if (blockIdx.x == 0 && threadIdx.x == 3 && a.U != nullptr) {
            double u = 0.0;
            for (int k = 0; k < P; ++k) u += a.U[k];
            atomicAdd(sv.est + 3, u);
        }
    }
}

template <int P>
static void launch_cart_t(const IntegratorArgs& a, const ModeConsts& mc, cudaStream_t s) {
    const int blocks = (a.n_dof + kIntThreads - 1) / kIntThreads;
    const size_t smem = (size_t)P * kIntThreads * sizeof(double);
    ensure_dyn_smem(integrator_cart_kernel<P, false>, (int)smem);
    ensure_dyn_smem(integrator_cart_kernel<P, true>, (int)smem);
    if (a.flags & I_OBABO) integrator_cart_kernel<P, true><<<blocks, kIntThreads, smem, s>>>(a, mc);
    else integrator_cart_kernel<P, false><<<blocks, kIntThreads, smem, s>>>(a, mc);
}

// v = p/m and p = m v per bead (the Cartesian method keeps v as it crosses the API)
__global__ void cart_convert_kernel(size_t n, int n_dof, const double* __restrict__ in, const double* __restrict__ mass,
                                    double* __restrict__ out, int forward) {
    const size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= n) return;
    const double m = mass[(t % n_dof) / 3];
    out[t] = forward ? in[t] / m : in[t] * m;
}
int launch_cart_convert(int P, int N, const double* in, const double* mass, double* out, int forward, cudaStream_t s) {
    const size_t n = (size_t)P * N * 3;
    cart_convert_kernel<<<(unsigned)((n + 255) / 256), 256, 0, s>>>(n, 3 * N, in, mass, out, forward);
    return 1;
}

int launch_integrator(int P, const IntegratorArgs& a, const ModeConsts& mc, cudaStream_t s) {
    // north_star's layout -- four lanes per atom-dimension, shuffles for the transforms (integrator4.cu) -- is parity-correct
    // but FP64-bound at twice this kernel's time; it runs only on request: PIMD_INT4=1
    if (P >= 16 && getenv("PIMD_INT4") != nullptr && launch_integrator4(P, a, mc, s)) return 1;
    if (a.flags & I_CART) {
        switch (P) {
            case 1: launch_cart_t<1>(a, mc, s); break;
            case 2: launch_cart_t<2>(a, mc, s); break;
            case 4: launch_cart_t<4>(a, mc, s); break;
            case 8: launch_cart_t<8>(a, mc, s); break;
            case 16: launch_cart_t<16>(a, mc, s); break;
            case 32: launch_cart_t<32>(a, mc, s); break;
            case 64: launch_cart_t<64>(a, mc, s); break;
            default: return 0;
        }
        return 1;
    }
    switch (P) {
        case 1: launch_int_t<1>(a, mc, s); break;
        case 2: launch_int_t<2>(a, mc, s); break;
        case 4: launch_int_t<4>(a, mc, s); break;
        case 8: launch_int_t<8>(a, mc, s); break;
        case 16: launch_int_t<16>(a, mc, s); break;
        case 32: launch_int_t<32>(a, mc, s); break;
        case 64: launch_int_t<64>(a, mc, s); break;
        default: return 0;
    }
    return 1;
}

// v~ = M (p/m)  and  p = m M^T v~  (API momenta are Cartesian; PAPER.md:L104 keeps v in NM form inside)
template <int P, bool kForward>
__global__ void nm_convert_kernel(int n_dof, const double* __restrict__ in, const double* __restrict__ mass,
                                  double* __restrict__ out) {
    const int e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= n_dof) return;
    const double m = mass[e / 3];
    double a[P];
#pragma unroll
    for (int k = 0; k < P; ++k) a[k] = in[(size_t)k * n_dof + e];
    if constexpr (kForward) {
#pragma unroll
        for (int k = 0; k < P; ++k) a[k] = a[k] / m;
        nm_forward<P>(a);
    } else {
        nm_inverse<P>(a);
#pragma unroll
        for (int k = 0; k < P; ++k) a[k] = a[k] * m;
    }
#pragma unroll
    for (int k = 0; k < P; ++k) out[(size_t)k * n_dof + e] = a[k];
}

template <bool kForward>
static void launch_conv(int P, int N, const double* in, const double* mass, double* out, cudaStream_t s) {
    const int n_dof = 3 * N, th = 128, bl = (n_dof + th - 1) / th;
    switch (P) {
        case 1: nm_convert_kernel<1, kForward><<<bl, th, 0, s>>>(n_dof, in, mass, out); break;
        case 2: nm_convert_kernel<2, kForward><<<bl, th, 0, s>>>(n_dof, in, mass, out); break;
        case 4: nm_convert_kernel<4, kForward><<<bl, th, 0, s>>>(n_dof, in, mass, out); break;
        case 8: nm_convert_kernel<8, kForward><<<bl, th, 0, s>>>(n_dof, in, mass, out); break;
        case 16: nm_convert_kernel<16, kForward><<<bl, th, 0, s>>>(n_dof, in, mass, out); break;
        case 32: nm_convert_kernel<32, kForward><<<bl, th, 0, s>>>(n_dof, in, mass, out); break;
        case 64: nm_convert_kernel<64, kForward><<<bl, th, 0, s>>>(n_dof, in, mass, out); break;
        default: break;
    }
}
int launch_to_nm_velocity(int P, int N, const double* p, const double* mass, double* vt, cudaStream_t s) {
    launch_conv<true>(P, N, p, mass, vt, s);
    return 1;
}
int launch_from_nm_momenta(int P, int N, const double* vt, const double* mass, double* p, cudaStream_t s) {
    launch_conv<false>(P, N, vt, mass, p, s);
    return 1;
}

// Test model U = sum_i 1/2 k |r_i|^2 (FP64): f = -k x, U^(k), Xi_ab = sum_i x_a f_b.
__global__ void harmonic_kernel(int N, double ks, const double* __restrict__ x, double* __restrict__ f,
                                double* __restrict__ U, double* __restrict__ Xi, double* __restrict__ Eatom) {
    const int k = blockIdx.y;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    double acc[10];
#pragma unroll
    for (int q = 0; q < 10; ++q) acc[q] = 0.0;
    if (i < N) {
        const size_t o = ((size_t)k * N + i) * 3;
        const double r[3] = {x[o], x[o + 1], x[o + 2]};
        double fr[3];
#pragma unroll
        for (int c = 0; c < 3; ++c) { fr[c] = -ks * r[c]; f[o + c] = fr[c]; }
        acc[9] = 0.5 * ks * (r[0] * r[0] + r[1] * r[1] + r[2] * r[2]);
        Eatom[(size_t)k * N + i] = acc[9];
#pragma unroll
        for (int c = 0; c < 3; ++c)
#pragma unroll
            for (int d = 0; d < 3; ++d) acc[3 * c + d] = r[c] * fr[d];
    }
#pragma unroll
    for (int q = 0; q < 10; ++q)
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) acc[q] += __shfl_xor_sync(0xffffffffu, acc[q], o);
    if ((threadIdx.x & 31) == 0) {
#pragma unroll
        for (int q = 0; q < 9; ++q) atomicAdd(Xi + k * 9 + q, acc[q]);
        atomicAdd(U + k, acc[9]);
    }
}

int launch_harmonic(int P, int N, double ks, const double* x, double* f, double* U, double* Xi, double* Eatom,
                     cudaStream_t s) {
    cudaMemsetAsync(U, 0, sizeof(double) * P, s);
    cudaMemsetAsync(Xi, 0, sizeof(double) * 9 * P, s);
    dim3 grid((N + 127) / 128, P);
    harmonic_kernel<<<grid, 128, 0, s>>>(N, ks, x, f, U, Xi, Eatom);
    return 1;
}

__global__ void debug_noise_kernel(uint32_t seed_lo, uint32_t seed_hi, uint32_t step_lo, uint32_t step_hi, int n,
                                   const int32_t* __restrict__ idx, uint32_t* __restrict__ words,
                                   double* __restrict__ eta) {
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= n) return;
    const uint32_t k = idx[3 * t], i = idx[3 * t + 1], al = idx[3 * t + 2];
    uint32_t w[4];
    philox4x32_10(step_lo, step_hi, i, 4u * (k >> 1) + al, seed_lo, seed_hi, w);
    for (int q = 0; q < 4; ++q) words[4 * t + q] = w[q];
    // both generators of the library: the four-wide branch-free one (integrator kernels, P >= 8) for even entries of the
    // request, the libm-based one (P < 8, barostat) for odd entries
    double ee, eo;
    if (t & 1) {
        philox_normal_pair(seed_lo, seed_hi, step_lo, step_hi, i, 4u * (k >> 1) + al, &ee, &eo);
    } else {
        double e4[4], o4[4];
        philox_normal_pairs4(seed_lo, seed_hi, step_lo, step_hi, i, 4u * (k >> 1) + al, e4, o4);
        ee = e4[0]; eo = o4[0];
    }
    eta[t] = (k & 1u) ? eo : ee;
}

int launch_debug_noise(uint64_t seed, uint64_t step, int n, const int32_t* idx, uint32_t* words, double* eta,
                        cudaStream_t s) {
    debug_noise_kernel<<<(n + 127) / 128, 128, 0, s>>>((uint32_t)seed, (uint32_t)(seed >> 32), (uint32_t)step,
                                                        (uint32_t)(step >> 32), n, idx, words, eta);
    return 1;
}

}  // namespace pimd
