// barostat.cu -- isotropic BZP barostat (Appendix E Eq. E1, E4-E7,
// Appendix A Eq. A12), readings DESIGN R-20 .. R-25.
//
// The cell has ONE degree of freedom, so everything the barostat does between two force evaluations is a
// function of five sums over the atoms taken right after the forces arrive (v~ still before the closing kick):
//   S_kin = sum_i m_i v~_i^(0)2         S_fv = sum_i F~_i^(0).v~_i^(0)       S_ff = sum_i |F~_i^(0)|^2 / m_i
//   S_cv  = sum_k sum_i (r_i^(k) - r_i^c).F_i^(k)                             Tr = sum_k Tr Xi^(k)
// baro_sums_kernel takes them (one thread per atom-dimension, all beads of it, like the integrator; block partials,
// no atomics);
// baro_update_kernel (one warp) then plays, in order, the closing E1(dt/2) of the step that ends, the B(dt/2) kick's
// effect on S_kin and S_fv (exact: the kick is v~ += h F~/m), the opening E1(dt/2) of the next step, the first
// E4-E6 half drift, E7, the second half drift -- leaving exp(+-h v_W) and sinh(h v_W)/v_W of both half drifts
// for the integrator kernel, which applies E4/E5 to the centroid mode in registers, and the new cell for the
// neighbour kernels.  The host never sees v_W or the cell inside a pimd_step call.
#include "common.cuh"
#include "philox.cuh"

namespace pimd {

constexpr int kBaroThreads = 128;

__global__ void __launch_bounds__(kBaroThreads)
baro_sums_kernel(const __grid_constant__ BaroArgs a) {
    const int e = blockIdx.x * kBaroThreads + threadIdx.x;
    double r[kBaroSums] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
    if (e < a.n_dof) {
        const size_t stride = (size_t)a.n_dof;
        const double m = a.mass[e / 3];
        double sx = 0.0, sf = 0.0, xf = 0.0;
        for (int k = 0; k < a.P; ++k) {
            const double xv = a.x[k * stride + e], fv = a.f[k * stride + e];
            sx += xv; sf += fv; xf += xv * fv;
        }
        const double inv_sqrtP = rsqrt((double)a.P);
        const double f0 = sf * inv_sqrtP;               // F~^(0) = sum_k F^(k) / sqrt(n)   (Eq. B1 row 0)
        const double v0 = a.vt[e];                      // v~^(0)
        r[0] = m * v0 * v0 * kMvv2e;                    // A12 first term
        r[1] = xf - (sx / (double)a.P) * sf;            // sum_k (r_k - r_c) F_k
        r[2] = f0 * v0;                                 // E1 third term
        r[3] = f0 * f0 / (m * kMvv2e);                  // E1 fourth term
        if (a.obabo) {
            // OBABO puts the centroid's thermostat between the closing and the opening E1, so the velocity sums of the
            // opening E1 are not a function of the closing ones: replay kick and O steps of the centroid mode here
            // (the normals are counter-based: the same ones the integrator kernel draws for mode 0)
            const int i = e / 3, alpha = e - 3 * i;
            const double sigma = sqrt(a.PkT_mvv / m);
            double v = v0, ee, eo;
            if (a.close) {
                v += (a.half_dt_mvv / m) * f0;
                if (a.thermostat) {
                    philox_normal_pair(a.seed_lo, a.seed_hi, a.cstep_lo, a.cstep_hi, (uint32_t)i, (uint32_t)alpha, &ee, &eo);
                    v = a.c1 * v + a.c2 * sigma * ee;
                }
            }
            r[4] = m * v * v * kMvv2e;                  // what the estimators' P_CV sees
            if (a.start && a.thermostat) {
                philox_normal_pair(a.seed_lo, a.seed_hi, a.step_lo, a.step_hi, (uint32_t)i, (uint32_t)alpha, &ee, &eo);
                v = a.c1 * v + a.c2 * sigma * ee;
            }
            r[5] = m * v * v * kMvv2e;
            r[6] = f0 * v;
        }
    }
    __shared__ double red[kBaroSums][kBaroThreads / 32];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1)
#pragma unroll
        for (int q = 0; q < kBaroSums; ++q) r[q] += __shfl_xor_sync(0xffffffffu, r[q], o);
    const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
    if (l == 0)
#pragma unroll
        for (int q = 0; q < kBaroSums; ++q) red[q][w] = r[q];
    __syncthreads();
    if (threadIdx.x < kBaroSums) {
        double t = 0.0;
#pragma unroll
        for (int q = 0; q < kBaroThreads / 32; ++q) t += red[threadIdx.x][q];
        a.partial[kBaroSums * blockIdx.x + threadIdx.x] = t;    // no atomics: the sums steer the dynamics, keep them reproducible
    }
}

// (e^{a} - e^{-a}) / (2 v_W) with a = h v_W, and its limit h (R-22: series below |a| = 1e-4)
__device__ __forceinline__ double sinh_over(double vW, double h) {
    const double x = h * vW;
    if (fabs(x) < 1e-4) return h * (1.0 + x * x / 6.0 + x * x * x * x / 120.0);
    return (exp(x) - exp(-x)) / (2.0 * vW);
}

__global__ void baro_update_kernel(const __grid_constant__ BaroArgs a) {
    // the block partials of the four sums, in a fixed order: lane-strided, then a shuffle tree
    double sum4[kBaroSums] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
    const int nblk = (a.n_dof + kBaroThreads - 1) / kBaroThreads;
    for (int b = threadIdx.x; b < nblk; b += 32)
#pragma unroll
        for (int q = 0; q < kBaroSums; ++q) sum4[q] += a.partial[kBaroSums * b + q];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1)
#pragma unroll
        for (int q = 0; q < kBaroSums; ++q) sum4[q] += __shfl_xor_sync(0xffffffffu, sum4[q], o);
    if (threadIdx.x != 0) return;
    double* st = a.state;
    double vW = st[BS_VW];
    double L[3] = {st[BS_LX], st[BS_LY], st[BS_LZ]};
    double Skin = sum4[0], Sfv = sum4[2];
    const double Scv = sum4[1], Sff = sum4[3];
    st[BS_SKIN] = sum4[0]; st[BS_SCV] = sum4[1]; st[BS_SFV] = sum4[2]; st[BS_SFF] = sum4[3];
    double tr = 0.0;
    for (int k = 0; k < a.P; ++k) tr += a.Xi[9 * k] + a.Xi[9 * k + 4] + a.Xi[9 * k + 8];
    const double V = L[0] * L[1] * L[2];
    const double h = a.h, nP = (double)a.P;
    auto press_v = [&]() {      // Eq. E1 over h; 3 n V P_CV = S_kin - S_cv + Tr (A12)
        const double pcv = (Skin - Scv + tr) / (3.0 * nP * V);
        vW = vW + (3.0 * h / a.W) * (nP * V * (pcv - a.p_ext) + a.nkT);
        vW = vW + (h * h / a.W) * Sfv;
        vW = vW + (h * h * h / (3.0 * a.W)) * Sff;
    };
    auto b_kick = [&]() {       // what B(h), v~0 += h F~0/m, does to the two velocity sums
        Skin = Skin + 2.0 * h * Sfv + h * h * Sff;
        Sfv = Sfv + h * Sff;
    };
    auto press_o = [&](uint32_t s_lo, uint32_t s_hi) {      // E7 (R-23), eta keyed (mode 0, atom N, dim 0)
        double ee, eo;
        philox_normal_pair(a.seed_lo, a.seed_hi, s_lo, s_hi, (uint32_t)a.N, 0u, &ee, &eo);
        vW = a.c1 * vW + a.c2sig * ee;
    };
    if (a.obabo) {
        // [E1, B](h) [O, E7](h) | [O, E7](h) [E1, B](h) [E4-E6 + A](dt)      (R-24)
        if (a.close) {
            press_v();
            if (a.thermostat) press_o(a.cstep_lo, a.cstep_hi);
        }
        st[BS_PCV] = (sum4[4] - Scv + tr) / (3.0 * nP * V);
        st[BS_TRXI] = tr;
        if (a.start) {
            if (a.thermostat) press_o(a.step_lo, a.step_hi);
            Skin = sum4[5]; Sfv = sum4[6];
            press_v();
            const double dt = 2.0 * h, e1 = exp(dt * vW);
            st[BS_EA1] = e1; st[BS_SH1] = sinh_over(vW, dt); st[BS_EM1] = exp(-dt * vW);
            st[BS_EA2] = 1.0; st[BS_SH2] = 0.0; st[BS_EM2] = 1.0;
            st[BS_LX] = L[0] * e1; st[BS_LY] = L[1] * e1; st[BS_LZ] = L[2] * e1;
        }
        st[BS_VW] = vW;
        return;
    }
    if (a.close) { press_v(); b_kick(); }
    st[BS_PCV] = (Skin - Scv + tr) / (3.0 * nP * V);       // A12 of the state the estimators see
    st[BS_TRXI] = tr;
    if (a.start) {
        press_v();
        const double e1 = exp(h * vW);
        st[BS_EA1] = e1; st[BS_SH1] = sinh_over(vW, h); st[BS_EM1] = exp(-h * vW);
        for (int c = 0; c < 3; ++c) L[c] *= e1;             // E6
        if (a.thermostat) press_o(a.step_lo, a.step_hi);    // E7 over dt
        const double e2 = exp(h * vW);
        st[BS_EA2] = e2; st[BS_SH2] = sinh_over(vW, h); st[BS_EM2] = exp(-h * vW);
        for (int c = 0; c < 3; ++c) L[c] *= e2;
        st[BS_LX] = L[0]; st[BS_LY] = L[1]; st[BS_LZ] = L[2];
    }
    st[BS_VW] = vW;
}

int launch_barostat(const BaroArgs& a, cudaStream_t s) {
    baro_sums_kernel<<<(a.n_dof + kBaroThreads - 1) / kBaroThreads, kBaroThreads, 0, s>>>(a);
    baro_update_kernel<<<1, 32, 0, s>>>(a);
    return 2;
}

size_t barostat_state_doubles(int n_dof) { return (size_t)BS_WIDTH + kBaroSums * (size_t)((n_dof + kBaroThreads - 1) / kBaroThreads); }

}  // namespace pimd
