// barostat.cu -- BZP barostat, isotropic and anisotropic (Appendix E
// Eq. E1-E7, Appendix A Eq. A12-A14), readings DESIGN R-20 .. R-25.
//
// The cell has one (iso) or three (aniso) degrees of freedom, so everything the barostat does between two force
// evaluations is a function of a few sums over the atoms, per Cartesian component a, taken right after the forces
// arrive (v~ still before the closing kick):
//   S_kin_a = sum_i m_i v~0_ia^2      S_fv_a = sum_i F~0_ia v~0_ia      S_ff_a = sum_i F~0_ia^2 / m_i
//   S_cv_a  = sum_k sum_i (r_ia^(k) - r_ia^c) F_ia^(k)                   Xi_aa = sum_k Xi_aa^(k)
// baro_sums_kernel takes them (one thread per atom-dimension, all beads of it, like the integrator; block partials,
// no atomics); baro_update_kernel (one warp) then plays, in order, the closing E1/E2(dt/2) of the step that ends,
// the B(dt/2) kick's effect on S_kin and S_fv (exact: the kick is v~ += h F~/m), the opening E1/E2(dt/2) of the next
// step, the first E4-E6 half drift, E7, the second half drift -- leaving exp(+-h v_W) and sinh(h v_W)/v_W of both
// half drifts, per component, for the integrator kernel, which applies E4/E5 to the centroid mode in registers, and
// the new cell for the neighbour kernels.  The host never sees v_W or the cell inside a pimd_step call.
// Isotropic mode sums the components (E1 = the trace of E2 with W three times larger) and keeps the three v_W equal.
#include "common.cuh"
#include "philox.cuh"

namespace pimd {

constexpr int kBaroThreads = 128;
constexpr int kBaroPart = 3 * kBaroSums;       // per block: [component][sum]

__global__ void __launch_bounds__(kBaroThreads)
baro_sums_kernel(const __grid_constant__ BaroArgs a) {
    const int e = blockIdx.x * kBaroThreads + threadIdx.x;
    double r[kBaroSums] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
    int alpha = 0;
    if (e < a.n_dof) {
        const size_t stride = (size_t)a.n_dof;
        const int i = e / 3;
        alpha = e - 3 * i;
        const double m = a.mass[i];
        double sx = 0.0, sf = 0.0, xf = 0.0;
        for (int k = 0; k < a.P; ++k) {
            const double xv = a.x[k * stride + e], fv = a.f[k * stride + e];
            sx += xv; sf += fv; xf += xv * fv;
        }
        const double inv_sqrtP = rsqrt((double)a.P);
        const double f0 = sf * inv_sqrtP;               // F~^(0) = sum_k F^(k) / sqrt(n)   (Eq. B1 row 0)
        const double v0 = a.vt[e];                      // v~^(0)
        r[0] = m * v0 * v0 * kMvv2e;                    // A12 / E3 first term
        r[1] = xf - (sx / (double)a.P) * sf;            // sum_k (r_k - r_c) F_k
        r[2] = f0 * v0;                                 // E1 / E2 third term
        r[3] = f0 * f0 / (m * kMvv2e);                  // E1 / E2 fourth term
        if (a.obabo) {
            // OBABO puts the centroid's thermostat between the closing and the opening E1, so the velocity sums of the
            // opening E1 are not a function of the closing ones: replay kick and O steps of the centroid mode here
            // (the normals are counter-based: the same ones the integrator kernel draws for mode 0)
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
    // per-component block sums: every lane contributes to its own component only
    __shared__ double red[3][kBaroSums][kBaroThreads / 32];
    const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
#pragma unroll
        for (int q = 0; q < kBaroSums; ++q) {
            double t = (alpha == c) ? r[q] : 0.0;
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
            if (l == 0) red[c][q][w] = t;
        }
    }
    __syncthreads();
    if (threadIdx.x < kBaroPart) {
        const int c = threadIdx.x / kBaroSums, q = threadIdx.x - c * kBaroSums;
        double t = 0.0;
#pragma unroll
        for (int g = 0; g < kBaroThreads / 32; ++g) t += red[c][q][g];
        a.partial[kBaroPart * blockIdx.x + threadIdx.x] = t;    // no atomics: the sums steer the dynamics, keep them reproducible
    }
}

// (e^{a} - e^{-a}) / (2 v_W) with a = h v_W, and its limit h (R-22: series below |a| = 1e-4)
__device__ __forceinline__ double sinh_over(double vW, double h) {
    const double x = h * vW;
    if (fabs(x) < 1e-4) return h * (1.0 + x * x / 6.0 + x * x * x * x / 120.0);
    return (exp(x) - exp(-x)) / (2.0 * vW);
}

__global__ void baro_update_kernel(const __grid_constant__ BaroArgs a) {
    // the block partials, in a fixed order: lane-strided, then a shuffle tree
    double S[3][kBaroSums];
    const int nblk = (a.n_dof + kBaroThreads - 1) / kBaroThreads;
#pragma unroll
    for (int c = 0; c < 3; ++c)
#pragma unroll
        for (int q = 0; q < kBaroSums; ++q) S[c][q] = 0.0;
    for (int b = threadIdx.x; b < nblk; b += 32) {          // a block's 21 partials are contiguous: independent loads
#pragma unroll
        for (int c = 0; c < 3; ++c)
#pragma unroll
            for (int q = 0; q < kBaroSums; ++q) S[c][q] += a.partial[kBaroPart * b + c * kBaroSums + q];
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1)
#pragma unroll
        for (int c = 0; c < 3; ++c)
#pragma unroll
            for (int q = 0; q < kBaroSums; ++q) S[c][q] += __shfl_xor_sync(0xffffffffu, S[c][q], o);
    double tr[3] = {0.0, 0.0, 0.0};
    for (int k = threadIdx.x; k < a.P; k += 32) { tr[0] += a.Xi[9 * k]; tr[1] += a.Xi[9 * k + 4]; tr[2] += a.Xi[9 * k + 8]; }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1)
#pragma unroll
        for (int c = 0; c < 3; ++c) tr[c] += __shfl_xor_sync(0xffffffffu, tr[c], o);
    if (threadIdx.x != 0) return;
    double* st = a.state;
    const double L[3] = {st[BS_LX], st[BS_LY], st[BS_LZ]};
    const double V = L[0] * L[1] * L[2];
    const double h = a.h, nP = (double)a.P;
    st[BS_TRXI] = tr[0] + tr[1] + tr[2];
    // diagonal of the centroid-virial stress (E3) of the state the estimators see: after the closing kick (and O)
    for (int c = 0; c < 3; ++c) {
        const double sk = a.obabo ? S[c][4] : (a.close ? S[c][0] + 2.0 * h * S[c][2] + h * h * S[c][3] : S[c][0]);
        st[BS_PCV + c] = (sk - S[c][1] + tr[c]) / (nP * V);
    }
    // isotropic: one cell velocity driven by the summed components (E1); anisotropic: one per component (E2)
    const int nd = a.aniso ? 3 : 1;
    if (!a.aniso) {
#pragma unroll
        for (int q = 0; q < kBaroSums; ++q) S[0][q] = S[0][q] + S[1][q] + S[2][q];
        tr[0] = tr[0] + tr[1] + tr[2];
    }
    if (a.est_slot != nullptr) {                // per-step record: the cell and the stress the estimators of this step see
        for (int c = 0; c < 3; ++c) { a.est_slot[kEstBaro + 3 + c] = L[c]; a.est_slot[kEstBaro + 6 + c] = st[BS_PCV + c]; }
        a.est_slot[kEstBaro + 9] = st[BS_TRXI];
    }
    const double dim = a.aniso ? 1.0 : 3.0;     // E1: 3 dt/W [..] with P_CV = trace/3;  E2: dt/W [..] with P_CV^aa
    for (int d = 0; d < nd; ++d) {
        double vW = st[BS_VW + d];
        double Skin = S[d][0], Sfv = S[d][2];
        const double Scv = S[d][1], Sff = S[d][3];
        auto press_v = [&]() {      // Eq. E1 / E2 over h; dim n V P_CV = S_kin - S_cv + Xi (A12 / E3)
            const double pcv = (Skin - Scv + tr[d]) / (dim * nP * V);
            vW = vW + (dim * h / a.W) * (nP * V * (pcv - a.p_ext) + a.nkT);
            vW = vW + (h * h / a.W) * Sfv;
            vW = vW + (h * h * h / (3.0 * a.W)) * Sff;
        };
        auto press_o = [&](uint32_t s_lo, uint32_t s_hi) {      // E7 (R-23), eta keyed (mode 0, atom N, dim d)
            double ee, eo;
            philox_normal_pair(a.seed_lo, a.seed_hi, s_lo, s_hi, (uint32_t)a.N, (uint32_t)d, &ee, &eo);
            vW = a.c1 * vW + a.c2sig * ee;
        };
        double* fac = st + BS_FAC + 6 * d;
        double vW_end = vW;
        if (a.obabo) {
            // [E1, B](h) [O, E7](h) | [O, E7](h) [E1, B](h) [E4-E6 + A](dt)      (R-24)
            if (a.close) {
                press_v();
                if (a.thermostat) press_o(a.cstep_lo, a.cstep_hi);
            }
            vW_end = vW;
            if (a.start) {
                if (a.thermostat) press_o(a.step_lo, a.step_hi);
                Skin = S[d][5]; Sfv = S[d][6];
                press_v();
                const double dt = 2.0 * h;
                fac[0] = exp(dt * vW); fac[1] = sinh_over(vW, dt); fac[2] = exp(-dt * vW);
                fac[3] = 1.0; fac[4] = 0.0; fac[5] = 1.0;
            }
        } else {
            if (a.close) {
                press_v();
                Skin = Skin + 2.0 * h * Sfv + h * h * Sff;     // what B(h), v~0 += h F~0/m, does to the two velocity sums
                Sfv = Sfv + h * Sff;
            }
            vW_end = vW;
            if (a.start) {
                press_v();
                fac[0] = exp(h * vW); fac[1] = sinh_over(vW, h); fac[2] = exp(-h * vW);
                if (a.thermostat) press_o(a.step_lo, a.step_hi);    // E7 over dt
                fac[3] = exp(h * vW); fac[4] = sinh_over(vW, h); fac[5] = exp(-h * vW);
            }
        }
        st[BS_VW + d] = vW;
        if (a.est_slot != nullptr)
            for (int c = d; c < (a.aniso ? d + 1 : 3); ++c) a.est_slot[kEstBaro + c] = vW_end;
    }
    if (!a.aniso) {
        // the integrator reads one factor set per component
        for (int d = 1; d < 3; ++d) {
            st[BS_VW + d] = st[BS_VW];
            if (a.start)
                for (int q = 0; q < 6; ++q) st[BS_FAC + 6 * d + q] = st[BS_FAC + q];
        }
    }
    if (a.start)                                               // E6, as the successive rescalings of the drifts
        for (int c = 0; c < 3; ++c) st[BS_LX + c] = (L[c] * st[BS_FAC + 6 * c]) * st[BS_FAC + 6 * c + 3];
}

int launch_barostat(const BaroArgs& a, cudaStream_t s) {
    baro_sums_kernel<<<(a.n_dof + kBaroThreads - 1) / kBaroThreads, kBaroThreads, 0, s>>>(a);
    baro_update_kernel<<<1, 32, 0, s>>>(a);
    return 2;
}

size_t barostat_state_doubles(int n_dof) {
    return (size_t)BS_WIDTH + kBaroPart * (size_t)((n_dof + kBaroThreads - 1) / kBaroThreads);
}

}  // namespace pimd
