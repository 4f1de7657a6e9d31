// embedding.cu -- F3 (embedding net forward + T_i = (1/N_sel) sum_rows G (x) R) and F5/F6 (embedding
// backward by forward-mode differentiation, pair gradient, force / virial scatter) of SURVEY 8(a).
// CUDA-core FP32 path: persistent CTAs walk the centre bead-atoms in type-sorted order, the weights of
// the (t_i, *) embedding nets stay resident in shared memory, one thread evaluates one neighbour row.
//   h1 = tanh(s W1 + b1); h2 = [h1,h1] + tanh(h1 W2 + b2); G = [h2,h2] + tanh(h2 W3 + b3)     (R-13)
//   T_i = (1/N_sel) sum_rows G_row (x) R_row                                                  (R-14)
// Backward: the net's input is the scalar s, so dG/ds is pushed forward through the same weights
// (G' = dG/ds); with dT_i from the fitting pass
//   dG = dT_i R / N_sel,  dR = dT_i^T G / N_sel,  ds = dG . G'
//   g = dU/dd = (ds + dR_0) s' d/r + (s'/r - s/r^2)(dR_1:3 . d) d/r + (s/r) dR_1:3            (R-16)
//   F_i += g, F_j -= g, Xi_ab -= d_a g_b
#include "common.cuh"

namespace pimd {

constexpr int kEmbThreads = 160;

template <int E1, int E2, int M1>
struct EmbLayout {
    static constexpr int E1p = (E1 + 3) / 4 * 4;
    static constexpr int E2p = (E2 + 3) / 4 * 4;
    static constexpr int oW1 = 0;
    static constexpr int ob1 = E1p;
    static constexpr int oW2t = 2 * E1p;              // [E2][E1p]
    static constexpr int ob2 = oW2t + E2 * E1p;       // [E2p]
    static constexpr int oW3t = ob2 + E2p;            // [M1][E2p]
    static constexpr int ob3 = oW3t + M1 * E2p;       // [M1]
    static constexpr int stride = (ob3 + M1 + 3) / 4 * 4;
};

__device__ __forceinline__ float act_tanh(float x) { return tanhf(x); }

struct EmbArgs {
    int P, N, ntypes, nsel, PN;
    int seloff[PIMD_MAX_TYPES + 1];
    const int* cen_idx; const int* types; const int* ncount;
    const NeighSlotA* slotA; const NeighSlotB* slotB;
    const float* emb_w;
    float* Tm; const float* dTm;
    double* f; double* Xi;
};

template <int E1, int E2, int M1>
__device__ __forceinline__ void load_weights(float* wts, const float* emb_w, int ti, int ntypes) {
    using LY = EmbLayout<E1, E2, M1>;
    const float4* src = reinterpret_cast<const float4*>(emb_w + (size_t)ti * ntypes * LY::stride);
    float4* dst = reinterpret_cast<float4*>(wts);
    for (int q = threadIdx.x; q < ntypes * LY::stride / 4; q += blockDim.x) dst[q] = src[q];
}

// row -> (tj, slot) for the compacted rows of one centre
__device__ __forceinline__ int row_to_slot(int row, const int* cnt, const int* seloff, int ntypes, int& tj) {
    int base = 0;
    tj = 0;
    for (int t = 0; t < ntypes; ++t) {
        if (row < base + cnt[t]) { tj = t; return seloff[t] + (row - base); }
        base += cnt[t];
    }
    return 0;
}

template <int E1, int E2, int M1>
__global__ void __launch_bounds__(kEmbThreads)
embed_fwd_kernel(const __grid_constant__ EmbArgs a) {
    using LY = EmbLayout<E1, E2, M1>;
    extern __shared__ __align__(16) float smem[];
    float* wts = smem;                                      // [ntypes][stride]
    float* Gs = wts + a.ntypes * LY::stride;                // [nsel][M1+1]
    float4* Rs = reinterpret_cast<float4*>(Gs + ((a.nsel * (M1 + 1) + 3) / 4 * 4));   // [nsel]
    __shared__ int cnt_s[PIMD_MAX_TYPES];

    const int per = (a.PN + gridDim.x - 1) / gridDim.x;
    const int r_begin = blockIdx.x * per, r_end = min(a.PN, r_begin + per);
    int cur_ti = -1;
    const float inv_nsel = 1.0f / (float)a.nsel;

    for (int r = r_begin; r < r_end; ++r) {
        const int ba = a.cen_idx[r];
        const int ti = a.types[ba % a.N];
        __syncthreads();                                    // previous centre's smem is free
        if (ti != cur_ti) { load_weights<E1, E2, M1>(wts, a.emb_w, ti, a.ntypes); cur_ti = ti; }
        if (threadIdx.x < a.ntypes) cnt_s[threadIdx.x] = a.ncount[(size_t)ba * a.ntypes + threadIdx.x];
        __syncthreads();
        int tot = 0;
        for (int t = 0; t < a.ntypes; ++t) tot += cnt_s[t];

        for (int row = threadIdx.x; row < tot; row += kEmbThreads) {
            int tj;
            const int slot = row_to_slot(row, cnt_s, a.seloff, a.ntypes, tj);
            const NeighSlotA A = a.slotA[(size_t)ba * a.nsel + slot];
            const NeighSlotB B = a.slotB[(size_t)ba * a.nsel + slot];
            const float s = A.s;
            const float sr = s * B.rinv;
            Rs[row] = make_float4(s, sr * A.dx, sr * A.dy, sr * A.dz);
            const float* W = wts + tj * LY::stride;
            float h1[LY::E1p];
#pragma unroll
            for (int k = 0; k < LY::E1p; ++k) h1[k] = (k < E1) ? act_tanh(fmaf(s, W[LY::oW1 + k], W[LY::ob1 + k])) : 0.f;
            float h2[LY::E2p];
#pragma unroll
            for (int n = 0; n < E2; ++n) {
                float acc = W[LY::ob2 + n];
                const float4* w4 = reinterpret_cast<const float4*>(W + LY::oW2t + n * LY::E1p);
#pragma unroll
                for (int k4 = 0; k4 < LY::E1p / 4; ++k4) {
                    const float4 w = w4[k4];
                    acc = fmaf(h1[4 * k4], w.x, acc); acc = fmaf(h1[4 * k4 + 1], w.y, acc);
                    acc = fmaf(h1[4 * k4 + 2], w.z, acc); acc = fmaf(h1[4 * k4 + 3], w.w, acc);
                }
                h2[n] = h1[n % E1] + act_tanh(acc);
            }
#pragma unroll
            for (int n = E2; n < LY::E2p; ++n) h2[n] = 0.f;
            float* Grow = Gs + row * (M1 + 1);
#pragma unroll 2
            for (int n = 0; n < M1; ++n) {
                float acc = W[LY::ob3 + n];
                const float4* w4 = reinterpret_cast<const float4*>(W + LY::oW3t + n * LY::E2p);
#pragma unroll
                for (int k4 = 0; k4 < LY::E2p / 4; ++k4) {
                    const float4 w = w4[k4];
                    acc = fmaf(h2[4 * k4], w.x, acc); acc = fmaf(h2[4 * k4 + 1], w.y, acc);
                    acc = fmaf(h2[4 * k4 + 2], w.z, acc); acc = fmaf(h2[4 * k4 + 3], w.w, acc);
                }
                Grow[n] = act_tanh(acc);
            }
#pragma unroll
            for (int n = 0; n < M1; ++n) Grow[n] += h2[n % E2];
        }
        __syncthreads();
        // T_i[m][c] = (1/N_sel) sum_rows G[row][m] R[row][c]
        for (int mm = threadIdx.x; mm < M1; mm += kEmbThreads) {
            float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
            for (int row = 0; row < tot; ++row) {
                const float g = Gs[row * (M1 + 1) + mm];
                const float4 R = Rs[row];
                acc.x = fmaf(g, R.x, acc.x); acc.y = fmaf(g, R.y, acc.y);
                acc.z = fmaf(g, R.z, acc.z); acc.w = fmaf(g, R.w, acc.w);
            }
            acc.x *= inv_nsel; acc.y *= inv_nsel; acc.z *= inv_nsel; acc.w *= inv_nsel;
            reinterpret_cast<float4*>(a.Tm)[(size_t)r * M1 + mm] = acc;
        }
    }
}

template <int E1, int E2, int M1>
__global__ void __launch_bounds__(kEmbThreads)
embed_bwd_kernel(const __grid_constant__ EmbArgs a) {
    using LY = EmbLayout<E1, E2, M1>;
    extern __shared__ __align__(16) float smem[];
    float* wts = smem;                                      // [ntypes][stride]
    float4* dTs = reinterpret_cast<float4*>(wts + a.ntypes * LY::stride);   // [M1]
    __shared__ int cnt_s[PIMD_MAX_TYPES];
    __shared__ double red[kEmbThreads / 32][12];

    const int per = (a.PN + gridDim.x - 1) / gridDim.x;
    const int r_begin = blockIdx.x * per, r_end = min(a.PN, r_begin + per);
    int cur_ti = -1;
    const float inv_nsel = 1.0f / (float)a.nsel;

    for (int r = r_begin; r < r_end; ++r) {
        const int ba = a.cen_idx[r];
        const int kbead = ba / a.N, i = ba - kbead * a.N;
        const int ti = a.types[i];
        __syncthreads();
        if (ti != cur_ti) { load_weights<E1, E2, M1>(wts, a.emb_w, ti, a.ntypes); cur_ti = ti; }
        if (threadIdx.x < a.ntypes) cnt_s[threadIdx.x] = a.ncount[(size_t)ba * a.ntypes + threadIdx.x];
        for (int q = threadIdx.x; q < M1; q += kEmbThreads) dTs[q] = reinterpret_cast<const float4*>(a.dTm)[(size_t)r * M1 + q];
        __syncthreads();
        int tot = 0;
        for (int t = 0; t < a.ntypes; ++t) tot += cnt_s[t];

        double gsum[3] = {0, 0, 0}, vir[9] = {0, 0, 0, 0, 0, 0, 0, 0, 0};
        for (int row = threadIdx.x; row < tot; row += kEmbThreads) {
            int tj;
            const int slot = row_to_slot(row, cnt_s, a.seloff, a.ntypes, tj);
            const NeighSlotA A = a.slotA[(size_t)ba * a.nsel + slot];
            const NeighSlotB B = a.slotB[(size_t)ba * a.nsel + slot];
            const float s = A.s;
            const float sr = s * B.rinv;
            const float R0 = s, R1 = sr * A.dx, R2 = sr * A.dy, R3 = sr * A.dz;
            const float* W = wts + tj * LY::stride;
            float h1[LY::E1p], h1p[LY::E1p];
#pragma unroll
            for (int k = 0; k < LY::E1p; ++k) {
                if (k < E1) {
                    const float w = W[LY::oW1 + k];
                    const float t = act_tanh(fmaf(s, w, W[LY::ob1 + k]));
                    h1[k] = t; h1p[k] = (1.f - t * t) * w;
                } else { h1[k] = 0.f; h1p[k] = 0.f; }
            }
            float h2[LY::E2p], h2p[LY::E2p];
#pragma unroll
            for (int n = 0; n < E2; ++n) {
                float acc = W[LY::ob2 + n], accp = 0.f;
                const float4* w4 = reinterpret_cast<const float4*>(W + LY::oW2t + n * LY::E1p);
#pragma unroll
                for (int k4 = 0; k4 < LY::E1p / 4; ++k4) {
                    const float4 w = w4[k4];
                    acc = fmaf(h1[4 * k4], w.x, acc); acc = fmaf(h1[4 * k4 + 1], w.y, acc);
                    acc = fmaf(h1[4 * k4 + 2], w.z, acc); acc = fmaf(h1[4 * k4 + 3], w.w, acc);
                    accp = fmaf(h1p[4 * k4], w.x, accp); accp = fmaf(h1p[4 * k4 + 1], w.y, accp);
                    accp = fmaf(h1p[4 * k4 + 2], w.z, accp); accp = fmaf(h1p[4 * k4 + 3], w.w, accp);
                }
                const float t = act_tanh(acc);
                h2[n] = h1[n % E1] + t;
                h2p[n] = h1p[n % E1] + (1.f - t * t) * accp;
            }
#pragma unroll
            for (int n = E2; n < LY::E2p; ++n) { h2[n] = 0.f; h2p[n] = 0.f; }
            // layer 3 contracted on the fly with dT_i:  ds = sum_n dG_n G'_n,  dR_c = sum_n dT[n][c] G_n
            float ds = 0.f, dR0 = 0.f, dR1 = 0.f, dR2 = 0.f, dR3 = 0.f;
#pragma unroll 2
            for (int n = 0; n < M1; ++n) {
                float acc = W[LY::ob3 + n], accp = 0.f;
                const float4* w4 = reinterpret_cast<const float4*>(W + LY::oW3t + n * LY::E2p);
#pragma unroll
                for (int k4 = 0; k4 < LY::E2p / 4; ++k4) {
                    const float4 w = w4[k4];
                    acc = fmaf(h2[4 * k4], w.x, acc); acc = fmaf(h2[4 * k4 + 1], w.y, acc);
                    acc = fmaf(h2[4 * k4 + 2], w.z, acc); acc = fmaf(h2[4 * k4 + 3], w.w, acc);
                    accp = fmaf(h2p[4 * k4], w.x, accp); accp = fmaf(h2p[4 * k4 + 1], w.y, accp);
                    accp = fmaf(h2p[4 * k4 + 2], w.z, accp); accp = fmaf(h2p[4 * k4 + 3], w.w, accp);
                }
                const float t = act_tanh(acc);
                const float4 dT = dTs[n];
                const float dG = fmaf(dT.x, R0, fmaf(dT.y, R1, fmaf(dT.z, R2, dT.w * R3)));
                ds = fmaf(dG, (1.f - t * t) * accp, ds);
                dR0 = fmaf(dT.x, t, dR0); dR1 = fmaf(dT.y, t, dR1); dR2 = fmaf(dT.z, t, dR2); dR3 = fmaf(dT.w, t, dR3);
            }
#pragma unroll
            for (int n = 0; n < M1; ++n) {               // skip-connection parts: G_n += h2[n%E2], G'_n += h2'[n%E2]
                const float4 dT = dTs[n];
                const float dG = fmaf(dT.x, R0, fmaf(dT.y, R1, fmaf(dT.z, R2, dT.w * R3)));
                const float g = h2[n % E2];
                ds = fmaf(dG, h2p[n % E2], ds);
                dR0 = fmaf(dT.x, g, dR0); dR1 = fmaf(dT.y, g, dR1); dR2 = fmaf(dT.z, g, dR2); dR3 = fmaf(dT.w, g, dR3);
            }
            ds *= inv_nsel; dR0 *= inv_nsel; dR1 *= inv_nsel; dR2 *= inv_nsel; dR3 *= inv_nsel;
            // pair gradient g = dU/dd
            const float rinv = B.rinv;
            const float dot = dR1 * A.dx + dR2 * A.dy + dR3 * A.dz;
            const float radial = (ds + dR0) * B.ds + (B.ds * rinv - s * rinv * rinv) * dot;
            const float rr = radial * rinv;
            const float gx = fmaf(rr, A.dx, sr * dR1), gy = fmaf(rr, A.dy, sr * dR2), gz = fmaf(rr, A.dz, sr * dR3);
            const int j = (int)(B.jcode & 0x7fffffu);
            double* fj = a.f + ((size_t)kbead * a.N + j) * 3;
            atomicAdd(fj, -(double)gx); atomicAdd(fj + 1, -(double)gy); atomicAdd(fj + 2, -(double)gz);
            gsum[0] += gx; gsum[1] += gy; gsum[2] += gz;
            const float dd[3] = {A.dx, A.dy, A.dz}, gg[3] = {gx, gy, gz};
#pragma unroll
            for (int p = 0; p < 3; ++p)
#pragma unroll
                for (int q = 0; q < 3; ++q) vir[3 * p + q] -= (double)(dd[p] * gg[q]);
        }
        // block reduction of F_i and the virial share
        double v12[12];
#pragma unroll
        for (int q = 0; q < 3; ++q) v12[q] = gsum[q];
#pragma unroll
        for (int q = 0; q < 9; ++q) v12[3 + q] = vir[q];
#pragma unroll
        for (int q = 0; q < 12; ++q)
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) v12[q] += __shfl_xor_sync(0xffffffffu, v12[q], o);
        if ((threadIdx.x & 31) == 0) {
#pragma unroll
            for (int q = 0; q < 12; ++q) red[threadIdx.x >> 5][q] = v12[q];
        }
        __syncthreads();
        if (threadIdx.x < 12) {
            double t = 0.0;
#pragma unroll
            for (int w = 0; w < kEmbThreads / 32; ++w) t += red[w][threadIdx.x];
            if (threadIdx.x < 3) atomicAdd(a.f + ((size_t)kbead * a.N + i) * 3 + threadIdx.x, t);
            else atomicAdd(a.Xi + kbead * 9 + (threadIdx.x - 3), t);
        }
    }
}

static EmbArgs make_args(Model& m, const ForceArgs& fa) {
    EmbArgs a;
    a.P = fa.P; a.N = fa.N; a.ntypes = fa.ntypes; a.nsel = m.nsel; a.PN = fa.P * fa.N;
    for (int t = 0; t <= PIMD_MAX_TYPES; ++t) a.seloff[t] = m.seloff[t];
    a.cen_idx = m.cen_idx; a.types = fa.types; a.ncount = m.ncount;
    a.slotA = m.slotA; a.slotB = m.slotB; a.emb_w = m.emb_w;
    a.Tm = m.Tm; a.dTm = m.dTm; a.f = fa.f; a.Xi = fa.Xi;
    return a;
}

using LY0 = EmbLayout<25, 50, 100>;

static size_t fwd_smem(const Model& m, int ntypes) {
    return sizeof(float) * ((size_t)ntypes * LY0::stride + ((size_t)m.nsel * 101 + 3) / 4 * 4) + sizeof(float4) * m.nsel;
}
static size_t bwd_smem(const Model& m, int ntypes) {
    return sizeof(float) * ((size_t)ntypes * LY0::stride) + sizeof(float4) * 100;
}
size_t embedding_smem_bytes(const Model& m, int ntypes) { return fwd_smem(m, ntypes); }

int embedding_forward(Model& m, const ForceArgs& fa, int n_sms, cudaStream_t s) {
    EmbArgs a = make_args(m, fa);
    const size_t smem = fwd_smem(m, fa.ntypes);
    cudaFuncSetAttribute(embed_fwd_kernel<25, 50, 100>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    const int grid = min(a.PN, n_sms * 2);
    embed_fwd_kernel<25, 50, 100><<<grid, kEmbThreads, smem, s>>>(a);
    return 1;
}

int embedding_backward(Model& m, const ForceArgs& fa, int n_sms, cudaStream_t s) {
    EmbArgs a = make_args(m, fa);
    const size_t smem = bwd_smem(m, fa.ntypes);
    cudaFuncSetAttribute(embed_bwd_kernel<25, 50, 100>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    const int grid = min(a.PN, n_sms * 2);
    embed_bwd_kernel<25, 50, 100><<<grid, kEmbThreads, smem, s>>>(a);
    return 1;
}

}  // namespace pimd
