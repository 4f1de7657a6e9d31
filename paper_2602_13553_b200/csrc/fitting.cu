// fitting.cu -- F4 of SURVEY 8(a): descriptor D_i = T_i (T_i^<)^T, fitting net forward and analytic
// backward, dT_i.  CUDA-core FP32 path (tiled SGEMM with fused epilogues); rows are the centre
// bead-atoms in type-sorted order so each centre type is one contiguous GEMM.
//   D[m*M2+m2] = sum_c T[m][c] T[m2][c]                                            (R-14)
//   y1 = tanh(D W1 + b1); y2 = y1 + tanh(y1 W2 + b2); y3 = y2 + tanh(y2 W3 + b3); E = y3.w4 + b4   (R-15)
//   backward: dy3 = w4; da_l = dy_l o (1 - t_l^2); dy_{l-1} = dy_l + da_l W_l^T; dD = da_1 W1^T
//   dT[m][c] = sum_{m2<M2} dD[m][m2] T[m2][c] + [m<M2] sum_{m1} dD[m1][m] T[m1][c]
#include "common.cuh"

namespace pimd {

// ---------------------------------------------------------------------------------------------
// descriptor and its backward
// ---------------------------------------------------------------------------------------------
template <int M1, int M2>
__global__ void __launch_bounds__(256) descriptor_kernel(int rows, const float* __restrict__ Tm, float* __restrict__ D) {
    __shared__ float4 Ts[M1];
    const int r = blockIdx.x;
    for (int q = threadIdx.x; q < M1; q += blockDim.x) Ts[q] = reinterpret_cast<const float4*>(Tm)[(size_t)r * M1 + q];
    __syncthreads();
    for (int o = threadIdx.x; o < M1 * M2; o += blockDim.x) {
        const float4 a = Ts[o / M2], b = Ts[o % M2];
        D[(size_t)r * (M1 * M2) + o] = a.x * b.x + a.y * b.y + a.z * b.z + a.w * b.w;
    }
}

template <int M1, int M2>
__global__ void __launch_bounds__(128) dT_kernel(int rows, const float* __restrict__ Tm, const float* __restrict__ dD,
                                                 float* __restrict__ dTm) {
    __shared__ float4 Ts[M1];
    __shared__ float dDs[M1 * M2];
    const int r = blockIdx.x;
    for (int q = threadIdx.x; q < M1; q += blockDim.x) Ts[q] = reinterpret_cast<const float4*>(Tm)[(size_t)r * M1 + q];
    for (int q = threadIdx.x; q < M1 * M2 / 4; q += blockDim.x)
        reinterpret_cast<float4*>(dDs)[q] = reinterpret_cast<const float4*>(dD)[(size_t)r * (M1 * M2 / 4) + q];
    __syncthreads();
    for (int mm = threadIdx.x; mm < M1; mm += blockDim.x) {
        float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
        for (int m2 = 0; m2 < M2; ++m2) {
            const float w = dDs[mm * M2 + m2];
            const float4 t = Ts[m2];
            acc.x = fmaf(w, t.x, acc.x); acc.y = fmaf(w, t.y, acc.y); acc.z = fmaf(w, t.z, acc.z); acc.w = fmaf(w, t.w, acc.w);
        }
        if (mm < M2) {
            for (int m1 = 0; m1 < M1; ++m1) {
                const float w = dDs[m1 * M2 + mm];
                const float4 t = Ts[m1];
                acc.x = fmaf(w, t.x, acc.x); acc.y = fmaf(w, t.y, acc.y); acc.z = fmaf(w, t.z, acc.z); acc.w = fmaf(w, t.w, acc.w);
            }
        }
        reinterpret_cast<float4*>(dTm)[(size_t)r * M1 + mm] = acc;
    }
}

// ---------------------------------------------------------------------------------------------
// tiled SGEMM  C[M x N] = epilogue(A[M x K] B[K x N]), row-major, K % 16 == 0
// ---------------------------------------------------------------------------------------------
enum : int {
    EPI_TANH_BIAS = 0,        // out0 = tanh(acc + bias)
    EPI_TANH_BIAS_SKIP = 1,   // t = tanh(acc + bias); out0 = t; out1 = add + t
    EPI_BWD = 2,              // y = add + acc; out0 = y (if non-null); out1 = y * (1 - tt^2)
    EPI_BWD_FIRST = 3,        // out1 = (add + acc) * (1 - tt^2)   (tt = y1 = tanh)
    EPI_PLAIN = 4             // out0 = acc
};

struct GemmArgs {
    int M, N, K;
    const float* A; int lda;
    const float* B; int ldb;
    const float* bias;        // [N]
    const float* add; int ldadd;
    const float* tt; int ldtt;
    float* out0; float* out1; int ldo;
};

constexpr int BM = 128, BN = 64, BK = 16;

template <int EPI>
__global__ void __launch_bounds__(256) sgemm_kernel(const __grid_constant__ GemmArgs g) {
    __shared__ __align__(16) float As[2][BK][BM + 4];
    __shared__ __align__(16) float Bs[2][BK][BN];
    const int tid = threadIdx.x;
    const int m0 = blockIdx.y * BM, n0 = blockIdx.x * BN;
    const int tx = tid & 15, ty = tid >> 4;               // 16 x 16 threads, each 8 (M) x 4 (N)
    float acc[8][4];
#pragma unroll
    for (int p = 0; p < 8; ++p)
#pragma unroll
        for (int q = 0; q < 4; ++q) acc[p][q] = 0.f;

    // global -> smem staging: A tile 128 x 16 = 512 float4 (2 per thread); B tile 16 x 64 = 256 float4 (1 per thread)
    const int a_row = tid >> 2, a_k4 = (tid & 3) * 4;       // rows a_row and a_row + 64
    const int b_k = tid >> 4, b_n4 = (tid & 15) * 4;
    float4 ra[2], rb;
    auto load_g = [&](int k0) {
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const int m = m0 + a_row + 64 * h;
            ra[h] = (m < g.M) ? *reinterpret_cast<const float4*>(g.A + (size_t)m * g.lda + k0 + a_k4)
                              : make_float4(0.f, 0.f, 0.f, 0.f);
        }
        const int n = n0 + b_n4;
        rb = (n < g.N) ? *reinterpret_cast<const float4*>(g.B + (size_t)(k0 + b_k) * g.ldb + n)
                       : make_float4(0.f, 0.f, 0.f, 0.f);
    };
    auto store_s = [&](int buf) {
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const int m = a_row + 64 * h;
            As[buf][a_k4 + 0][m] = ra[h].x; As[buf][a_k4 + 1][m] = ra[h].y;
            As[buf][a_k4 + 2][m] = ra[h].z; As[buf][a_k4 + 3][m] = ra[h].w;
        }
        *reinterpret_cast<float4*>(&Bs[buf][b_k][b_n4]) = rb;
    };
    load_g(0);
    store_s(0);
    __syncthreads();
    const int nk = g.K / BK;
    for (int kt = 0; kt < nk; ++kt) {
        const int buf = kt & 1;
        if (kt + 1 < nk) load_g((kt + 1) * BK);
#pragma unroll
        for (int kk = 0; kk < BK; ++kk) {
            const float4 a0 = *reinterpret_cast<const float4*>(&As[buf][kk][ty * 4]);
            const float4 a1 = *reinterpret_cast<const float4*>(&As[buf][kk][64 + ty * 4]);
            const float4 b = *reinterpret_cast<const float4*>(&Bs[buf][kk][tx * 4]);
            const float av[8] = {a0.x, a0.y, a0.z, a0.w, a1.x, a1.y, a1.z, a1.w};
            const float bv[4] = {b.x, b.y, b.z, b.w};
#pragma unroll
            for (int p = 0; p < 8; ++p)
#pragma unroll
                for (int q = 0; q < 4; ++q) acc[p][q] = fmaf(av[p], bv[q], acc[p][q]);
        }
        if (kt + 1 < nk) store_s(buf ^ 1);
        __syncthreads();
    }
    // epilogue: rows m0 + ty*4 + p (p<4) and m0 + 64 + ty*4 + (p-4); cols n0 + tx*4 + q
    const int n = n0 + tx * 4;
    if (n >= g.N) return;
    float4 bias = make_float4(0.f, 0.f, 0.f, 0.f);
    if (EPI == EPI_TANH_BIAS || EPI == EPI_TANH_BIAS_SKIP) bias = *reinterpret_cast<const float4*>(g.bias + n);
#pragma unroll
    for (int p = 0; p < 8; ++p) {
        const int m = m0 + (p < 4 ? ty * 4 + p : 64 + ty * 4 + (p - 4));
        if (m >= g.M) continue;
        float4 v = make_float4(acc[p][0], acc[p][1], acc[p][2], acc[p][3]);
        if (EPI == EPI_TANH_BIAS) {
            v.x = tanhf(v.x + bias.x); v.y = tanhf(v.y + bias.y); v.z = tanhf(v.z + bias.z); v.w = tanhf(v.w + bias.w);
            *reinterpret_cast<float4*>(g.out0 + (size_t)m * g.ldo + n) = v;
        } else if (EPI == EPI_TANH_BIAS_SKIP) {
            v.x = tanhf(v.x + bias.x); v.y = tanhf(v.y + bias.y); v.z = tanhf(v.z + bias.z); v.w = tanhf(v.w + bias.w);
            *reinterpret_cast<float4*>(g.out0 + (size_t)m * g.ldo + n) = v;
            const float4 ad = *reinterpret_cast<const float4*>(g.add + (size_t)m * g.ldadd + n);
            v.x += ad.x; v.y += ad.y; v.z += ad.z; v.w += ad.w;
            *reinterpret_cast<float4*>(g.out1 + (size_t)m * g.ldo + n) = v;
        } else if (EPI == EPI_BWD || EPI == EPI_BWD_FIRST) {
            const float4 ad = *reinterpret_cast<const float4*>(g.add + (size_t)m * g.ldadd + n);
            v.x += ad.x; v.y += ad.y; v.z += ad.z; v.w += ad.w;
            if (EPI == EPI_BWD) *reinterpret_cast<float4*>(g.out0 + (size_t)m * g.ldo + n) = v;
            const float4 t = *reinterpret_cast<const float4*>(g.tt + (size_t)m * g.ldtt + n);
            v.x *= (1.f - t.x * t.x); v.y *= (1.f - t.y * t.y); v.z *= (1.f - t.z * t.z); v.w *= (1.f - t.w * t.w);
            *reinterpret_cast<float4*>(g.out1 + (size_t)m * g.ldo + n) = v;
        } else {
            *reinterpret_cast<float4*>(g.out0 + (size_t)m * g.ldo + n) = v;
        }
    }
}

template <int EPI>
static void launch_gemm(const GemmArgs& g, cudaStream_t s) {
    dim3 grid((g.N + BN - 1) / BN, (g.M + BM - 1) / BM);
    sgemm_kernel<EPI><<<grid, 256, 0, s>>>(g);
}

// E_i = y3 . w4 + b4; U^(k) += E_i; also the seed of the backward pass: dy3 = w4, da3 = w4 o (1 - t3^2).
// One warp per row.
__global__ void __launch_bounds__(128)
energy_kernel(int row0, int rows, int NF, int N, const float* __restrict__ Y3, const float* __restrict__ T3,
              const float* __restrict__ w4, const float* __restrict__ b4, const int* __restrict__ cen_idx,
              double* __restrict__ Eatom, double* __restrict__ U, float* __restrict__ dA3, float* __restrict__ dY3) {
    const int r = row0 + ((blockIdx.x * blockDim.x + threadIdx.x) >> 5);
    const int lane = threadIdx.x & 31;
    if (r >= row0 + rows) return;
    float acc = 0.f;
    for (int n = lane; n < NF; n += 32) {
        const float w = w4[n];
        acc = fmaf(Y3[(size_t)r * NF + n], w, acc);
        const float t = T3[(size_t)r * NF + n];
        dA3[(size_t)r * NF + n] = w * (1.f - t * t);
        dY3[(size_t)r * NF + n] = w;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    if (lane == 0) {
        const int ba = cen_idx[r];
        const double e = (double)(acc + b4[0]);
        Eatom[ba] = e;
        atomicAdd(U + ba / N, e);
    }
}

int fitting_forward_backward(Model& m, const ForceArgs& a, cudaStream_t s) {
    const int PN = a.P * a.N;
    const int NF = m.NF, ND = m.ND;
    int launches = 2;
    if (m.use_tc && m.tc_ready && m.M1 == 100 && m.M2 == 16) {
        // one launch per layer for all centre types; descriptor fused into layer 1, energy into layer 3, dD -> dT
        launches = fitting_chain_tc(m, a, s);
        return launches;
    }
    descriptor_kernel<100, 16><<<PN, 256, 0, s>>>(PN, m.Tm, m.D);
    for (int t = 0; t < a.ntypes; ++t) {
        const int row0 = m.type_row0[t], rows = m.type_row0[t + 1] - row0;
        if (rows == 0) continue;
        launches += 7;
        const size_t oF = (size_t)row0 * NF, oD = (size_t)row0 * ND;
        GemmArgs g{};
        // layer 1: Y1 = tanh(D W1 + b1)
        g.M = rows; g.N = NF; g.K = ND; g.A = m.D + oD; g.lda = ND; g.B = m.fit_w[t][0]; g.ldb = NF;
        g.bias = m.fit_b[t][0]; g.out0 = m.Y1 + oF; g.ldo = NF;
        launch_gemm<EPI_TANH_BIAS>(g, s);
        // layer 2: T2 = tanh(Y1 W2 + b2); Y2 = Y1 + T2
        g = GemmArgs{};
        g.M = rows; g.N = NF; g.K = NF; g.A = m.Y1 + oF; g.lda = NF; g.B = m.fit_w[t][1]; g.ldb = NF;
        g.bias = m.fit_b[t][1]; g.add = m.Y1 + oF; g.ldadd = NF; g.out0 = m.T2 + oF; g.out1 = m.Y2 + oF; g.ldo = NF;
        launch_gemm<EPI_TANH_BIAS_SKIP>(g, s);
        // layer 3: T3 = tanh(Y2 W3 + b3); Y3 = Y2 + T3
        g = GemmArgs{};
        g.M = rows; g.N = NF; g.K = NF; g.A = m.Y2 + oF; g.lda = NF; g.B = m.fit_w[t][2]; g.ldb = NF;
        g.bias = m.fit_b[t][2]; g.add = m.Y2 + oF; g.ldadd = NF; g.out0 = m.T3 + oF; g.out1 = m.Y3 + oF; g.ldo = NF;
        launch_gemm<EPI_TANH_BIAS_SKIP>(g, s);
        // E_i, U^(k); da3 -> G1, dy3 -> G2
        energy_kernel<<<(rows * 32 + 127) / 128, 128, 0, s>>>(row0, rows, NF, a.N, m.Y3, m.T3, m.fit_w[t][3],
                                                              m.fit_b[t][3], m.cen_idx, a.Eatom, a.U, m.G1, m.G2);
        // dy2 = dy3 + da3 W3^T -> Y3 ; da2 = dy2 o (1 - t2^2) -> T3
        g = GemmArgs{};
        g.M = rows; g.N = NF; g.K = NF; g.A = m.G1 + oF; g.lda = NF; g.B = m.fit_wT[t][2]; g.ldb = NF;
        g.add = m.G2 + oF; g.ldadd = NF; g.tt = m.T2 + oF; g.ldtt = NF; g.out0 = m.Y3 + oF; g.out1 = m.T3 + oF; g.ldo = NF;
        launch_gemm<EPI_BWD>(g, s);
        // dy1 = dy2 + da2 W2^T ; da1 = dy1 o (1 - y1^2) -> G1
        g = GemmArgs{};
        g.M = rows; g.N = NF; g.K = NF; g.A = m.T3 + oF; g.lda = NF; g.B = m.fit_wT[t][1]; g.ldb = NF;
        g.add = m.Y3 + oF; g.ldadd = NF; g.tt = m.Y1 + oF; g.ldtt = NF; g.out1 = m.G1 + oF; g.ldo = NF;
        launch_gemm<EPI_BWD_FIRST>(g, s);
        // dD = da1 W1^T
        g = GemmArgs{};
        g.M = rows; g.N = ND; g.K = NF; g.A = m.G1 + oF; g.lda = NF; g.B = m.fit_wT[t][0]; g.ldb = ND;
        g.out0 = m.dD + oD; g.ldo = ND;
        launch_gemm<EPI_PLAIN>(g, s);
    }
    dT_kernel<100, 16><<<PN, 128, 0, s>>>(PN, m.Tm, m.dD, m.dTm);
    return launches;
}

}  // namespace pimd
