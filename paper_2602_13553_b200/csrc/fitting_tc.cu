// fitting_tc.cu -- the fitting-net GEMMs of F4 on the 5th-generation tensor cores.
//
//   C[M x N] = epilogue( A[M x K] . Bt[N x K]^T ),  FP32 in / FP32 out, computed as 3xTF32:
//   a = a_hi + a_lo, b = b_hi + b_lo (hi = top 10 mantissa bits, lo = exact remainder)
//   a.b ~= a_hi.b_hi + a_lo.b_hi + a_hi.b_lo     (FP32 accumulate in TMEM; dropped term ~2^-22)
// which keeps the force error at the FP32 level (single-pass TF32 fails north_star's 1e-4).
//
// One CTA computes a 256 x BN tile (two M = 128 accumulators, 2 x BN <= 512 TMEM columns) so that every
// weight tile is used for 256 rows.  Warp roles (192 threads):
//   warp 0   TMA producer: raw FP32 A (2 boxes 16 x 128) and B (box 16 x BN) tiles, SWIZZLE_64B, 3 stages
//   warp 1   TMEM allocation + single-thread tcgen05.mma issue (12 MMAs of 128 x BN x 8 per stage)
//   warps 2-5 split hi/lo in shared memory (elementwise, so the swizzled layout is preserved), then the
//            epilogue: tcgen05.ld accumulators -> bias / tanh / skip / derivative -> global
#include "common.cuh"
#include "tc_gemm.cuh"

namespace pimd {

using namespace tc;

enum : int { TEPI_TANH_BIAS = 0, TEPI_TANH_BIAS_SKIP = 1, TEPI_BWD = 2, TEPI_BWD_FIRST = 3, TEPI_PLAIN = 4 };

struct TcGemmArgs {
    int M, N, K;               // N = logical columns of C (multiple of BN chunks handled by grid.x)
    const float* bias;
    const float* add; int ldadd;
    const float* tt; int ldtt;
    float* out0; float* out1; int ldo;
};

constexpr int kTcThreads = 192;
constexpr int kTcStages = 3;
constexpr int kTcBK = 16;                 // floats per K block = 64 B rows (SWIZZLE_64B)

template <int BN>
struct TcSmem {
    static constexpr int kABytes = 128 * 64;                      // one 128-row half
    static constexpr int kBBytes = BN * 64;
    static constexpr int oAhi = 0, oAlo = 2 * kABytes, oBhi = 4 * kABytes, oBlo = 4 * kABytes + kBBytes;
    static constexpr int kStage = 4 * kABytes + 2 * kBBytes;
    static constexpr int kTotal = kTcStages * kStage + 1024 /*align slack*/ + 256 /*barriers*/;
};

template <int BN, int EPI>
__global__ void __launch_bounds__(kTcThreads, 1)
gemm3xtf32_kernel(const __grid_constant__ CUtensorMap mapA, const __grid_constant__ CUtensorMap mapB,
                  const __grid_constant__ TcGemmArgs g) {
    using SM = TcSmem<BN>;
    extern __shared__ uint8_t smem_raw[];
    uint8_t* smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);   // keeps the shared address space
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem + kTcStages * SM::kStage);
    uint64_t* full = bars;                     // [stages] TMA -> split warps
    uint64_t* ready = bars + kTcStages;        // [stages] split warps -> MMA
    uint64_t* empty = bars + 2 * kTcStages;    // [stages] MMA -> TMA
    uint64_t* tmem_full = bars + 3 * kTcStages;
    uint32_t* tmem_ptr = reinterpret_cast<uint32_t*>(bars + 3 * kTcStages + 1);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int m0 = blockIdx.y * 256, n0 = blockIdx.x * BN;
    const int nk = g.K / kTcBK;

    if (warp == 0 && lane == 0) {
        tma_prefetch_desc(&mapA);
        tma_prefetch_desc(&mapB);
        for (int s = 0; s < kTcStages; ++s) { mbar_init(full + s, 1); mbar_init(ready + s, 128); mbar_init(empty + s, 1); }
        mbar_init(tmem_full, 1);
        fence_barrier_init();
    }
    if (warp == 1) tmem_alloc(tmem_ptr, 512);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_ptr;

    if (warp == 0) {
        if (lane == 0) {
            for (int kb = 0; kb < nk; ++kb) {
                const int s = kb % kTcStages, ph = (kb / kTcStages) & 1;
                mbar_wait(empty + s, ph ^ 1);
                uint8_t* st = smem + s * SM::kStage;
                mbar_arrive_expect_tx(full + s, 2 * SM::kABytes + SM::kBBytes);
                tma_load_2d(st + SM::oAhi, &mapA, full + s, kb * kTcBK, m0);
                tma_load_2d(st + SM::oAhi + SM::kABytes, &mapA, full + s, kb * kTcBK, m0 + 128);
                tma_load_2d(st + SM::oBhi, &mapB, full + s, kb * kTcBK, n0);
            }
        }
    } else if (warp == 1) {
        if (lane == 0) {
            constexpr uint32_t idesc = make_idesc_tf32(128, BN);
            for (int kb = 0; kb < nk; ++kb) {
                const int s = kb % kTcStages, ph = (kb / kTcStages) & 1;
                mbar_wait(ready + s, ph);
                tc_fence_after();
                const uint32_t st = smem_u32(smem + s * SM::kStage);
#pragma unroll
                for (int h = 0; h < 2; ++h) {
                    const uint32_t d = tmem_base + h * 256;
#pragma unroll
                    for (int ks = 0; ks < 2; ++ks) {
                        const uint64_t a_hi = make_smem_desc_kmajor(st + SM::oAhi + h * SM::kABytes + ks * 32, 64);
                        const uint64_t a_lo = make_smem_desc_kmajor(st + SM::oAlo + h * SM::kABytes + ks * 32, 64);
                        const uint64_t b_hi = make_smem_desc_kmajor(st + SM::oBhi + ks * 32, 64);
                        const uint64_t b_lo = make_smem_desc_kmajor(st + SM::oBlo + ks * 32, 64);
                        umma_tf32(d, a_hi, b_hi, idesc, (kb | ks) ? 1u : 0u);
                        umma_tf32(d, a_lo, b_hi, idesc, 1u);
                        umma_tf32(d, a_hi, b_lo, idesc, 1u);
                    }
                }
                umma_commit(empty + s);
            }
            umma_commit(tmem_full);
        }
    } else {
        // ---- split hi / lo in place (128 threads) ----
        const int t = threadIdx.x - 64;
        for (int kb = 0; kb < nk; ++kb) {
            const int s = kb % kTcStages, ph = (kb / kTcStages) & 1;
            mbar_wait(full + s, ph);
            uint8_t* st = smem + s * SM::kStage;
            float4* a_hi = reinterpret_cast<float4*>(st + SM::oAhi);
            float4* a_lo = reinterpret_cast<float4*>(st + SM::oAlo);
#pragma unroll
            for (int q = 0; q < (2 * SM::kABytes / 16) / 128; ++q) {
                const int idx = t + q * 128;
                const float4 v = a_hi[idx];
                float4 hi, lo;
                hi.x = __uint_as_float(__float_as_uint(v.x) & 0xFFFFE000u); lo.x = v.x - hi.x;
                hi.y = __uint_as_float(__float_as_uint(v.y) & 0xFFFFE000u); lo.y = v.y - hi.y;
                hi.z = __uint_as_float(__float_as_uint(v.z) & 0xFFFFE000u); lo.z = v.z - hi.z;
                hi.w = __uint_as_float(__float_as_uint(v.w) & 0xFFFFE000u); lo.w = v.w - hi.w;
                a_hi[idx] = hi;
                a_lo[idx] = lo;
            }
            float4* b_hi = reinterpret_cast<float4*>(st + SM::oBhi);
            float4* b_lo = reinterpret_cast<float4*>(st + SM::oBlo);
            for (int idx = t; idx < SM::kBBytes / 16; idx += 128) {
                const float4 v = b_hi[idx];
                float4 hi, lo;
                hi.x = __uint_as_float(__float_as_uint(v.x) & 0xFFFFE000u); lo.x = v.x - hi.x;
                hi.y = __uint_as_float(__float_as_uint(v.y) & 0xFFFFE000u); lo.y = v.y - hi.y;
                hi.z = __uint_as_float(__float_as_uint(v.z) & 0xFFFFE000u); lo.z = v.z - hi.z;
                hi.w = __uint_as_float(__float_as_uint(v.w) & 0xFFFFE000u); lo.w = v.w - hi.w;
                b_hi[idx] = hi;
                b_lo[idx] = lo;
            }
            fence_proxy_async_smem();
            mbar_arrive(ready + s);
        }
        // ---- epilogue ----
        mbar_wait(tmem_full, 0);
        tc_fence_after();
        const int quarter = warp & 3;                      // TMEM lane quarter this warp may access
#pragma unroll 1
        for (int h = 0; h < 2; ++h) {
            const int m = m0 + h * 128 + quarter * 32 + lane;
            const bool row_ok = m < g.M;
#pragma unroll 1
            for (int c = 0; c < BN / 16; ++c) {
                uint32_t v[16];
                tmem_ld16(tmem_base + ((uint32_t)(quarter * 32) << 16) + h * 256 + c * 16, v);
                tmem_ld_wait();
                const int n = n0 + c * 16;
                if (!row_ok || n >= g.N) continue;
                float r[16];
#pragma unroll
                for (int q = 0; q < 16; ++q) r[q] = __uint_as_float(v[q]);
                if (EPI == TEPI_TANH_BIAS || EPI == TEPI_TANH_BIAS_SKIP) {
#pragma unroll
                    for (int q = 0; q < 16; ++q) r[q] = tanhf(r[q] + __ldg(g.bias + n + q));
                }
                float4* o0 = (g.out0 != nullptr) ? reinterpret_cast<float4*>(g.out0 + (size_t)m * g.ldo + n) : nullptr;
                float4* o1 = (g.out1 != nullptr) ? reinterpret_cast<float4*>(g.out1 + (size_t)m * g.ldo + n) : nullptr;
                if (EPI == TEPI_TANH_BIAS || EPI == TEPI_PLAIN) {
#pragma unroll
                    for (int q = 0; q < 4; ++q) o0[q] = make_float4(r[4 * q], r[4 * q + 1], r[4 * q + 2], r[4 * q + 3]);
                } else if (EPI == TEPI_TANH_BIAS_SKIP) {
                    const float4* ad = reinterpret_cast<const float4*>(g.add + (size_t)m * g.ldadd + n);
#pragma unroll
                    for (int q = 0; q < 4; ++q) {
                        o0[q] = make_float4(r[4 * q], r[4 * q + 1], r[4 * q + 2], r[4 * q + 3]);
                        const float4 a4 = ad[q];
                        o1[q] = make_float4(r[4 * q] + a4.x, r[4 * q + 1] + a4.y, r[4 * q + 2] + a4.z, r[4 * q + 3] + a4.w);
                    }
                } else {   // TEPI_BWD, TEPI_BWD_FIRST
                    const float4* ad = reinterpret_cast<const float4*>(g.add + (size_t)m * g.ldadd + n);
                    const float4* tt = reinterpret_cast<const float4*>(g.tt + (size_t)m * g.ldtt + n);
#pragma unroll
                    for (int q = 0; q < 4; ++q) {
                        const float4 a4 = ad[q], t4 = tt[q];
                        float4 y = make_float4(r[4 * q] + a4.x, r[4 * q + 1] + a4.y, r[4 * q + 2] + a4.z, r[4 * q + 3] + a4.w);
                        if (EPI == TEPI_BWD) o0[q] = y;
                        y.x *= (1.f - t4.x * t4.x); y.y *= (1.f - t4.y * t4.y);
                        y.z *= (1.f - t4.z * t4.z); y.w *= (1.f - t4.w * t4.w);
                        o1[q] = y;
                    }
                }
            }
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 1) tmem_dealloc(tmem_base, 512);
}

// ---------------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static EncodeTiledFn get_encode() {
    static EncodeTiledFn fn = nullptr;
    if (!fn) {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) == cudaSuccess &&
            qres == cudaDriverEntryPointSuccess)
            fn = reinterpret_cast<EncodeTiledFn>(p);
    }
    return fn;
}

// row-major FP32 matrix [rows][cols] with leading dimension ld (floats); box = 16 floats x box_rows, SWIZZLE_64B
bool tc_make_map(CUtensorMap* map, const float* base, uint64_t rows, uint64_t cols, uint64_t ld, uint32_t box_rows) {
    EncodeTiledFn enc = get_encode();
    if (!enc) return false;
    cuuint64_t dims[2] = {cols, rows};
    cuuint64_t strides[1] = {ld * sizeof(float)};
    cuuint32_t box[2] = {(cuuint32_t)kTcBK, box_rows};
    cuuint32_t estr[2] = {1, 1};
    return enc(map, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, const_cast<float*>(base), dims, strides, box, estr,
               CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_64B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
               CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

template <int BN, int EPI>
static cudaError_t launch_tc(const CUtensorMap& mapA, const CUtensorMap& mapB, const TcGemmArgs& g, cudaStream_t s) {
    using SM = TcSmem<BN>;
    static bool attr = false;
    if (!attr) {
        cudaError_t e = cudaFuncSetAttribute(gemm3xtf32_kernel<BN, EPI>, cudaFuncAttributeMaxDynamicSharedMemorySize, SM::kTotal);
        if (e != cudaSuccess) return e;
        attr = true;
    }
    dim3 grid((g.N + BN - 1) / BN, (g.M + 255) / 256);
    gemm3xtf32_kernel<BN, EPI><<<grid, kTcThreads, SM::kTotal, s>>>(mapA, mapB, g);
    return cudaGetLastError();
}

// C = epi(A Bt^T): A [M][K] (lda), Bt [N][K] (ldb) row-major FP32.  bn = 240 (N == 240) or 160 (N % 160 == 0).
cudaError_t tc_gemm(int epi, int bn, const CUtensorMap& mapA, const CUtensorMap& mapB, const TcGemmArgs& g, cudaStream_t s) {
    if (bn == 240) {
        switch (epi) {
            case TEPI_TANH_BIAS: return launch_tc<240, TEPI_TANH_BIAS>(mapA, mapB, g, s);
            case TEPI_TANH_BIAS_SKIP: return launch_tc<240, TEPI_TANH_BIAS_SKIP>(mapA, mapB, g, s);
            case TEPI_BWD: return launch_tc<240, TEPI_BWD>(mapA, mapB, g, s);
            case TEPI_BWD_FIRST: return launch_tc<240, TEPI_BWD_FIRST>(mapA, mapB, g, s);
            case TEPI_PLAIN: return launch_tc<240, TEPI_PLAIN>(mapA, mapB, g, s);
        }
    } else if (bn == 160) {
        if (epi == TEPI_PLAIN) return launch_tc<160, TEPI_PLAIN>(mapA, mapB, g, s);
    }
    return cudaErrorInvalidValue;
}


bool tc_setup_maps(Model& m, int ntypes) {
    const int NF = m.NF, ND = m.ND;
    if (NF != 240 || ND % 160 != 0) return false;
    for (int t = 0; t < ntypes; ++t) {
        const uint64_t row0 = m.type_row0[t], rows = m.type_row0[t + 1] - m.type_row0[t];
        if (rows == 0) continue;
        bool ok = true;
        ok &= tc_make_map(&m.mapA_D[t], m.D + row0 * ND, rows, ND, ND, 128);
        ok &= tc_make_map(&m.mapA_Y1[t], m.Y1 + row0 * NF, rows, NF, NF, 128);
        ok &= tc_make_map(&m.mapA_Y2[t], m.Y2 + row0 * NF, rows, NF, NF, 128);
        ok &= tc_make_map(&m.mapA_G1[t], m.G1 + row0 * NF, rows, NF, NF, 128);
        ok &= tc_make_map(&m.mapA_T3[t], m.T3 + row0 * NF, rows, NF, NF, 128);
        ok &= tc_make_map(&m.mapB_fwd[t][0], m.fit_wT[t][0], NF, ND, ND, 240);
        ok &= tc_make_map(&m.mapB_fwd[t][1], m.fit_wT[t][1], NF, NF, NF, 240);
        ok &= tc_make_map(&m.mapB_fwd[t][2], m.fit_wT[t][2], NF, NF, NF, 240);
        ok &= tc_make_map(&m.mapB_bwd[t][0], m.fit_w[t][0], ND, NF, NF, 160);
        ok &= tc_make_map(&m.mapB_bwd[t][1], m.fit_w[t][1], NF, NF, NF, 240);
        ok &= tc_make_map(&m.mapB_bwd[t][2], m.fit_w[t][2], NF, NF, NF, 240);
        if (!ok) return false;
    }
    m.tc_ready = true;
    return true;
}

// the six GEMMs of one centre type on the tensor cores; same buffers and epilogues as the CUDA-core path
int fitting_gemms_tc(Model& m, int t, cudaStream_t s) {
    const int NF = m.NF, ND = m.ND;
    const int row0 = m.type_row0[t], rows = m.type_row0[t + 1] - row0;
    const size_t oF = (size_t)row0 * NF, oD = (size_t)row0 * ND;
    TcGemmArgs g{};
    g.M = rows; g.N = NF; g.K = ND; g.bias = m.fit_b[t][0]; g.out0 = m.Y1 + oF; g.ldo = NF;
    tc_gemm(TEPI_TANH_BIAS, 240, m.mapA_D[t], m.mapB_fwd[t][0], g, s);
    g = TcGemmArgs{};
    g.M = rows; g.N = NF; g.K = NF; g.bias = m.fit_b[t][1]; g.add = m.Y1 + oF; g.ldadd = NF;
    g.out0 = m.T2 + oF; g.out1 = m.Y2 + oF; g.ldo = NF;
    tc_gemm(TEPI_TANH_BIAS_SKIP, 240, m.mapA_Y1[t], m.mapB_fwd[t][1], g, s);
    g = TcGemmArgs{};
    g.M = rows; g.N = NF; g.K = NF; g.bias = m.fit_b[t][2]; g.add = m.Y2 + oF; g.ldadd = NF;
    g.out0 = m.T3 + oF; g.out1 = m.Y3 + oF; g.ldo = NF;
    tc_gemm(TEPI_TANH_BIAS_SKIP, 240, m.mapA_Y2[t], m.mapB_fwd[t][2], g, s);
    return 3;
}
int fitting_gemms_tc_bwd(Model& m, int t, cudaStream_t s) {
    const int NF = m.NF, ND = m.ND;
    const int row0 = m.type_row0[t], rows = m.type_row0[t + 1] - row0;
    const size_t oF = (size_t)row0 * NF, oD = (size_t)row0 * ND;
    TcGemmArgs g{};
    // dy2 = dy3 + da3 W3^T -> Y3 ; da2 = dy2 o (1 - t2^2) -> T3       (A = G1 = da3)
    g.M = rows; g.N = NF; g.K = NF; g.add = m.G2 + oF; g.ldadd = NF; g.tt = m.T2 + oF; g.ldtt = NF;
    g.out0 = m.Y3 + oF; g.out1 = m.T3 + oF; g.ldo = NF;
    tc_gemm(TEPI_BWD, 240, m.mapA_G1[t], m.mapB_bwd[t][2], g, s);
    // dy1 = dy2 + da2 W2^T ; da1 = dy1 o (1 - y1^2) -> G1                (A = T3 = da2)
    g = TcGemmArgs{};
    g.M = rows; g.N = NF; g.K = NF; g.add = m.Y3 + oF; g.ldadd = NF; g.tt = m.Y1 + oF; g.ldtt = NF;
    g.out1 = m.G1 + oF; g.ldo = NF;
    tc_gemm(TEPI_BWD_FIRST, 240, m.mapA_T3[t], m.mapB_bwd[t][1], g, s);
    // dD = da1 W1^T                                                     (A = G1 = da1)
    g = TcGemmArgs{};
    g.M = rows; g.N = ND; g.K = NF; g.out0 = m.dD + oD; g.ldo = ND;
    tc_gemm(TEPI_PLAIN, 160, m.mapA_G1[t], m.mapB_bwd[t][0], g, s);
    return 3;
}

// parity hook: C[M][N] = A[M][K] Bt[N][K]^T through the tensor-core kernel (N == 240 or N % 160 == 0, K % 16 == 0)
int debug_tc_gemm(int M, int N, int K, const float* A, const float* Bt, float* C, cudaStream_t s) {
    const int bn = (N == 240) ? 240 : 160;
    if ((bn == 160 && N % 160 != 0) || K % 16 != 0) return -1;
    CUtensorMap ma, mb;
    if (!tc_make_map(&ma, A, M, K, K, 128)) return -2;
    if (!tc_make_map(&mb, Bt, N, K, K, bn)) return -2;
    TcGemmArgs g{};
    g.M = M; g.N = N; g.K = K; g.out0 = C; g.ldo = N;
    return tc_gemm(TEPI_PLAIN, bn, ma, mb, g, s) == cudaSuccess ? 0 : -3;
}

}  // namespace pimd
