// fitting_tc.cu -- the fitting-net GEMMs of F4 on the 5th-generation tensor cores.
// One launch per layer covers the rows of all centre types (tiles numbered type by type).
//
//   C[M x N] = epilogue( A[M x K] . Bt[N x K]^T ),  FP32 in / FP32 out, computed as 3xTF32:
//   a = a_hi + a_lo, b = b_hi + b_lo (hi = top 10 mantissa bits, lo = exact remainder)
//   a.b ~= a_hi.b_hi + a_lo.b_hi + a_hi.b_lo     (FP32 accumulate in TMEM; dropped term ~2^-22)
// which keeps the force error at the FP32 level (single-pass TF32 fails north_star's 1e-4).
//
// One CTA computes a (128 NH) x BN tile (NH accumulators of M = 128 in TMEM).  Warp roles (192 threads):
//   warp 0   TMA producer: raw FP32 A (NH boxes 16 x 128) and the PRE-SPLIT weights B_hi, B_lo (boxes 16 x BN),
//            SWIZZLE_64B, ST stages
//   warp 1   TMEM allocation + single-thread tcgen05.mma issue (6 NH MMAs of 128 x BN x 8 per stage)
//   warps 2-5 split A into hi/lo in shared memory (elementwise, so the swizzled layout is preserved), then
//            the epilogue: tcgen05.ld accumulators -> bias / tanh / skip / derivative / energy -> global
// Two CTAs share an SM (2 x 256 TMEM columns, 2 x 2 stages), so one CTA's epilogue runs under the other's MMAs.
#include <algorithm>
#include <type_traits>
#include <cstdlib>
#include <cuda_fp16.h>
#include "common.cuh"
#include "tc_gemm.cuh"

namespace pimd {

using namespace tc;

enum : int { TEPI_TANH_BIAS = 0, TEPI_TANH_BIAS_SKIP = 1, TEPI_BWD_VEC = 2, TEPI_BWD_FIRST = 3, TEPI_PLAIN = 4, TEPI_L3E = 5 };

constexpr int kMaxT = PIMD_MAX_TYPES;

// one launch covers the rows of ALL centre types: M tiles are numbered type by type
struct TcMaps {
    CUtensorMap A[kMaxT];       // activations of type t: [rows_t][K], box 16 x 128
    CUtensorMap Bhi[kMaxT];     // weights of type t, TF32 hi part: [N][K] (K-major), box 16 x BN
    CUtensorMap Blo[kMaxT];     // exact remainder
};

struct TcGemmArgs {
    int tile_off;                   // first M tile of this launch (the chain runs in tile ranges on two streams)
    int ntypes, N, K;               // N = logical columns of C (grid.x chunks of BN)
    int tile0[kMaxT + 1];           // first M tile of each type
    int row0[kMaxT + 1];            // first (type-sorted) row of each type
    const float* bias[kMaxT];
    const float* vec[kMaxT];        // TEPI_L3E: w4 ; TEPI_BWD_VEC: dy3 = w4 (a row vector)
    const float* b4[kMaxT];
    const float* add; int ldadd;    // matrices indexed by the global (type-sorted) row
    const float* tt; int ldtt;
    float* out0; float* out1; int ldo;
    const int* cen_idx; double* Eatom; double* U; int natoms;    // TEPI_L3E
    float scale;                    // TEPI_BWD_FIRST: da1 is stored as FP16 hi / lo of scale * da1
};

constexpr int kTcThreads = 192;
constexpr int kTcBK = 16;                 // floats per K block = 64 B rows (SWIZZLE_64B)

template <int BN, int NH, int ST>
struct TcSmem {
    static constexpr int kABytes = 128 * 64;                      // one 128-row half
    static constexpr int kBBytes = BN * 64;
    static constexpr int oAhi = 0, oAlo = NH * kABytes, oBhi = 2 * NH * kABytes, oBlo = 2 * NH * kABytes + kBBytes;
    static constexpr int kStage = 2 * NH * kABytes + 2 * kBBytes;
    static constexpr int kEpiOff = ST * kStage + 256;                       // 4 warps x 32 x 20 floats: epilogue transpose
    static constexpr int kTotal = ST * kStage + 256 /*barriers*/ + 4 * 32 * 20 * 4 + 1024 /*align slack*/;
    static constexpr int kTmemCols = (NH * BN <= 256) ? 256 : 512;
};

// BN: N tile; EPI: epilogue; NH: 128-row halves per CTA; ST: pipeline stages; OCC: CTAs per SM
template <int BN, int EPI, int NH, int ST, int OCC>
__global__ void __launch_bounds__(kTcThreads, OCC)
gemm3xtf32_kernel(const __grid_constant__ TcMaps maps, const __grid_constant__ TcGemmArgs g) {
    using SM = TcSmem<BN, NH, ST>;
    extern __shared__ uint8_t smem_raw[];
    uint8_t* smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);   // keeps the shared address space
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem + ST * SM::kStage);
    uint64_t* full = bars;                     // [stages] TMA -> split warps (A) and MMA (B)
    uint64_t* ready = bars + ST;               // [stages] split warps -> MMA
    uint64_t* empty = bars + 2 * ST;           // [stages] MMA -> TMA
    uint64_t* tmem_full = bars + 3 * ST;
    uint32_t* tmem_ptr = reinterpret_cast<uint32_t*>(bars + 3 * ST + 1);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int tile = (int)blockIdx.y + g.tile_off;
    int ty = 0;
#pragma unroll
    for (int t = 1; t < kMaxT; ++t)
        if (t < g.ntypes && tile >= g.tile0[t]) ty = t;
    const int m0 = (tile - g.tile0[ty]) * (128 * NH), n0 = blockIdx.x * BN;
    const int rows_t = g.row0[ty + 1] - g.row0[ty];
    const int nk = g.K / kTcBK;
    const CUtensorMap* mapA = &maps.A[ty];
    const CUtensorMap* mapBhi = &maps.Bhi[ty];
    const CUtensorMap* mapBlo = &maps.Blo[ty];

    if (warp == 0 && lane == 0) {
        tma_prefetch_desc(mapA);
        tma_prefetch_desc(mapBhi);
        tma_prefetch_desc(mapBlo);
        for (int s = 0; s < ST; ++s) { mbar_init(full + s, 1); mbar_init(ready + s, 128); mbar_init(empty + s, 1); }
        mbar_init(tmem_full, 1);
        fence_barrier_init();
    }
    if (warp == 1) tmem_alloc(tmem_ptr, SM::kTmemCols);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_ptr;

    if (warp == 0) {
        if (lane == 0) {
            for (int kb = 0; kb < nk; ++kb) {
                const int s = kb % ST, ph = (kb / ST) & 1;
                mbar_wait(empty + s, ph ^ 1);
                uint8_t* st = smem + s * SM::kStage;
                mbar_arrive_expect_tx(full + s, NH * SM::kABytes + 2 * SM::kBBytes);
#pragma unroll
                for (int h = 0; h < NH; ++h) tma_load_2d(st + SM::oAhi + h * SM::kABytes, mapA, full + s, kb * kTcBK, m0 + 128 * h);
                tma_load_2d(st + SM::oBhi, mapBhi, full + s, kb * kTcBK, n0);
                tma_load_2d(st + SM::oBlo, mapBlo, full + s, kb * kTcBK, n0);
            }
        }
    } else if (warp == 1) {
        if (lane == 0) {
            constexpr uint32_t idesc = make_idesc_tf32(128, BN);
            for (int kb = 0; kb < nk; ++kb) {
                const int s = kb % ST, ph = (kb / ST) & 1;
                mbar_wait(ready + s, ph);
                tc_fence_after();
                const uint32_t st = smem_u32(smem + s * SM::kStage);
#pragma unroll
                for (int h = 0; h < NH; ++h) {
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
        // ---- split A into hi / lo in place (128 threads; elementwise, so the swizzled layout is preserved;
        //      the weights arrive pre-split) ----
        const int t = threadIdx.x - 64;
        for (int kb = 0; kb < nk; ++kb) {
            const int s = kb % ST, ph = (kb / ST) & 1;
            mbar_wait(full + s, ph);
            uint8_t* st = smem + s * SM::kStage;
            float4* a_hi = reinterpret_cast<float4*>(st + SM::oAhi);
            float4* a_lo = reinterpret_cast<float4*>(st + SM::oAlo);
#pragma unroll
            for (int q = 0; q < (NH * SM::kABytes / 16) / 128; ++q) {
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
            fence_proxy_async_smem();
            mbar_arrive(ready + s);
        }
        // ---- epilogue.  tcgen05.ld hands every lane one ROW of the accumulator; row-per-lane global accesses
        // would touch 32 different 128 B lines per instruction (the L1 tag stage then bounds the epilogue), so each
        // 32 x 16 chunk goes through a per-warp shared-memory patch and comes back as lane <-> (row l/4 + 8 j,
        // columns 4 (l % 4) .. + 3), j = 0..3: a warp-wide float4 access then covers 8 rows x 64 contiguous bytes.
        // All epilogue math is elementwise, so it runs in that layout; `add` / `tt` are fetched one chunk ahead. ----
        mbar_wait(tmem_full, 0);
        tc_fence_after();
        const int quarter = warp & 3;                      // TMEM lane quarter this warp may access
        constexpr bool kAdd = (EPI == TEPI_TANH_BIAS_SKIP || EPI == TEPI_L3E || EPI == TEPI_BWD_FIRST);
        constexpr bool kTt = (EPI == TEPI_BWD_VEC || EPI == TEPI_BWD_FIRST);
        constexpr bool kTanh = (EPI == TEPI_TANH_BIAS || EPI == TEPI_TANH_BIAS_SKIP || EPI == TEPI_L3E);
        float* patch = reinterpret_cast<float*>(smem + SM::kEpiOff) + (warp - 2) * (32 * 20);
        const int lr = lane >> 2, lc = 4 * (lane & 3);     // my row (+ 8 j) and column offset inside a chunk
        const float4 zero4 = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll 1
        for (int h = 0; h < NH; ++h) {
            const int mbase = m0 + h * 128 + quarter * 32;         // first row of this warp inside the type
            bool ok[4];
            size_t mrow[4];
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                ok[j] = mbase + lr + 8 * j < rows_t;
                mrow[j] = (size_t)(g.row0[ty] + (ok[j] ? mbase + lr + 8 * j : 0));
            }
            float e_acc[4] = {0.f, 0.f, 0.f, 0.f};
            float4 adn[4], ttn[4];
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                adn[j] = (kAdd && ok[j] && n0 < g.N) ? *reinterpret_cast<const float4*>(g.add + mrow[j] * g.ldadd + n0 + lc) : zero4;
                ttn[j] = (kTt && ok[j] && n0 < g.N) ? *reinterpret_cast<const float4*>(g.tt + mrow[j] * g.ldtt + n0 + lc) : zero4;
            }
#pragma unroll 1
            for (int c = 0; c < BN / 16; ++c) {
                uint32_t v[16];
                tmem_ld16(tmem_base + ((uint32_t)(quarter * 32) << 16) + h * 256 + c * 16, v);
                float4 ad[4], t4[4];
#pragma unroll
                for (int j = 0; j < 4; ++j) { ad[j] = adn[j]; t4[j] = ttn[j]; }
                const int n = n0 + c * 16;
                const bool more = (c + 1 < BN / 16) && (n + 16 < g.N);
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    if (kAdd) adn[j] = (more && ok[j]) ? *reinterpret_cast<const float4*>(g.add + mrow[j] * g.ldadd + n + 16 + lc) : zero4;
                    if (kTt) ttn[j] = (more && ok[j]) ? *reinterpret_cast<const float4*>(g.tt + mrow[j] * g.ldtt + n + 16 + lc) : zero4;
                }
                tmem_ld_wait();
                // transpose through the patch: row `lane` in, (row lr + 8 j, columns lc..lc+3) out
#pragma unroll
                for (int q = 0; q < 4; ++q)
                    *reinterpret_cast<float4*>(patch + lane * 20 + 4 * q) =
                        make_float4(__uint_as_float(v[4 * q]), __uint_as_float(v[4 * q + 1]), __uint_as_float(v[4 * q + 2]), __uint_as_float(v[4 * q + 3]));
                __syncwarp();
                float4 r[4];
#pragma unroll
                for (int j = 0; j < 4; ++j) r[j] = *reinterpret_cast<const float4*>(patch + (lr + 8 * j) * 20 + lc);
                __syncwarp();
                if (n >= g.N) continue;
                if (kTanh) {
                    const float4 b4 = __ldg(reinterpret_cast<const float4*>(g.bias[ty] + n + lc));
#pragma unroll
                    for (int j = 0; j < 4; ++j) {
                        r[j].x = tanh_fast(r[j].x + b4.x); r[j].y = tanh_fast(r[j].y + b4.y);
                        r[j].z = tanh_fast(r[j].z + b4.z); r[j].w = tanh_fast(r[j].w + b4.w);
                    }
                }
                float4 w = zero4;
                if (EPI == TEPI_L3E || EPI == TEPI_BWD_VEC) w = __ldg(reinterpret_cast<const float4*>(g.vec[ty] + n + lc));
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    if (!ok[j]) continue;
                    float4* o0 = (g.out0 != nullptr) ? reinterpret_cast<float4*>(g.out0 + mrow[j] * g.ldo + n + lc) : nullptr;
                    float4* o1 = (g.out1 != nullptr) ? reinterpret_cast<float4*>(g.out1 + mrow[j] * g.ldo + n + lc) : nullptr;
                    if (EPI == TEPI_TANH_BIAS || EPI == TEPI_PLAIN) {
                        *o0 = r[j];
                    } else if (EPI == TEPI_TANH_BIAS_SKIP) {
                        *o0 = r[j];
                        *o1 = make_float4(r[j].x + ad[j].x, r[j].y + ad[j].y, r[j].z + ad[j].z, r[j].w + ad[j].w);
                    } else if (EPI == TEPI_L3E) {
                        // y3 = y2 + t3 ; E_i += y3 . w4 ; seed of the backward pass da3 = w4 o (1 - t3^2) -> out1
                        e_acc[j] = fmaf(ad[j].x + r[j].x, w.x, e_acc[j]);
                        e_acc[j] = fmaf(ad[j].y + r[j].y, w.y, e_acc[j]);
                        e_acc[j] = fmaf(ad[j].z + r[j].z, w.z, e_acc[j]);
                        e_acc[j] = fmaf(ad[j].w + r[j].w, w.w, e_acc[j]);
                        *o1 = make_float4(w.x * (1.f - r[j].x * r[j].x), w.y * (1.f - r[j].y * r[j].y),
                                          w.z * (1.f - r[j].z * r[j].z), w.w * (1.f - r[j].w * r[j].w));
                    } else {   // TEPI_BWD_VEC (add = the row vector w4), TEPI_BWD_FIRST
                        const float4 a4 = (EPI == TEPI_BWD_VEC) ? w : ad[j];
                        const float4 tq = t4[j];
                        float4 y = make_float4(r[j].x + a4.x, r[j].y + a4.y, r[j].z + a4.z, r[j].w + a4.w);
                        if (EPI == TEPI_BWD_VEC) *o0 = y;
                        y.x *= (1.f - tq.x * tq.x); y.y *= (1.f - tq.y * tq.y);
                        y.z *= (1.f - tq.z * tq.z); y.w *= (1.f - tq.w * tq.w);
                        if (EPI == TEPI_BWD_FIRST) {
                            // da1 feeds dd_dt_kernel only: stored as FP16 hi (-> out1) / lo (-> out0) of scale * da1,
                            // [rows][240] halfs (the power-of-two scale keeps the values in FP16's normal range)
                            const __half2 h01 = __floats2half2_rn(y.x * g.scale, y.y * g.scale);
                            const __half2 h23 = __floats2half2_rn(y.z * g.scale, y.w * g.scale);
                            const float2 f01 = __half22float2(h01), f23 = __half22float2(h23);
                            const __half2 l01 = __floats2half2_rn(y.x * g.scale - f01.x, y.y * g.scale - f01.y);
                            const __half2 l23 = __floats2half2_rn(y.z * g.scale - f23.x, y.w * g.scale - f23.y);
                            __half* ph = reinterpret_cast<__half*>(g.out1) + mrow[j] * g.ldo + n + lc;
                            __half* pl = reinterpret_cast<__half*>(g.out0) + mrow[j] * g.ldo + n + lc;
                            *reinterpret_cast<uint2*>(ph) = make_uint2(*reinterpret_cast<const uint32_t*>(&h01), *reinterpret_cast<const uint32_t*>(&h23));
                            *reinterpret_cast<uint2*>(pl) = make_uint2(*reinterpret_cast<const uint32_t*>(&l01), *reinterpret_cast<const uint32_t*>(&l23));
                        } else {
                            *o1 = y;
                        }
                    }
                }
            }
            if (EPI == TEPI_L3E) {
                // E_i = y3 . w4 + b4: the four lanes of a row add their column shares; lane 4 r then owns rows
                // r + 8 j.  U^(bead) += E_i with one atomic per warp when all its rows share the bead.
                double esum = 0.0;
                int bead_u = -1;
                bool uniform = true;
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    float e = e_acc[j];
                    e += __shfl_xor_sync(0xffffffffu, e, 1);
                    e += __shfl_xor_sync(0xffffffffu, e, 2);
                    const bool mine = ok[j] && (lane & 3) == 0;
                    const int ba = mine ? g.cen_idx[mrow[j]] : 0;
                    const double ed = mine ? (double)(e + __ldg(g.b4[ty])) : 0.0;
                    if (mine) g.Eatom[ba] = ed;
                    const int bead = mine ? ba / g.natoms : -1;
                    const int bmax = __reduce_max_sync(0xffffffffu, bead);
                    const bool same = __all_sync(0xffffffffu, bead < 0 || bead == bmax);
                    if (same && (bead_u < 0 || bmax < 0 || bmax == bead_u)) {
                        esum += ed;
                        if (bmax >= 0) bead_u = bmax;
                    } else {
                        uniform = false;
                        if (mine) atomicAdd(g.U + bead, ed);
                    }
                }
                (void)uniform;
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) esum += __shfl_xor_sync(0xffffffffu, esum, o);
                if (lane == 0 && bead_u >= 0) atomicAdd(g.U + bead_u, esum);
            }
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 1) tmem_dealloc(tmem_base, SM::kTmemCols);
}

// ---------------------------------------------------------------------------------------------
// Layer 1 fused with the descriptor (F3 -> F4 hand-over): Y1 = tanh(D W1 + b1) with
// D[i][16 m1 + m2] = T[i][m1] . T[i][m2] (R-14) produced on the fly -- K block kb of the A operand is exactly
// m1 = kb, so the producer thread of row i needs T[i][kb] (one float4 per K block) and T[i][0:16] (registers).
// D (rows x 1600, 315 MB at configs[2]) is neither written nor read.  The weights arrive pre-split by TMA.
// ---------------------------------------------------------------------------------------------
struct L1Args {
    int tile_off;
    int ntypes, K;
    int tile0[kMaxT + 1];
    int row0[kMaxT + 1];
    const float* bias[kMaxT];
    const float* Tm;      // [rows][100][4]
    float* out; int ldo;  // Y1 (FP32), or
    uint8_t* out_img;     // when set: Y1 as the operand image of fit_mid_kernel, [tile] x 128 KB: [hi | lo][K block 8][128 rows x 64 B, SWIZZLE_64B order]
    const uint8_t* wimg[kMaxT];       // W1^T x 64 as shared-memory images, [K block of 32][hi | lo][240 rows x 64 B]
    int M1;
};

// FP16-split operands (kind::f16, three passes, FP32 accumulate; see embedding_tc.cu): D is scaled by 256 and W1 by
// 64 (exact powers of two) so that hi and lo stay in FP16's normal range -- |D| <= 4 (3 x 1.2)^2 ~ 52 by
// construction (|G| <= 3, |R| <= ~1.2, at most N_sel rows), so 256 |D| < 65504 -- and the epilogue multiplies the
// accumulator by 2^-14.  A stage holds K = 32 (two m1 values): 50 stages of 6 MMAs instead of 100.
constexpr int kL1BN = 240, kL1ST = 4;
constexpr int kL1Threads = 320;         // warp 0: TMA, warp 1: MMA issue, warps 2-9: operand producers + epilogue
constexpr float kL1DScale = 256.f, kW1Scale = 64.f;
struct L1Smem {
    static constexpr int kABytes = 128 * 64, kBBytes = kL1BN * 64;        // 64 B rows = 32 halfs, SWIZZLE_64B
    static constexpr int oAhi = 0, oAlo = kABytes, oBhi = 2 * kABytes, oBlo = 2 * kABytes + kBBytes;
    static constexpr int kStage = 2 * kABytes + 2 * kBBytes;               // 47104
    static constexpr int oBias = kL1ST * kStage;                           // float [240]
    static constexpr int oBars = oBias + kL1BN * 4;
    static constexpr int kTotal = oBars + 256 + 1024;
};

__global__ void __launch_bounds__(kL1Threads, 1)
l1_desc_kernel(const __grid_constant__ TcMaps maps, const __grid_constant__ L1Args g) {
    using SM = L1Smem;
    constexpr int ST = kL1ST, BN = kL1BN;
    extern __shared__ uint8_t smem_raw[];
    uint8_t* smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem + SM::oBars);
    uint64_t* full = bars;                     // TMA (weights) -> MMA
    uint64_t* ready = bars + ST;               // producer threads (A = D block) -> MMA
    uint64_t* empty = bars + 2 * ST;           // MMA -> TMA and producers
    uint64_t* tmem_full = bars + 3 * ST;
    uint32_t* tmem_ptr = reinterpret_cast<uint32_t*>(bars + 3 * ST + 1);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int tile = (int)blockIdx.x + g.tile_off;
    int ty = 0;
#pragma unroll
    for (int t = 1; t < kMaxT; ++t)
        if (t < g.ntypes && tile >= g.tile0[t]) ty = t;
    const int m0 = (tile - g.tile0[ty]) * 128;
    const int rows_t = g.row0[ty + 1] - g.row0[ty];
    const int nk = g.K / 32;                   // K = 16 m1: two m1 per stage

    if (warp == 0 && lane == 0) {
        for (int s = 0; s < ST; ++s) { mbar_init(full + s, 1); mbar_init(ready + s, 256); mbar_init(empty + s, 1); }
        mbar_init(tmem_full, 1);
        fence_barrier_init();
    }
    if (warp == 1) tmem_alloc(tmem_ptr, 256);
    if (threadIdx.x < BN) reinterpret_cast<float*>(smem + SM::oBias)[threadIdx.x] = __ldg(g.bias[ty] + threadIdx.x);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_ptr;

    // control warps: all 32 lanes run the loop converged, one elected lane issues (tc_gemm.cuh)
    if (warp == 0) {
        const uint8_t* wimg = g.wimg[ty];
        int s = 0, ph = 1;
        for (int kb = 0; kb < nk; ++kb) {
            mbar_wait(empty + s, ph);
            bulk_load_expect_elect(smem + s * SM::kStage + SM::oBhi, wimg + (size_t)kb * (2 * SM::kBBytes), 2 * SM::kBBytes, full + s);
            if (++s == ST) { s = 0; ph ^= 1; }
        }
    } else if (warp == 1) {
        constexpr uint32_t idesc = make_idesc_f16(128, BN);
        const uint32_t sb = smem_u32(smem);
        const uint64_t dAh = make_smem_desc_kmajor(sb + SM::oAhi, 64), dAl = make_smem_desc_kmajor(sb + SM::oAlo, 64);
        const uint64_t dBh = make_smem_desc_kmajor(sb + SM::oBhi, 64), dBl = make_smem_desc_kmajor(sb + SM::oBlo, 64);
        int s = 0, ph = 0;
        for (int kb = 0; kb < nk; ++kb) {
            mbar_wait(full + s, ph);
            mbar_wait(ready + s, ph);
            tc_fence_after();
            const uint64_t so = (uint64_t)((s * SM::kStage) >> 4);
            umma_f16_elect(tmem_base, dAh + so, dBh + so, idesc, kb ? 1u : 0u);
            umma_f16_elect(tmem_base, dAl + so, dBh + so, idesc, 1u);
            umma_f16_elect(tmem_base, dAh + so, dBl + so, idesc, 1u);
            umma_f16_elect(tmem_base, dAh + so + 2, dBh + so + 2, idesc, 1u);
            umma_f16_elect(tmem_base, dAl + so + 2, dBh + so + 2, idesc, 1u);
            umma_f16_elect(tmem_base, dAh + so + 2, dBl + so + 2, idesc, 1u);
            umma_commit_elect(empty + s);
            if (++s == ST) { s = 0; ph ^= 1; }
        }
        umma_commit_elect(tmem_full);
    } else {
        // two warps per TMEM lane quarter (a warp alone on its scheduler cannot hide the latency of its own loads and
        // conversions; the round-2 profile had the tensor pipe 46 % active behind four producer warps): warp `half`
        // of a quarter produces m1 = 2 kb + half of every stage and takes the epilogue chunks c = half, half + 2, ...
        const int quarter = warp & 3, half = (warp - 2) >> 2;
        const int row = quarter * 32 + lane;                   // tile row = TMEM lane
        const int ml = m0 + row;
        const bool row_ok = ml < rows_t;
        const size_t m = (size_t)(g.row0[ty] + (row_ok ? ml : 0));
        const float4* Trow = reinterpret_cast<const float4*>(g.Tm) + m * g.M1;
        const float4 zero4 = make_float4(0.f, 0.f, 0.f, 0.f);
        float4 T2[16];
#pragma unroll
        for (int m2 = 0; m2 < 16; ++m2) {
            T2[m2] = row_ok ? __ldg(Trow + m2) : zero4;
            T2[m2].x *= kL1DScale; T2[m2].y *= kL1DScale; T2[m2].z *= kL1DScale; T2[m2].w *= kL1DScale;   // D x 256
        }
        // SWIZZLE_64B K-major block: 64 B rows (32 halfs), 16 B chunk index XOR ((row >> 1) & 3)
        const int rbase = row * 64, sw = (row >> 1) & 3;
        auto load_T1 = [&](int kb) { return (row_ok && kb < nk) ? __ldg(Trow + 2 * kb + half) : zero4; };
        // T[i][m1] is fetched three stages ahead of its use into three named registers; the loop is unrolled by hand
        // so that no register that is the target of a load in flight gets moved (a rotation Ta = Tb; Tb = Tc; ... makes
        // every move wait for the load behind it, which cut the prefetch distance to one stage in the first version)
        float4 Ta = load_T1(0), Tb = load_T1(1), Tc = load_T1(2);
        auto stage = [&](int kb, const float4 Ta) {
            const int s = kb % ST, ph = (kb / ST) & 1;
            uint32_t hi[8], lo[8];                              // K indices 16 half .. 16 half + 15 of the stage, packed in pairs
#pragma unroll
            for (int q = 0; q < 8; ++q) {
                const int m2 = 2 * q;
                const float d0 = Ta.x * T2[m2].x + Ta.y * T2[m2].y + Ta.z * T2[m2].z + Ta.w * T2[m2].w;
                const float d1 = Ta.x * T2[m2 + 1].x + Ta.y * T2[m2 + 1].y + Ta.z * T2[m2 + 1].z + Ta.w * T2[m2 + 1].w;
                const __half2 h = __floats2half2_rn(d0, d1);
                const float2 hf = __half22float2(h);
                const __half2 l = __floats2half2_rn(d0 - hf.x, d1 - hf.y);
                hi[q] = *reinterpret_cast<const uint32_t*>(&h);
                lo[q] = *reinterpret_cast<const uint32_t*>(&l);
            }
            mbar_wait(empty + s, ph ^ 1);                       // the MMAs that read this stage have retired
            uint8_t* st = smem + s * SM::kStage;
#pragma unroll
            for (int c2 = 0; c2 < 2; ++c2) {
                const int off = rbase + (((2 * half + c2) ^ sw) << 4);
                *reinterpret_cast<uint4*>(st + SM::oAhi + off) = make_uint4(hi[4 * c2], hi[4 * c2 + 1], hi[4 * c2 + 2], hi[4 * c2 + 3]);
                *reinterpret_cast<uint4*>(st + SM::oAlo + off) = make_uint4(lo[4 * c2], lo[4 * c2 + 1], lo[4 * c2 + 2], lo[4 * c2 + 3]);
            }
            fence_proxy_async_smem();
            mbar_arrive(ready + s);
        };
        for (int kb = 0; kb < nk; kb += 3) {
            stage(kb, Ta);
            Ta = load_T1(kb + 3);
            if (kb + 1 < nk) stage(kb + 1, Tb);
            Tb = load_T1(kb + 4);
            if (kb + 2 < nk) stage(kb + 2, Tc);
            Tc = load_T1(kb + 5);
        }
        // ---- epilogue: Y1 = tanh(acc 2^-14 + b1) ----
        mbar_wait(tmem_full, 0);
        tc_fence_after();
        float* orow = g.out + m * g.ldo;
        constexpr float kInv = 1.f / (kL1DScale * kW1Scale);
#pragma unroll 1
        for (int c = half; c < BN / 16; c += 2) {
            uint32_t v[16];
            tmem_ld16(tmem_base + ((uint32_t)(quarter * 32) << 16) + c * 16, v);
            float bv[16];
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                const float4 b4 = reinterpret_cast<const float4*>(smem + SM::oBias + c * 64)[q];
                bv[4 * q] = b4.x; bv[4 * q + 1] = b4.y; bv[4 * q + 2] = b4.z; bv[4 * q + 3] = b4.w;
            }
            tmem_ld_wait();
            if (!row_ok) continue;
            float r[16];
#pragma unroll
            for (int q = 0; q < 16; ++q) r[q] = tanh_fast(fmaf(__uint_as_float(v[q]), kInv, bv[q]));
            if (g.out_img) {
                // the stage memory is idle (tmem_full: every MMA has retired): the image of this tile is put together there
                uint32_t hi[8], lo[8];
#pragma unroll
                for (int q = 0; q < 8; ++q) {
                    const __half2 h = __floats2half2_rn(r[2 * q], r[2 * q + 1]);
                    const float2 hf = __half22float2(h);
                    const __half2 l = __floats2half2_rn(r[2 * q] - hf.x, r[2 * q + 1] - hf.y);
                    hi[q] = *reinterpret_cast<const uint32_t*>(&h);
                    lo[q] = *reinterpret_cast<const uint32_t*>(&l);
                }
                const int base = (c >> 1) * (128 * 64) + rbase, ci = 2 * (c & 1);
                const int o0 = base + ((ci ^ sw) << 4), o1 = base + (((ci + 1) ^ sw) << 4);
                *reinterpret_cast<uint4*>(smem + o0) = make_uint4(hi[0], hi[1], hi[2], hi[3]);
                *reinterpret_cast<uint4*>(smem + o1) = make_uint4(hi[4], hi[5], hi[6], hi[7]);
                *reinterpret_cast<uint4*>(smem + 65536 + o0) = make_uint4(lo[0], lo[1], lo[2], lo[3]);
                *reinterpret_cast<uint4*>(smem + 65536 + o1) = make_uint4(lo[4], lo[5], lo[6], lo[7]);
                continue;
            }
#pragma unroll
            for (int q = 0; q < 4; ++q)
                reinterpret_cast<float4*>(orow + c * 16)[q] = make_float4(r[4 * q], r[4 * q + 1], r[4 * q + 2], r[4 * q + 3]);
        }
        if (g.out_img) {
            fence_proxy_async_smem();
            asm volatile("bar.sync 5, 256;" ::: "memory");
            if (warp == 2 && lane == 0) {
                uint8_t* img = g.out_img + (size_t)tile * 131072;
                bulk_store(img, smem, 65536);
                bulk_store(img + 65536, smem + 65536, 65536);
                bulk_commit();
                bulk_wait_read0();             // shared memory may go once it has been read; the writes complete with the grid
            }
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 1) tmem_dealloc(tmem_base, 256);
}

// ---------------------------------------------------------------------------------------------
// The same layer with the A operand in TENSOR MEMORY (tcgen05.mma TS mode; the path of the fused chain).  The D block
// of a stage is produced by the thread that owns the row = TMEM lane, so it goes where it was made: tcgen05.st into
// a 4-stage ring of 32 columns (16 hi + 16 lo, two FP16 per column) behind the accumulator -- no swizzle, no proxy
// fence, no shared-memory traffic for A -- and the 128 KB of shared memory this frees hold SEVEN weight stages
// instead of four: the weight stream through a 4-deep ring was what this kernel waited for (24.9 us with MMAs and
// producers switched off, profiles/r2_README.md).
// ---------------------------------------------------------------------------------------------
struct L1TsSmem {
    static constexpr int kST = 7;                                          // weight stages
    static constexpr int kBBytes = kL1BN * 64;                             // one copy (hi or lo) of a K block of 32: 64 B rows, SWIZZLE_64B
    static constexpr int kStage = 2 * kBBytes;                             // 30720
    static constexpr int oBias = kST * kStage;                             // float [240]
    static constexpr int oBars = oBias + kL1BN * 4;
    static constexpr int kTotal = oBars + 256 + 1024;
};
static_assert(L1TsSmem::kTotal <= 232448 && L1TsSmem::oBias >= 131072, "shared memory budget / room for the y1 image");
constexpr int kL1AST = 4, kL1ACol = 256;      // A ring: stage s at TMEM columns 256 + 32 s (hi: +0..15, lo: +16..31)

__global__ void __launch_bounds__(kL1Threads, 1)
l1_desc_ts_kernel(const __grid_constant__ L1Args g) {
    using SM = L1TsSmem;
    constexpr int ST = SM::kST, AST = kL1AST, BN = kL1BN;
    extern __shared__ uint8_t smem_raw[];
    uint8_t* smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem + SM::oBars);
    uint64_t* b_full = bars;                   // [ST]  weights landed -> MMA
    uint64_t* b_empty = bars + ST;             // [ST]  MMA -> TMA
    uint64_t* a_ready = bars + 2 * ST;         // [AST] producers -> MMA (count 256)
    uint64_t* a_empty = bars + 2 * ST + AST;   // [AST] MMA -> producers
    uint64_t* tmem_full = bars + 2 * ST + 2 * AST;
    uint64_t* blk_done = bars + 2 * ST + 2 * AST + 1;   // [8] epilogue -> store: K block kb of the y1 image is complete (count 256)
    uint32_t* tmem_ptr = reinterpret_cast<uint32_t*>(bars + 2 * ST + 2 * AST + 9);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int tile = (int)blockIdx.x + g.tile_off;
    int ty = 0;
#pragma unroll
    for (int t = 1; t < kMaxT; ++t)
        if (t < g.ntypes && tile >= g.tile0[t]) ty = t;
    const int m0 = (tile - g.tile0[ty]) * 128;
    const int rows_t = g.row0[ty + 1] - g.row0[ty];
    const int nk = g.K / 32;                   // K = 16 m1: two m1 per stage

    if (warp == 0 && lane == 0) {
        for (int s = 0; s < ST; ++s) { mbar_init(b_full + s, 1); mbar_init(b_empty + s, 1); }
        for (int s = 0; s < AST; ++s) { mbar_init(a_ready + s, 256); mbar_init(a_empty + s, 1); }
        mbar_init(tmem_full, 1);
        for (int kb = 0; kb < 8; ++kb) mbar_init(blk_done + kb, 256);
        fence_barrier_init();
    }
    if (warp == 1) tmem_alloc(tmem_ptr, 512);
    if (threadIdx.x < BN) reinterpret_cast<float*>(smem + SM::oBias)[threadIdx.x] = __ldg(g.bias[ty] + threadIdx.x);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_ptr;

    // control warps: all 32 lanes run the loop converged, one elected lane issues (tc_gemm.cuh)
    if (warp == 0) {
        const uint8_t* wimg = g.wimg[ty];
        int s = 0, ph = 1;
        for (int kb = 0; kb < nk; ++kb) {
            mbar_wait(b_empty + s, ph);
            bulk_load_expect_elect(smem + s * SM::kStage, wimg + (size_t)kb * SM::kStage, SM::kStage, b_full + s);
            if (++s == ST) { s = 0; ph ^= 1; }
        }
        // the y1 image leaves K block by K block, behind the epilogue (a single 128 KB store at the end took 2.4 us)
        uint8_t* img = g.out_img + (size_t)tile * 131072;
        for (int kb = 0; kb < 8; ++kb) {
            mbar_wait(blk_done + kb, 0);
            if (lane == 0) {
                bulk_store(img + kb * 8192, smem + kb * 8192, 8192);
                bulk_store(img + 65536 + kb * 8192, smem + 65536 + kb * 8192, 8192);
                bulk_commit();
            }
        }
        if (lane == 0) bulk_wait_read0();      // shared memory may go once it has been read; the writes complete with the grid
    } else if (warp == 1) {
        constexpr uint32_t idesc = make_idesc_f16(128, BN);
        const uint32_t sb = smem_u32(smem);
        const uint64_t dBh = make_smem_desc_kmajor(sb, 64), dBl = make_smem_desc_kmajor(sb + SM::kBBytes, 64);
        int s = 0, ph = 0;
        for (int kb = 0; kb < nk; ++kb) {
            const int sa = kb & (AST - 1), pa = (kb / AST) & 1;
            mbar_wait(b_full + s, ph);
            mbar_wait(a_ready + sa, pa);
            tc_fence_after();
            const uint64_t bo = (uint64_t)((s * SM::kStage) >> 4);
            const uint32_t acol = tmem_base + kL1ACol + 32 * sa;
            umma_f16_ts_elect(tmem_base, acol, dBh + bo, idesc, kb ? 1u : 0u);
            umma_f16_ts_elect(tmem_base, acol + 16, dBh + bo, idesc, 1u);
            umma_f16_ts_elect(tmem_base, acol, dBl + bo, idesc, 1u);
            umma_f16_ts_elect(tmem_base, acol + 8, dBh + bo + 2, idesc, 1u);
            umma_f16_ts_elect(tmem_base, acol + 24, dBh + bo + 2, idesc, 1u);
            umma_f16_ts_elect(tmem_base, acol + 8, dBl + bo + 2, idesc, 1u);
            umma_commit_elect(a_empty + sa);
            umma_commit_elect(b_empty + s);
            if (++s == ST) { s = 0; ph ^= 1; }
        }
        umma_commit_elect(tmem_full);
    } else {
        // two warps per TMEM lane quarter: warp `half` of a quarter produces m1 = 2 kb + half of every stage (= k-step
        // `half` of the stage: 8 columns of hi, 8 of lo) and takes the epilogue chunks c = half, half + 2, ...
        const int quarter = warp & 3, half = (warp - 2) >> 2;
        const int row = quarter * 32 + lane;                   // tile row = TMEM lane
        const int ml = m0 + row;
        const bool row_ok = ml < rows_t;
        const size_t m = (size_t)(g.row0[ty] + (row_ok ? ml : 0));
        const float4* Trow = reinterpret_cast<const float4*>(g.Tm) + m * g.M1;
        const float4 zero4 = make_float4(0.f, 0.f, 0.f, 0.f);
        const uint32_t lanefield = ((uint32_t)(quarter * 32)) << 16;
        float4 T2[16];
#pragma unroll
        for (int m2 = 0; m2 < 16; ++m2) {
            T2[m2] = row_ok ? __ldg(Trow + m2) : zero4;
            T2[m2].x *= kL1DScale; T2[m2].y *= kL1DScale; T2[m2].z *= kL1DScale; T2[m2].w *= kL1DScale;   // D x 256
        }
        auto load_T1 = [&](int kb) { return (row_ok && kb < nk) ? __ldg(Trow + 2 * kb + half) : zero4; };
        // T[i][m1] three stages ahead in three named registers, loop unrolled by hand (no moves of registers with a load in flight)
        float4 Ta = load_T1(0), Tb = load_T1(1), Tc = load_T1(2);
        auto stage = [&](int kb, const float4 Ta) {
            const int sa = kb & (AST - 1), pa = (kb / AST) & 1;
            uint32_t hi[8], lo[8];                              // K indices 16 half .. 16 half + 15 of the stage, two per word
#pragma unroll
            for (int q = 0; q < 8; ++q) {
                const int m2 = 2 * q;
                const float d0 = Ta.x * T2[m2].x + Ta.y * T2[m2].y + Ta.z * T2[m2].z + Ta.w * T2[m2].w;
                const float d1 = Ta.x * T2[m2 + 1].x + Ta.y * T2[m2 + 1].y + Ta.z * T2[m2 + 1].z + Ta.w * T2[m2 + 1].w;
                const __half2 h = __floats2half2_rn(d0, d1);
                const float2 hf = __half22float2(h);
                const __half2 l = __floats2half2_rn(d0 - hf.x, d1 - hf.y);
                hi[q] = *reinterpret_cast<const uint32_t*>(&h);
                lo[q] = *reinterpret_cast<const uint32_t*>(&l);
            }
            mbar_wait(a_empty + sa, pa ^ 1);                    // the MMAs that read this A stage have retired
            tc_fence_after();
            const uint32_t col = tmem_base + lanefield + kL1ACol + 32 * sa + 8 * half;
            tmem_st8(col, hi);
            tmem_st8(col + 16, lo);
            tmem_st_wait();
            tc_fence_before();
            mbar_arrive(a_ready + sa);
        };
        for (int kb = 0; kb < nk; kb += 3) {
            stage(kb, Ta);
            Ta = load_T1(kb + 3);
            if (kb + 1 < nk) stage(kb + 1, Tb);
            Tb = load_T1(kb + 4);
            if (kb + 2 < nk) stage(kb + 2, Tc);
            Tc = load_T1(kb + 5);
        }
        // ---- epilogue: Y1 = tanh(acc 2^-14 + b1), assembled as the operand image of fit_mid_kernel in the (now idle:
        // tmem_full says every MMA has retired) weight stages and handed over with one bulk store ----
        mbar_wait(tmem_full, 0);
        tc_fence_after();
        constexpr float kInv = 1.f / (kL1DScale * kW1Scale);
        const int rbase = row * 64, sw = (row >> 1) & 3;
#pragma unroll 1
        for (int c = half; c < BN / 16; c += 2) {
            uint32_t v[16];
            tmem_ld16(tmem_base + lanefield + c * 16, v);
            float bv[16];
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                const float4 b4 = reinterpret_cast<const float4*>(smem + SM::oBias + c * 64)[q];
                bv[4 * q] = b4.x; bv[4 * q + 1] = b4.y; bv[4 * q + 2] = b4.z; bv[4 * q + 3] = b4.w;
            }
            tmem_ld_wait();
            if (!row_ok) { mbar_arrive(blk_done + (c >> 1)); continue; }
            uint32_t hi[8], lo[8];
#pragma unroll
            for (int q = 0; q < 8; ++q) {
                const float r0 = tanh_fast(fmaf(__uint_as_float(v[2 * q]), kInv, bv[2 * q]));
                const float r1 = tanh_fast(fmaf(__uint_as_float(v[2 * q + 1]), kInv, bv[2 * q + 1]));
                const __half2 h = __floats2half2_rn(r0, r1);
                const float2 hf = __half22float2(h);
                const __half2 l = __floats2half2_rn(r0 - hf.x, r1 - hf.y);
                hi[q] = *reinterpret_cast<const uint32_t*>(&h);
                lo[q] = *reinterpret_cast<const uint32_t*>(&l);
            }
            const int base = (c >> 1) * (128 * 64) + rbase, ci = 2 * (c & 1);
            const int o0 = base + ((ci ^ sw) << 4), o1 = base + (((ci + 1) ^ sw) << 4);
            *reinterpret_cast<uint4*>(smem + o0) = make_uint4(hi[0], hi[1], hi[2], hi[3]);
            *reinterpret_cast<uint4*>(smem + o1) = make_uint4(hi[4], hi[5], hi[6], hi[7]);
            *reinterpret_cast<uint4*>(smem + 65536 + o0) = make_uint4(lo[0], lo[1], lo[2], lo[3]);
            *reinterpret_cast<uint4*>(smem + 65536 + o1) = make_uint4(lo[4], lo[5], lo[6], lo[7]);
            fence_proxy_async_smem();
            mbar_arrive(blk_done + (c >> 1));
        }
        if (half == 1) mbar_arrive(blk_done + 7);      // 15 chunks: the last K block holds only chunk 14 (a half-0 chunk)
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 1) tmem_dealloc(tmem_base, 512);
}

// ---------------------------------------------------------------------------------------------
// dD = da1 W1^T fused with the descriptor backward (F4 -> F5 hand-over): dD (rows x 1600, 315 MB at
// configs[2]) never reaches HBM.  One CTA owns 128 rows and walks the 10 column chunks of 160 = 10 m1 x 16 m2;
// the epilogue thread of row i contracts each accumulator chunk with T_i on the fly (R-14):
//   dT[i][m][c] = sum_{m2<16} dD[i][m,m2] T[i][m2][c]  +  [m<16] sum_{m1} dD[i][m1,m] T[i][m1][c]
// first term: complete inside a chunk, stored at once; second term: 16 x 4 register accumulators over all
// chunks, added to the rows m < 16 at the end (same thread, program order).  T[i][0:16] sits in shared memory.
// ---------------------------------------------------------------------------------------------
struct DdDtArgs {
    int tile_off;
    int ntypes, K, nchunks;
    int tile0[kMaxT + 1];
    int row0[kMaxT + 1];
    const float* Tm;      // [rows][100][4]
    float* dTm;           // [rows][100][4]
    int M1;               // 100
    float inv_scale;      // 1 / (bwd_scale x W1 scale): the operands are FP16-split images of scaled values
    const uint8_t* wimg[kMaxT];   // W1 x 64 as shared-memory images, [chunk of 160 rows][K block of 32][hi | lo][160 rows x 64 B]
    const uint8_t* a_img;         // when set: da1 as fit_mid_kernel's image, [tile] x 128 KB: [K block 8][hi | lo][128 rows x 64 B]; else the TMA maps
};

// A (= da1) arrives pre-split as well (the producing epilogue writes hi and lo), so nothing stands between TMA
// and MMA: warps 0 / 1 run ahead through the chunks, alternating between two TMEM accumulator buffers, while
// the four epilogue warps contract the previous chunk.
struct DdMaps {
    CUtensorMap Ahi[kMaxT], Alo[kMaxT], Bhi[kMaxT], Blo[kMaxT];
};

constexpr int kDdBN = 160, kDdST = 5;
struct DdSmem {
    static constexpr int kABytes = 128 * 64, kBBytes = kDdBN * 64;
    static constexpr int oAhi = 0, oAlo = kABytes, oBhi = 2 * kABytes, oBlo = 2 * kABytes + kBBytes;
    static constexpr int kStage = 2 * kABytes + 2 * kBBytes;               // 36864
    static constexpr int oT2 = kDdST * kStage;                             // float4 [16][128]
    static constexpr int oBars = oT2 + 16 * 128 * 16;
    static constexpr int kTotal = oBars + 256 + 1024;
};

__global__ void __launch_bounds__(kL1Threads, 1)
dd_dt_kernel(const __grid_constant__ DdMaps maps, const __grid_constant__ DdDtArgs g) {
    using SM = DdSmem;
    constexpr int ST = kDdST, BN = kDdBN;
    extern __shared__ uint8_t smem_raw[];
    uint8_t* smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem + SM::oBars);
    uint64_t* full = bars;                     // [ST] TMA -> MMA
    uint64_t* empty = bars + ST;               // [ST] MMA -> TMA
    uint64_t* tmem_full = bars + 2 * ST;       // [2]  MMA -> epilogue
    uint64_t* tmem_empty = bars + 2 * ST + 2;  // [2]  epilogue -> MMA
    uint32_t* tmem_ptr = reinterpret_cast<uint32_t*>(bars + 2 * ST + 4);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int tile = (int)blockIdx.x + g.tile_off;
    int ty = 0;
#pragma unroll
    for (int t = 1; t < kMaxT; ++t)
        if (t < g.ntypes && tile >= g.tile0[t]) ty = t;
    const int m0 = (tile - g.tile0[ty]) * 128;
    const int rows_t = g.row0[ty + 1] - g.row0[ty];
    const int nk = (g.K + 31) / 32, nch = g.nchunks;    // K blocks of 32 halfs; the last one is zero-filled past K

    if (warp == 0 && lane == 0) {
        tma_prefetch_desc(&maps.Ahi[ty]);
        tma_prefetch_desc(&maps.Alo[ty]);
        for (int s = 0; s < ST; ++s) { mbar_init(full + s, 1); mbar_init(empty + s, 1); }
        for (int b = 0; b < 2; ++b) { mbar_init(tmem_full + b, 1); mbar_init(tmem_empty + b, 256); }
        fence_barrier_init();
    }
    if (warp == 1) tmem_alloc(tmem_ptr, 512);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_ptr;

    // The two control warps run their loops with all 32 lanes converged and let one elected lane issue (tc_gemm.cuh):
    // with N = 160 an MMA lasts 80 clk, which the single-lane form of the issue loop did not keep up with.
    if (warp == 0) {
        if (g.a_img) {
            const uint8_t* aimg = g.a_img + (size_t)tile * 131072;
            const uint8_t* wimg = g.wimg[ty];
            int s = 0, ph = 1;
            for (int nc = 0; nc < nch; ++nc)
                for (int kb = 0; kb < nk; ++kb) {
                    mbar_wait(empty + s, ph);
                    uint8_t* st = smem + s * SM::kStage;
                    // one barrier, two copies: the expect_tx of the first covers both
                    asm volatile(
                        "{\n\t"
                        ".reg .pred q;\n\t"
                        "elect.sync _|q, 0xffffffff;\n\t"
                        "@q mbarrier.arrive.expect_tx.shared::cta.b64 _, [%6], %5;\n\t"
                        "@q cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%6];\n\t"
                        "@q cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%3], [%4], %7, [%6];\n\t"
                        "}" ::"r"(smem_u32(st + SM::oAhi)),
                        "l"(aimg + kb * (2 * SM::kABytes)), "r"(2 * SM::kABytes), "r"(smem_u32(st + SM::oBhi)),
                        "l"(wimg + (size_t)(nc * nk + kb) * (2 * SM::kBBytes)), "r"(2 * SM::kABytes + 2 * SM::kBBytes), "r"(smem_u32(full + s)),
                        "r"(2 * SM::kBBytes)
                        : "memory");
                    if (++s == ST) { s = 0; ph ^= 1; }
                }
        } else if (lane == 0) {
            for (int it = 0; it < nch * nk; ++it) {
                const int nc = it / nk, kb = it - nc * nk;
                const int s = it % ST, ph = (it / ST) & 1;
                mbar_wait(empty + s, ph ^ 1);
                uint8_t* st = smem + s * SM::kStage;
                mbar_arrive_expect_tx(full + s, 2 * SM::kABytes + 2 * SM::kBBytes);
                tma_load_2d(st + SM::oAhi, &maps.Ahi[ty], full + s, kb * 32, m0);
                tma_load_2d(st + SM::oAlo, &maps.Alo[ty], full + s, kb * 32, m0);
                bulk_load(st + SM::oBhi, g.wimg[ty] + (size_t)it * (2 * SM::kBBytes), 2 * SM::kBBytes, full + s);
                (void)nc;
            }
        }
    } else if (warp == 1) {
        constexpr uint32_t idesc = make_idesc_f16(128, BN);
        // descriptors of stage 0; stage s and k-step ks add (s kStage + 32 ks) >> 4 to the address field
        const uint32_t sb = smem_u32(smem);
        const uint64_t dAh = make_smem_desc_kmajor(sb + SM::oAhi, 64), dAl = make_smem_desc_kmajor(sb + SM::oAlo, 64);
        const uint64_t dBh = make_smem_desc_kmajor(sb + SM::oBhi, 64), dBl = make_smem_desc_kmajor(sb + SM::oBlo, 64);
        const bool short_last = (g.K & 31) != 0;      // K = 240: the last block holds one k-step (the image has no zero padding behind it)
        int s = 0, ph = 0;
        for (int nc = 0; nc < nch; ++nc) {
            const int buf = nc & 1;
            if (nc >= 2) {                     // the epilogue has drained this buffer (chunk nc - 2)
                mbar_wait(tmem_empty + buf, ((nc >> 1) - 1) & 1);
                tc_fence_after();
            }
            const uint32_t dcol = tmem_base + buf * 256;
            for (int kb = 0; kb < nk; ++kb) {
                mbar_wait(full + s, ph);
                tc_fence_after();
                const uint64_t so = (uint64_t)((s * SM::kStage) >> 4);
                umma_f16_elect(dcol, dAh + so, dBh + so, idesc, kb ? 1u : 0u);
                umma_f16_elect(dcol, dAl + so, dBh + so, idesc, 1u);
                umma_f16_elect(dcol, dAh + so, dBl + so, idesc, 1u);
                if (!(short_last && kb == nk - 1)) {
                    umma_f16_elect(dcol, dAh + so + 2, dBh + so + 2, idesc, 1u);
                    umma_f16_elect(dcol, dAl + so + 2, dBh + so + 2, idesc, 1u);
                    umma_f16_elect(dcol, dAh + so + 2, dBl + so + 2, idesc, 1u);
                }
                umma_commit_elect(empty + s);
                if (++s == ST) { s = 0; ph ^= 1; }
            }
            umma_commit_elect(tmem_full + buf);
        }
    } else {
        // Two warps per TMEM lane quarter (a warp alone on its scheduler ran this loop at 0.16 IPC); warp `half` owns the
        // m2 values 8 half .. 8 half + 7 of every m1 group: its eight T[i][m2] and second-term sums stay in registers
        // (no shared-memory read per product, the stall that dominated the first two versions), and it reads only its
        // eight accumulator columns of each group.  The first term is a sum over all sixteen m2: the two warps swap
        // the halves they do not finalise through shared memory (warp `half` finalises j = 5 half .. 5 half + 4).
        constexpr int NJ = BN / 16, JH = NJ / 2;               // 10 m1 values per chunk, 5 finalised per warp
        const int quarter = warp & 3;
        auto epilogue = [&](auto half_c) {
        constexpr int half = decltype(half_c)::value;          // compile-time: it selects registers below
        const int ml = m0 + quarter * 32 + lane;               // my row inside the type (TMEM lane)
        const bool row_ok = ml < rows_t;
        const size_t m = (size_t)(g.row0[ty] + (row_ok ? ml : 0));
        const float4* Trow = reinterpret_cast<const float4*>(g.Tm) + m * g.M1;
        float4* dTrow = reinterpret_cast<float4*>(g.dTm) + m * g.M1;
        const float4 zero4 = make_float4(0.f, 0.f, 0.f, 0.f);
        float4 T2[8], accB[8];
#pragma unroll
        for (int k = 0; k < 8; ++k) { T2[k] = row_ok ? __ldg(Trow + 8 * half + k) : zero4; accB[k] = zero4; }
        float4 T1[NJ];                                          // T[i][m1] of the chunk; refilled for the next chunk as it is used up
#pragma unroll
        for (int j = 0; j < NJ; ++j) T1[j] = row_ok ? __ldg(Trow + j) : zero4;
        const float inv_scale = g.inv_scale;
        // exchange buffer [writer half][jj][row] (float4), in the place of the former T[i][0:16] copy
        float4* xw = reinterpret_cast<float4*>(smem + SM::oT2) + half * (JH * 128) + (quarter * 32 + lane);
        const float4* xr = reinterpret_cast<const float4*>(smem + SM::oT2) + (1 - half) * (JH * 128) + (quarter * 32 + lane);
        const int bar_id = 1 + quarter;

        for (int nc = 0; nc < nch; ++nc) {
            const int buf = nc & 1;
            const bool more = row_ok && nc + 1 < nch;
            mbar_wait(tmem_full + buf, (nc >> 1) & 1);
            tc_fence_after();
            const uint32_t dcol = tmem_base + ((uint32_t)(quarter * 32) << 16) + buf * 256 + 8 * half;
            float4 keep[JH];
            uint32_t vq[2][8];                                  // the next group's columns are in flight while this one is contracted
            tmem_ld8(dcol, vq[0]);
#pragma unroll
            for (int j = 0; j < NJ; ++j) {
                tmem_ld_wait();
                if (j + 1 < NJ) tmem_ld8(dcol + (j + 1) * 16, vq[(j + 1) & 1]);
                const uint32_t* v = vq[j & 1];
                float4 accA = zero4;
                const float4 t1 = T1[j];
#pragma unroll
                for (int k = 0; k < 8; ++k) {
                    const float d = __uint_as_float(v[k]);      // the common factor 1 / scale is applied at the stores
                    accA.x = fmaf(d, T2[k].x, accA.x); accA.y = fmaf(d, T2[k].y, accA.y);
                    accA.z = fmaf(d, T2[k].z, accA.z); accA.w = fmaf(d, T2[k].w, accA.w);
                    accB[k].x = fmaf(d, t1.x, accB[k].x); accB[k].y = fmaf(d, t1.y, accB[k].y);
                    accB[k].z = fmaf(d, t1.z, accB[k].z); accB[k].w = fmaf(d, t1.w, accB[k].w);
                }
                T1[j] = more ? __ldg(Trow + (nc + 1) * NJ + j) : zero4;
                if (j >= JH * half && j < JH * half + JH) keep[j - JH * half] = accA;      // mine to finalise
                else xw[(j - JH * (1 - half)) * 128] = accA;                                // my partner's
            }
            tc_fence_before();
            mbar_arrive(tmem_empty + buf);
            asm volatile("bar.sync %0, 64;" ::"r"(bar_id) : "memory");
            if (row_ok) {
#pragma unroll
                for (int jj = 0; jj < JH; ++jj) {
                    const float4 x = xr[jj * 128];
                    dTrow[nc * NJ + JH * half + jj] = make_float4((keep[jj].x + x.x) * inv_scale, (keep[jj].y + x.y) * inv_scale,
                                                                   (keep[jj].z + x.z) * inv_scale, (keep[jj].w + x.w) * inv_scale);
                }
            }
            asm volatile("bar.sync %0, 64;" ::"r"(bar_id) : "memory");     // the buffer is free again; orders the stores too
        }
        // second term: complete in this warp for its eight m2 (it saw every m1); the rows m < 16 it is added to were
        // stored above by either warp of the quarter, ordered by the barrier that closed the last chunk
        if (row_ok) {
#pragma unroll
            for (int k = 0; k < 8; ++k) {
                float4 o = dTrow[8 * half + k];
                o.x = fmaf(accB[k].x, inv_scale, o.x); o.y = fmaf(accB[k].y, inv_scale, o.y);
                o.z = fmaf(accB[k].z, inv_scale, o.z); o.w = fmaf(accB[k].w, inv_scale, o.w);
                dTrow[8 * half + k] = o;
            }
        }
        };
        if (warp < 6) epilogue(std::integral_constant<int, 0>{});
        else epilogue(std::integral_constant<int, 1>{});
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

// row-major FP16 matrix [rows][cols] with leading dimension ld (halfs); box = 32 halfs x box_rows, SWIZZLE_64B;
// columns past `cols` read as zero (the K = 240 operands are walked in 8 blocks of 32)
bool tc_make_map_h(CUtensorMap* map, const uint16_t* base, uint64_t rows, uint64_t cols, uint64_t ld, uint32_t box_rows) {
    EncodeTiledFn enc = get_encode();
    if (!enc) return false;
    cuuint64_t dims[2] = {cols, rows};
    cuuint64_t strides[1] = {ld * 2};
    cuuint32_t box[2] = {32, box_rows};
    cuuint32_t estr[2] = {1, 1};
    return enc(map, CU_TENSOR_MAP_DATA_TYPE_FLOAT16, 2, const_cast<uint16_t*>(base), dims, strides, box, estr,
               CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_64B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
               CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// operand images of the first fitting layer (see kmajor_image in fitting_mid.cu): W is [ND][NF] row-major, WT [NF][ND]
size_t l1_wimg_bytes(int ND) { return (size_t)(ND / 32) * 2 * L1Smem::kBBytes; }
void l1_build_wimg(const float* WT, int ND, uint8_t* img) {
    for (int kb = 0; kb < ND / 32; ++kb) kmajor_image(WT, kL1BN, ND, 0, kL1BN, 32 * kb, 32, kW1Scale, img + (size_t)kb * 2 * L1Smem::kBBytes);
}
size_t dd_wimg_bytes(int ND) { return (size_t)(ND / kDdBN) * 8 * 2 * DdSmem::kBBytes; }
void dd_build_wimg(const float* W, int ND, uint8_t* img) {
    for (int nc = 0; nc < ND / kDdBN; ++nc)
        for (int kb = 0; kb < 8; ++kb)
            kmajor_image(W, ND, kL1BN, nc * kDdBN, kDdBN, 32 * kb, 32, kW1Scale, img + (size_t)(nc * 8 + kb) * 2 * DdSmem::kBBytes);
}

// FP16 split of scale * w: hi = fp16(v), lo = fp16(v - hi)
__global__ void split_hi_lo_h_kernel(size_t n, const float* __restrict__ w, float scale, __half* __restrict__ hi,
                                     __half* __restrict__ lo) {
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const float v = w[i] * scale;
    const __half h = __float2half_rn(v);
    hi[i] = h;
    lo[i] = __float2half_rn(v - __half2float(h));
}
void tc_split_weights_h(size_t n, const float* w, float scale, uint16_t* hi, uint16_t* lo, cudaStream_t s) {
    split_hi_lo_h_kernel<<<(unsigned)((n + 255) / 256), 256, 0, s>>>(n, w, scale, reinterpret_cast<__half*>(hi),
                                                                      reinterpret_cast<__half*>(lo));
}

// w = hi + lo, hi = top 10 mantissa bits (what kind::tf32 reads), lo the exact remainder
__global__ void split_hi_lo_kernel(size_t n, const float* __restrict__ w, float* __restrict__ hi, float* __restrict__ lo) {
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const float v = w[i];
    const float h = __uint_as_float(__float_as_uint(v) & 0xFFFFE000u);
    hi[i] = h;
    lo[i] = v - h;
}
void tc_split_weights(size_t n, const float* w, float* hi, float* lo, cudaStream_t s) {
    split_hi_lo_kernel<<<(unsigned)((n + 255) / 256), 256, 0, s>>>(n, w, hi, lo);
}

constexpr int kNH = 1, kST = 4, kOCC = 1;     // 128-row tiles, 2 stages, 2 CTAs per SM (one's epilogue under the other's MMAs)

template <int BN, int EPI>
static cudaError_t launch_tc(const TcMaps& maps, const TcGemmArgs& g, int mtiles, cudaStream_t s) {
    using SM = TcSmem<BN, kNH, kST>;
    ensure_dyn_smem(gemm3xtf32_kernel<BN, EPI, kNH, kST, kOCC>, SM::kTotal);
    dim3 grid((g.N + BN - 1) / BN, mtiles);
    gemm3xtf32_kernel<BN, EPI, kNH, kST, kOCC><<<grid, kTcThreads, SM::kTotal, s>>>(maps, g);
    return cudaGetLastError();
}

// C = epi(A Bt^T) for all centre types at once.  bn = 240 (N == 240) or 160 (N % 160 == 0).
static cudaError_t tc_gemm(int epi, int bn, const TcMaps& maps, const TcGemmArgs& g, int mtiles, cudaStream_t s) {
    if (bn == 240) {
        switch (epi) {
            case TEPI_TANH_BIAS: return launch_tc<240, TEPI_TANH_BIAS>(maps, g, mtiles, s);
            case TEPI_TANH_BIAS_SKIP: return launch_tc<240, TEPI_TANH_BIAS_SKIP>(maps, g, mtiles, s);
            case TEPI_L3E: return launch_tc<240, TEPI_L3E>(maps, g, mtiles, s);
            case TEPI_BWD_VEC: return launch_tc<240, TEPI_BWD_VEC>(maps, g, mtiles, s);
            case TEPI_BWD_FIRST: return launch_tc<240, TEPI_BWD_FIRST>(maps, g, mtiles, s);
            case TEPI_PLAIN: return launch_tc<240, TEPI_PLAIN>(maps, g, mtiles, s);
        }
    } else if (bn == 160) {
        if (epi == TEPI_PLAIN) return launch_tc<160, TEPI_PLAIN>(maps, g, mtiles, s);
    }
    return cudaErrorInvalidValue;
}

// tile / row bookkeeping shared by all launches of a model
static int fill_types(const Model& m, int ntypes, TcGemmArgs& g) {
    g.ntypes = ntypes;
    int tiles = 0;
    for (int t = 0; t <= kMaxT; ++t) {
        g.tile0[t] = tiles;
        g.row0[t] = m.type_row0[t < ntypes ? t : ntypes];
        if (t < ntypes) tiles += (m.type_row0[t + 1] - m.type_row0[t] + 128 * kNH - 1) / (128 * kNH);
    }
    return tiles;
}

bool tc_setup_maps(Model& m, int ntypes) {
    const int NF = m.NF, ND = m.ND;
    if (NF != 240 || ND % 160 != 0) return false;
    bool ok = true;
    {   // da1 as FP16 hi / lo lives in D's storage (D is not materialised on this path); buffers of its own, because
        // the tile ranges of the chain run on different streams and a half-precision row r does not alias row r of
        // a float buffer
        const size_t S = (size_t)m.type_row0[ntypes] * NF;
        m.da1_h_hi = reinterpret_cast<uint16_t*>(m.D);
        m.da1_h_lo = m.da1_h_hi + S;
    }
    for (int t = 0; t < ntypes; ++t) {
        const uint64_t row0 = m.type_row0[t];
        uint64_t rows = m.type_row0[t + 1] - m.type_row0[t];
        if (rows == 0) rows = 1;                          // keep the descriptor valid; no tile ever uses it
        ok &= tc_make_map(&m.mapA_D[t], m.D + row0 * ND, rows, ND, ND, 128);
        ok &= tc_make_map(&m.mapA_Y1[t], m.Y1 + row0 * NF, rows, NF, NF, 128);
        ok &= tc_make_map(&m.mapA_Y2[t], m.Y2 + row0 * NF, rows, NF, NF, 128);
        ok &= tc_make_map(&m.mapA_G1[t], m.G1 + row0 * NF, rows, NF, NF, 128);
        ok &= tc_make_map(&m.mapA_G2[t], m.G2 + row0 * NF, rows, NF, NF, 128);
        ok &= tc_make_map_h(&m.mapAh_G1[t], m.da1_h_hi + row0 * NF, rows, NF, NF, 128);
        ok &= tc_make_map_h(&m.mapAh_G2[t], m.da1_h_lo + row0 * NF, rows, NF, NF, 128);
        ok &= tc_make_map(&m.mapA_T3[t], m.T3 + row0 * NF, rows, NF, NF, 128);
        for (int l = 0; l < 3; ++l) {
            const uint64_t nin = (l == 0) ? ND : NF;
            // forward: Bt = W_l^T [out][in];  backward: Bt = W_l [in][out]
            ok &= tc_make_map(&m.mapB_fwd_hi[t][l], m.fit_wT_hi[t][l], NF, nin, nin, 240);
            ok &= tc_make_map(&m.mapB_fwd_lo[t][l], m.fit_wT_lo[t][l], NF, nin, nin, 240);
            ok &= tc_make_map(&m.mapB_bwd_hi[t][l], m.fit_w_hi[t][l], nin, NF, NF, l == 0 ? 160 : 240);
            ok &= tc_make_map(&m.mapB_bwd_lo[t][l], m.fit_w_lo[t][l], nin, NF, NF, l == 0 ? 160 : 240);
        }
    }
    if (!ok) return false;
    m.tc_ready = true;
    return true;
}

static void gather_maps(TcMaps& mp, const CUtensorMap* A, const CUtensorMap (*Bhi)[3], const CUtensorMap (*Blo)[3], int l, int ntypes) {
    for (int t = 0; t < ntypes; ++t) { mp.A[t] = A[t]; mp.Bhi[t] = Bhi[t][l]; mp.Blo[t] = Blo[t][l]; }
    for (int t = ntypes; t < kMaxT; ++t) { mp.A[t] = A[0]; mp.Bhi[t] = Bhi[0][l]; mp.Blo[t] = Blo[0][l]; }
}

// the whole fitting chain of all centre types on the tensor cores: 3 forward GEMMs (the third also yields
// E_i, U and the seed of the backward pass), 3 backward GEMMs.  Returns the number of launches.
// tiles [t0, t0 + nt_) of the chain on stream s
static int chain_range(Model& m, const ForceArgs& fa, int t0, int ntl, cudaStream_t s) {
    const int NF = m.NF, ND = m.ND, nt = fa.ntypes;
    TcGemmArgs g{};
    TcMaps mp;
    fill_types(m, nt, g);
    auto base = [&]() { TcGemmArgs q{}; fill_types(m, nt, q); q.tile_off = t0; return q; };
    static const bool old_chain = getenv("PIMD_FIT_OLD") != nullptr;      // A/B partner: the round-1 chain of four GEMM launches
    const bool fused = m.mid_ready && !old_chain;
    // layer 1: Y1 = tanh(D W1 + b1), D produced on the fly from T
    {
        L1Args a1{};
        a1.tile_off = t0;
        a1.ntypes = nt; a1.K = ND; a1.Tm = m.Tm; a1.out = m.Y1; a1.ldo = NF; a1.M1 = m.M1;
        if (fused) a1.out_img = m.y1_img;
        for (int t = 0; t <= kMaxT; ++t) { a1.tile0[t] = g.tile0[t]; a1.row0[t] = g.row0[t]; }
        for (int t = 0; t < nt; ++t) a1.bias[t] = m.fit_b[t][0];
        for (int t = 0; t < kMaxT; ++t) { const int q = t < nt ? t : 0; mp.A[t] = m.mapA_D[q]; mp.Bhi[t] = m.mapA_D[q]; mp.Blo[t] = m.mapA_D[q]; a1.wimg[t] = m.l1_wimg[q]; }
        static const bool l1_ss = getenv("PIMD_L1_SS") != nullptr;            // A/B partner: the A operand through shared memory
        if (fused && !l1_ss) l1_desc_ts_kernel<<<ntl, kL1Threads, L1TsSmem::kTotal, s>>>(a1);
        else l1_desc_kernel<<<ntl, kL1Threads, L1Smem::kTotal, s>>>(mp, a1);
    }
    if (fused) {
        // layers 2 and 3, the energy and their backward products in one kernel (fitting_mid.cu)
        fitting_mid_launch(m, fa, t0, ntl, s);
    } else {
    // layer 2: T2 = tanh(Y1 W2 + b2); Y2 = Y1 + T2
    g = base(); g.N = NF; g.K = NF; g.add = m.Y1; g.ldadd = NF; g.out0 = m.T2; g.out1 = m.Y2; g.ldo = NF;
    for (int t = 0; t < nt; ++t) g.bias[t] = m.fit_b[t][1];
    gather_maps(mp, m.mapA_Y1, m.mapB_fwd_hi, m.mapB_fwd_lo, 1, nt);
    tc_gemm(TEPI_TANH_BIAS_SKIP, 240, mp, g, ntl, s);
    // layer 3 + energy: t3 = tanh(Y2 W3 + b3); y3 = Y2 + t3; E_i = y3.w4 + b4; da3 = w4 o (1 - t3^2) -> G1
    g = base(); g.N = NF; g.K = NF; g.add = m.Y2; g.ldadd = NF; g.out1 = m.G1; g.ldo = NF;
    g.cen_idx = m.cen_idx; g.Eatom = fa.Eatom; g.U = fa.U; g.natoms = fa.N;
    for (int t = 0; t < nt; ++t) { g.bias[t] = m.fit_b[t][2]; g.vec[t] = m.fit_w[t][3]; g.b4[t] = m.fit_b[t][3]; }
    gather_maps(mp, m.mapA_Y2, m.mapB_fwd_hi, m.mapB_fwd_lo, 2, nt);
    tc_gemm(TEPI_L3E, 240, mp, g, ntl, s);
    // dy2 = dy3 + da3 W3^T -> Y3 ; da2 = dy2 o (1 - t2^2) -> T3       (A = G1 = da3, dy3 = w4)
    g = base(); g.N = NF; g.K = NF; g.tt = m.T2; g.ldtt = NF; g.out0 = m.Y3; g.out1 = m.T3; g.ldo = NF;
    for (int t = 0; t < nt; ++t) g.vec[t] = m.fit_w[t][3];
    gather_maps(mp, m.mapA_G1, m.mapB_bwd_hi, m.mapB_bwd_lo, 2, nt);
    tc_gemm(TEPI_BWD_VEC, 240, mp, g, ntl, s);
    // dy1 = dy2 + da2 W2^T ; da1 = dy1 o (1 - y1^2) -> G1                (A = T3 = da2)
    g = base(); g.N = NF; g.K = NF; g.add = m.Y3; g.ldadd = NF; g.tt = m.Y1; g.ldtt = NF; g.out1 = reinterpret_cast<float*>(m.da1_h_hi); g.out0 = reinterpret_cast<float*>(m.da1_h_lo); g.ldo = NF; g.scale = m.bwd_scale;
    gather_maps(mp, m.mapA_T3, m.mapB_bwd_hi, m.mapB_bwd_lo, 1, nt);
    tc_gemm(TEPI_BWD_FIRST, 240, mp, g, ntl, s);
    }
    // dD = da1 W1^T contracted with T on the fly -> dT                   (A = G1 = da1)
    {
        DdDtArgs d{};
        d.tile_off = t0;
        d.ntypes = nt; d.K = NF; d.nchunks = ND / kDdBN; d.Tm = m.Tm; d.dTm = m.dTm; d.M1 = m.M1; d.inv_scale = 1.f / (m.bwd_scale * kW1Scale);
        for (int t = 0; t <= kMaxT; ++t) { d.tile0[t] = g.tile0[t]; d.row0[t] = g.row0[t]; }
        DdMaps dm;
        for (int t = 0; t < kMaxT; ++t) {
            const int q = t < nt ? t : 0;
            dm.Ahi[t] = m.mapAh_G1[q]; dm.Alo[t] = m.mapAh_G2[q];
            dm.Bhi[t] = dm.Ahi[t]; dm.Blo[t] = dm.Alo[t];
            d.wimg[t] = m.dd_wimg[q];
            d.a_img = fused ? m.da1_img : nullptr;
        }
        dd_dt_kernel<<<ntl, kL1Threads, DdSmem::kTotal, s>>>(dm, d);
    }
    return fused ? 3 : 6;
}

// The whole fitting chain of all centre types on the tensor cores: 3 kernels per tile range (6 with PIMD_FIT_OLD).  Every kernel of
// the chain is row-local, so the tiles are cut into ranges that run on separate streams: the tail wave of one
// range's kernel (384 tiles on 148 SMs are 2.6 waves) is filled by the other range's kernels.
int fitting_chain_tc(Model& m, const ForceArgs& fa, cudaStream_t s) {
    TcGemmArgs g{};
    const int tiles = fill_types(m, fa.ntypes, g);
    ensure_dyn_smem(l1_desc_kernel, L1Smem::kTotal);
    ensure_dyn_smem(l1_desc_ts_kernel, L1TsSmem::kTotal);
    ensure_dyn_smem(dd_dt_kernel, DdSmem::kTotal);
    if (!m.aux_stream[0]) {
        if (const char* e = getenv("PIMD_CHAIN_STREAMS")) m.chain_streams = std::min(std::max(atoi(e), 1), (int)Model::kChainStreams);
        for (int q = 0; q < Model::kChainStreams - 1; ++q) {
            cudaStreamCreateWithFlags(&m.aux_stream[q], cudaStreamNonBlocking);
            cudaEventCreateWithFlags(&m.ev_join[q], cudaEventDisableTiming);
        }
        cudaEventCreateWithFlags(&m.ev_fork, cudaEventDisableTiming);
    }
    const int NR = m.chain_streams;
    if (tiles < 2 * NR) {
        return chain_range(m, fa, 0, tiles, s);
    }
    cudaEventRecord(m.ev_fork, s);
    int launches = 0;
    for (int q = 0; q < NR; ++q) {
        const int t0 = (int)((long long)tiles * q / NR), t1 = (int)((long long)tiles * (q + 1) / NR);
        cudaStream_t sq = (q == 0) ? s : m.aux_stream[q - 1];
        if (q > 0) cudaStreamWaitEvent(sq, m.ev_fork, 0);
        launches += chain_range(m, fa, t0, t1 - t0, sq);
        if (q > 0) cudaEventRecord(m.ev_join[q - 1], sq);
    }
    for (int q = 1; q < NR; ++q) cudaStreamWaitEvent(s, m.ev_join[q - 1], 0);
    return launches;
}

// parity hook: C[M][N] = A[M][K] Bt[N][K]^T through the tensor-core kernel (N == 240 or N % 160 == 0, K % 16 == 0)
int debug_tc_gemm(int M, int N, int K, const float* A, const float* Bt, float* C, cudaStream_t s) {
    const int bn = (N == 240) ? 240 : 160;
    if ((bn == 160 && N % 160 != 0) || K % 16 != 0) return -1;
    float *hi = nullptr, *lo = nullptr;
    if (cudaMalloc(&hi, sizeof(float) * (size_t)N * K) != cudaSuccess) return -4;
    if (cudaMalloc(&lo, sizeof(float) * (size_t)N * K) != cudaSuccess) { cudaFree(hi); return -4; }
    tc_split_weights((size_t)N * K, Bt, hi, lo, s);
    TcMaps mp;
    CUtensorMap ma, mh, ml;
    int rc = 0;
    if (!tc_make_map(&ma, A, M, K, K, 128) || !tc_make_map(&mh, hi, N, K, K, bn) || !tc_make_map(&ml, lo, N, K, K, bn)) rc = -2;
    if (rc == 0) {
        for (int t = 0; t < kMaxT; ++t) { mp.A[t] = ma; mp.Bhi[t] = mh; mp.Blo[t] = ml; }
        TcGemmArgs g{};
        g.ntypes = 1; g.N = N; g.K = K; g.out0 = C; g.ldo = N;
        const int tiles = (M + 128 * kNH - 1) / (128 * kNH);
        for (int t = 0; t <= kMaxT; ++t) { g.tile0[t] = t == 0 ? 0 : tiles; g.row0[t] = t == 0 ? 0 : M; }
        rc = tc_gemm(TEPI_PLAIN, bn, mp, g, tiles, s) == cudaSuccess ? 0 : -3;
    }
    cudaStreamSynchronize(s);
    cudaFree(hi); cudaFree(lo);
    return rc;
}

}  // namespace pimd
