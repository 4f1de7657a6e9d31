// fitting_mid.cu -- the four 240 x 240 products of the fitting net (F4 of SURVEY 8(a): layers 2 and 3 forward, their two
// backward products) as ONE kernel per 128-row tile, chained on chip:
//   phase 0   t2 = tanh(y1 W2 + b2),  y2 = y1 + t2                                    (R-15)
//   phase 1   t3 = tanh(y2 W3 + b3),  y3 = y2 + t3,  E_i = y3 . w4 + b4,  da3 = w4 o (1 - t3^2)
//   phase 2   dy2 = w4 + da3 W3^T,    da2 = dy2 o (1 - t2^2)
//   phase 3   dy1 = dy2 + da2 W2^T,   da1 = dy1 o (1 - y1^2)     -> FP16 hi / lo for dd_dt_kernel
// Round 1 ran these as four launches of a 3xTF32 GEMM kernel per tile range (12-16 launches per evaluation, each
// 25-30 us with the tensor pipe 23-27 % active: prologue / epilogue bound) with every activation crossing HBM as FP32
// between them.  Here the A operand of every phase -- y1, y2, da3, da2 as FP16 hi / lo pairs (three-pass split
// products with FP32 accumulation, as everywhere in this library) -- stays RESIDENT in shared memory (128 KB): phase 0
// loads it by TMA, the epilogue of phase p rewrites it in place as the operand of phase p + 1.  The weights stream
// through a 5-stage TMA ring one k-step (16) at a time and the ring runs ahead into the next phase while an epilogue
// works.  Only t2 / dy2 (one FP32 buffer, rewritten in place) and the two ends (y1 in, da1 out) touch global memory.
#include <cuda_fp16.h>
#include "common.cuh"
#include "tc_gemm.cuh"

namespace pimd {

using namespace tc;

namespace mid {
constexpr int kThreads = 320;          // warp 0: TMA, warp 1: MMA issue + TMEM, warps 2-9: epilogue (two per TMEM lane quarter)
constexpr int kN = 240, kKS = 15;      // N = K = 240: 15 k-steps of 16
constexpr int kST = 5;
constexpr int kAcopy = 8 * 128 * 64;   // one copy of the A operand: 8 K blocks of 32 halfs, 128 rows x 64 B (SWIZZLE_64B)
constexpr int kBcopy = kN * 32;        // one copy of one k-step of the weights: 240 rows x 32 B (SWIZZLE_32B)
constexpr int kStage = 2 * kBcopy;
constexpr int oAhi = 0, oAlo = kAcopy, oB = 2 * kAcopy;
constexpr int oPatch = oB + kST * kStage;
constexpr int oEsh = oPatch + 8 * 32 * 20 * 4;   // float [128]: energy shares of the second warp of a quarter
constexpr int oBars = oEsh + 128 * 4;
constexpr int kSmem = oBars + 256 + 1024;
static_assert(kSmem <= 232448, "shared memory budget");
constexpr float kWScale = 64.f;        // the weights are split as FP16 pairs of 64 w
}  // namespace mid

struct MidMaps {
    CUtensorMap Ahi[PIMD_MAX_TYPES], Alo[PIMD_MAX_TYPES];      // y1 pair of type t: [rows_t][240] halfs, box 32 x 128, SWIZZLE_64B
    CUtensorMap B[PIMD_MAX_TYPES][4][2];                       // phase p, hi / lo: [240][240] halfs, box 16 x 240, SWIZZLE_32B
};

struct MidArgs {
    int tile_off, ntypes;
    int tile0[PIMD_MAX_TYPES + 1], row0[PIMD_MAX_TYPES + 1];
    const float* b2[PIMD_MAX_TYPES];
    const float* b3[PIMD_MAX_TYPES];
    const float* w4[PIMD_MAX_TYPES];
    const float* b4[PIMD_MAX_TYPES];
    const __half* y1_hi; const __half* y1_lo;                  // [rows][240], global type-sorted rows
    float* t2;                                                 // [rows][240]: t2 after phase 0, dy2 after phase 2
    __half* da1_hi; __half* da1_lo;                            // [rows][240]: bwd_scale * da1
    const int* cen_idx; double* Eatom; double* U; int natoms;
    float bwd_scale;
};

// byte offset of element (row, n) inside one copy of the resident A operand
__device__ __forceinline__ int mid_aoff(int row, int n) {
    return (n >> 5) * (128 * 64) + row * 64 + ((((n & 31) >> 3) ^ ((row >> 1) & 3)) << 4) + (n & 7) * 2;
}
__device__ __forceinline__ float4 mid_load_op(const uint8_t* smem, int row, int n) {
    const int off = mid_aoff(row, n);
    const uint2 h = *reinterpret_cast<const uint2*>(smem + mid::oAhi + off), l = *reinterpret_cast<const uint2*>(smem + mid::oAlo + off);
    const float2 h0 = __half22float2(*reinterpret_cast<const __half2*>(&h.x)), h1 = __half22float2(*reinterpret_cast<const __half2*>(&h.y));
    const float2 l0 = __half22float2(*reinterpret_cast<const __half2*>(&l.x)), l1 = __half22float2(*reinterpret_cast<const __half2*>(&l.y));
    return make_float4(h0.x + l0.x, h0.y + l0.y, h1.x + l1.x, h1.y + l1.y);
}
__device__ __forceinline__ void mid_split4(float4 v, uint2& hi, uint2& lo) {
    const __half2 a = __floats2half2_rn(v.x, v.y), b = __floats2half2_rn(v.z, v.w);
    const float2 fa = __half22float2(a), fb = __half22float2(b);
    const __half2 c = __floats2half2_rn(v.x - fa.x, v.y - fa.y), d = __floats2half2_rn(v.z - fb.x, v.w - fb.y);
    hi = make_uint2(*reinterpret_cast<const uint32_t*>(&a), *reinterpret_cast<const uint32_t*>(&b));
    lo = make_uint2(*reinterpret_cast<const uint32_t*>(&c), *reinterpret_cast<const uint32_t*>(&d));
}
__device__ __forceinline__ void mid_store_op(uint8_t* smem, int row, int n, float4 v) {
    const int off = mid_aoff(row, n);
    uint2 hi, lo;
    mid_split4(v, hi, lo);
    *reinterpret_cast<uint2*>(smem + mid::oAhi + off) = hi;
    *reinterpret_cast<uint2*>(smem + mid::oAlo + off) = lo;
}
__device__ __forceinline__ float4 mid_tanh4(float4 v) {
    return make_float4(tanh_fast(v.x), tanh_fast(v.y), tanh_fast(v.z), tanh_fast(v.w));
}

__global__ void __launch_bounds__(mid::kThreads, 1)
fit_mid_kernel(const __grid_constant__ MidMaps maps, const __grid_constant__ MidArgs g) {
    using namespace mid;
    extern __shared__ uint8_t smem_raw[];
    uint8_t* smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem + oBars);
    uint64_t* full = bars;                    // [kST] TMA (weights) -> MMA
    uint64_t* empty = bars + kST;             // [kST] MMA -> TMA
    uint64_t* a_full = bars + 2 * kST;        // TMA (y1) -> MMA, once
    uint64_t* a_ready = bars + 2 * kST + 1;   // epilogue -> MMA: the operand of the next phase is in place (count 256)
    uint64_t* acc_full = bars + 2 * kST + 2;  // MMA -> epilogue
    uint32_t* tmem_ptr = reinterpret_cast<uint32_t*>(bars + 2 * kST + 3);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int tile = (int)blockIdx.x + g.tile_off;
    int ty = 0;
#pragma unroll
    for (int t = 1; t < PIMD_MAX_TYPES; ++t)
        if (t < g.ntypes && tile >= g.tile0[t]) ty = t;
    const int m0 = (tile - g.tile0[ty]) * 128;
    const int rows_t = g.row0[ty + 1] - g.row0[ty];

    if (warp == 0 && lane == 0) {
        tma_prefetch_desc(&maps.Ahi[ty]);
        tma_prefetch_desc(&maps.Alo[ty]);
        for (int s = 0; s < kST; ++s) { mbar_init(full + s, 1); mbar_init(empty + s, 1); }
        mbar_init(a_full, 1);
        mbar_init(a_ready, 256);
        mbar_init(acc_full, 1);
        fence_barrier_init();
    }
    if (warp == 1) tmem_alloc(tmem_ptr, 256);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = *tmem_ptr;

    if (warp == 0) {
        if (lane == 0) {
            // the resident A operand: y1 as FP16 hi / lo, 8 K blocks of 32 (columns past 240 are zero-filled)
            mbar_arrive_expect_tx(a_full, 2 * kAcopy);
            for (int kb = 0; kb < 8; ++kb) {
                tma_load_2d(smem + oAhi + kb * (128 * 64), &maps.Ahi[ty], a_full, kb * 32, m0);
                tma_load_2d(smem + oAlo + kb * (128 * 64), &maps.Alo[ty], a_full, kb * 32, m0);
            }
            // the weights of the four phases, one k-step per stage; the ring runs ahead across the phase boundaries
            for (int it = 0; it < 4 * kKS; ++it) {
                const int p = it / kKS, ks = it - p * kKS;
                const int s = it % kST, ph = (it / kST) & 1;
                mbar_wait(empty + s, ph ^ 1);
                uint8_t* st = smem + oB + s * kStage;
                mbar_arrive_expect_tx(full + s, kStage);
                tma_load_2d(st, &maps.B[ty][p][0], full + s, ks * 16, 0);
                tma_load_2d(st + kBcopy, &maps.B[ty][p][1], full + s, ks * 16, 0);
            }
        }
    } else if (warp == 1) {
        if (lane == 0) {
            constexpr uint32_t idesc = make_idesc_f16(128, kN);
            const uint32_t a_hi = smem_u32(smem + oAhi), a_lo = smem_u32(smem + oAlo);
            for (int p = 0; p < 4; ++p) {
                if (p == 0) mbar_wait(a_full, 0);
                else mbar_wait(a_ready, (p - 1) & 1);
                tc_fence_after();
                for (int ks = 0; ks < kKS; ++ks) {
                    const int it = p * kKS + ks;
                    const int s = it % kST, ph = (it / kST) & 1;
                    mbar_wait(full + s, ph);
                    tc_fence_after();
                    const uint32_t aoff = (uint32_t)((ks >> 1) * (128 * 64) + (ks & 1) * 32);
                    const uint32_t st = smem_u32(smem + oB + s * kStage);
                    const uint64_t dah = make_smem_desc_kmajor(a_hi + aoff, 64), dal = make_smem_desc_kmajor(a_lo + aoff, 64);
                    const uint64_t dbh = make_smem_desc_kmajor(st, 32), dbl = make_smem_desc_kmajor(st + kBcopy, 32);
                    umma_f16(tmem, dah, dbh, idesc, ks ? 1u : 0u);
                    umma_f16(tmem, dal, dbh, idesc, 1u);
                    umma_f16(tmem, dah, dbl, idesc, 1u);
                    umma_commit(empty + s);
                }
                umma_commit(acc_full);
            }
        }
    } else {
        // ---- epilogues.  A 32 x 16 accumulator chunk goes through a per-warp shared-memory patch and comes back as
        // lane <-> (rows lr + 8 j, columns lc .. lc + 3), j = 0..3, so that global accesses are 64 contiguous bytes per
        // row (fitting_tc.cu has the same transpose); all epilogue math is elementwise and runs in that layout ----
        // two warps per TMEM lane quarter (one warp alone on its scheduler cannot hide the latencies of this loop):
        // warp `half` of a quarter takes the column chunks c = half, half + 2, ...
        const int quarter = warp & 3, half = (warp - 2) >> 2;
        float* patch = reinterpret_cast<float*>(smem + oPatch) + (warp - 2) * (32 * 20);
        const int lr = lane >> 2, lc = 4 * (lane & 3);
        const uint32_t lanefield = ((uint32_t)(quarter * 32)) << 16;
        bool ok[4];
        int trow[4];
        size_t grow[4];
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            trow[j] = quarter * 32 + lr + 8 * j;
            ok[j] = m0 + trow[j] < rows_t;
            grow[j] = (size_t)(g.row0[ty] + (ok[j] ? m0 + trow[j] : 0));
        }
        const float S = g.bwd_scale, inv_w = 1.f / kWScale, inv_ws = 1.f / (kWScale * S);
        const float4 zero4 = make_float4(0.f, 0.f, 0.f, 0.f);
        float e_acc[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll 1
        for (int p = 0; p < 4; ++p) {
            mbar_wait(acc_full, p & 1);
            tc_fence_after();
            // operands of this phase's elementwise part that come from global memory, fetched one chunk ahead
            float4 aux[4];
            uint2 yh[4], yl[4];
            auto fetch = [&](int c) {
                const int n = 16 * c + lc;
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    aux[j] = zero4; yh[j] = make_uint2(0u, 0u); yl[j] = yh[j];
                    if (!ok[j]) continue;
                    if (p >= 2) aux[j] = *reinterpret_cast<const float4*>(g.t2 + grow[j] * kN + n);        // t2 (p = 2), dy2 (p = 3)
                    if (p == 3) {
                        yh[j] = *reinterpret_cast<const uint2*>(g.y1_hi + grow[j] * kN + n);
                        yl[j] = *reinterpret_cast<const uint2*>(g.y1_lo + grow[j] * kN + n);
                    }
                }
            };
            fetch(half);
#pragma unroll 1
            for (int c = half; c < kN / 16; c += 2) {
                uint32_t v[16];
                tmem_ld16(tmem + lanefield + c * 16, v);
                float4 ax[4];
                uint2 yhc[4], ylc[4];
#pragma unroll
                for (int j = 0; j < 4; ++j) { ax[j] = aux[j]; yhc[j] = yh[j]; ylc[j] = yl[j]; }
                if (c + 2 < kN / 16) fetch(c + 2);
                tmem_ld_wait();
#pragma unroll
                for (int q = 0; q < 4; ++q)
                    *reinterpret_cast<float4*>(patch + lane * 20 + 4 * q) =
                        make_float4(__uint_as_float(v[4 * q]), __uint_as_float(v[4 * q + 1]), __uint_as_float(v[4 * q + 2]), __uint_as_float(v[4 * q + 3]));
                __syncwarp();
                float4 r[4];
#pragma unroll
                for (int j = 0; j < 4; ++j) r[j] = *reinterpret_cast<const float4*>(patch + (lr + 8 * j) * 20 + lc);
                __syncwarp();
                const int n = 16 * c + lc;
                const float4 w4v = __ldg(reinterpret_cast<const float4*>(g.w4[ty] + n));
                if (p == 0) {
                    const float4 b = __ldg(reinterpret_cast<const float4*>(g.b2[ty] + n));
#pragma unroll
                    for (int j = 0; j < 4; ++j) {
                        const float4 t = mid_tanh4(make_float4(fmaf(r[j].x, inv_w, b.x), fmaf(r[j].y, inv_w, b.y), fmaf(r[j].z, inv_w, b.z), fmaf(r[j].w, inv_w, b.w)));
                        const float4 y1 = mid_load_op(smem, trow[j], n);
                        if (ok[j]) *reinterpret_cast<float4*>(g.t2 + grow[j] * kN + n) = t;
                        mid_store_op(smem, trow[j], n, make_float4(y1.x + t.x, y1.y + t.y, y1.z + t.z, y1.w + t.w));
                    }
                } else if (p == 1) {
                    const float4 b = __ldg(reinterpret_cast<const float4*>(g.b3[ty] + n));
#pragma unroll
                    for (int j = 0; j < 4; ++j) {
                        const float4 t = mid_tanh4(make_float4(fmaf(r[j].x, inv_w, b.x), fmaf(r[j].y, inv_w, b.y), fmaf(r[j].z, inv_w, b.z), fmaf(r[j].w, inv_w, b.w)));
                        const float4 y2 = mid_load_op(smem, trow[j], n);
                        e_acc[j] = fmaf(y2.x + t.x, w4v.x, fmaf(y2.y + t.y, w4v.y, fmaf(y2.z + t.z, w4v.z, fmaf(y2.w + t.w, w4v.w, e_acc[j]))));
                        mid_store_op(smem, trow[j], n, make_float4(S * w4v.x * (1.f - t.x * t.x), S * w4v.y * (1.f - t.y * t.y),
                                                                    S * w4v.z * (1.f - t.z * t.z), S * w4v.w * (1.f - t.w * t.w)));
                    }
                } else if (p == 2) {
#pragma unroll
                    for (int j = 0; j < 4; ++j) {
                        const float4 t = ax[j];
                        const float4 dy = make_float4(fmaf(r[j].x, inv_ws, w4v.x), fmaf(r[j].y, inv_ws, w4v.y), fmaf(r[j].z, inv_ws, w4v.z), fmaf(r[j].w, inv_ws, w4v.w));
                        if (ok[j]) *reinterpret_cast<float4*>(g.t2 + grow[j] * kN + n) = dy;               // dy2 replaces t2
                        mid_store_op(smem, trow[j], n, make_float4(S * dy.x * (1.f - t.x * t.x), S * dy.y * (1.f - t.y * t.y),
                                                                    S * dy.z * (1.f - t.z * t.z), S * dy.w * (1.f - t.w * t.w)));
                    }
                } else {
#pragma unroll
                    for (int j = 0; j < 4; ++j) {
                        if (!ok[j]) continue;
                        const float4 d2 = ax[j];
                        const float2 h0 = __half22float2(*reinterpret_cast<const __half2*>(&yhc[j].x)), h1 = __half22float2(*reinterpret_cast<const __half2*>(&yhc[j].y));
                        const float2 l0 = __half22float2(*reinterpret_cast<const __half2*>(&ylc[j].x)), l1 = __half22float2(*reinterpret_cast<const __half2*>(&ylc[j].y));
                        const float4 y1 = make_float4(h0.x + l0.x, h0.y + l0.y, h1.x + l1.x, h1.y + l1.y);
                        const float4 da = make_float4(S * fmaf(r[j].x, inv_ws, d2.x) * (1.f - y1.x * y1.x), S * fmaf(r[j].y, inv_ws, d2.y) * (1.f - y1.y * y1.y),
                                                      S * fmaf(r[j].z, inv_ws, d2.z) * (1.f - y1.z * y1.z), S * fmaf(r[j].w, inv_ws, d2.w) * (1.f - y1.w * y1.w));
                        uint2 hi, lo;
                        mid_split4(da, hi, lo);
                        *reinterpret_cast<uint2*>(g.da1_hi + grow[j] * kN + n) = hi;
                        *reinterpret_cast<uint2*>(g.da1_lo + grow[j] * kN + n) = lo;
                    }
                }
            }
            if (p == 1) {
                // E_i = y3 . w4 + b4: the four lanes of a row add their column shares; U^(bead) += E_i with one atomic
                // per warp when all its rows share the bead (as in fitting_tc.cu)
                float* esh = reinterpret_cast<float*>(smem + oEsh);
                float er[4];
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    float e = e_acc[j];
                    e += __shfl_xor_sync(0xffffffffu, e, 1);
                    e += __shfl_xor_sync(0xffffffffu, e, 2);
                    er[j] = e;
                    if (half == 1 && (lane & 3) == 0) esh[trow[j]] = e;
                }
                asm volatile("bar.sync %0, 64;" ::"r"(1 + quarter) : "memory");     // the two warps of this quarter
                double esum = 0.0;
                int bead_u = -1;
                if (half == 0) {
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    const float e = er[j] + esh[trow[j]];
                    const bool mine = ok[j] && (lane & 3) == 0;
                    const int ba = mine ? g.cen_idx[grow[j]] : 0;
                    const double ed = mine ? (double)(e + __ldg(g.b4[ty])) : 0.0;
                    if (mine) g.Eatom[ba] = ed;
                    const int bead = mine ? ba / g.natoms : -1;
                    const int bmax = __reduce_max_sync(0xffffffffu, bead);
                    const bool same = __all_sync(0xffffffffu, bead < 0 || bead == bmax);
                    if (same && (bead_u < 0 || bmax < 0 || bmax == bead_u)) {
                        esum += ed;
                        if (bmax >= 0) bead_u = bmax;
                    } else if (mine) {
                        atomicAdd(g.U + bead, ed);
                    }
                }
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) esum += __shfl_xor_sync(0xffffffffu, esum, o);
                if (lane == 0 && bead_u >= 0) atomicAdd(g.U + bead_u, esum);
                }
            }
            if (p < 3) {
                fence_proxy_async_smem();          // the rewritten operand is read by the next phase's MMAs (async proxy)
                tc_fence_before();
                mbar_arrive(a_ready);
            }
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 1) tmem_dealloc(tmem, 256);
}

// ---- host side ----
bool fitting_mid_setup(Model& m, int ntypes) {
    const int NF = m.NF;
    m.mid_ready = false;
    if (NF != mid::kN) return false;
    const size_t S = (size_t)m.type_row0[ntypes] * NF;
    m.y1_h_hi = reinterpret_cast<uint16_t*>(m.Y1);            // the pair takes exactly the bytes of the FP32 buffer
    m.y1_h_lo = m.y1_h_hi + S;
    bool ok = true;
    for (int t = 0; t < ntypes; ++t) {
        const uint64_t row0 = m.type_row0[t];
        uint64_t rows = m.type_row0[t + 1] - m.type_row0[t];
        if (rows == 0) rows = 1;
        ok &= tc_make_map_h(&m.mapMidA_hi[t], m.y1_h_hi + row0 * NF, rows, NF, NF, 128);
        ok &= tc_make_map_h(&m.mapMidA_lo[t], m.y1_h_lo + row0 * NF, rows, NF, NF, 128);
        for (int p = 0; p < 4; ++p)
            for (int h = 0; h < 2; ++h) ok &= tc_make_map_h16(&m.mapMidB[t][p][h], m.wmid_h[t][p][h], NF, NF, NF, mid::kN);
    }
    m.mid_ready = ok;
    return ok;
}

void fitting_mid_launch(Model& m, const ForceArgs& fa, int tile_off, int ntiles, cudaStream_t s) {
    const int nt = fa.ntypes;
    MidMaps mp;
    MidArgs g{};
    g.tile_off = tile_off;
    g.ntypes = nt;
    int tiles = 0;
    for (int t = 0; t <= PIMD_MAX_TYPES; ++t) {
        g.tile0[t] = tiles;
        g.row0[t] = m.type_row0[t < nt ? t : nt];
        if (t < nt) tiles += (m.type_row0[t + 1] - m.type_row0[t] + 127) / 128;
    }
    for (int t = 0; t < PIMD_MAX_TYPES; ++t) {
        const int q = t < nt ? t : 0;
        mp.Ahi[t] = m.mapMidA_hi[q];
        mp.Alo[t] = m.mapMidA_lo[q];
        for (int p = 0; p < 4; ++p)
            for (int h = 0; h < 2; ++h) mp.B[t][p][h] = m.mapMidB[q][p][h];
        g.b2[t] = m.fit_b[q][1]; g.b3[t] = m.fit_b[q][2]; g.w4[t] = m.fit_w[q][3]; g.b4[t] = m.fit_b[q][3];
    }
    g.y1_hi = reinterpret_cast<const __half*>(m.y1_h_hi);
    g.y1_lo = reinterpret_cast<const __half*>(m.y1_h_lo);
    g.t2 = m.T2;
    g.da1_hi = reinterpret_cast<__half*>(m.da1_h_hi);
    g.da1_lo = reinterpret_cast<__half*>(m.da1_h_lo);
    g.cen_idx = m.cen_idx; g.Eatom = fa.Eatom; g.U = fa.U; g.natoms = fa.N;
    g.bwd_scale = m.bwd_scale;
    ensure_dyn_smem(fit_mid_kernel, mid::kSmem);
    fit_mid_kernel<<<ntiles, mid::kThreads, mid::kSmem, s>>>(mp, g);
}

}  // namespace pimd
