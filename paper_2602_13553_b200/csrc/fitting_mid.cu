// fitting_mid.cu -- the four 240 x 240 products of the fitting net (F4 of SURVEY 8(a): layers 2 and 3 forward, their two
// backward products) as ONE kernel per 128-row tile, chained on chip:
//   phase 0   t2 = tanh(y1 W2 + b2),  y2 = y1 + t2                                    (R-15)
//   phase 1   t3 = tanh(y2 W3 + b3),  y3 = y2 + t3,  E_i = y3 . w4 + b4,  da3 = w4 o (1 - t3^2)
//   phase 2   dy2 = w4 + da3 W3^T,    da2 = dy2 o (1 - t2^2)
//   phase 3   dy1 = dy2 + da2 W2^T,   da1 = dy1 o (1 - y1^2)     -> FP16 hi / lo for dd_dt_kernel
// Round 1 ran these as four launches of a 3xTF32 GEMM kernel per tile range (12-16 launches per evaluation, each
// 25-30 us with the tensor pipe a quarter active: prologue / epilogue bound) with every activation crossing HBM as
// FP32 between them.  Here the A operand of every phase -- y1, y2, da3, da2 as FP16 hi / lo pairs (three-pass split
// products with FP32 accumulation, as everywhere in this library) -- stays RESIDENT in shared memory (128 KB): it
// arrives as one bulk copy of the image l1_desc_kernel left in global memory, the epilogue of phase p rewrites it in
// place, 16 columns at a time, as the operand of phase p + 1, and the last epilogue hands it to dd_dt_kernel as an
// image again.  Chunk c of an epilogue's output is k-step c of the next product, so the MMAs of phase p + 1 start
// behind the epilogue of phase p chunk by chunk (one mbarrier per chunk) into the second accumulator buffer instead
// of waiting for the whole operand.  The weights stream through a 5-stage ring, one pre-swizzled image of a k-step
// per bulk copy, and run ahead across the phase boundaries.  Per-element state that outlives a phase (t2 -> dy2,
// 1 - y1^2) sits in a tile-private scratch laid out [chunk][float4][row], so the row-per-lane epilogue threads
// read and write it coalesced.
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
constexpr int oVec = oB + kST * kStage;          // float [3][240]: b2, b3, w4 of this tile's centre type
constexpr int oEx = oVec + 3 * kN * 4;           // float [128]: energy shares of the second warp of a quarter
constexpr int oBars = oEx + 128 * 4;
constexpr int kSmem = oBars + 384 + 1024;          // 43 barriers + the TMEM address
static_assert(kSmem <= 232448, "shared memory budget");
constexpr float kWScale = 64.f;        // the weights are split as FP16 pairs of 64 w
constexpr int kScratch = kKS * 4 * 128 * 16;     // bytes per tile of one scratch array: [chunk 15][float4 4][row 128]
constexpr int kImage = 2 * kAcopy;               // bytes per tile of an operand image in global memory
}  // namespace mid

struct MidArgs {
    int tile_off, ntypes;
    int tile0[PIMD_MAX_TYPES + 1], row0[PIMD_MAX_TYPES + 1];
    const float* b2[PIMD_MAX_TYPES];
    const float* b3[PIMD_MAX_TYPES];
    const float* w4[PIMD_MAX_TYPES];
    const float* b4[PIMD_MAX_TYPES];
    const uint8_t* wimg[PIMD_MAX_TYPES];                       // weight images, [phase][k-step] x kStage bytes
    const uint8_t* y1_img;                                     // [tile] x kImage: [hi | lo][K block 8][128 rows x 64 B]
    uint8_t* da1_img;                                          // [tile] x kImage: [K block 8][hi | lo][128 rows x 64 B], bwd_scale * da1
    float4* sc_t2; float4* sc_g1;                              // [tile] x kScratch
    const int* cen_idx; double* Eatom; double* U; int natoms;
    float bwd_scale;
};

// 16 consecutive halfs (columns 16 c .. 16 c + 15 of row `row`) inside one copy of the resident operand: two
// 16-byte pieces at K block c >> 1, chunk indices 2 (c & 1) and 2 (c & 1) + 1, XOR-swizzled by the row
__device__ __forceinline__ void mid_chunk_off(int row, int c, int& o0, int& o1) {
    const int base = (c >> 1) * (128 * 64) + row * 64, sw = (row >> 1) & 3, ci = 2 * (c & 1);
    o0 = base + ((ci ^ sw) << 4);
    o1 = base + (((ci + 1) ^ sw) << 4);
}
__device__ __forceinline__ void mid_unpack8(uint4 h, uint4 l, float* o) {
    const uint32_t hw[4] = {h.x, h.y, h.z, h.w}, lw[4] = {l.x, l.y, l.z, l.w};
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        const float2 a = __half22float2(*reinterpret_cast<const __half2*>(&hw[q])), b = __half22float2(*reinterpret_cast<const __half2*>(&lw[q]));
        o[2 * q] = a.x + b.x; o[2 * q + 1] = a.y + b.y;
    }
}
__device__ __forceinline__ void mid_load16(const uint8_t* smem, int row, int c, float* o) {
    int o0, o1;
    mid_chunk_off(row, c, o0, o1);
    mid_unpack8(*reinterpret_cast<const uint4*>(smem + mid::oAhi + o0), *reinterpret_cast<const uint4*>(smem + mid::oAlo + o0), o);
    mid_unpack8(*reinterpret_cast<const uint4*>(smem + mid::oAhi + o1), *reinterpret_cast<const uint4*>(smem + mid::oAlo + o1), o + 8);
}
__device__ __forceinline__ void mid_store16(uint8_t* smem, int row, int c, const float* v) {
    int o0, o1;
    mid_chunk_off(row, c, o0, o1);
    uint32_t hi[8], lo[8];
#pragma unroll
    for (int q = 0; q < 8; ++q) {
        const __half2 h = __floats2half2_rn(v[2 * q], v[2 * q + 1]);
        const float2 hf = __half22float2(h);
        const __half2 l = __floats2half2_rn(v[2 * q] - hf.x, v[2 * q + 1] - hf.y);
        hi[q] = *reinterpret_cast<const uint32_t*>(&h);
        lo[q] = *reinterpret_cast<const uint32_t*>(&l);
    }
    *reinterpret_cast<uint4*>(smem + mid::oAhi + o0) = make_uint4(hi[0], hi[1], hi[2], hi[3]);
    *reinterpret_cast<uint4*>(smem + mid::oAhi + o1) = make_uint4(hi[4], hi[5], hi[6], hi[7]);
    *reinterpret_cast<uint4*>(smem + mid::oAlo + o0) = make_uint4(lo[0], lo[1], lo[2], lo[3]);
    *reinterpret_cast<uint4*>(smem + mid::oAlo + o1) = make_uint4(lo[4], lo[5], lo[6], lo[7]);
}

__global__ void __launch_bounds__(mid::kThreads, 1)
fit_mid_kernel(const __grid_constant__ MidArgs g) {
    using namespace mid;
    extern __shared__ uint8_t smem_raw[];
    uint8_t* smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem + oBars);
    uint64_t* full = bars;                    // [kST] weights landed -> MMA
    uint64_t* empty = bars + kST;             // [kST] MMA -> TMA
    uint64_t* a_full = bars + 2 * kST;        // [8] K block kb of the y1 image landed -> MMA, epilogue
    uint64_t* acc_full = bars + 2 * kST + 8;  // [2] MMA -> epilogue, one per accumulator buffer
    uint64_t* chunk_ready = bars + 2 * kST + 10;  // [kKS] epilogue -> MMA: columns 16 c .. 16 c + 15 of the next operand are in place (count 128)
    uint64_t* blk_done = bars + 2 * kST + 10 + kKS;   // [8] last epilogue -> store: K block kb of the da1 image is complete (count 256)
    uint32_t* tmem_ptr = reinterpret_cast<uint32_t*>(bars + 2 * kST + 18 + kKS);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int tile = (int)blockIdx.x + g.tile_off;
    int ty = 0;
#pragma unroll
    for (int t = 1; t < PIMD_MAX_TYPES; ++t)
        if (t < g.ntypes && tile >= g.tile0[t]) ty = t;
    const int m0 = (tile - g.tile0[ty]) * 128;
    const int rows_t = g.row0[ty + 1] - g.row0[ty];

    if (warp == 0 && lane == 0) {
        for (int s = 0; s < kST; ++s) { mbar_init(full + s, 1); mbar_init(empty + s, 1); }
        for (int kb = 0; kb < 8; ++kb) mbar_init(a_full + kb, 1);
        mbar_init(acc_full, 1);
        mbar_init(acc_full + 1, 1);
        for (int c = 0; c < kKS; ++c) mbar_init(chunk_ready + c, 128);
        for (int kb = 0; kb < 8; ++kb) mbar_init(blk_done + kb, 256);
        fence_barrier_init();
    }
    if (warp == 1) tmem_alloc(tmem_ptr, 512);
    {   // the row vectors of the epilogues: read from shared memory, not through a global load per chunk (a cold
        // L2 round trip in front of every chunk was the largest stall of the first version)
        float* vec = reinterpret_cast<float*>(smem + oVec);
        for (int i = threadIdx.x; i < 3 * kN; i += kThreads) {
            const int w = i / kN, n = i - w * kN;
            vec[i] = __ldg((w == 0 ? g.b2[ty] : w == 1 ? g.b3[ty] : g.w4[ty]) + n);
        }
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = *tmem_ptr;

    // control warps: all 32 lanes run the loop converged, one elected lane issues (tc_gemm.cuh)
    if (warp == 0) {
        // the resident A operand: the y1 image of this tile, FP16 hi then lo (columns 240..255 of the last K block are never read)
        // one barrier per K block, so that the first product starts when 16 of the 128 KB are there
        for (int kb = 0; kb < 8; ++kb) {
            const uint8_t* img = g.y1_img + (size_t)tile * kImage + kb * 8192;
            asm volatile(
                "{\n\t"
                ".reg .pred q;\n\t"
                "elect.sync _|q, 0xffffffff;\n\t"
                "@q mbarrier.arrive.expect_tx.shared::cta.b64 _, [%4], %5;\n\t"
                "@q cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %6, [%4];\n\t"
                "@q cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%2], [%3], %6, [%4];\n\t"
                "}" ::"r"(smem_u32(smem + oAhi + kb * 8192)),
                "l"(img), "r"(smem_u32(smem + oAlo + kb * 8192)), "l"(img + kAcopy), "r"(smem_u32(a_full + kb)), "r"(16384), "r"(8192)
                : "memory");
        }
        // the weights of the four phases, one k-step per stage; the ring runs ahead across the phase boundaries
        const uint8_t* wimg = g.wimg[ty];
        int s = 0, ph = 1;
        for (int it = 0; it < 4 * kKS; ++it) {
            mbar_wait(empty + s, ph);
            bulk_load_expect_elect(smem + oB + s * kStage, wimg + (size_t)it * kStage, kStage, full + s);
            if (++s == kST) { s = 0; ph ^= 1; }
        }
        // after the last product the operand holds bwd_scale * da1: out as the image dd_dt_kernel loads, K block by K
        // block behind the last epilogue, hi next to lo
        uint8_t* img = g.da1_img + (size_t)tile * kImage;
        for (int kb = 0; kb < 8; ++kb) {
            mbar_wait(blk_done + kb, 0);
            if (lane == 0) {
                bulk_store(img + kb * 16384, smem + oAhi + kb * 8192, 8192);
                bulk_store(img + kb * 16384 + 8192, smem + oAlo + kb * 8192, 8192);
                bulk_commit();
            }
        }
        if (lane == 0) bulk_wait_read0();      // shared memory may go once it has been read; the writes complete with the grid
    } else if (warp == 1) {
        constexpr uint32_t idesc = make_idesc_f16(128, kN);
        const uint32_t sb = smem_u32(smem);
        const uint64_t dAh = make_smem_desc_kmajor(sb + oAhi, 64), dAl = make_smem_desc_kmajor(sb + oAlo, 64);
        const uint64_t dBh = make_smem_desc_kmajor(sb + oB, 32), dBl = make_smem_desc_kmajor(sb + oB + kBcopy, 32);
        int s = 0, ph = 0;
        for (int p = 0; p < 4; ++p) {
            const uint32_t acc = tmem + (uint32_t)(p & 1) * 256;
            for (int ks = 0; ks < kKS; ++ks) {
                if (p > 0) mbar_wait(chunk_ready + ks, (p - 1) & 1);     // k-step ks of this operand = chunk ks of the last epilogue
                else if (!(ks & 1)) mbar_wait(a_full + (ks >> 1), 0);
                mbar_wait(full + s, ph);
                tc_fence_after();
                const uint64_t ao = (uint64_t)(((ks >> 1) * (128 * 64) + (ks & 1) * 32) >> 4), bo = (uint64_t)((s * kStage) >> 4);
                umma_f16_elect(acc, dAh + ao, dBh + bo, idesc, ks ? 1u : 0u);
                umma_f16_elect(acc, dAl + ao, dBh + bo, idesc, 1u);
                umma_f16_elect(acc, dAh + ao, dBl + bo, idesc, 1u);
                umma_commit_elect(empty + s);
                if (++s == kST) { s = 0; ph ^= 1; }
            }
            umma_commit_elect(acc_full + (p & 1));
        }
    } else {
        // ---- epilogues: thread <-> tile row (= TMEM lane); two warps per lane quarter, warp `half` of a quarter takes the
        // column chunks c = half, half + 2, ... ----
        const int quarter = warp & 3, half = (warp - 2) >> 2;
        const int row = quarter * 32 + lane;
        const bool row_ok = m0 + row < rows_t;
        const uint32_t lanefield = ((uint32_t)(quarter * 32)) << 16;
        const float* vec = reinterpret_cast<const float*>(smem + oVec);
        const float S = g.bwd_scale, inv_w = 1.f / kWScale, inv_ws = 1.f / (kWScale * S);
        float4* t2s = g.sc_t2 + (size_t)tile * (kScratch / 16) + row;      // + (4 c + q) * 128
        float4* g1s = g.sc_g1 + (size_t)tile * (kScratch / 16) + row;
        float e_acc = 0.f;
        for (int kb = 0; kb < 8; ++kb) mbar_wait(a_full + kb, 0);   // phase 0 reads y1 from the operand
#pragma unroll 1
        for (int p = 0; p < 4; ++p) {
            mbar_wait(acc_full + (p & 1), (p >> 1) & 1);
            tc_fence_after();
            const uint32_t acc = tmem + lanefield + (uint32_t)(p & 1) * 256;
            float4 na[4] = {}, nb[4] = {};                     // scratch values of the chunk after this one, in flight
            auto fetch = [&](int c) {
                if (p < 2 || c >= kKS) return;
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    na[q] = t2s[(4 * c + q) * 128];
                    if (p == 3) nb[q] = g1s[(4 * c + q) * 128];
                }
            };
            fetch(half);
#pragma unroll 1
            for (int c = half; c < kKS; c += 2) {
                uint32_t v[16];
                tmem_ld16(acc + c * 16, v);
                float a[16], b[16], o[16];
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    a[4 * q] = na[q].x; a[4 * q + 1] = na[q].y; a[4 * q + 2] = na[q].z; a[4 * q + 3] = na[q].w;
                    b[4 * q] = nb[q].x; b[4 * q + 1] = nb[q].y; b[4 * q + 2] = nb[q].z; b[4 * q + 3] = nb[q].w;
                }
                fetch(c + 2);
                float w4v[16];
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    const float4 w = *reinterpret_cast<const float4*>(vec + 2 * kN + 16 * c + 4 * q);
                    w4v[4 * q] = w.x; w4v[4 * q + 1] = w.y; w4v[4 * q + 2] = w.z; w4v[4 * q + 3] = w.w;
                }
                tmem_ld_wait();
                if (p == 0) {
                    float y1[16];
                    mid_load16(smem, row, c, y1);
                    float4 tq[4], gq[4];
#pragma unroll
                    for (int q = 0; q < 16; ++q) {
                        const float t = tanh_fast(fmaf(__uint_as_float(v[q]), inv_w, vec[16 * c + q]));
                        o[q] = y1[q] + t;
                        reinterpret_cast<float*>(tq)[q] = t;
                        reinterpret_cast<float*>(gq)[q] = fmaf(-y1[q], y1[q], 1.f);
                    }
#pragma unroll
                    for (int q = 0; q < 4; ++q) { t2s[(4 * c + q) * 128] = tq[q]; g1s[(4 * c + q) * 128] = gq[q]; }
                } else if (p == 1) {
                    float y2[16];
                    mid_load16(smem, row, c, y2);
#pragma unroll
                    for (int q = 0; q < 16; ++q) {
                        const float t = tanh_fast(fmaf(__uint_as_float(v[q]), inv_w, vec[kN + 16 * c + q]));
                        e_acc = fmaf(y2[q] + t, w4v[q], e_acc);
                        o[q] = S * w4v[q] * fmaf(-t, t, 1.f);
                    }
                } else if (p == 2) {
                    float4 dq[4];
#pragma unroll
                    for (int q = 0; q < 16; ++q) {
                        const float dy = fmaf(__uint_as_float(v[q]), inv_ws, w4v[q]);
                        reinterpret_cast<float*>(dq)[q] = dy;
                        o[q] = S * dy * fmaf(-a[q], a[q], 1.f);
                    }
#pragma unroll
                    for (int q = 0; q < 4; ++q) t2s[(4 * c + q) * 128] = dq[q];             // dy2 replaces t2
                } else {
#pragma unroll
                    for (int q = 0; q < 16; ++q) o[q] = S * fmaf(__uint_as_float(v[q]), inv_ws, a[q]) * b[q];
                }
                mid_store16(smem, row, c, o);
                fence_proxy_async_smem();          // read next by the MMAs of phase p + 1 / the bulk store (async proxy)
                if (p < 3) {
                    tc_fence_before();
                    mbar_arrive(chunk_ready + c);
                } else {
                    mbar_arrive(blk_done + (c >> 1));
                }
            }
            if (p == 3 && half == 1) mbar_arrive(blk_done + 7);     // 15 chunks: the last K block holds only chunk 14 (a half-0 chunk)
            if (p == 1) {
                // E_i = y3 . w4 + b4: the two warps of a quarter hold shares over their chunks; U^(bead) += E_i with one
                // atomic per warp when all its rows share the bead
                float* ex = reinterpret_cast<float*>(smem + oEx);
                if (half == 1) ex[row] = e_acc;
                asm volatile("bar.sync %0, 64;" ::"r"(1 + quarter) : "memory");
                if (half == 0) {
                    const size_t grow = (size_t)(g.row0[ty] + (row_ok ? m0 + row : 0));
                    const int ba = row_ok ? g.cen_idx[grow] : 0;
                    const int bead = row_ok ? ba / g.natoms : -1;
                    const double ed = row_ok ? (double)(e_acc + ex[row] + __ldg(g.b4[ty])) : 0.0;
                    if (row_ok) g.Eatom[ba] = ed;
                    const int bmax = __reduce_max_sync(0xffffffffu, bead);
                    if (__all_sync(0xffffffffu, bead < 0 || bead == bmax)) {
                        double esum = ed;
#pragma unroll
                        for (int of = 16; of > 0; of >>= 1) esum += __shfl_xor_sync(0xffffffffu, esum, of);
                        if (lane == 0 && bmax >= 0) atomicAdd(g.U + bmax, esum);
                    } else if (row_ok) {
                        atomicAdd(g.U + bead, ed);
                    }
                }
            }
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 1) tmem_dealloc(tmem, 512);
}

// ---- host side ----
// Shared-memory image of rows [n0, n0 + nr) x columns [k0, k0 + kc) of scale * Bt ([N][K] row-major, zero past K)
// as a K-major MMA operand: FP16 hi part then lo part, each nr rows of 2 kc bytes with the 16-byte chunks XOR-swizzled
// the way the matrix descriptor expects (kc = 16: SWIZZLE_32B, chunk ^= (row >> 2) & 1; kc = 32: SWIZZLE_64B,
// chunk ^= (row >> 1) & 3).  A bulk copy of the image into a stage is then all the load there is.
size_t kmajor_image_bytes(int nrows, int kc) { return (size_t)2 * nrows * kc * 2; }
void kmajor_image(const float* Bt, int N, int K, int n0, int nr, int k0, int kc, float scale, uint8_t* img) {
    const int rb = 2 * kc;
    uint16_t* hi = reinterpret_cast<uint16_t*>(img);
    uint16_t* lo = reinterpret_cast<uint16_t*>(img + (size_t)nr * rb);
    for (int r = 0; r < nr; ++r)
        for (int k = 0; k < kc; ++k) {
            const float v = (n0 + r < N && k0 + k < K) ? Bt[(size_t)(n0 + r) * K + k0 + k] * scale : 0.f;
            const __half h = __float2half_rn(v);
            const __half l = __float2half_rn(v - __half2float(h));
            const int sw = (kc == 32) ? ((r >> 1) & 3) : ((r >> 2) & 1);
            const int off = r * rb + (((k >> 3) ^ sw) << 4) + (k & 7) * 2;
            hi[off / 2] = *reinterpret_cast<const uint16_t*>(&h);
            lo[off / 2] = *reinterpret_cast<const uint16_t*>(&l);
        }
}
size_t mid_wimg_bytes() { return (size_t)4 * mid::kKS * mid::kStage; }
// phases: y1 W2 (Bt = W2^T), y2 W3 (W3^T), da3 W3^T (Bt = W3), da2 W2^T (W2); W row-major [in][out], WT [out][in]
void mid_build_wimg(const float* W2, const float* W2T, const float* W3, const float* W3T, uint8_t* img) {
    const float* Bt[4] = {W2T, W3T, W3, W2};
    for (int p = 0; p < 4; ++p)
        for (int ks = 0; ks < mid::kKS; ++ks)
            kmajor_image(Bt[p], mid::kN, mid::kN, 0, mid::kN, 16 * ks, 16, mid::kWScale, img + (size_t)(p * mid::kKS + ks) * mid::kStage);
}

bool fitting_mid_setup(Model& m, int ntypes) {
    m.mid_ready = m.NF == mid::kN && m.y1_img && m.da1_img && m.mid_t2 && m.mid_g1 && m.mid_wimg[0];
    (void)ntypes;
    return m.mid_ready;
}
size_t mid_image_bytes() { return mid::kImage; }
size_t mid_scratch_bytes() { return mid::kScratch; }

void fitting_mid_launch(Model& m, const ForceArgs& fa, int tile_off, int ntiles, cudaStream_t s) {
    const int nt = fa.ntypes;
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
        g.wimg[t] = m.mid_wimg[q];
        g.b2[t] = m.fit_b[q][1]; g.b3[t] = m.fit_b[q][2]; g.w4[t] = m.fit_w[q][3]; g.b4[t] = m.fit_b[q][3];
    }
    g.y1_img = m.y1_img;
    g.da1_img = m.da1_img;
    g.sc_t2 = m.mid_t2;
    g.sc_g1 = m.mid_g1;
    g.cen_idx = m.cen_idx; g.Eatom = fa.Eatom; g.U = fa.U; g.natoms = fa.N;
    g.bwd_scale = m.bwd_scale;
    ensure_dyn_smem(fit_mid_kernel, mid::kSmem);
    fit_mid_kernel<<<ntiles, mid::kThreads, mid::kSmem, s>>>(g);
}

}  // namespace pimd
