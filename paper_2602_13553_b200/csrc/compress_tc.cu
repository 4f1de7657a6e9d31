// compress_tc.cu -- SURVEY 8(f) NEXT-3: the compressed ("tabulated") embedding net, the model variant the paper's own
// timings were taken with ("We use a compressed DP model", L262; ref. 41 is only cited; DESIGN R-28).
//
// R-28: per ordered type pair (t_i, t_j) the embedding net G(s) -- a function of ONE scalar -- is replaced on the
// uniform grid s in [0, 2], stride h = 0.05 (40 intervals) by the quintic Hermite polynomial that matches G, G', G''
// at both nodes.  With u = (s - s_n)/h in [0, 1]:   G~_m(s) = sum_{p<6} C[iv][p][m] u^p.
//
// What is computed is R-14 / R-16 with G~ for G.  HOW it is computed is not a per-row table lookup: because G~ is a
// polynomial in u with ROW-independent coefficients, the two contractions over the rows of a centre factor through
// per-centre MOMENTS (K = (t_j, interval, power) = 2 x 40 x 6 = 480):
//   forward   T_i[m][c]  = 1/N_sel sum_K C[K][m] Mom_i[K][c],   Mom_i[K][c] = sum_{rows in bucket K} u^p R_row[c]
//   backward  Q_i[K][c]  = sum_m dT_i[m][c] C[K][m];   per row:  dR[c] = 1/N_sel sum_p u^p Q_i[K(row), p][c]
//                                                                 ds    = 1/(N_sel h) sum_c R[c] sum_p p u^{p-1} Q_i[..][c]
// so a row costs O(24) operations instead of O(100 x 18), and the O(480 x 100 x 4) per-centre products are dense
// GEMMs with ONE constant operand -- the table.  On sm_100a the table lives in TENSOR MEMORY for the whole kernel as
// the A operand of tcgen05.mma (FP16 hi / lo images, 480 of the 512 TMEM columns forward, 448 backward), the
// per-centre moments / dT are the small shared-memory B operand (N = 32 = 8 centres x 4 components), accumulators take
// the remaining TMEM columns.  Products are the three-pass FP16 split of embedding_tc.cu (FP32 accumulate).
// Neither the moments nor Q ever touch HBM.
#include <cmath>
#include <cstring>
#include <cuda_fp16.h>
#include "common.cuh"
#include "tc_gemm.cuh"

namespace pimd {

using namespace tc;

namespace cmp {
constexpr int NI = 40, NP = 6, KB = NI * NP;       // intervals, coefficients, K per neighbour type
constexpr int M1 = 100;                            // channels
constexpr int MAXT = 2;                            // neighbour types the TMEM-resident table has room for
constexpr int K = MAXT * KB;                       // 480
constexpr float kInvH = 20.0f;                     // 1 / stride
constexpr float kSHi = 2.0f;
constexpr int TC = 8;                              // centres per tile  -> N = 32 operand rows (centre, component)
constexpr int NROW = 4 * TC;
// forward TMEM image of centre type t_i: A[lane = channel m][k], two halfs per 32-bit column
constexpr int FW_COLS = K / 2;                     // 240 columns per copy (hi, lo)
constexpr int FW_D = 2 * FW_COLS;                  // accumulator columns 480..511
// backward: four M tiles of 120 table rows (k = 120 j + lane), K = channels padded to 112
constexpr int BW_MT = 4, BW_ROWS = 120, BW_KP = 112, BW_COLS = BW_KP / 2;    // 56 columns per copy
constexpr int BW_D = BW_MT * 2 * BW_COLS;          // 448: two accumulator buffers of 32 columns
// shared memory, forward
constexpr int STG = 488;                           // floats per (centre, component) row of the FP32 moment stage:
                                                   // 488 = 8 mod 32 keeps lane (p, c) on bank 8c + 6b + p
constexpr int F_STAGE = TC * 4 * STG * 4;          // 62,464
constexpr int F_OPB = 8 * NROW * 128;              // one copy: 8 K blocks of 64 halfs x 32 rows x 128 B = 32 KB
constexpr int F_ROWBUF = 32 * 25 * 4;              // per warp: 32 rows x (24 products + bucket)
constexpr int F_WARPS = 2 * TC;                    // moment warps: (centre, neighbour type)
constexpr int F_THREADS = (F_WARPS + 4) * 32;      // + the tensor warpgroup
constexpr int F_SMEM = 1024 + 2 * F_OPB + F_STAGE + F_WARPS * F_ROWBUF + 256;
// backward
constexpr int B_Q = TC * K * 16;                   // one Q buffer: [centre][k] float4 = 61,440
constexpr int B_OPB = 2 * NROW * 128;              // one copy: 2 K blocks x 32 rows x 128 B = 8 KB
constexpr int B_WARPS = 2 * TC;
constexpr int B_THREADS = (B_WARPS + 4) * 32;
constexpr int B_SMEM = 1024 + 2 * B_OPB + 2 * B_Q + 256;
static_assert(F_SMEM <= 232448 && B_SMEM <= 232448, "shared memory budget");
}  // namespace cmp

__device__ __forceinline__ void cmp_bar_sync(int id, int nthreads) {
    asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}

// eight floats -> one 16-byte chunk of FP16 hi and one of FP16 lo (hi = fp16(v), lo = fp16(v - hi))
__device__ __forceinline__ void split8(const float* v, uint4& hi, uint4& lo) {
    uint32_t h[4], l[4];
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        const __half2 hh = __floats2half2_rn(v[2 * q], v[2 * q + 1]);
        const float2 hf = __half22float2(hh);
        const __half2 ll = __floats2half2_rn(v[2 * q] - hf.x, v[2 * q + 1] - hf.y);
        h[q] = *reinterpret_cast<const uint32_t*>(&hh);
        l[q] = *reinterpret_cast<const uint32_t*>(&ll);
    }
    hi = make_uint4(h[0], h[1], h[2], h[3]);
    lo = make_uint4(l[0], l[1], l[2], l[3]);
}

struct CmpArgs {
    int PN, N, ntypes, nsel;
    int seloff[PIMD_MAX_TYPES + 1];
    int type_row0[PIMD_MAX_TYPES + 1];
    int n_of_type[PIMD_MAX_TYPES];
    const int* cen_idx;        // [PN] type-sorted centre row -> bead-atom k*N + i
    const int* ncount;         // [PN][ntypes]
    const NeighSlotA* slotA;
    const NeighSlotB* slotB;
    const uint32_t* img_fw;    // [ntypes][128 lanes][2 hi/lo][FW_COLS]           (the column order of tensor memory)
    const uint32_t* img_bw;    // [ntypes][128 lanes][BW_MT][2 hi/lo][BW_COLS]
    float* Tm;                 // [PN rows][100][4]
    const float* dTm;
    double* f;                 // [P][N][3]
    double* cpart;             // [PN][9]
    int* overflow;             // bit 2 (value 4): a row outside the table (s > 2)
    uint32_t* need;            // [PN / TC + ntypes + 1] per tile of 8 centres, written by the forward kernel: bit tj = some row
                               // of neighbour type tj sits in the upper 20 positions (backward: which M tiles to compute)
    float inv_nsel;
};

// The table image of one centre type, [128 lanes][ncols] words in global memory with the column order of tensor memory,
// is written to TMEM columns [0, ncols) by ALL warps of the CTA: warp w serves lane quarter w % 4 (the quarter it may
// address) and every (nwarps / 4)-th chunk of 8 columns; two chunks of loads are in flight before their stores.
__device__ __forceinline__ void cmp_load_image(uint32_t tmem, const uint32_t* __restrict__ img, int ncols, int warp, int lane, int nwarps) {
    const int quarter = warp & 3, slice = warp >> 2, nslice = nwarps >> 2;
    const uint32_t lanefield = ((uint32_t)(quarter * 32)) << 16;
    const uint4* src = reinterpret_cast<const uint4*>(img + (size_t)(quarter * 32 + lane) * ncols);
    const int nch = ncols >> 3;
    for (int ch0 = slice; ch0 < nch; ch0 += 2 * nslice) {
        const int ch1 = ch0 + nslice;
        const uint4 x0 = __ldg(src + 2 * ch0), x1 = __ldg(src + 2 * ch0 + 1);
        uint4 y0 = x0, y1 = x1;
        if (ch1 < nch) { y0 = __ldg(src + 2 * ch1); y1 = __ldg(src + 2 * ch1 + 1); }
        {
            const uint32_t v[8] = {x0.x, x0.y, x0.z, x0.w, x1.x, x1.y, x1.z, x1.w};
            tmem_st8(tmem + lanefield + ch0 * 8, v);
        }
        if (ch1 < nch) {                                                // warp-uniform
            const uint32_t v[8] = {y0.x, y0.y, y0.z, y0.w, y1.x, y1.y, y1.z, y1.w};
            tmem_st8(tmem + lanefield + ch1 * 8, v);
        }
    }
    tmem_st_wait();
}

// Position of interval iv inside the K order of the images.  Liquid water populates intervals 0..13 (r > 1.45 A) and
// 20, 21 (the O-H bond, s ~ 1.05); the order 0..13, 20, 21, 14..19, 22..39 puts all of them into the first 20
// positions = the first M tile of a neighbour type in the backward kernel and the first 8 k-steps in the forward one,
// so that the remaining MMAs are issued only for tiles that hold a row elsewhere (close contacts).
__host__ __device__ __forceinline__ int cmp_pos(int iv) { return iv < 14 ? iv : (iv < 20 ? iv + 2 : (iv < 22 ? iv - 6 : iv)); }

// interval and normalised offset of a row (R-28): iv = min(floor(s / h), 39), u = s / h - iv
__device__ __forceinline__ void cmp_locate(float s, int& iv, float& u) {
    iv = min((int)(s * cmp::kInvH), cmp::NI - 1);
    u = fmaf(s, cmp::kInvH, -(float)iv);
}

// The CTAs are dealt out to the centre types in proportion to their tile counts, so that a CTA loads ONE table image into
// tensor memory instead of one per type (the image load is ~8 us of a ~220 us kernel, per type).  Returns the CTA's index
// and the number of CTAs inside the share of type ti (bid < 0: none of this type's tiles are mine).  With fewer than two
// CTAs per type every CTA walks every type, as before.
__device__ __forceinline__ void cmp_cta_share(const CmpArgs& a, int ti, int& bid, int& gsz) {
    const int G = (int)gridDim.x, nt = a.ntypes;
    int ntile[PIMD_MAX_TYPES], tot = 0, live = 0;
#pragma unroll
    for (int t = 0; t < PIMD_MAX_TYPES; ++t) {
        ntile[t] = t < nt ? (a.type_row0[t + 1] - a.type_row0[t] + cmp::TC - 1) / cmp::TC : 0;
        tot += ntile[t];
        live += ntile[t] > 0 ? 1 : 0;
    }
    if (G < 2 * live || live < 2) { bid = (int)blockIdx.x; gsz = G; return; }
    int c0 = 0, pre = 0, left = live;
    bid = -1; gsz = 1;
#pragma unroll
    for (int t = 0; t < PIMD_MAX_TYPES; ++t) {
        if (ntile[t] == 0) continue;
        pre += ntile[t];
        --left;
        int c1 = (int)(((long long)G * pre + tot / 2) / tot);
        c1 = max(c1, c0 + 1);                              // at least one CTA for a type that has tiles ..
        c1 = min(c1, G - left);                            // .. and for every type still to come
        if (left == 0) c1 = G;
        if (t == ti && (int)blockIdx.x >= c0 && (int)blockIdx.x < c1) { bid = (int)blockIdx.x - c0; gsz = c1 - c0; }
        c0 = c1;
    }
}

// -------------------------------------------------------------------------------------------------
// forward: T_i = 1/N_sel  C^T Mom_i
// -------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(cmp::F_THREADS, 1)
cmp_fwd_kernel(const __grid_constant__ CmpArgs a) {
    using namespace cmp;
    extern __shared__ uint8_t smem_raw[];
    uint8_t* smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
    uint8_t* opB_hi = smem;
    uint8_t* opB_lo = smem + F_OPB;
    float* stage = reinterpret_cast<float*>(smem + 2 * F_OPB);
    float* rowbuf_all = reinterpret_cast<float*>(smem + 2 * F_OPB + F_STAGE);
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem + 2 * F_OPB + F_STAGE + F_WARPS * F_ROWBUF);
    uint64_t* ready = bars;            // moment warps -> MMA issuer: the operand buffer holds this tile   (count F_WARPS)
    uint64_t* opfree = bars + 1;       // MMAs of the tile have read the operand buffer                      (commit)
    uint64_t* mma_done = bars + 2;     // accumulator complete                                               (commit)
    uint64_t* d_free = bars + 3;       // epilogue has read the accumulator                                  (count 128)
    uint32_t* kmask = reinterpret_cast<uint32_t*>(bars + 4);      // [F_WARPS] k-steps with non-zero moments
    uint32_t* upm = kmask + F_WARPS;                               // [F_WARPS] the warp saw a row in the upper 20 positions
    uint32_t* tmem_ptr = upm + F_WARPS;

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (threadIdx.x == 0) {
        mbar_init(ready, F_WARPS);
        mbar_init(opfree, 1);
        mbar_init(mma_done, 1);
        mbar_init(d_free, 128);
        fence_barrier_init();
    }
    if (warp == F_WARPS) tmem_alloc(tmem_ptr, 512);
    // zero the FP32 stage once (the conversion re-zeroes what it reads) and both operand copies (K padding)
    for (int q = threadIdx.x; q < (2 * F_OPB + F_STAGE) / 16; q += F_THREADS)
        reinterpret_cast<uint4*>(smem)[q] = make_uint4(0u, 0u, 0u, 0u);
    fence_proxy_async_smem();
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = *tmem_ptr;
    constexpr uint32_t idesc = make_idesc_f16(128, NROW);
    const int nt = a.ntypes;
    uint32_t it = 0;                   // tiles this CTA has processed (all roles count alike)

    for (int ti = 0; ti < nt; ++ti) {
        const int row0 = a.type_row0[ti], row1 = a.type_row0[ti + 1];
        const int ntile = (row1 - row0 + TC - 1) / TC;
        int bid, gsz;
        cmp_cta_share(a, ti, bid, gsz);
        if (bid < 0 || ntile == 0) continue;               // CTA-uniform
        // ---- the table of centre type t_i goes into tensor memory (all MMAs of the previous type have retired:
        //      every role has passed its last tile, whose epilogue waited for mma_done) ----
        __syncthreads();
        cmp_load_image(tmem, a.img_fw + (size_t)ti * 128 * (2 * FW_COLS), 2 * FW_COLS, warp, lane, F_THREADS / 32);
        tc_fence_before();
        __syncthreads();
        tc_fence_after();

        if (warp < F_WARPS) {
            // ================= moment warps: (centre cl, neighbour type tj) =================
            const int cl = warp >> 1, tj = warp & 1;
            float* stg = stage + cl * 4 * STG;                       // [4 c][STG], shared by the two warps of the centre
            float* rowbuf = rowbuf_all + warp * (F_ROWBUF / 4);      // (they own disjoint k ranges)
            const int p = lane >> 2, c = lane & 3;
            // Row data is prefetched one tile ahead into registers and the (centre, count) pair two tiles ahead: all 16
            // moment warps of a CTA reach the same point of a tile together, so an exposed cen_idx -> ncount -> slot
            // load chain (three dependent L2 / HBM round trips) would be paid by the whole SM at once.
            struct RowF { float dx, dy, dz, s, rinv; };
            auto meta = [&](int tile, size_t& s0, int& n) {
                const int r = row0 + tile * TC + cl;
                s0 = 0; n = 0;
                if (tile < ntile && r < row1 && tj < nt) {
                    const int ba = __ldg(a.cen_idx + r);
                    n = __ldg(a.ncount + (size_t)ba * nt + tj);
                    s0 = (size_t)ba * a.nsel + a.seloff[tj];
                }
            };
            auto load_row = [&](size_t slot) {
                const float4 A = __ldg(reinterpret_cast<const float4*>(a.slotA) + slot);
                RowF R;
                R.dx = A.x; R.dy = A.y; R.dz = A.z; R.s = A.w; R.rinv = __ldg(&a.slotB[slot].rinv);
                return R;
            };
            auto load_rows = [&](size_t s0, int n, RowF (&R)[3]) {
#pragma unroll
                for (int b = 0; b < 3; ++b)
                    if (32 * b + lane < n) R[b] = load_row(s0 + 32 * b + lane);
            };
            const int hotk = tj * NI * NP;                           // bucket (tj, interval 0): two thirds of all rows
            // one batch of up to 32 rows: lane = row writes its 24 products u^p R_c, then lane = (p, c) adds them up
            bool up = false;
            auto batch = [&](const RowF& R, int nb, float& acc0) {
                // rows of the hot bucket (interval 0 of this neighbour type) are compacted to the front of the row buffer:
                // their sum needs no bucket lookup and no read-modify-write, only independent loads and adds
                const bool act = lane < nb;
                int iv = 0; float u = 0.f;
                const float s = act ? R.s : 0.f;
                if (act) {
                    if (s > kSHi) {                              // outside the table: an error, not an extrapolation (R-28)
                        atomicOr(a.overflow, 4);
                        atomicMin(reinterpret_cast<unsigned*>(a.overflow) + 1, (unsigned)a.overflow[2]);
                    }
                    cmp_locate(s, iv, u);
                }
                const int pos = cmp_pos(iv);
                const bool hot = act && pos == 0;
                const unsigned hm = __ballot_sync(0xffffffffu, hot), cm = __ballot_sync(0xffffffffu, act && !hot);
                const unsigned lt = (1u << lane) - 1u;
                const int nh = __popc(hm);
                if (act) {
                    up |= pos >= NI / 2;
                    const float sr = s * R.rinv;
                    const float Rv[4] = {s, sr * R.dx, sr * R.dy, sr * R.dz};
                    float* rb = rowbuf + (hot ? __popc(hm & lt) : nh + __popc(cm & lt)) * 25;
                    float pw = 1.f;
#pragma unroll
                    for (int pp = 0; pp < NP; ++pp) {
#pragma unroll
                        for (int cc = 0; cc < 4; ++cc) rb[pp * 4 + cc] = pw * Rv[cc];
                        pw *= u;
                    }
                    rb[24] = __int_as_float((tj * NI + pos) * NP);
                }
                __syncwarp();
                if (lane < 24) {
                    float h0 = 0.f, h1 = 0.f, h2 = 0.f, h3 = 0.f;
                    int q = 0;
                    for (; q + 4 <= nh; q += 4) {
                        h0 += rowbuf[q * 25 + lane]; h1 += rowbuf[(q + 1) * 25 + lane];
                        h2 += rowbuf[(q + 2) * 25 + lane]; h3 += rowbuf[(q + 3) * 25 + lane];
                    }
                    for (; q < nh; ++q) h0 += rowbuf[q * 25 + lane];
                    acc0 += (h0 + h1) + (h2 + h3);
                    for (q = nh; q < nb; ++q) {
                        const float v = rowbuf[q * 25 + lane];
                        const int k0 = __float_as_int(rowbuf[q * 25 + 24]);
                        stg[c * STG + k0 + p] += v;
                    }
                }
                __syncwarp();
            };
            size_t s0c, s0n; int nc, nn;
            RowF cur[3];
            meta(bid, s0c, nc);
            load_rows(s0c, nc, cur);
            meta(bid + gsz, s0n, nn);
            for (int tile = bid; tile < ntile; tile += gsz, ++it) {
                RowF nxt[3];
                load_rows(s0n, nn, nxt);                             // the next tile's rows are in flight during this one
                size_t s0nn; int nnn;
                meta(tile + 2 * gsz, s0nn, nnn);
                float acc0 = 0.f;
#pragma unroll
                for (int b = 0; b < 3; ++b)
                    if (32 * b < nc) batch(cur[b], min(32, nc - 32 * b), acc0);
                for (int q0 = 96; q0 < nc; q0 += 32) {               // sel > 96: not prefetched
                    RowF R = {0.f, 0.f, 0.f, 0.f, 1.f};
                    if (q0 + lane < nc) R = load_row(s0c + q0 + lane);
                    batch(R, min(32, nc - q0), acc0);
                }
                if (lane < 24) stg[c * STG + hotk + p] += acc0;
#pragma unroll
                for (int b = 0; b < 3; ++b) cur[b] = nxt[b];
                s0c = s0n; nc = nn; s0n = s0nn; nn = nnn;
                // ---- my half of the centre's moments -> FP16 hi / lo operand rows 4 cl + c (K-major, SWIZZLE_128B),
                //      once the MMAs of the previous tile have read the buffer; the stage is zeroed on the way ----
                __syncwarp();
                if (it > 0) mbar_wait(opfree, (it - 1) & 1);
                uint32_t km = 0;
                for (int ch = lane; ch < 4 * (KB / 8); ch += 32) {
                    const int cc = ch / (KB / 8), kk = tj * KB + (ch - cc * (KB / 8)) * 8;
                    float* src = stg + cc * STG + kk;
                    const float4 v0 = *reinterpret_cast<const float4*>(src), v1 = *reinterpret_cast<const float4*>(src + 4);
                    *reinterpret_cast<float4*>(src) = make_float4(0.f, 0.f, 0.f, 0.f);
                    *reinterpret_cast<float4*>(src + 4) = make_float4(0.f, 0.f, 0.f, 0.f);
                    const float v[8] = {v0.x, v0.y, v0.z, v0.w, v1.x, v1.y, v1.z, v1.w};
                    const bool nz = (v0.x != 0.f) | (v0.y != 0.f) | (v0.z != 0.f) | (v0.w != 0.f) | (v1.x != 0.f) |
                                    (v1.y != 0.f) | (v1.z != 0.f) | (v1.w != 0.f);
                    if (nz) km |= 1u << (kk >> 4);
                    uint4 hi, lo;
                    split8(v, hi, lo);
                    const int row = 4 * cl + cc, kb = kk >> 6, chunk = (kk & 63) >> 3;
                    const int off = kb * (NROW * 128) + row * 128 + ((chunk ^ (row & 7)) << 4);
                    *reinterpret_cast<uint4*>(opB_hi + off) = hi;
                    *reinterpret_cast<uint4*>(opB_lo + off) = lo;
                }
                km = __reduce_or_sync(0xffffffffu, km);
                fence_proxy_async_smem();
                __syncwarp();
                const bool upw = __any_sync(0xffffffffu, up);
                up = false;
                if (lane == 0) {
                    kmask[warp] = km;
                    upm[warp] = upw ? 1u : 0u;
                    mbar_arrive(ready);
                }
            }
        } else {
            // ================= tensor warpgroup: MMA issue (one thread) + epilogue (TMEM lane = channel) =================
            const int wq = warp - F_WARPS;
            const int m = wq * 32 + lane;
            const uint32_t lanefield = ((uint32_t)(wq * 32)) << 16;
            for (int tile = bid; tile < ntile; tile += gsz, ++it) {
                if (wq == 0) {
                    mbar_wait(ready, it & 1);
                    if (it > 0) mbar_wait(d_free, (it - 1) & 1);
                    tc_fence_after();
                    {   // all 32 lanes run the (uniform) loop, one elected lane issues
                        uint32_t km = 1u, nd = 0u;                 // k-step 0 always: the accumulator is always written
                        for (int w = 0; w < F_WARPS; ++w) { km |= kmask[w]; nd |= upm[w] << (w & 1); }
                        if (lane == 0) a.need[row0 / TC + ti + tile] = nd;
                        const uint64_t dbh0 = make_smem_desc_kmajor(smem_u32(opB_hi), 128), dbl0 = make_smem_desc_kmajor(smem_u32(opB_lo), 128);
                        uint32_t acc = 0;
                        for (int ks = 0; ks < K / 16; ++ks) {
                            if (!((km >> ks) & 1u)) continue;
                            const uint64_t bo = (uint64_t)(((ks >> 2) * (NROW * 128) + (ks & 3) * 32) >> 4);
                            const uint32_t ahi = tmem + ks * 8, alo = tmem + FW_COLS + ks * 8;
                            umma_f16_ts_elect(tmem + FW_D, ahi, dbh0 + bo, idesc, acc);
                            umma_f16_ts_elect(tmem + FW_D, alo, dbh0 + bo, idesc, 1u);
                            umma_f16_ts_elect(tmem + FW_D, ahi, dbl0 + bo, idesc, 1u);
                            acc = 1u;
                        }
                        umma_commit_elect(opfree);
                        umma_commit_elect(mma_done);
                    }
                    __syncwarp();
                }
                mbar_wait(mma_done, it & 1);
                tc_fence_after();
                uint32_t v[32];
                tmem_ld32(tmem + lanefield + FW_D, v);
                tmem_ld_wait();
                tc_fence_before();
                mbar_arrive(d_free);
                if (m < M1) {
#pragma unroll
                    for (int cl = 0; cl < TC; ++cl) {
                        const int r = row0 + tile * TC + cl;
                        if (r < row1)
                            *reinterpret_cast<float4*>(a.Tm + ((size_t)r * M1 + m) * 4) =
                                make_float4(__uint_as_float(v[4 * cl]) * a.inv_nsel, __uint_as_float(v[4 * cl + 1]) * a.inv_nsel,
                                            __uint_as_float(v[4 * cl + 2]) * a.inv_nsel, __uint_as_float(v[4 * cl + 3]) * a.inv_nsel);
                    }
                }
            }
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == F_WARPS) tmem_dealloc(tmem, 512);
}

// -------------------------------------------------------------------------------------------------
// backward: Q_i = C dT_i in tensor memory -> shared memory; rows: dR, ds, pair gradient, force and virial
// -------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(cmp::B_THREADS, 1)
cmp_bwd_kernel(const __grid_constant__ CmpArgs a) {
    using namespace cmp;
    extern __shared__ uint8_t smem_raw[];
    uint8_t* smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
    uint8_t* opB_hi = smem;
    uint8_t* opB_lo = smem + B_OPB;
    float4* Qs = reinterpret_cast<float4*>(smem + 2 * B_OPB);                  // [2 buffers][TC][K]
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem + 2 * B_OPB + 2 * B_Q);
    uint64_t* qfull = bars;            // [2] tensor group -> row warps (count 128)
    uint64_t* qempty = bars + 2;       // [2] row warps -> tensor group (count B_WARPS)
    uint64_t* dfull = bars + 4;        // [2] MMAs of an M tile complete (commit)
    float* inv_scale = reinterpret_cast<float*>(bars + 6);                     // [TC]
    uint32_t* tmem_ptr = reinterpret_cast<uint32_t*>(inv_scale + TC);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (threadIdx.x == 0) {
        for (int b = 0; b < 2; ++b) { mbar_init(qfull + b, 128); mbar_init(qempty + b, B_WARPS); mbar_init(dfull + b, 1); }
        fence_barrier_init();
    }
    if (warp == B_WARPS) tmem_alloc(tmem_ptr, 512);
    for (int q = threadIdx.x; q < 2 * B_OPB / 16; q += B_THREADS) reinterpret_cast<uint4*>(smem)[q] = make_uint4(0u, 0u, 0u, 0u);
    fence_proxy_async_smem();
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = *tmem_ptr;
    constexpr uint32_t idesc = make_idesc_f16(128, NROW);
    const int nt = a.ntypes;
    uint32_t it = 0, ndf0 = 0u, ndf1 = 0u;  // tiles processed; completed uses of each accumulator buffer

    for (int ti = 0; ti < nt; ++ti) {
        const int row0 = a.type_row0[ti], row1 = a.type_row0[ti + 1];
        const int ntile = (row1 - row0 + TC - 1) / TC;
        int bid, gsz;
        cmp_cta_share(a, ti, bid, gsz);
        if (bid < 0 || ntile == 0) continue;               // CTA-uniform
        __syncthreads();
        cmp_load_image(tmem, a.img_bw + (size_t)ti * 128 * BW_D, BW_D, warp, lane, B_THREADS / 32);
        tc_fence_before();
        __syncthreads();
        tc_fence_after();

        if (warp >= B_WARPS) {
            // ================= tensor warpgroup =================
            const int wq = warp - B_WARPS, t = wq * 32 + lane;
            const uint32_t lanefield = ((uint32_t)(wq * 32)) << 16;
            // dT of my (centre, 8 channels) piece, fetched one tile ahead
            const int cl = t >> 4, n0 = (t & 15) * 8;
            auto load_dT = [&](int tile, float4 (&x)[8]) {
                const int r = row0 + tile * TC + cl;
#pragma unroll
                for (int q = 0; q < 8; ++q)
                    x[q] = (tile < ntile && r < row1 && n0 + q < M1)
                               ? __ldg(reinterpret_cast<const float4*>(a.dTm) + (size_t)r * M1 + n0 + q)
                               : make_float4(0.f, 0.f, 0.f, 0.f);
            };
            float4 x[8];
            load_dT(bid, x);
            uint32_t nd_next = (bid < ntile) ? __ldg(a.need + row0 / TC + ti + bid) : 0u;
            for (int tile = bid; tile < ntile; tile += gsz, ++it) {
                const int buf = it & 1;
                // ---- dT of the tile's centres -> operand rows (centre, c), K = channel; scaled per centre by the
                //      power of two that brings max |dT| to [1, 2) (FP16 range; undone when Q is written) ----
                {
                    float mx = 0.f;
#pragma unroll
                    for (int q = 0; q < 8; ++q)
                        mx = fmaxf(mx, fmaxf(fmaxf(fabsf(x[q].x), fabsf(x[q].y)), fmaxf(fabsf(x[q].z), fabsf(x[q].w))));
#pragma unroll
                    for (int o = 8; o > 0; o >>= 1) mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, o));
                    const uint32_t e = (__float_as_uint(mx) >> 23) & 0xffu;
                    const float sc = (e == 0u || e >= 254u) ? 1.f : __uint_as_float((254u - e) << 23);     // 2^(127 - e)
                    if ((t & 15) == 0) inv_scale[cl] = (e == 0u || e >= 254u) ? 1.f : __uint_as_float(e << 23);
                    if (n0 < BW_KP) {
#pragma unroll
                        for (int c = 0; c < 4; ++c) {
                            float v[8];
#pragma unroll
                            for (int q = 0; q < 8; ++q) v[q] = (c == 0 ? x[q].x : c == 1 ? x[q].y : c == 2 ? x[q].z : x[q].w) * sc;
                            uint4 hi, lo;
                            split8(v, hi, lo);
                            const int row = 4 * cl + c, kb = n0 >> 6, chunk = (n0 & 63) >> 3;
                            const int off = kb * (NROW * 128) + row * 128 + ((chunk ^ (row & 7)) << 4);
                            *reinterpret_cast<uint4*>(opB_hi + off) = hi;
                            *reinterpret_cast<uint4*>(opB_lo + off) = lo;
                        }
                    }
                }
                load_dT(tile + gsz, x);                        // next tile's dT in flight under this tile's MMAs
                fence_proxy_async_smem();
                if (it >= 2) mbar_wait(qempty + buf, ((it >> 1) - 1) & 1);     // the row warps have left this Q buffer
                tc_fence_before();
                cmp_bar_sync(1, 128);
                auto issue = [&](int j, int db) {
                    if (t < 32) {                          // converged warp, one elected lane issues
                        tc_fence_after();
                        const uint64_t dbh0 = make_smem_desc_kmajor(smem_u32(opB_hi), 128), dbl0 = make_smem_desc_kmajor(smem_u32(opB_lo), 128);
                        const uint32_t d = tmem + BW_D + db * NROW;
#pragma unroll
                        for (int ks = 0; ks < BW_KP / 16; ++ks) {
                            const uint64_t bo = (uint64_t)(((ks >> 2) * (NROW * 128) + (ks & 3) * 32) >> 4);
                            const uint32_t ahi = tmem + j * 2 * BW_COLS + ks * 8, alo = ahi + BW_COLS;
                            umma_f16_ts_elect(d, ahi, dbh0 + bo, idesc, ks ? 1u : 0u);
                            umma_f16_ts_elect(d, alo, dbh0 + bo, idesc, 1u);
                            umma_f16_ts_elect(d, ahi, dbl0 + bo, idesc, 1u);
                        }
                        umma_commit_elect(dfull + db);
                    }
                };
                // M tiles of this tile of centres: the lower 20 positions of both neighbour types always (j = 0, 2), the
                // upper ones (j = 1, 3) only when a row sits there.  Two accumulator buffers, used in turn.
                const uint32_t nd = nd_next;
                nd_next = (tile + gsz < ntile) ? __ldg(a.need + row0 / TC + ti + tile + gsz) : 0u;
                const int nj = 2 + (int)(nd & 1u) + (int)((nd >> 1) & 1u);
                auto jof = [&](int idx) { return idx == 0 ? 0 : idx == 1 ? 2 : (idx == 2 ? ((nd & 1u) ? 1 : 3) : 3); };
                issue(0, 0);
                issue(2, 1);
                float4* Qb = Qs + (size_t)buf * (TC * K);
#pragma unroll 1
                for (int idx = 0; idx < nj; ++idx) {
                    const int db = idx & 1, j = jof(idx);
                    mbar_wait(dfull + db, (db ? ndf1 : ndf0) & 1);
                    if (db) ++ndf1; else ++ndf0;
                    tc_fence_after();
                    uint32_t v[32];
                    tmem_ld32(tmem + lanefield + BW_D + db * NROW, v);
                    tmem_ld_wait();
                    if (t < BW_ROWS) {
#pragma unroll
                        for (int cl2 = 0; cl2 < TC; ++cl2) {
                            const float is = inv_scale[cl2];
                            Qb[cl2 * K + j * BW_ROWS + t] = make_float4(__uint_as_float(v[4 * cl2]) * is, __uint_as_float(v[4 * cl2 + 1]) * is,
                                                                        __uint_as_float(v[4 * cl2 + 2]) * is, __uint_as_float(v[4 * cl2 + 3]) * is);
                        }
                    }
                    if (idx + 2 < nj) {
                        tc_fence_before();
                        cmp_bar_sync(1, 128);                       // every thread has read this accumulator buffer
                        issue(jof(idx + 2), db);
                    }
                }
                tc_fence_before();
                mbar_arrive(qfull + buf);                           // release: my Q stores are visible to the waiters
                cmp_bar_sync(1, 128);                               // inv_scale / operand rows are free for the next tile
            }
        } else {
            // ================= row warps: (centre cl, neighbour type tj), lane = row =================
            const int cl = warp >> 1, tj = warp & 1;
            const float inv_h = kInvH;
            struct RowB { float dx, dy, dz, s, dsw, rinv; uint32_t jcode; };
            auto meta = [&](int tile, int& r, int& ba, int& n) {
                r = row0 + tile * TC + cl;
                ba = 0; n = 0;
                if (tile < ntile && r < row1 && tj < nt) {
                    ba = __ldg(a.cen_idx + r);
                    n = __ldg(a.ncount + (size_t)ba * nt + tj);
                }
            };
            auto load_row = [&](size_t slot) {
                const float4 A = __ldg(reinterpret_cast<const float4*>(a.slotA) + slot);
                const float4 B = __ldg(reinterpret_cast<const float4*>(a.slotB) + slot);
                RowB R;
                R.dx = A.x; R.dy = A.y; R.dz = A.z; R.s = A.w; R.dsw = B.x; R.rinv = B.y; R.jcode = __float_as_uint(B.z);
                return R;
            };
            int rn, ban, nn;
            meta(bid, rn, ban, nn);
            for (int tile = bid; tile < ntile; tile += gsz, ++it) {
                const int buf = it & 1;
                const int r = rn, ba = ban, n = nn;
                const size_t s0 = (size_t)ba * a.nsel + a.seloff[tj];
                // my rows are loaded BEFORE the wait for Q (their latency hides under the tensor group's work on this
                // tile), the next tile's (centre, count) pair behind them
                RowB rows[3];
#pragma unroll
                for (int b = 0; b < 3; ++b)
                    if (32 * b + lane < n) rows[b] = load_row(s0 + 32 * b + lane);
                meta(tile + gsz, rn, ban, nn);
                mbar_wait(qfull + buf, (it >> 1) & 1);
                if (n > 0) {
                    const float4* Qc = Qs + (size_t)buf * (TC * K) + cl * K + tj * KB;
                    double* fb = a.f + (size_t)(ba / a.N) * a.N * 3;
                    float acc[12];
#pragma unroll
                    for (int q = 0; q < 12; ++q) acc[q] = 0.f;
                    auto one = [&](const RowB& R) {
                        const float s = R.s, dsw = R.dsw, rinv = R.rinv;
                        int iv; float u;
                        cmp_locate(s, iv, u);
                        const float4* Q = Qc + cmp_pos(iv) * NP;
                        const float4 q5 = Q[5], q4 = Q[4], q3 = Q[3], q2 = Q[2], q1 = Q[1], q0v = Q[0];
                        // A_c = sum_p u^p Q_p[c],  D_c = sum_p p u^(p-1) Q_p[c]  (Horner)
                        float Av[4], Dv[4];
                        const float a5[4] = {q5.x, q5.y, q5.z, q5.w}, a4[4] = {q4.x, q4.y, q4.z, q4.w}, a3[4] = {q3.x, q3.y, q3.z, q3.w};
                        const float a2[4] = {q2.x, q2.y, q2.z, q2.w}, a1[4] = {q1.x, q1.y, q1.z, q1.w}, a0[4] = {q0v.x, q0v.y, q0v.z, q0v.w};
#pragma unroll
                        for (int c = 0; c < 4; ++c) {
                            float v = a5[c];
                            v = fmaf(v, u, a4[c]); v = fmaf(v, u, a3[c]); v = fmaf(v, u, a2[c]); v = fmaf(v, u, a1[c]); v = fmaf(v, u, a0[c]);
                            Av[c] = v;
                            float d = 5.f * a5[c];
                            d = fmaf(d, u, 4.f * a4[c]); d = fmaf(d, u, 3.f * a3[c]); d = fmaf(d, u, 2.f * a2[c]); d = fmaf(d, u, a1[c]);
                            Dv[c] = d;
                        }
                        const float sr = s * rinv;
                        const float R0 = s, R1 = sr * R.dx, R2 = sr * R.dy, R3 = sr * R.dz;
                        const float w = a.inv_nsel;
                        const float ds = (R0 * Dv[0] + R1 * Dv[1] + R2 * Dv[2] + R3 * Dv[3]) * (w * inv_h);
                        const float dR0 = Av[0] * w, dR1 = Av[1] * w, dR2 = Av[2] * w, dR3 = Av[3] * w;
                        // pair gradient g = dU/dd (R-16), as in embedding_tc.cu
                        const float dot = dR1 * R.dx + dR2 * R.dy + dR3 * R.dz;
                        const float radial = (ds + dR0) * dsw + (dsw * rinv - s * rinv * rinv) * dot;
                        const float rr = radial * rinv;
                        const float gx = fmaf(rr, R.dx, sr * dR1), gy = fmaf(rr, R.dy, sr * dR2), gz = fmaf(rr, R.dz, sr * dR3);
                        double* fj = fb + (size_t)(R.jcode & 0x7fffffu) * 3;
                        atomicAdd(fj, -(double)gx); atomicAdd(fj + 1, -(double)gy); atomicAdd(fj + 2, -(double)gz);
                        acc[0] += gx; acc[1] += gy; acc[2] += gz;
                        const float dd[3] = {R.dx, R.dy, R.dz}, gg[3] = {gx, gy, gz};
#pragma unroll
                        for (int xq = 0; xq < 3; ++xq)
#pragma unroll
                            for (int y = 0; y < 3; ++y) acc[3 + 3 * xq + y] -= dd[xq] * gg[y];
                    };
#pragma unroll
                    for (int b = 0; b < 3; ++b)
                        if (32 * b + lane < n) one(rows[b]);
                    for (int q0 = 96; q0 < n; q0 += 32)              // sel > 96: not prefetched
                        if (q0 + lane < n) one(load_row(s0 + q0 + lane));
#pragma unroll
                    for (int q = 0; q < 12; ++q)
#pragma unroll
                        for (int o = 16; o > 0; o >>= 1) acc[q] += __shfl_xor_sync(0xffffffffu, acc[q], o);
                    if (lane == 0) {
                        double* fi = a.f + (size_t)ba * 3;
                        atomicAdd(fi, (double)acc[0]); atomicAdd(fi + 1, (double)acc[1]); atomicAdd(fi + 2, (double)acc[2]);
                        double* cp = a.cpart + (size_t)r * 9;
#pragma unroll
                        for (int q = 0; q < 9; ++q) atomicAdd(cp + q, (double)acc[3 + q]);
                    }
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(qempty + buf);
            }
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == B_WARPS) tmem_dealloc(tmem, 512);
}

// Xi^(k) = sum of the per-centre virial shares of bead k (one block per bead)
__global__ void __launch_bounds__(256)
cmp_virial_reduce_kernel(int ntypes, CmpArgs a, double* __restrict__ Xi) {
    const int k = blockIdx.x;
    double acc[9];
#pragma unroll
    for (int q = 0; q < 9; ++q) acc[q] = 0.0;
    for (int tt = 0; tt < ntypes; ++tt) {
        const int r0 = a.type_row0[tt] + k * a.n_of_type[tt];
        for (int r = r0 + threadIdx.x; r < r0 + a.n_of_type[tt]; r += 256) {
#pragma unroll
            for (int q = 0; q < 9; ++q) acc[q] += a.cpart[(size_t)r * 9 + q];
        }
    }
    __shared__ double red[8][9];
#pragma unroll
    for (int q = 0; q < 9; ++q)
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) acc[q] += __shfl_xor_sync(0xffffffffu, acc[q], o);
    if ((threadIdx.x & 31) == 0)
        for (int q = 0; q < 9; ++q) red[threadIdx.x >> 5][q] = acc[q];
    __syncthreads();
    if (threadIdx.x < 9) {
        double s = 0.0;
        for (int w = 0; w < 8; ++w) s += red[w][threadIdx.x];
        Xi[k * 9 + threadIdx.x] = s;
    }
}

// -------------------------------------------------------------------------------------------------
// host side: tables (FP64) -> tensor-memory images
// -------------------------------------------------------------------------------------------------
// value, first and second s-derivative of the embedding net of one pair (R-13) at s, by forward-mode differentiation;
// w = W1[1][25], b1, W2[25][50], b2, W3[50][100], b3 (row-major in x out)
static void cmp_net_d2(const double* w, double s, double* y, double* y1, double* y2) {
    const int dims[4] = {1, 25, 50, 100};
    std::vector<double> h(1, s), h1(1, 1.0), h2(1, 0.0);
    size_t pos = 0;
    for (int l = 0; l < 3; ++l) {
        const int nin = dims[l], nout = dims[l + 1];
        const double* W = w + pos;
        const double* b = W + (size_t)nin * nout;
        pos += (size_t)nin * nout + nout;
        std::vector<double> o(nout), o1(nout), o2(nout);
        for (int n = 0; n < nout; ++n) {
            double z = b[n], z1 = 0.0, z2 = 0.0;
            for (int k = 0; k < nin; ++k) {
                const double wk = W[(size_t)k * nout + n];
                z += h[k] * wk; z1 += h1[k] * wk; z2 += h2[k] * wk;
            }
            const double t = std::tanh(z), u = 1.0 - t * t;
            double v = t, v1 = u * z1, v2 = u * z2 - 2.0 * t * u * z1 * z1;
            if (nout == 2 * nin) { v += h[n % nin]; v1 += h1[n % nin]; v2 += h2[n % nin]; }
            else if (nout == nin) { v += h[n]; v1 += h1[n]; v2 += h2[n]; }
            o[n] = v; o1[n] = v1; o2[n] = v2;
        }
        h.swap(o); h1.swap(o1); h2.swap(o2);
    }
    for (int n = 0; n < cmp::M1; ++n) { y[n] = h[n]; y1[n] = h1[n]; y2[n] = h2[n]; }
}

// coefficients in the normalised variable u = (s - s_n)/h:  C[iv][p][m]  (R-28: quintic Hermite, value and two
// derivatives at both nodes)
static void cmp_pair_table(const double* w_pair, std::vector<double>& C) {
    using namespace cmp;
    const double h = 1.0 / (double)kInvH;
    std::vector<double> y((NI + 1) * M1), y1((NI + 1) * M1), y2((NI + 1) * M1);
    for (int n = 0; n <= NI; ++n) cmp_net_d2(w_pair, h * n, &y[(size_t)n * M1], &y1[(size_t)n * M1], &y2[(size_t)n * M1]);
    C.assign((size_t)NI * NP * M1, 0.0);
    for (int iv = 0; iv < NI; ++iv)
        for (int m = 0; m < M1; ++m) {
            const double a0 = y[(size_t)iv * M1 + m], a1 = h * y1[(size_t)iv * M1 + m], a2 = 0.5 * h * h * y2[(size_t)iv * M1 + m];
            const double b0 = y[(size_t)(iv + 1) * M1 + m], b1 = h * y1[(size_t)(iv + 1) * M1 + m], b2 = h * h * y2[(size_t)(iv + 1) * M1 + m];
            const double D0 = b0 - (a0 + a1 + a2), D1 = b1 - (a1 + 2.0 * a2), D2 = b2 - 2.0 * a2;
            double* c = &C[(size_t)iv * NP * M1];
            c[0 * M1 + m] = a0; c[1 * M1 + m] = a1; c[2 * M1 + m] = a2;
            c[3 * M1 + m] = 10.0 * D0 - 4.0 * D1 + 0.5 * D2;
            c[4 * M1 + m] = -15.0 * D0 + 7.0 * D1 - D2;
            c[5 * M1 + m] = 6.0 * D0 - 3.0 * D1 + 0.5 * D2;
        }
}

size_t cmp_image_words_fw(int ntypes) { return (size_t)ntypes * 2 * 128 * cmp::FW_COLS; }
size_t cmp_image_words_bw(int ntypes) { return (size_t)ntypes * 2 * cmp::BW_MT * 128 * cmp::BW_COLS; }

// w_emb: the embedding weights of all ordered pairs in the C-ABI packing order (6450 doubles per pair)
void cmp_build_images(const double* w_emb, int ntypes, uint32_t* img_fw, uint32_t* img_bw) {
    using namespace cmp;
    const size_t per_pair = (size_t)2 * 25 + 25 * 50 + 50 + 50 * 100 + 100;
    memset(img_fw, 0, cmp_image_words_fw(ntypes) * 4);
    memset(img_bw, 0, cmp_image_words_bw(ntypes) * 4);
    auto put = [](uint32_t* word, int half_idx, float v, bool lo_part) {
        const __half hi = __float2half_rn(v);
        const __half val = lo_part ? __float2half_rn(v - __half2float(hi)) : hi;
        uint16_t bits;
        memcpy(&bits, &val, 2);
        *word = (*word & ~(0xffffu << (16 * half_idx))) | ((uint32_t)bits << (16 * half_idx));
    };
    std::vector<double> C;
    for (int ti = 0; ti < ntypes; ++ti)
        for (int tj = 0; tj < ntypes; ++tj) {
            cmp_pair_table(w_emb + (size_t)(ti * ntypes + tj) * per_pair, C);
            for (int iv = 0; iv < NI; ++iv)
                for (int p = 0; p < NP; ++p)
                    for (int m = 0; m < M1; ++m) {
                        const float v = (float)C[((size_t)iv * NP + p) * M1 + m];
                        const int k = tj * KB + cmp_pos(iv) * NP + p;
                        for (int copy = 0; copy < 2; ++copy) {
                            put(img_fw + (((size_t)ti * 128 + m) * 2 + copy) * FW_COLS + (k >> 1), k & 1, v, copy == 1);
                            const int j = k / BW_ROWS, lanek = k - j * BW_ROWS;
                            put(img_bw + ((((size_t)ti * 128 + lanek) * BW_MT + j) * 2 + copy) * BW_COLS + (m >> 1), m & 1, v, copy == 1);
                        }
                    }
        }
}

static CmpArgs make_cmp_args(Model& m, const ForceArgs& fa) {
    CmpArgs a;
    a.PN = fa.P * fa.N; a.N = fa.N; a.ntypes = fa.ntypes; a.nsel = m.nsel;
    for (int t = 0; t <= PIMD_MAX_TYPES; ++t) { a.seloff[t] = m.seloff[t]; a.type_row0[t] = m.type_row0[t]; }
    for (int t = 0; t < PIMD_MAX_TYPES; ++t) a.n_of_type[t] = (t < fa.ntypes) ? m.n_of_type[t] : 0;
    a.cen_idx = m.cen_idx; a.ncount = m.ncount; a.slotA = m.slotA; a.slotB = m.slotB;
    a.img_fw = m.cmp_img_fw; a.img_bw = m.cmp_img_bw;
    a.Tm = m.Tm; a.dTm = m.dTm; a.f = fa.f; a.cpart = m.cpart; a.overflow = m.overflow; a.need = m.cmp_need;
    a.inv_nsel = 1.0f / (float)m.nsel;
    return a;
}

int compressed_forward(Model& m, const ForceArgs& fa, int n_sms, cudaStream_t s) {
    CmpArgs a = make_cmp_args(m, fa);
    ensure_dyn_smem(cmp_fwd_kernel, cmp::F_SMEM);
    cmp_fwd_kernel<<<n_sms, cmp::F_THREADS, cmp::F_SMEM, s>>>(a);
    return 1;
}

int compressed_backward(Model& m, const ForceArgs& fa, int n_sms, cudaStream_t s) {
    CmpArgs a = make_cmp_args(m, fa);
    ensure_dyn_smem(cmp_bwd_kernel, cmp::B_SMEM);
    cudaMemsetAsync(m.cpart, 0, sizeof(double) * (size_t)a.PN * 9, s);
    cmp_bwd_kernel<<<n_sms, cmp::B_THREADS, cmp::B_SMEM, s>>>(a);
    cmp_virial_reduce_kernel<<<fa.P, 256, 0, s>>>(fa.ntypes, a, fa.Xi);
    return 2;
}

}  // namespace pimd
