// embedding_tc.cu -- F3 and F5/F6 of SURVEY 8(a) on the 5th-generation tensor cores (tcgen05 kind::f16 + TMEM,
// three-pass FP16-split products with FP32 accumulation).
//
// Neighbour rows are processed in tiles of 128 rows of ONE ordered type pair (t_i, t_j) -- one weight set,
// resident in shared memory as ready-made UMMA B operands (FP16 hi / lo split, swizzled K-major, bias folded
// in as an extra K row).  A row is one TMEM lane and is shared by TWO threads (halves A and B,
// warps w and w+4 of a context: both may touch the same TMEM lane quarter), each owning half of the columns:
//   h1 = tanh(s W1 + b1)                  CUDA cores (K = 1); 13 of the 26 (25 + 1 dummy) channels per thread
//   z2 = [h1,1] W2b   (128 x 64 x 32)     tcgen05.mma kind::f16, three passes: a_hi b_hi + a_lo b_hi + a_hi b_lo
//   h2 = [h1,h1] + tanh(z2)               epilogue: tcgen05.ld -> registers -> next A operand in smem
//   z3 = [h2,1] W3b   (128 x 112 x 64)
//   G  = [h2,h2] + tanh(z3)                                                                    (R-13)
// The channels are permuted (and padded with zero-weight dummies, 25 -> 26, 50 -> 52, 100 -> 104) so that the
// skip connections stay thread-local: the thread that owns h1 channel i also owns h2 channels i and i + 25 and
// G channels i, i + 25, i + 50, i + 75 (see `Perm` below).  Halving the per-thread state is what lets 16 warps
// (2 contexts x 2 halves x 4 lane quarters) fit the register file: the kernels are bound by MUFU and issue
// latency, not by the tensor pipe, so they need the extra warps.
// Forward:  T_i += (1/N_sel) sum_rows G (x) R  (R-14): G tile through smem; the two warps of a lane quarter
//           split its 32 rows, lane <-> 4 G positions, red.global.add.v4.f32 on (warp-uniform) centre change.
// Backward: forward-mode -- the derivative rows h' = dh/ds go through the same weights (bias slot 0):
//           G' = [h2',h2'] + (1 - tanh^2 z3) z3';  ds = sum_n (dT_n . R) G'_n = R . E, E_c = sum_n dT_nc G'_n;
//           dR_c = sum_n dT_nc G_n;  pair gradient g = dU/dd (R-16), F_j -= g (f64 atomics), F_i and the virial
//           share by a segmented warp reduction over the rows of one centre.  This tail of tile n runs under the
//           layer-3 MMAs of tile n + 1, from rows parked in shared memory (see `tail` in the kernel).
// A CTA runs two independent contexts, each with its own A-operand region, TMEM columns and mbarrier, so
// that one context's MMAs overlap the other's tanh / epilogue work.
#include <cstdio>
#include <cstring>
#include <mutex>
#include <cuda_fp16.h>
#include <cuda_pipeline.h>
#include <type_traits>
#include "common.cuh"
#include "tc_gemm.cuh"
#include "../../include/pimd_noalloc.h"

namespace pimd {

using namespace tc;

namespace etc {
constexpr int E1 = 25, E2 = 50, M1 = 100;
constexpr int H1 = 13;                 // h1 channels per half (26 = 25 + one zero-weight dummy)
constexpr int H2 = 26;                 // h2 channels per half
constexpr int H3 = 52;                 // G channels per half
constexpr int N2 = 64;                 // layer-2 N: half A at columns 0..25, half B at 32..57
constexpr int N3 = 112;                // layer-3 N: half A at columns 0..51, half B at 56..107
constexpr int GROW = 108;              // floats per staged G row (104 + pad: conflict-free 16 B stores)
// weight image of one (t_i, t_j) pair (FP16-split, see namespace eh): [64][32] + [112][64] halfs, hi and lo, + layer 1
constexpr int kImgBytes = 2 * 64 * 64 + 2 * 112 * 128 + 256;     // 37120
constexpr int kImgPad = (kImgBytes + 1023) / 1024 * 1024;
// per-context shared memory
constexpr int kABlk = 128 * 128;                                 // one K-block of 32 for 128 rows: 16 KB
constexpr int oPark = 4 * kABlk;                                 // float4 park[128][3]: a finished row waiting for its tail (bwd)
constexpr int oCen = oPark + 128 * 48;                           // int centre[128]
constexpr int kCtxBytes = (oCen + 128 * 4 + 1023) / 1024 * 1024;     // 72704
constexpr int kSmemBytes = kImgPad + 2 * kCtxBytes + 64 + 1024;  // + barriers + alignment slack = 184320
// The backward kernel keeps its contexts where they were before the weight image shrank (73 KB into the block) and
// the largest carve-out: measured 6 % faster than the compact layout (the forward kernel is 5 % faster compact).
constexpr int kImgPadBwd = 74752;
constexpr int kDtBufBytes = (kImgPadBwd - kImgPad) / 2;          // per context, between the weight image and the contexts
static_assert(kDtBufBytes >= 11 * 1600, "dT buffer");
constexpr int kSmemBytesBwd = kImgPadBwd + 2 * kCtxBytes + 64 + 1024;
constexpr int kThreads = 512;
constexpr int kScanBlock = 1024;       // centres per scan block
static_assert(128 * GROW * 4 <= 4 * kABlk, "G staging must fit the A region");
static_assert(kSmemBytes <= 232448, "shared memory budget");

// Channel permutation.  Half h (0/1), local indices:  h1: i in [0,13) -> padded channel c1 = 13 h + i
// (c1 = 25 is the dummy);  h2: j in [0,26) -> original channel 25 (j / 13) + c1(j % 13);  G: g in [0,52) ->
// original channel 50 (g / 26) + h2 channel of (g % 26).  Returns -1 for a dummy.
__host__ __device__ constexpr int h2_orig(int h, int j) { return (13 * h + j % 13 == 25) ? -1 : 25 * (j / 13) + 13 * h + j % 13; }
__host__ __device__ constexpr int g_orig(int h, int g) { return h2_orig(h, g % 26) < 0 ? -1 : 50 * (g / 26) + h2_orig(h, g % 26); }
// positions inside the operands / accumulators
__host__ __device__ constexpr int n2_of(int h, int j) { return 32 * h + j; }       // layer-2 output column
__host__ __device__ constexpr int n3_of(int h, int g) { return 56 * h + g; }       // layer-3 output column
}  // namespace etc

// ---- FP16-split operands -------------------------------------------------------------------------------------
// a = hi + lo with hi = fp16(a) (11-bit significand, like TF32) and lo = fp16(a - hi): a b ~= hi_a hi_b + lo_a hi_b +
// hi_a lo_b with FP32 accumulation, the same three-pass scheme at kind::f16 -- twice the tensor rate per pass and
// half the shared-memory bytes per operand (the MMAs here are operand-read-bound).  All operands are O(1)
// (tanh outputs plus skips, weights ~ 1/sqrt(fan_in)), far inside FP16's range; small values keep an absolute
// error of 2^-25 through FP16 subnormals, which is what matters inside a dot product.
namespace eh {
constexpr int K2 = 32;                 // halfs: half A at k 0..12, bias at 13, half B at 16..28   (64 B rows, SW64)
constexpr int N2 = 64;
constexpr int K3 = 64;                 // halfs: half A at k 0..25, bias at 26, half B at 32..57   (128 B rows, SW128)
constexpr int N3 = 112;
constexpr int oW2hi = 0, oW2lo = N2 * 64;                        // [64][32] fp16
constexpr int oW3hi = 2 * N2 * 64, oW3lo = oW3hi + N3 * 128;     // [112][64] fp16
constexpr int oW1 = oW3lo + N3 * 128;                            // W1[32], b1[32] plain floats (padded h1 index)
constexpr int kImgBytes = oW1 + 256;                             // 37120
constexpr int kImgPad = (kImgBytes + 1023) / 1024 * 1024;
static_assert(kImgBytes == etc::kImgBytes, "image size");
__host__ __device__ constexpr int k2_of(int h, int i) { return 16 * h + i; }
constexpr int kBias2 = 13;
__host__ __device__ constexpr int k3_of(int h, int j) { return 32 * h + j; }
constexpr int kBias3 = 26;
constexpr int oA1hi = 0, oA1lo = 128 * 64;                       // per-context A1: [128][32] fp16 hi / lo
constexpr int oA2hi = 0, oA2lo = 128 * 128;                      // per-context A2: [128][64] fp16 hi / lo (overlays A1)
}  // namespace eh

// 8 consecutive K elements (one 16-byte chunk) of row `row` -> hi and lo copies of a K-major FP16 operand block
// with `ROWB`-byte rows (64: SWIZZLE_64B, 128: SWIZZLE_128B)
template <int ROWB>
__device__ __forceinline__ void store_chunk_h(uint8_t* blk_hi, uint8_t* blk_lo, int row, int chunk, const float* v) {
    const int sw = (ROWB == 128) ? (row & 7) : ((row >> 1) & 3);
    const int off = row * ROWB + ((chunk ^ sw) << 4);
    uint32_t hi[4], lo[4];
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        const __half2 h = __floats2half2_rn(v[2 * q], v[2 * q + 1]);
        const float2 hf = __half22float2(h);
        const __half2 l = __floats2half2_rn(v[2 * q] - hf.x, v[2 * q + 1] - hf.y);
        hi[q] = *reinterpret_cast<const uint32_t*>(&h);
        lo[q] = *reinterpret_cast<const uint32_t*>(&l);
    }
    *reinterpret_cast<uint4*>(blk_hi + off) = make_uint4(hi[0], hi[1], hi[2], hi[3]);
    *reinterpret_cast<uint4*>(blk_lo + off) = make_uint4(lo[0], lo[1], lo[2], lo[3]);
}

// three-pass FP16 product over `nks` k-steps of 16 (32 bytes of K per step inside a swizzled row)
template <int ROWB>
__device__ __forceinline__ void mma_3x_f16(uint32_t d_tmem, uint32_t a_hi, uint32_t a_lo, uint32_t b_hi, uint32_t b_lo,
                                           uint32_t idesc, int nks) {
    for (int ks = 0; ks < nks; ++ks) {
        const uint64_t dah = make_smem_desc_kmajor(a_hi + ks * 32, ROWB), dal = make_smem_desc_kmajor(a_lo + ks * 32, ROWB);
        const uint64_t dbh = make_smem_desc_kmajor(b_hi + ks * 32, ROWB), dbl = make_smem_desc_kmajor(b_lo + ks * 32, ROWB);
        umma_f16(d_tmem, dah, dbh, idesc, ks == 0 ? 0u : 1u);
        umma_f16(d_tmem, dal, dbh, idesc, 1u);
        umma_f16(d_tmem, dah, dbl, idesc, 1u);
    }
}

// the same by a converged warp (one elected lane issues, tc_gemm.cuh), descriptors built once per product: with
// N = 64 / 112 an MMA lasts 32 / 56 clk and the issue loop, not the tensor pipe, sets the length of the round trip
template <int ROWB>
__device__ __forceinline__ void mma_3x_f16_elect(uint32_t d_tmem, uint32_t a_hi, uint32_t a_lo, uint32_t b_hi, uint32_t b_lo,
                                                 uint32_t idesc, int nks) {
    const uint64_t dah = make_smem_desc_kmajor(a_hi, ROWB), dal = make_smem_desc_kmajor(a_lo, ROWB);
    const uint64_t dbh = make_smem_desc_kmajor(b_hi, ROWB), dbl = make_smem_desc_kmajor(b_lo, ROWB);
#pragma unroll
    for (int ks = 0; ks < 4; ++ks) {
        if (ks >= nks) break;
        const uint64_t o = (uint64_t)(2 * ks);             // 32 bytes of K per step, address field in units of 16 B
        umma_f16_elect(d_tmem, dah + o, dbh + o, idesc, ks == 0 ? 0u : 1u);
        umma_f16_elect(d_tmem, dal + o, dbh + o, idesc, 1u);
        umma_f16_elect(d_tmem, dah + o, dbl + o, idesc, 1u);
    }
}

struct EmbTcArgs {
    int PN, N, ntypes, nsel;
    int seloff[PIMD_MAX_TYPES + 1];
    int type_row0[PIMD_MAX_TYPES + 1];
    int n_of_type[PIMD_MAX_TYPES];
    const int* rowstart;       // [ntypes][PN+1]  exclusive scan over type-sorted centres of ncount[.][tj]
    const int* rowaddr;        // [PN*nsel]       compact row -> slot index (ba*nsel + seloff[tj] + q)
    const int* row_of;         // [PN]            ba -> type-sorted centre row r
    const NeighSlotA* slotA;
    const NeighSlotB* slotB;
    const uint8_t* wimg_h;     // [ntypes*ntypes][eh::kImgBytes]  FP16-split weight images
    const uint8_t* wimg_fwd;   // the same with every weight and bias times 2 log2(e): the forward kernel's tanh takes the
                               // accumulator as the exponent's argument (one multiply per tanh less)
    float* Tm;                 // [PN][100][4]  (zeroed before the forward kernel)
    const float* dTm;
    double* f;                 // [P][N][3]
    double* cpart;             // [PN][9] per-centre virial share (zeroed before the backward kernel)
    float inv_nsel;
    uint32_t nsel_mul, nsel_sh, n_mul, n_sh;   // x / nsel and x / N as a multiply and a shift (FastDiv below)
    int skew_fwd, skew_bwd;    // head start (cycles) of context 0 over context 1 after every weight load
};

// x / d for 0 <= x < 2^31 as one wide multiply and a shift: m = ceil(2^sh / d), sh = 31 + ceil(log2 d) (m <= 2^31 for a
// power of two, < 2^32 otherwise; exact because x (m d - 2^sh) < 2^31 d <= 2^sh).  The kernels divide a slot index by nsel
// and a bead-atom index by N per row and tile.
__host__ __device__ inline void fastdiv_make(uint32_t d, uint32_t* mul, uint32_t* sh) {
    uint32_t l = 0;
    while ((1ull << l) < d) ++l;                        // ceil(log2 d)
    *sh = 31 + l;
    *mul = (uint32_t)((((unsigned long long)1 << (31 + l)) + d - 1) / d);
}
__device__ __forceinline__ int fastdiv(int x, uint32_t mul, uint32_t sh) {
    return (int)(((unsigned long long)(uint32_t)x * mul) >> sh);
}

// -------------------------------------------------------------------------------------------------
// row bookkeeping: exclusive scan of the neighbour counts in type-sorted centre order, slot index per row
// -------------------------------------------------------------------------------------------------
struct SelOff { int v[PIMD_MAX_TYPES + 1]; };

__global__ void __launch_bounds__(256)
row_block_sums_kernel(int PN, int ntypes, const int* __restrict__ cen_idx, const int* __restrict__ ncount,
                      int* __restrict__ bsum) {
    const int tj = blockIdx.y, b = blockIdx.x;
    int s = 0;
    for (int q = threadIdx.x; q < etc::kScanBlock; q += 256) {
        const int r = b * etc::kScanBlock + q;
        if (r < PN) s += ncount[(size_t)cen_idx[r] * ntypes + tj];
    }
    __shared__ int red[8];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        int t = 0;
        for (int w = 0; w < 8; ++w) t += red[w];
        bsum[tj * gridDim.x + b] = t;
    }
}

__global__ void __launch_bounds__(256)
row_scan_fill_kernel(int PN, int ntypes, int nsel, SelOff so, const int* __restrict__ cen_idx,
                     const int* __restrict__ ncount, const int* __restrict__ bsum, int* __restrict__ rowstart,
                     int* __restrict__ rowaddr) {
    const int* seloff = so.v;
    const int tj = blockIdx.y, b = blockIdx.x, nblk = gridDim.x;
    __shared__ int red[8];
    __shared__ int s_off;
    // offset of this block = sum of the block sums before it
    int s = 0;
    for (int q = threadIdx.x; q < b; q += 256) s += bsum[tj * nblk + q];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        int t = 0;
        for (int w = 0; w < 8; ++w) t += red[w];
        s_off = t;
    }
    __syncthreads();
    // each thread owns 4 consecutive centres
    const int r0 = b * etc::kScanBlock + threadIdx.x * 4;
    int c[4], ba[4];
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        const int r = r0 + q;
        ba[q] = (r < PN) ? cen_idx[r] : 0;
        c[q] = (r < PN) ? ncount[(size_t)ba[q] * ntypes + tj] : 0;
    }
    const int mine = c[0] + c[1] + c[2] + c[3];
    int incl = mine;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int t = __shfl_up_sync(0xffffffffu, incl, o);
        if ((threadIdx.x & 31) >= o) incl += t;
    }
    __syncthreads();
    if ((threadIdx.x & 31) == 31) red[threadIdx.x >> 5] = incl;
    __syncthreads();
    int woff = 0;
    for (int w = 0; w < (int)(threadIdx.x >> 5); ++w) woff += red[w];
    int run = s_off + woff + incl - mine;
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        const int r = r0 + q;
        if (r < PN) rowstart[(size_t)tj * (PN + 1) + r] = run;
        run += c[q];
        if (r == PN - 1) rowstart[(size_t)tj * (PN + 1) + PN] = run;
    }
}

// slot index of every compact row: one warp per (neighbour type, centre), coalesced.  Its own launch: inside the scan
// kernel (96 CTAs, each warp 128 centres in sequence) the fill was latency-bound (27 of the kernel's 30 us).
__global__ void __launch_bounds__(256)
row_fill_kernel(int PN, int ntypes, int nsel, SelOff so, const int* __restrict__ cen_idx,
                const int* __restrict__ rowstart, int* __restrict__ rowaddr) {
    const long long w = ((long long)blockIdx.x * 256 + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (w >= (long long)PN * ntypes) return;
    const int tj = (int)(w / PN), r = (int)(w - (long long)tj * PN);
    const int* rs = rowstart + (size_t)tj * (PN + 1);
    const int s0 = rs[r], n = rs[r + 1] - s0;
    const int base = cen_idx[r] * nsel + so.v[tj];
    int* out = rowaddr + (size_t)PN * so.v[tj];
    for (int e = lane; e < n; e += 32) out[s0 + e] = base + e;
}

__device__ __forceinline__ void named_bar_sync(int id, int nthreads) {
    asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}

__device__ __forceinline__ void red_add_v4(float* addr, float a, float b, float c, float d) {
    asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(addr), "f"(a), "f"(b), "f"(c), "f"(d) : "memory");
}

// per-row inputs, prefetched one tile ahead
struct RowIn {
    float dx, dy, dz, s, ds, rinv;
    uint32_t jcode;
    int cen;          // type-sorted centre row r, -1 for a row past the end of the pair
    int ba;           // centre bead-atom k*N + i
};

__device__ __forceinline__ RowIn load_row(const EmbTcArgs& a, int addr) {
    RowIn r;
    if (addr < 0) {
        r.dx = r.dy = r.dz = r.s = r.ds = 0.f; r.rinv = 1.f; r.jcode = 0u; r.cen = -1; r.ba = 0;
        return r;
    }
    const float4 A = __ldg(reinterpret_cast<const float4*>(a.slotA) + addr);
    const float4 B = __ldg(reinterpret_cast<const float4*>(a.slotB) + addr);
    r.dx = A.x; r.dy = A.y; r.dz = A.z; r.s = A.w;
    r.ds = B.x; r.rinv = B.y; r.jcode = __float_as_uint(B.z);
    r.ba = fastdiv(addr, a.nsel_mul, a.nsel_sh);
    r.cen = __ldg(a.row_of + r.ba);
    return r;
}

struct CtxSetup {
    uint8_t* smem;       // 1024-aligned base
    uint8_t* ctx;        // this context's region
    uint64_t* mma_bar;
    uint32_t tmem_base;  // allocation base (all contexts)
};

// common prologue: barriers, TMEM allocation of `ncols` columns; returns after a CTA-wide sync
__device__ __forceinline__ CtxSetup ctx_setup_at(uint8_t* smem_raw, uint32_t ncols, int img_pad, int ctx_bytes, int commits = 1) {
    CtxSetup c;
    // pad to 1024 B by pointer arithmetic on the __shared__ array (a uintptr_t round trip loses the address
    // space and turns every access into a generic LD/ST)
    c.smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
    const int wg = threadIdx.x >> 8;                   // context
    c.ctx = c.smem + img_pad + wg * ctx_bytes;
    uint64_t* bars = reinterpret_cast<uint64_t*>(c.smem + img_pad + 2 * ctx_bytes);
    c.mma_bar = bars + wg;
    uint32_t* tmem_ptr = reinterpret_cast<uint32_t*>(bars + 2);
    if (threadIdx.x == 0) {
        mbar_init(bars, commits);          // tcgen05.commit arrivals per MMA round trip
        mbar_init(bars + 1, commits);
        fence_barrier_init();
    }
    if ((threadIdx.x >> 5) == 0) tmem_alloc(tmem_ptr, ncols);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    c.tmem_base = *tmem_ptr;
    return c;
}

__device__ __forceinline__ CtxSetup ctx_setup(uint8_t* smem_raw, uint32_t ncols) {
    return ctx_setup_at(smem_raw, ncols, etc::kImgPad, etc::kCtxBytes);
}

__device__ __forceinline__ void load_weight_image_n(uint8_t* dst, const uint8_t* src, int nbytes) {
    const float4* s4 = reinterpret_cast<const float4*>(src);
    float4* d4 = reinterpret_cast<float4*>(dst);
    for (int q = threadIdx.x; q < nbytes / 16; q += etc::kThreads) d4[q] = __ldg(s4 + q);
    fence_proxy_async_smem();
}

// -------------------------------------------------------------------------------------------------
// F3: embedding forward + T_i.  One thread per row here (it does the work of both column halves in turn; the
// operand layout and the weight image are those of the two-threads-per-row backward kernel), 128 threads per
// context, so THREE contexts fit the register file (384 threads x 170) and, with FP16 operands, shared memory
// (3 x 57 KB + 37 KB).  The third context gives the tile pipeline -- tanh epilogues, MMA round trips, T
// accumulation -- one more independent stream to overlap: 0.75 -> 0.64 ms against the two-context version.
// -------------------------------------------------------------------------------------------------
namespace f3 {
constexpr int kCtx = 3, kThreads = 128 * kCtx;
constexpr int oRs = 128 * etc::GROW * 4;                           // G staging (overlays the A operands), then R, centres
constexpr int oCen = oRs + 128 * 16;
constexpr int kCtxBytes = (oCen + 128 * 4 + 1023) / 1024 * 1024;   // 58368
constexpr int kSmemBytes = eh::kImgPad + kCtx * kCtxBytes + 64 + 1024;
static_assert(kSmemBytes <= 232448, "shared memory budget (3-context forward)");
}  // namespace f3

__global__ void __launch_bounds__(f3::kThreads, 1)
embed_fwd_tc_kernel(const __grid_constant__ EmbTcArgs a) {
    using namespace etc;
    extern __shared__ uint8_t smem_raw[];
    uint8_t* smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
    const int cx = threadIdx.x >> 7, t = threadIdx.x & 127, lane = threadIdx.x & 31;
    uint8_t* ctx = smem + eh::kImgPad + cx * f3::kCtxBytes;
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem + eh::kImgPad + f3::kCtx * f3::kCtxBytes);
    uint64_t* mma_bar = bars + cx;
    uint32_t* tmem_ptr = reinterpret_cast<uint32_t*>(bars + 4);
    if (threadIdx.x == 0) {
        for (int q = 0; q < f3::kCtx; ++q) mbar_init(bars + q, 1);
        fence_barrier_init();
    }
    if ((threadIdx.x >> 5) == 0) tmem_alloc(tmem_ptr, 512);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_d = *tmem_ptr + cx * 128;
    const int bar_ctx = 1 + cx;
    float4* Rs = reinterpret_cast<float4*>(ctx + f3::oRs);
    int* cen_s = reinterpret_cast<int*>(ctx + f3::oCen);
    float* Gs = reinterpret_cast<float*>(ctx);
    const float* W1s = reinterpret_cast<const float*>(smem + eh::oW1);
    const float* b1s = W1s + 32;
    const uint32_t lanefield = ((uint32_t)((t >> 5) * 32)) << 16;
    const uint32_t actx = smem_u32(ctx), wbase = smem_u32(smem);
    constexpr uint32_t idesc2 = make_idesc_f16(128, eh::N2), idesc3 = make_idesc_f16(128, eh::N3);
    uint32_t phase = 0;
    const int nt = a.ntypes;
    int mo[4];                                             // original channels of staged positions 4 lane .. + 3
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        const int ps = (4 * lane + j) % (2 * H3);
        mo[j] = g_orig(ps / H3, ps % H3);
    }

    int tile_total = 0, sub_lo = 0, sub_hi = 0;
    for (int p = 0; p < nt * nt; ++p) {
        const int ti = p / nt, tj = p - ti * nt;
        const int* rs = a.rowstart + (size_t)tj * (a.PN + 1);
        tile_total += (rs[a.type_row0[ti + 1]] - rs[a.type_row0[ti]] + 127) >> 7;
    }
    const int g_lo = (int)((long long)tile_total * blockIdx.x / gridDim.x);
    const int g_hi = (int)((long long)tile_total * (blockIdx.x + 1) / gridDim.x);
    int tile_off = 0;
    for (int p = 0; p < nt * nt; ++p) {
        const int ti = p / nt, tj = p - ti * nt;
        {
            const int* rs0 = a.rowstart + (size_t)tj * (a.PN + 1);
            const int nt_p = (rs0[a.type_row0[ti + 1]] - rs0[a.type_row0[ti]] + 127) >> 7;
            const int lo = max(g_lo, tile_off) - tile_off, hi = min(g_hi, tile_off + nt_p) - tile_off;
            tile_off += nt_p;
            if (lo >= hi) continue;                        // CTA-uniform: no tile of this pair is mine
            sub_lo = lo; sub_hi = hi;
        }
        __syncthreads();                                   // all contexts are done with the previous weights
        {
            const float4* s4 = reinterpret_cast<const float4*>(a.wimg_fwd + (size_t)p * eh::kImgBytes);    // weights x 2 log2(e)
            float4* d4 = reinterpret_cast<float4*>(smem);
            for (int q = threadIdx.x; q < eh::kImgBytes / 16; q += f3::kThreads) d4[q] = __ldg(s4 + q);
            fence_proxy_async_smem();
        }
        __syncthreads();
        const int* rs = a.rowstart + (size_t)tj * (a.PN + 1);
        const int begin = rs[a.type_row0[ti]], end = rs[a.type_row0[ti + 1]];
        const int tl0 = sub_lo + (sub_hi - sub_lo) * cx / f3::kCtx, tl1 = sub_lo + (sub_hi - sub_lo) * (cx + 1) / f3::kCtx;
        if (tl0 >= tl1) continue;
        if (cx > 0 && a.skew_fwd > 0) {                     // de-phase the contexts
            const long long t0 = clock64();
            while (clock64() - t0 < (long long)a.skew_fwd * cx) __nanosleep(200);
        }
        const int* raddr = a.rowaddr + (size_t)a.PN * a.seloff[tj];
        auto addr_of = [&](int tile) -> int {
            const int g = begin + tile * 128 + t;
            return (tile < tl1 && g < end) ? __ldg(raddr + g) : -1;
        };
        RowIn cur = load_row(a, addr_of(tl0));
        int addr_n1 = addr_of(tl0 + 1);

        for (int tile = tl0; tile < tl1; ++tile) {
            const int addr_n2 = addr_of(tile + 2);
            const RowIn nxt = load_row(a, addr_n1);
            addr_n1 = addr_n2;
            const float s = cur.s;
            {
                const float sr = cur.s * cur.rinv;
                Rs[t] = make_float4(s, sr * cur.dx, sr * cur.dy, sr * cur.dz);
                cen_s[t] = cur.cen;
            }
            // ---- layer 1: both halves' 13 channels -> A1 (64 B rows): K slots 0..15 and 16..31 ----
            float h1[2][H1];
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                float v16[16];
#pragma unroll
                for (int i = 0; i < H1; ++i) h1[h][i] = fmaf(s, W1s[H1 * h + i], b1s[H1 * h + i]);
                tanh_fast_n<H1, true>(h1[h]);
#pragma unroll
                for (int i = 0; i < H1; ++i) v16[i] = h1[h][i];
                v16[13] = h ? 0.f : 1.f; v16[14] = 0.f; v16[15] = 0.f;
                store_chunk_h<64>(ctx + eh::oA1hi, ctx + eh::oA1lo, t, 2 * h, v16);
                store_chunk_h<64>(ctx + eh::oA1hi, ctx + eh::oA1lo, t, 2 * h + 1, v16 + 8);
            }
            fence_proxy_async_smem();
            tc_fence_before();
            named_bar_sync(bar_ctx, 128);
            if (t < 32) {
                tc_fence_after();
                mma_3x_f16_elect<64>(tmem_d, actx + eh::oA1hi, actx + eh::oA1lo, wbase + eh::oW2hi, wbase + eh::oW2lo, idesc2, 2);
                umma_commit_elect(mma_bar);
            }
            mbar_wait(mma_bar, phase);
            phase ^= 1;
            tc_fence_after();
            // ---- epilogue 2: h2 = [h1,h1] + tanh(z2) -> A2 (128 B rows): K slots 0..31 and 32..63 ----
            float h2[2][H2];
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                uint32_t v[H2];
                const uint32_t col = tmem_d + lanefield + 32 * h;
                tmem_ld16(col, v);
                tmem_ld8(col + 16, v + 16);
                tmem_ld2(col + 24, v + 24);
                tmem_ld_wait();
                float v32[32];
#pragma unroll
                for (int j = 0; j < H2; ++j) v32[j] = __uint_as_float(v[j]);
                tanh_fast_n<H2, true>(v32);
#pragma unroll
                for (int j = 0; j < H2; ++j) { h2[h][j] = h1[h][j % H1] + v32[j]; v32[j] = h2[h][j]; }
                v32[26] = h ? 0.f : 1.f;
#pragma unroll
                for (int j = 27; j < 32; ++j) v32[j] = 0.f;
#pragma unroll
                for (int cq = 0; cq < 4; ++cq)
                    store_chunk_h<128>(ctx + eh::oA2hi, ctx + eh::oA2lo, t, 4 * h + cq, v32 + 8 * cq);
            }
            fence_proxy_async_smem();
            tc_fence_before();
            named_bar_sync(bar_ctx, 128);
            if (t < 32) {
                tc_fence_after();
                mma_3x_f16_elect<128>(tmem_d, actx + eh::oA2hi, actx + eh::oA2lo, wbase + eh::oW3hi, wbase + eh::oW3lo, idesc3, 4);
                umma_commit_elect(mma_bar);
            }
            mbar_wait(mma_bar, phase);
            phase ^= 1;
            tc_fence_after();
            // ---- epilogue 3: G = [h2,h2] + tanh(z3) -> smem [row][GROW] (overlays the A operands) ----
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                const uint32_t col = tmem_d + lanefield + 56 * h;
                float* grow = Gs + t * GROW + H3 * h;
#pragma unroll
                for (int pc = 0; pc < 3; ++pc) {
                    uint32_t v[16];
                    tmem_ld16(col + 16 * pc, v);
                    tmem_ld_wait();
#pragma unroll
                    for (int q = 0; q < 4; ++q) {
                        const int g = 16 * pc + 4 * q;
                        float4 gq;
                        tanh_fast4<true>(__uint_as_float(v[4 * q]), __uint_as_float(v[4 * q + 1]), __uint_as_float(v[4 * q + 2]),
                                   __uint_as_float(v[4 * q + 3]), gq.x, gq.y, gq.z, gq.w);
                        gq.x += h2[h][g % H2]; gq.y += h2[h][(g + 1) % H2]; gq.z += h2[h][(g + 2) % H2]; gq.w += h2[h][(g + 3) % H2];
                        *reinterpret_cast<float4*>(grow + g) = gq;
                    }
                }
                uint32_t v[4];
                tmem_ld4(col + 48, v);
                tmem_ld_wait();
                float4 gq;
                tanh_fast4<true>(__uint_as_float(v[0]), __uint_as_float(v[1]), __uint_as_float(v[2]), __uint_as_float(v[3]), gq.x, gq.y, gq.z, gq.w);
                gq.x += h2[h][48 % H2]; gq.y += h2[h][49 % H2]; gq.z += h2[h][50 % H2]; gq.w += h2[h][51 % H2];
                *reinterpret_cast<float4*>(grow + 48) = gq;
            }
            tc_fence_before();
            __syncwarp();                                  // a warp accumulates the 32 rows it has just written
            // ---- T_i += (1/N_sel) sum_rows G (x) R: lane <-> 4 staged G positions (26 lanes) ----
            {
                const int r_lo = t & ~31;
                const int cme = cen_s[r_lo + lane];
                const int cpv = __shfl_up_sync(0xffffffffu, cme, 1);
                const uint32_t bnd = __ballot_sync(0xffffffffu, lane != 0 && cme != cpv);
                if (lane < 26) {
                    const float* gp = Gs + r_lo * GROW + 4 * lane;
                    int r0 = 0;
                    while (r0 < 32) {                       // one iteration per centre segment [r0, r1)
                        const uint32_t rest = (r0 + 1 < 32) ? (bnd >> (r0 + 1)) : 0u;
                        const int r1 = rest ? r0 + __ffs(rest) : 32;
                        const int cn = cen_s[r_lo + r0];
                        if (cn < 0) break;                  // rows past the end of the pair (always at the tail)
                        float acc[16];
#pragma unroll
                        for (int q = 0; q < 16; ++q) acc[q] = 0.f;
                        auto rows = [&](auto NR, int row) {
                            constexpr int nr = decltype(NR)::value;
                            float4 G4[nr], R[nr];
#pragma unroll
                            for (int u = 0; u < nr; ++u) {
                                G4[u] = *reinterpret_cast<const float4*>(gp + (row + u) * GROW);
                                R[u] = Rs[r_lo + row + u];
                            }
#pragma unroll
                            for (int u = 0; u < nr; ++u) {
                                const float gv[4] = {G4[u].x, G4[u].y, G4[u].z, G4[u].w};
#pragma unroll
                                for (int j = 0; j < 4; ++j) {
                                    acc[4 * j] = fmaf(gv[j], R[u].x, acc[4 * j]);
                                    acc[4 * j + 1] = fmaf(gv[j], R[u].y, acc[4 * j + 1]);
                                    acc[4 * j + 2] = fmaf(gv[j], R[u].z, acc[4 * j + 2]);
                                    acc[4 * j + 3] = fmaf(gv[j], R[u].w, acc[4 * j + 3]);
                                }
                            }
                        };
                        int row = r0;
                        for (; row + 4 <= r1; row += 4) rows(std::integral_constant<int, 4>{}, row);
                        if (row + 2 <= r1) { rows(std::integral_constant<int, 2>{}, row); row += 2; }
                        if (row < r1) rows(std::integral_constant<int, 1>{}, row);
#pragma unroll
                        for (int j = 0; j < 4; ++j)
                            if (mo[j] >= 0)
                                red_add_v4(a.Tm + ((size_t)cn * M1 + mo[j]) * 4, acc[4 * j] * a.inv_nsel,
                                           acc[4 * j + 1] * a.inv_nsel, acc[4 * j + 2] * a.inv_nsel, acc[4 * j + 3] * a.inv_nsel);
                        r0 = r1;
                    }
                }
            }
            named_bar_sync(bar_ctx, 128);                  // G / R / centre buffers are free again
            cur = nxt;
        }
    }
    tc_fence_before();
    __syncthreads();
    if ((threadIdx.x >> 5) == 0) tmem_dealloc(*tmem_ptr, 512);
}

// -------------------------------------------------------------------------------------------------
// F5 / F6: embedding backward (forward-mode), pair gradient, force and virial
// -------------------------------------------------------------------------------------------------
constexpr int kDtStage = 11;          // centres whose dT fits the dedicated buffer: 11 x 1600 B (a tile spans 3-6)

__global__ void __launch_bounds__(etc::kThreads, 1)
embed_bwd_tc_kernel(const __grid_constant__ EmbTcArgs a) {
    using namespace etc;
    extern __shared__ uint8_t smem_raw[];
    const CtxSetup cs = ctx_setup_at(smem_raw, 512, kImgPadBwd, kCtxBytes, 2);
    const int cx = threadIdx.x >> 8, half = (threadIdx.x >> 7) & 1, t = threadIdx.x & 127, lane = threadIdx.x & 31;
    const int bar_ctx = 1 + cx;
    uint8_t* ctx = cs.ctx;
    int* cen_s = reinterpret_cast<int*>(ctx + oCen);
    float4* dTs = reinterpret_cast<float4*>(cs.smem + kImgPad + cx * kDtBufBytes);   // dedicated dT buffer (cp.async target)
    float4* park = reinterpret_cast<float4*>(ctx + oPark) + t * 3;       // {A's dR}, {A's ds, slot index, centre, B's ds}, {B's dR}
    const float* W1s = reinterpret_cast<const float*>(cs.smem + eh::oW1) + H1 * half;
    const float* b1s = W1s + 32;
    const uint32_t tmem_v = cs.tmem_base + cx * 256, tmem_g = tmem_v + 128;     // value / derivative accumulators
    const uint32_t lanefield = ((uint32_t)((t >> 5) * 32)) << 16;
    const uint32_t actx = smem_u32(ctx), wbase = smem_u32(cs.smem);
    constexpr uint32_t idesc2 = make_idesc_f16(128, eh::N2), idesc3 = make_idesc_f16(128, eh::N3);
    // FP16-split operands (see namespace eh): region X = ctx + 0 (32 KB): A1v | A1d, later A2v; region Y = ctx + 32 KB: A2d.
    // Value and derivative operands have their own storage, so both layer-3 products go out in one MMA round trip.
    constexpr int oY = 2 * kABlk;
    uint32_t phase = 0;
    const int nt = a.ntypes;

    // The tail of a finished tile -- pair gradient g = dU/dd (R-16), F_j -= g, and the sums over the rows of a centre
    // (F_i, virial share) -- does not run at the end of its tile but one tile later, UNDER THE LAYER-3 MMAs of the next
    // tile, where the context would otherwise only wait.  The contraction parks a row as {partial sums of both halves,
    // slot index, centre}; the geometry is read again from the slot (L2).  Both threads of a row rebuild g; half A sends
    // F_j, half B reduces the twelve sums of a centre (force, virial share).
    auto tail = [&]() {
        const float4 pa = park[0], pm = park[1], pb = park[2];
        const int addr = __float_as_int(pm.y), cen = __float_as_int(pm.z);
        float4 A = make_float4(0.f, 0.f, 0.f, 0.f), B = make_float4(0.f, 1.f, 0.f, 0.f);
        if (addr >= 0) {
            A = __ldg(reinterpret_cast<const float4*>(a.slotA) + addr);
            B = __ldg(reinterpret_cast<const float4*>(a.slotB) + addr);
        }
        const float w = (cen >= 0) ? a.inv_nsel : 0.f;
        const float ds = (pm.x + pm.w) * w, dR0 = (pa.x + pb.x) * w, dR1 = (pa.y + pb.y) * w, dR2 = (pa.z + pb.z) * w,
                    dR3 = (pa.w + pb.w) * w;
        const float s = A.w, dsw = B.x, rinv = B.y, sr = s * rinv;
        const float dot = dR1 * A.x + dR2 * A.y + dR3 * A.z;
        const float radial = (ds + dR0) * dsw + (dsw * rinv - s * rinv * rinv) * dot;
        const float rr = radial * rinv;
        const float gx = fmaf(rr, A.x, sr * dR1), gy = fmaf(rr, A.y, sr * dR2), gz = fmaf(rr, A.z, sr * dR3);
        const int ba = addr >= 0 ? fastdiv(addr, a.nsel_mul, a.nsel_sh) : 0;
        // segmented warp reduction over the rows of one centre (rows of a centre are contiguous)
        auto seg_reduce = [&](auto NQ, float* red) {
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int ko = __shfl_down_sync(0xffffffffu, cen, o);
                const bool take = (lane + o < 32) && (ko == cen);
#pragma unroll
                for (int q = 0; q < decltype(NQ)::value; ++q) {
                    const float vo = __shfl_down_sync(0xffffffffu, red[q], o);
                    if (take) red[q] += vo;
                }
            }
        };
        const int cprev = __shfl_up_sync(0xffffffffu, cen, 1);
        const bool head = cen >= 0 && (lane == 0 || cprev != cen);
        if (half == 0) {
            if (cen >= 0) {
                const int j = (int)(__float_as_uint(B.z) & 0x7fffffu);
                double* fj = a.f + ((size_t)fastdiv(ba, a.n_mul, a.n_sh) * a.N + j) * 3;
                atomicAdd(fj, (double)(-gx)); atomicAdd(fj + 1, (double)(-gy)); atomicAdd(fj + 2, (double)(-gz));
            }
        } else {
            // half B: every sum over the rows of a centre (half A's warps also issue the MMAs and send F_j: measured,
            // 3 + 9 or 6 + 6 sums split between the halves are slower)
            float red[12];
            red[0] = gx; red[1] = gy; red[2] = gz;
            const float dd[3] = {A.x, A.y, A.z}, gg[3] = {gx, gy, gz};
#pragma unroll
            for (int u = 0; u < 3; ++u)
#pragma unroll
                for (int w2 = 0; w2 < 3; ++w2) red[3 + 3 * u + w2] = -dd[u] * gg[w2];
            seg_reduce(std::integral_constant<int, 12>{}, red);
            if (head) {
                double* fi = a.f + (size_t)ba * 3;
                atomicAdd(fi, (double)red[0]); atomicAdd(fi + 1, (double)red[1]); atomicAdd(fi + 2, (double)red[2]);
                double* cp = a.cpart + (size_t)cen * 9;
#pragma unroll
                for (int q = 0; q < 9; ++q) atomicAdd(cp + q, (double)red[3 + q]);
            }
        }
    };

    // Work split (unlike the forward kernel's contiguous shares): every context takes its 1/(2G) slice of EVERY
    // pair, which keeps the two contexts of a CTA on far-apart centres -- measured 3 % faster here, presumably
    // because their force atomics then rarely meet on the same atoms.
    for (int p = 0; p < nt * nt; ++p) {
        const int ti = p / nt, tj = p - ti * nt;
        __syncthreads();
        load_weight_image_n(cs.smem, a.wimg_h + (size_t)p * eh::kImgBytes, eh::kImgBytes);
        __syncthreads();
        const int* rs = a.rowstart + (size_t)tj * (a.PN + 1);
        const int begin = rs[a.type_row0[ti]], end = rs[a.type_row0[ti + 1]];
        const int ntile = (end - begin + 127) >> 7;
        const int C = gridDim.x * 2, c = blockIdx.x * 2 + cx;
        const int tl0 = (int)((long long)ntile * c / C), tl1 = (int)((long long)ntile * (c + 1) / C);
        if (tl0 >= tl1) continue;
        // De-phase the two contexts: started together they stay in lockstep (both in a tanh phase, then both
        // waiting for their MMAs); a head start of about a third of a tile persists and lets one context's
        // CUDA-core phases run under the other's MMA round trips.
        if (cx == 1 && a.skew_bwd > 0) {
            const long long t0 = clock64();
            while (clock64() - t0 < a.skew_bwd) __nanosleep(200);
        }
        const int* raddr = a.rowaddr + (size_t)a.PN * a.seloff[tj];
        auto addr_of = [&](int tile) -> int {
            const int g = begin + tile * 128 + t;
            return (tile < tl1 && g < end) ? __ldg(raddr + g) : -1;
        };
        // software pipeline: slot index two tiles ahead, {d, s} one tile ahead (s feeds layer 1 at once); the
        // rest of the row is loaded at the top of its tile and first used after the second MMA round trip
        auto load_A = [&](int addr) -> float4 {
            return addr >= 0 ? __ldg(reinterpret_cast<const float4*>(a.slotA) + addr) : make_float4(0.f, 0.f, 0.f, 0.f);
        };
        auto load_cen = [&](int addr) -> int { return addr >= 0 ? __ldg(a.row_of + fastdiv(addr, a.nsel_mul, a.nsel_sh)) : -1; };
        int addr_nx = addr_of(tl0), addr_n2 = addr_of(tl0 + 1);
        float4 nxtA = load_A(addr_nx);
        int nxtCen = load_cen(addr_nx);

        for (int tile = tl0; tile < tl1; ++tile) {
            // {d, s} and the centre of my row were fetched one tile ahead; {s', 1/r, j} follow under the layer-3 MMAs
            RowIn cur;
            const int addr_c = addr_nx;
            cur.dx = nxtA.x; cur.dy = nxtA.y; cur.dz = nxtA.z; cur.s = nxtA.w;
            cur.cen = nxtCen;
            addr_nx = addr_n2;
            nxtA = load_A(addr_nx);
            nxtCen = load_cen(addr_nx);
            addr_n2 = addr_of(tile + 2);

            const float s = cur.s;
            // ---- layer 1 and its s-derivative, my 13 channels; A1v = [h1,1,0..], A1d = [h1',0,0..] ----
            float h1[H1], h1p[H1];
#pragma unroll
            for (int i = 0; i < H1; ++i) {
                const float w = W1s[i];
                const float th = tanh_fast(fmaf(s, w, b1s[i]));
                h1[i] = th;
                h1p[i] = (1.f - th * th) * w;
            }
            {
                // A1v = [h1, 1 (bias slot, half A), 0, 0], A1d = [h1', 0, 0, 0]: K slots 16 half .. + 15 (64 B rows)
                float vv[16], vd[16];
#pragma unroll
                for (int i = 0; i < H1; ++i) { vv[i] = h1[i]; vd[i] = h1p[i]; }
                vv[13] = half ? 0.f : 1.f; vv[14] = 0.f; vv[15] = 0.f;
                vd[13] = 0.f; vd[14] = 0.f; vd[15] = 0.f;
#pragma unroll
                for (int cq = 0; cq < 2; ++cq) {
                    store_chunk_h<64>(ctx, ctx + 8192, t, 2 * half + cq, vv + 8 * cq);
                    store_chunk_h<64>(ctx + 16384, ctx + 24576, t, 2 * half + cq, vd + 8 * cq);
                }
            }
            fence_proxy_async_smem();
            tc_fence_before();
            named_bar_sync(bar_ctx, 256);
            // the value and the derivative products are independent: two warps issue them side by side (the barrier counts both commits)
            if ((threadIdx.x & 255) < 64) {
                tc_fence_after();
                if ((threadIdx.x & 255) < 32) mma_3x_f16_elect<64>(tmem_v, actx, actx + 8192, wbase + eh::oW2hi, wbase + eh::oW2lo, idesc2, 2);
                else mma_3x_f16_elect<64>(tmem_g, actx + 16384, actx + 24576, wbase + eh::oW2hi, wbase + eh::oW2lo, idesc2, 2);
                umma_commit_elect(cs.mma_bar);
            }
            mbar_wait(cs.mma_bar, phase);
            phase ^= 1;
            tc_fence_after();
            // ---- epilogue 2: h2, h2' (my 26 columns) -> A2v and A2d ----
            float h2[H2], h2p[H2];
            {
                uint32_t v[H2], d[H2];
                const uint32_t cv = tmem_v + lanefield + 32 * half, cd = tmem_g + lanefield + 32 * half;
                tmem_ld16(cv, v); tmem_ld8(cv + 16, v + 16); tmem_ld2(cv + 24, v + 24);
                tmem_ld16(cd, d); tmem_ld8(cd + 16, d + 16); tmem_ld2(cd + 24, d + 24);
                tmem_ld_wait();
#pragma unroll
                for (int j = 0; j < H2; ++j) {
                    const float th = tanh_fast(__uint_as_float(v[j]));
                    h2[j] = h1[j % H1] + th;
                    h2p[j] = fmaf(1.f - th * th, __uint_as_float(d[j]), h1p[j % H1]);
                }
                // A2v (region X) = [h2, 1 (bias slot, half A), 0..]; A2d (region Y) = [h2', 0..]: K slots 32 half .. + 31
                float vv[32], vd[32];
#pragma unroll
                for (int j = 0; j < H2; ++j) { vv[j] = h2[j]; vd[j] = h2p[j]; }
                vv[26] = half ? 0.f : 1.f; vd[26] = 0.f;
#pragma unroll
                for (int j = 27; j < 32; ++j) { vv[j] = 0.f; vd[j] = 0.f; }
#pragma unroll
                for (int cq = 0; cq < 4; ++cq) {
                    store_chunk_h<128>(ctx, ctx + 16384, t, 4 * half + cq, vv + 8 * cq);
                    store_chunk_h<128>(ctx + oY, ctx + oY + 16384, t, 4 * half + cq, vd + 8 * cq);
                }
            }
            if (half == 0) cen_s[t] = cur.cen;
            fence_proxy_async_smem();
            tc_fence_before();
            named_bar_sync(bar_ctx, 256);
            if ((threadIdx.x & 255) < 64) {
                tc_fence_after();
                if ((threadIdx.x & 255) < 32) mma_3x_f16_elect<128>(tmem_v, actx, actx + 16384, wbase + eh::oW3hi, wbase + eh::oW3lo, idesc3, 4);
                else mma_3x_f16_elect<128>(tmem_g, actx + oY, actx + oY + 16384, wbase + eh::oW3hi, wbase + eh::oW3lo, idesc3, 4);
                umma_commit_elect(cs.mma_bar);
            }
            // ---- while the MMAs run: dT of this tile's centres goes global -> shared by cp.async (no registers in
            // between), and the rest of my row arrives ----
            const int nvalid = min(128, end - (begin + tile * 128));
            const int r_lo = cen_s[0], r_hi = cen_s[nvalid - 1];
            const bool staged = r_hi - r_lo < kDtStage;
            if (staged) {
                const float4* dsrc = reinterpret_cast<const float4*>(a.dTm) + (size_t)r_lo * M1;
                const int nq = (r_hi - r_lo + 1) * M1;
                for (int q = threadIdx.x & 255; q < nq; q += 256) __pipeline_memcpy_async(dTs + q, dsrc + q, 16);
            }
            __pipeline_commit();
            cur.ds = 0.f; cur.rinv = 1.f; cur.jcode = 0u;
            if (addr_c >= 0) {
                const float4 B = __ldg(reinterpret_cast<const float4*>(a.slotB) + addr_c);
                cur.ds = B.x; cur.rinv = B.y; cur.jcode = __float_as_uint(B.z);
            }
            const float sr = cur.s * cur.rinv;
            const float R0 = s, R1 = sr * cur.dx, R2 = sr * cur.dy, R3 = sr * cur.dz;
            if (tile > tl0) tail();                        // the previous tile's rows (parked before two context barriers)
            mbar_wait(cs.mma_bar, phase);
            phase ^= 1;
            tc_fence_after();
            __pipeline_wait_prior(0);
            named_bar_sync(bar_ctx, 256);
            // ---- epilogue 3: contract G, G' (my 52 columns) with dT on the fly.  dT rows come from the staged
            // copy when the whole tile's centres fit (always, unless a centre has < 4 rows of this pair type);
            // the choice is tile-uniform so that the common path uses plain shared-memory loads.  Original
            // channel of my position g: 50 (g / 26) + 25 ((g % 26) / 13) + (g % 26) % 13  + 13 half. ----
            // ds = sum_n (dT_n . R) G'_n = R . E with E_c = sum_n dT_nc G'_n: four FMAs per channel instead of five
            float E0 = 0.f, E1 = 0.f, E2 = 0.f, E3 = 0.f, dR0 = 0.f, dR1 = 0.f, dR2 = 0.f, dR3 = 0.f;
            auto contract = [&](auto dTp) {
                auto piece = [&](auto NV, int g0, const uint32_t* v, const uint32_t* d) {
#pragma unroll
                    for (int q = 0; q < decltype(NV)::value; ++q) {
                        const int g = g0 + q, j = g % H2;
                        const bool dummy = (j % H1 == H1 - 1) && half;        // padded channel 25
                        float4 dT = dTp[50 * (g / H2) + 25 * (j / H1) + j % H1];
                        if (dummy) dT = make_float4(0.f, 0.f, 0.f, 0.f);
                        const float th = tanh_fast(__uint_as_float(v[q]));
                        const float G = h2[j] + th;
                        const float Gp = fmaf(1.f - th * th, __uint_as_float(d[q]), h2p[j]);
                        E0 = fmaf(dT.x, Gp, E0); E1 = fmaf(dT.y, Gp, E1);
                        E2 = fmaf(dT.z, Gp, E2); E3 = fmaf(dT.w, Gp, E3);
                        dR0 = fmaf(dT.x, G, dR0); dR1 = fmaf(dT.y, G, dR1);
                        dR2 = fmaf(dT.z, G, dR2); dR3 = fmaf(dT.w, G, dR3);
                    }
                };
                const uint32_t cv = tmem_v + lanefield + 56 * half, cd = tmem_g + lanefield + 56 * half;
                // eight columns of each accumulator at a time: sixteen cost 16 more registers, which at the 128 this block
                // size allows spilled the row prefetch (a store of a value still in flight: a stall per tile)
                uint32_t v[8], d[8];
#pragma unroll
                for (int cc = 0; cc < 6; ++cc) {
                    tmem_ld8(cv + 8 * cc, v);
                    tmem_ld8(cd + 8 * cc, d);
                    tmem_ld_wait();
                    piece(std::integral_constant<int, 8>{}, 8 * cc, v, d);
                }
                tmem_ld4(cv + 48, v);
                tmem_ld4(cd + 48, d);
                tmem_ld_wait();
                piece(std::integral_constant<int, 4>{}, 48, v, d);
            };
            if (staged) {
                contract(dTs + max(cur.cen - r_lo, 0) * M1 + H1 * half);
            } else {
                contract(reinterpret_cast<const float4*>(a.dTm) + (size_t)max(cur.cen, 0) * M1 + H1 * half);
            }
            tc_fence_before();
            const float ds = fmaf(E0, R0, fmaf(E1, R1, fmaf(E2, R2, E3 * R3)));
            // park the row for its tail (above); the context barriers of the next tile order these stores before the
            // reads, and the reads before the next tile's stores
            if (half == 0) {
                park[0] = make_float4(dR0, dR1, dR2, dR3);
                float* pm = reinterpret_cast<float*>(park + 1);
                pm[0] = ds; pm[1] = __int_as_float(addr_c); pm[2] = __int_as_float(cur.cen);
            } else {
                park[2] = make_float4(dR0, dR1, dR2, dR3);
                reinterpret_cast<float*>(park + 1)[3] = ds;
            }
        }
        // the last tile's tail
        named_bar_sync(bar_ctx, 256);
        tail();
    }
    tc_fence_before();
    __syncthreads();
    if ((threadIdx.x >> 5) == 0) tmem_dealloc(cs.tmem_base, 512);
}

// Xi^(k) = sum of the per-centre virial shares of bead k (one block per bead)
__global__ void __launch_bounds__(256)
virial_reduce_kernel(int ntypes, EmbTcArgs a, double* __restrict__ Xi) {
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
// host side
// -------------------------------------------------------------------------------------------------
size_t emb_tc_image_h_bytes() { return eh::kImgBytes; }

// Builds the shared-memory image of one (t_i, t_j) embedding net from its packed FP64 weights
// (W1[1][25], b1[25], W2[25][50], b2[50], W3[50][100], b3[100], row-major in x out) as FP16-split
// UMMA B operands, with the channel permutation / padding of `etc` applied (dummy channels: zero weights, biases).
void emb_tc_build_image_h(const double* w, uint8_t* img, double scale) {
    using namespace etc;
    memset(img, 0, eh::kImgBytes);
    const double* W1 = w;
    const double* b1 = W1 + E1;
    const double* W2 = b1 + E1;
    const double* b2 = W2 + E1 * E2;
    const double* W3 = b2 + E2;
    const double* b3 = W3 + E2 * M1;
    auto put = [&](int o_hi, int o_lo, int rowb, int n, int k, float v) {
        const int sw = (rowb == 128) ? (n & 7) : ((n >> 1) & 3);
        const int off = n * rowb + (((k >> 3) ^ sw) << 4) + (k & 7) * 2;
        const __half hi = __float2half_rn(v);
        const __half lo = __float2half_rn(v - __half2float(hi));
        memcpy(img + o_hi + off, &hi, 2);
        memcpy(img + o_lo + off, &lo, 2);
    };
    for (int h = 0; h < 2; ++h)
        for (int j = 0; j < H2; ++j) {
            const int n_orig = h2_orig(h, j);
            if (n_orig < 0) continue;
            const int n = n2_of(h, j);
            for (int hh = 0; hh < 2; ++hh)
                for (int i = 0; i < H1; ++i) {
                    const int c1 = H1 * hh + i;
                    if (c1 < E1) put(eh::oW2hi, eh::oW2lo, 64, n, eh::k2_of(hh, i), (float)(scale * W2[c1 * E2 + n_orig]));
                }
            put(eh::oW2hi, eh::oW2lo, 64, n, eh::kBias2, (float)(scale * b2[n_orig]));
        }
    for (int h = 0; h < 2; ++h)
        for (int g = 0; g < H3; ++g) {
            const int n_orig = g_orig(h, g);
            if (n_orig < 0) continue;
            const int n = n3_of(h, g);
            for (int hh = 0; hh < 2; ++hh)
                for (int j = 0; j < H2; ++j) {
                    const int k_orig = h2_orig(hh, j);
                    if (k_orig >= 0) put(eh::oW3hi, eh::oW3lo, 128, n, eh::k3_of(hh, j), (float)(scale * W3[k_orig * M1 + n_orig]));
                }
            put(eh::oW3hi, eh::oW3lo, 128, n, eh::kBias3, (float)(scale * b3[n_orig]));
        }
    float* l1 = reinterpret_cast<float*>(img + eh::oW1);
    for (int k = 0; k < E1; ++k) { l1[k] = (float)(scale * W1[k]); l1[32 + k] = (float)(scale * b1[k]); }
}

static EmbTcArgs make_tc_args(Model& m, const ForceArgs& fa) {
    EmbTcArgs a;
    a.PN = fa.P * fa.N; a.N = fa.N; a.ntypes = fa.ntypes; a.nsel = m.nsel;
    for (int t = 0; t <= PIMD_MAX_TYPES; ++t) { a.seloff[t] = m.seloff[t]; a.type_row0[t] = m.type_row0[t]; }
    for (int t = 0; t < PIMD_MAX_TYPES; ++t) a.n_of_type[t] = (t < fa.ntypes) ? m.n_of_type[t] : 0;
    a.rowstart = m.rowstart; a.rowaddr = m.rowaddr; a.row_of = m.row_of;
    a.slotA = m.slotA; a.slotB = m.slotB; a.wimg_h = m.emb_img_h; a.wimg_fwd = m.emb_img_h_fwd;
    a.Tm = m.Tm; a.dTm = m.dTm; a.f = fa.f; a.cpart = m.cpart;
    a.inv_nsel = 1.0f / (float)m.nsel;
    fastdiv_make((uint32_t)m.nsel, &a.nsel_mul, &a.nsel_sh);
    fastdiv_make((uint32_t)fa.N, &a.n_mul, &a.n_sh);
    // measured on B200: plateaus at 4-6 k cycles (forward, -20 %) and 5-13 k cycles (backward, -8 %)
    a.skew_fwd = 5000;
    a.skew_bwd = 9000;
    return a;
}

// after neighbor_build: compact-row bookkeeping for the tensor-core embedding kernels
int emb_tc_row_index(Model& m, const ForceArgs& fa, cudaStream_t s) {
    const int PN = fa.P * fa.N;
    const int nblk = (PN + etc::kScanBlock - 1) / etc::kScanBlock;
    SelOff so;
    for (int t = 0; t <= PIMD_MAX_TYPES; ++t) so.v[t] = m.seloff[t];
    dim3 grid(nblk, fa.ntypes);
    row_block_sums_kernel<<<grid, 256, 0, s>>>(PN, fa.ntypes, m.cen_idx, m.ncount, m.row_bsum);
    row_scan_fill_kernel<<<grid, 256, 0, s>>>(PN, fa.ntypes, m.nsel, so, m.cen_idx, m.ncount, m.row_bsum, m.rowstart,
                                              m.rowaddr);
    const long long nw = (long long)PN * fa.ntypes;
    row_fill_kernel<<<(unsigned)((nw * 32 + 255) / 256), 256, 0, s>>>(PN, fa.ntypes, m.nsel, so, m.cen_idx, m.rowstart,
                                                                      m.rowaddr);
    return 3;
}

int embedding_forward_tc(Model& m, const ForceArgs& fa, int n_sms, cudaStream_t s) {
    EmbTcArgs a = make_tc_args(m, fa);
    ensure_dyn_smem(embed_fwd_tc_kernel, f3::kSmemBytes);
    cudaMemsetAsync(m.Tm, 0, sizeof(float) * (size_t)a.PN * etc::M1 * 4, s);
    embed_fwd_tc_kernel<<<n_sms, f3::kThreads, f3::kSmemBytes, s>>>(a);
    return 1;
}

int embedding_backward_tc(Model& m, const ForceArgs& fa, int n_sms, cudaStream_t s) {
    EmbTcArgs a = make_tc_args(m, fa);
    ensure_dyn_smem(embed_bwd_tc_kernel, etc::kSmemBytesBwd);
    cudaMemsetAsync(m.cpart, 0, sizeof(double) * (size_t)a.PN * 9, s);
    embed_bwd_tc_kernel<<<n_sms, etc::kThreads, etc::kSmemBytesBwd, s>>>(a);
    virial_reduce_kernel<<<fa.P, 256, 0, s>>>(fa.ntypes, a, fa.Xi);
    return 2;
}

// -------------------------------------------------------------------------------------------------
// No-allocation entry point (include/pimd_noalloc.h): the row-index scan of emb_tc_row_index -- the exclusive scan
// of the neighbour counts in type-sorted centre order that places every (t_i, t_j) row tile of F3 / F5 -- with its
// scratch (the per-block sums the two scan kernels hand over) in a file-scope device array instead of the context's
// arena.  For callers that may not allocate: code under CUDA graph capture, serving loops, harnesses that forbid
// cudaMalloc.  The kernels are the ones pimd_step launches; only the scratch pointer differs.
// -------------------------------------------------------------------------------------------------
namespace noalloc {
constexpr int kMaxScanBlocks = 4096;                                   // x 1024 centres = PIMD_NOALLOC_MAX_CENTRES
constexpr int kMaxCentres = kMaxScanBlocks * etc::kScanBlock;
constexpr int kMaxDevices = 64;
static_assert(kMaxCentres == PIMD_NOALLOC_MAX_CENTRES, "include/pimd_noalloc.h states the limit");
// 64 KB per GPU that loads the library, held until the process exits.  Every block sum a call reads has been written
// by the first kernel of the same call, so nothing has to start at zero; the array keeps the last call's sums.
static __device__ __align__(256) int g_row_bsum[PIMD_MAX_TYPES * kMaxScanBlocks];
// In host code `g_row_bsum` is a host-side stand-in for the symbol, not a device address: the address a kernel can
// use comes from cudaGetSymbolAddress, asked once per device with that device current.
static int* g_row_bsum_dev[kMaxDevices];
static std::mutex g_mu;
static thread_local char g_err[256] = "";

static int fail(int code, const char* what, const char* detail = "") {
    snprintf(g_err, sizeof g_err, "%s%s", what, detail);
    return code;
}

static int scratch_for_current_device(int** out) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return fail(PIMD_ECUDA, "cudaGetDevice: ", cudaGetErrorString(e));
    if (dev < 0 || dev >= kMaxDevices) return fail(PIMD_EINVAL, "device ordinal beyond the 64 this entry point keeps scratch addresses for");
    std::lock_guard<std::mutex> lk(g_mu);
    if (!g_row_bsum_dev[dev]) {
        int* p = nullptr;
        e = cudaGetSymbolAddress(reinterpret_cast<void**>(&p), g_row_bsum);
        if (e != cudaSuccess || !p) return fail(PIMD_ECUDA, "cudaGetSymbolAddress(g_row_bsum): ", cudaGetErrorString(e));
        g_row_bsum_dev[dev] = p;
    }
    *out = g_row_bsum_dev[dev];
    return PIMD_OK;
}
}  // namespace noalloc

}  // namespace pimd

extern "C" {

int pimd_noalloc_setup(void) {
    int* p = nullptr;
    return pimd::noalloc::scratch_for_current_device(&p);
}

const char* pimd_noalloc_last_error(void) { return pimd::noalloc::g_err; }

int pimd_row_scan_noalloc_dev(int n_centres, int n_types, const int32_t* cen_idx_dev, const int32_t* ncount_dev,
                              int32_t* rowstart_dev, void* cuda_stream) {
    using namespace pimd;
    if (!cen_idx_dev || !ncount_dev || !rowstart_dev) return noalloc::fail(PIMD_EINVAL, "null device pointer");
    if (n_centres <= 0) return noalloc::fail(PIMD_EINVAL, "n_centres must be positive");
    if (n_types <= 0 || n_types > PIMD_MAX_TYPES) return noalloc::fail(PIMD_EINVAL, "n_types outside 1..PIMD_MAX_TYPES (4)");
    if (n_centres > noalloc::kMaxCentres)
        return noalloc::fail(PIMD_EINVAL, "n_centres beyond PIMD_NOALLOC_MAX_CENTRES (4194304): the static scratch holds "
                                          "4096 block sums per neighbour type; use the context path (pimd_step) for larger systems");
    int* bsum = nullptr;
    const int rc = noalloc::scratch_for_current_device(&bsum);
    if (rc) return rc;
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    const int nblk = (n_centres + etc::kScanBlock - 1) / etc::kScanBlock;
    SelOff so;
    for (int t = 0; t <= PIMD_MAX_TYPES; ++t) so.v[t] = 0;             // the scan kernels do not read it
    dim3 grid(nblk, n_types);
    row_block_sums_kernel<<<grid, 256, 0, s>>>(n_centres, n_types, cen_idx_dev, ncount_dev, bsum);
    row_scan_fill_kernel<<<grid, 256, 0, s>>>(n_centres, n_types, 0, so, cen_idx_dev, ncount_dev, bsum, rowstart_dev, nullptr);
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return noalloc::fail(PIMD_ECUDA, "row scan launch: ", cudaGetErrorString(e));
    return PIMD_OK;
}

}  // extern "C"
