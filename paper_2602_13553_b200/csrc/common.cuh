// common.cuh -- internal declarations shared by the translation units of libpimd_b200.
// Product code (CUDA, sm_100a).  Shares nothing with oracle/.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>
#include <stddef.h>
#include <string>
#include <vector>
#include "../../include/pimd.h"
#include "../../include/pimd_debug.h"

namespace pimd {

// Physical constants: PAPER.md:L458 prints h and mvv2e; k_B is DESIGN R-9.
constexpr double kHPlanck = 4.135667403e-3;                       // eV ps
constexpr double kHbar    = kHPlanck / (2.0 * 3.14159265358979323846);
constexpr double kMvv2e   = 1.0364269e-4;                         // eV / ((g/mol)(A/ps)^2)
constexpr double kKB      = 8.617333262e-5;                       // eV / K

constexpr int kMaxBeads = 64;
constexpr int kEstCap   = 4096;     // estimator history slots per pimd_step call
constexpr int kEstWidth = 16;       // K_ring, S_ring, sum x.f - x~0.f~0, U_sum; barostat record at kEstBaro
constexpr int kEstBaro  = 4;        // v_W[3], L[3], diag P_CV[3] (eV/A^3), sum_k Tr Xi: the cell at the END of the step

// integrator launch flags
enum : int { I_BCLOSE = 1, I_EST = 2, I_START = 4, I_OBABO = 8, I_COMACC = 16, I_COMSUB = 32, I_CART = 64,
              I_NOISE_PER_MODE = 128 /* timing only: one Philox draw per mode (DESIGN R-10 A/B) */ };

// Per-mode constants of the A and O steps (DESIGN R-3, R-5), kernel parameter.
struct ModeConsts {
    double cosA[kMaxBeads];      // cos(omega_k dt/2)
    double sinA_w[kMaxBeads];    // sin(omega_k dt/2)/omega_k   (k = 0: dt/2)
    double msinA_w[kMaxBeads];   // -omega_k sin(omega_k dt/2)
    double c1[kMaxBeads];        // exp(-dt gamma_k)
    double c2[kMaxBeads];        // sqrt(1 - c1^2)
    double om2[kMaxBeads];       // omega_k^2
};

struct IntegratorArgs {
    int      N;                  // atoms
    int      n_dof;              // 3N
    int      flags;
    int      thermostat;         // 0 = NVE (O step skipped)
    double   half_dt_mvv;        // (dt/2)/mvv2e : multiply by f~/m to get the B kick
    double   PkT_mvv;            // P k_B T / mvv2e : sigma_i^2 = this / m_i
    uint32_t seed_lo, seed_hi, step_lo, step_hi;   // step = the step this launch OPENS
    uint32_t cstep_lo, cstep_hi;                   // OBABO: the step this launch CLOSES, bit 31 of word 1 set (second O)
    const double* x_in;  const double* vt_in;  const double* f;
    double*  x_out;      double* vt_out;
    const double* mass;          // [N] per atom
    const double* U;             // [P] bead energies (for the U_sum slot), may be null
    double*  est;                // [kEstWidth] accumulators of this step's slot, may be null
    double*  com;                // [3] fixcom: sum_i m_i v~_0,i per component (I_COMACC adds, I_COMSUB reads)
    double   inv_mtot;           // 1 / sum_i m_i
    double   wP2;                // omega_n^2 (Cartesian method: ring-spring force)
    const double* baro;          // barostat state (BaroSlot layout) or null: centroid drift by Eq. E4/E5
    // Graph replay (api.cu): when ctl != null the step counter and the estimator slot are NOT launch arguments but are
    // read from the device -- ctl[0] = the step this launch opens (advanced once per force evaluation by
    // wrap_bin_kernel), ctl[1] = the absolute step whose estimators go to history slot 0 -- so that one captured
    // launch sequence serves every step of a pimd_step call.
    int      prefetch_ahead;     // blocks ahead whose inputs this block prefetches into L2 (0 = none)
    const long long* ctl;
    double*  est_base;           // estimator history [kEstCap][kEstWidth]
    double*  est_scratch;        // slot for steps outside the recorded window
};

// Barostat state on the device (Appendix E; DESIGN R-20..R-25), doubles:
enum BaroSlot { BS_VW = 0 /* [3], equal in isotropic mode */, BS_LX = 3, BS_LY = 4, BS_LZ = 5,
                BS_PCV = 6 /* [3] diagonal of Eq. E3, eV/A^3 */, BS_TRXI = 9,
                BS_FAC = 10 /* [3][6]: e^{h v}, sinh(h v)/v, e^{-h v} of the first and the second half drift */,
                BS_WIDTH = 32 };
struct BaroArgs {
    int P, N, n_dof;
    int close, start, thermostat;
    int aniso;                   // one cell velocity per Cartesian component (Eq. E2-E3) instead of one (E1)
    int obabo;                   // OBABO: O(dt/2) twice around the kicks, one drift of dt (R-24)
    double h;                    // dt/2
    double W, p_ext;             // barostat mass (eV ps^2), target pressure (eV/A^3)
    double nkT;                  // n k_B T
    double c1, c2sig;            // E7 over the O step's length (dt, OBABO dt/2): exp(-l gamma0), sqrt(1-c1^2) sqrt(n k_B T / W)
    double c2;                   // sqrt(1-c1^2): the centroid mode's own O coefficients are the same c1, c2 (tau_0)
    double half_dt_mvv, PkT_mvv; // as IntegratorArgs
    uint32_t seed_lo, seed_hi, step_lo, step_hi;
    uint32_t cstep_lo, cstep_hi; // OBABO: the step this launch closes, bit 31 of word 1 set
    const double* x; const double* vt; const double* f; const double* mass; const double* Xi;
    double* state;               // [BS_WIDTH]
    double* est_slot;            // estimator slot of the step this launch closes (barostat record at kEstBaro), or null
    double* partial;             // [blocks][3][kBaroSums] block partials of the sums, per Cartesian component
};
constexpr int kBaroSums = 7;     // S_kin, S_cv, S_fv, S_ff, and (OBABO) S_kin after kick + closing O, S_kin and S_fv after the opening O
int launch_barostat(const BaroArgs& a, cudaStream_t s);

// Opt-in to more than 48 KB of dynamic shared memory, once per (kernel, device): the attribute belongs to the
// kernel's image on ONE device, so a process-wide "done" flag would leave a second device without it.
void ensure_dyn_smem_impl(const void* kernel, int bytes);
template <typename K>
inline void ensure_dyn_smem(K kernel, int bytes) { ensure_dyn_smem_impl(reinterpret_cast<const void*>(kernel), bytes); }
size_t barostat_state_doubles(int n_dof);    // BS_WIDTH + the partials

int launch_integrator(int P, const IntegratorArgs& a, const ModeConsts& mc, cudaStream_t s);
int launch_integrator4(int P, const IntegratorArgs& a, const ModeConsts& mc, cudaStream_t s);   // 0: not taken
int launch_cart_convert(int P, int N, const double* in, const double* mass, double* out, int forward, cudaStream_t s);
int launch_to_nm_velocity(int P, int N, const double* p_cart, const double* mass, double* vt, cudaStream_t s);
int launch_from_nm_momenta(int P, int N, const double* vt, const double* mass, double* p_cart, cudaStream_t s);
int launch_harmonic(int P, int N, double k_spring, const double* x, double* f, double* U, double* Xi,
                     double* Eatom, cudaStream_t s);
int launch_debug_noise(uint64_t seed, uint64_t step, int n, const int32_t* idx_dev, uint32_t* words_dev,
                        double* eta_dev, cudaStream_t s);

// ---------------------------------------------------------------------------------------------
// se_e2_a model on the device
// ---------------------------------------------------------------------------------------------
struct NeighSlotA { float dx, dy, dz, s; };          // environment row pieces (FP32 from FP64)
struct NeighSlotB { float ds, rinv; uint32_t jcode; float pad; };   // jcode = j | shiftcode << 23

struct Model {
    bool     set = false;
    static constexpr int kChainStreams = 8; // at most; tile ranges of the fitting chain run on chain_streams streams (fitting_tc.cu)
    int      chain_streams = 4;             // measured at configs[2]: 1: 0.613, 2: 0.542, 3: 0.543, 4: 0.532, 6: 0.550, 8: 0.549 ms
    cudaStream_t aux_stream[kChainStreams - 1] = {};
    cudaEvent_t  ev_fork = nullptr, ev_join[kChainStreams - 1] = {};
    pimd_model_desc d;
    int      nsel = 0;
    int      seloff[PIMD_MAX_TYPES + 1];
    int      M1 = 0, M2 = 0, E1 = 0, E2 = 0, NF = 0, ND = 0;   // 100,16,25,50,240,1600
    // geometry of the cell grid
    int      ncell[3]; int ncells = 0; int R[3];
    // device buffers
    float*   emb_w = nullptr;          // [ntypes*ntypes][emb_stride] packed for the kernels
    int      emb_stride = 0;
    float*   fit_w[PIMD_MAX_TYPES][4];     // W[in][out] row-major
    float*   fit_wT[PIMD_MAX_TYPES][4];    // W^T: [out][in] row-major (backward GEMM operand)
    float*   fit_b[PIMD_MAX_TYPES][4];
    int*     cen_idx = nullptr;        // [PN] sorted row -> k*N+i  (order [type][bead][atom of type])
    int*     row_of = nullptr;         // [PN] inverse
    int      type_row0[PIMD_MAX_TYPES + 1];   // first sorted row of each centre type
    int      n_of_type[PIMD_MAX_TYPES];
    int*     cell_count = nullptr;     // [P][ncells+1]
    int*     cell_start = nullptr;     // [P][ncells+1]
    int*     cell_fill = nullptr;      // [P][ncells]
    int*     cell_id = nullptr;        // [PN]
    int*     cell_tmp = nullptr;       // [PN] unsorted members
    double*  wtmp = nullptr;           // [PN][3] wrapped coordinates
    double4* wsorted = nullptr;        // [PN] cell-ordered {w, idx|type}
    int*     ncount = nullptr;         // [PN][ntypes]
    NeighSlotA* slotA = nullptr;       // [PN][nsel]
    NeighSlotB* slotB = nullptr;
    int*     overflow = nullptr;       // device flag
    float*   Tm = nullptr;             // [PN rows][M1][4]
    float*   dTm = nullptr;
    float*   D = nullptr;              // [rows][ND]
    float*   dD = nullptr;
    float*   Y1 = nullptr, *T2 = nullptr, *Y2 = nullptr, *T3 = nullptr, *Y3 = nullptr;   // [rows][NF]
    float*   G1 = nullptr, *G2 = nullptr;   // backward scratch [rows][NF]
    // tensor-core path (fitting_tc.cu): TMA tensor maps per centre type
    bool     use_tc = true;
    bool     tc_ready = false;
    CUtensorMap mapA_D[PIMD_MAX_TYPES], mapA_Y1[PIMD_MAX_TYPES], mapA_Y2[PIMD_MAX_TYPES], mapA_G1[PIMD_MAX_TYPES],
                mapA_T3[PIMD_MAX_TYPES], mapA_G2[PIMD_MAX_TYPES];
    CUtensorMap mapB_fwd_hi[PIMD_MAX_TYPES][3], mapB_fwd_lo[PIMD_MAX_TYPES][3];   // W_l^T  [out][in], TF32 hi / lo
    CUtensorMap mapB_bwd_hi[PIMD_MAX_TYPES][3], mapB_bwd_lo[PIMD_MAX_TYPES][3];   // W_l    [in][out]
    float*   fit_w_hi[PIMD_MAX_TYPES][3], *fit_w_lo[PIMD_MAX_TYPES][3];           // pre-split weights (layers 1..3)
    float*   fit_wT_hi[PIMD_MAX_TYPES][3], *fit_wT_lo[PIMD_MAX_TYPES][3];
    // FP16-split images of the first fitting layer (x kW1Scale) for the two K = 1600 / N = 1600 kernels
    uint8_t* l1_wimg[PIMD_MAX_TYPES];    // W1^T: one image per K block of 32 (l1_desc_kernel's B operand, one bulk copy per stage)
    uint8_t* dd_wimg[PIMD_MAX_TYPES];    // W1: one image per (chunk of 160 rows, K block of 32) (dd_dt_kernel's B operand)
    CUtensorMap mapAh_G1[PIMD_MAX_TYPES], mapAh_G2[PIMD_MAX_TYPES];           // da1 as FP16 hi / lo (x bwd_scale)
    uint16_t* da1_h_hi = nullptr, *da1_h_lo = nullptr;   // [rows][240] halfs, carved out of D
    float    bwd_scale = 1.f;          // power of two that brings the backward activations to O(1..16)
    // fused middle of the fitting chain (fitting_mid.cu): operand images handed from kernel to kernel (per 128-row
    // tile: y1 from l1_desc_kernel, bwd_scale * da1 to dd_dt_kernel), tile-private scratch, weight images
    bool     mid_ready = false;
    uint8_t* y1_img = nullptr, *da1_img = nullptr;      // [tiles] x mid_image_bytes()
    float4*  mid_t2 = nullptr, *mid_g1 = nullptr;       // [tiles] x mid_scratch_bytes()
    uint8_t* mid_wimg[PIMD_MAX_TYPES];   // [phase 4][k-step 15][hi | lo][240 rows x 32 B, SWIZZLE_32B order]: one bulk copy per k-step
    // tensor-core embedding path (embedding_tc.cu)
    bool     use_tc_emb = true;
    bool     tc_emb_ready = false;
    uint8_t* emb_img_h = nullptr;      // [ntypes*ntypes][emb_tc_image_h_bytes()] FP16-split shared-memory images of the nets
    uint8_t* emb_img_h_fwd = nullptr;  // the same, weights x 2 log2(e) (forward kernel)
    int*     rowstart = nullptr;       // [ntypes][PN+1] exclusive scan of ncount[.][tj] over type-sorted centres
    int*     rowaddr = nullptr;        // [PN*nsel] compact row -> slot index
    int*     row_bsum = nullptr;       // [ntypes][ceil(PN/1024)] scan block sums
    double*  cpart = nullptr;          // [PN][9] per-centre virial share
    // compressed (tabulated) embedding, SURVEY 8(f) NEXT-3 (compress_tc.cu)
    bool     compressed = false;
    uint32_t* cmp_img_fw = nullptr;    // tensor-memory images of the tables: forward A operand per centre type
    uint32_t* cmp_img_bw = nullptr;    // backward A operand (four M tiles) per centre type
    uint32_t* cmp_need = nullptr;      // [PN / 8 + ntypes + 1] per tile: which upper M tiles the backward kernel needs
};

struct ForceArgs {
    int P, N, ntypes;
    double box[3];
    const double* box_dev; // barostat: the cell lives on the device ([3] doubles) and box[] is ignored; else null
    const double* x;      // [P][N][3]
    const int* types;     // [N]
    double* f;            // [P][N][3]
    double* U;            // [P]
    double* Xi;           // [P][9]
    double* Eatom;        // [P][N]
    long long* ctl;       // device step counter (graph replay) or null
};

int neighbor_build(Model& m, const ForceArgs& a, cudaStream_t s);
int embedding_forward(Model& m, const ForceArgs& a, int n_sms, cudaStream_t s);
int fitting_forward_backward(Model& m, const ForceArgs& a, cudaStream_t s);
int embedding_backward(Model& m, const ForceArgs& a, int n_sms, cudaStream_t s);
size_t embedding_smem_bytes(const Model& m, int ntypes);
bool tc_setup_maps(Model& m, int ntypes);
void tc_split_weights(size_t n, const float* w, float* hi, float* lo, cudaStream_t s);
void tc_split_weights_h(size_t n, const float* w, float scale, uint16_t* hi, uint16_t* lo, cudaStream_t s);
int fitting_chain_tc(Model& m, const ForceArgs& a, cudaStream_t s);
bool tc_make_map_h(CUtensorMap* map, const uint16_t* base, uint64_t rows, uint64_t cols, uint64_t ld, uint32_t box_rows);
bool fitting_mid_setup(Model& m, int ntypes);
size_t kmajor_image_bytes(int nrows, int kc);
void kmajor_image(const float* Bt, int N, int K, int n0, int nr, int k0, int kc, float scale, uint8_t* img);
size_t mid_wimg_bytes();
size_t mid_image_bytes();
size_t mid_scratch_bytes();
size_t l1_wimg_bytes(int ND);
void l1_build_wimg(const float* WT, int ND, uint8_t* img);
size_t dd_wimg_bytes(int ND);
void dd_build_wimg(const float* W, int ND, uint8_t* img);
void mid_build_wimg(const float* W2, const float* W2T, const float* W3, const float* W3T, uint8_t* img);
void fitting_mid_launch(Model& m, const ForceArgs& a, int tile_off, int ntiles, cudaStream_t s);
size_t emb_tc_image_h_bytes();
void emb_tc_build_image_h(const double* w_pair, uint8_t* img, double scale = 1.0);
int emb_tc_row_index(Model& m, const ForceArgs& a, cudaStream_t s);
int embedding_forward_tc(Model& m, const ForceArgs& a, int n_sms, cudaStream_t s);
int embedding_backward_tc(Model& m, const ForceArgs& a, int n_sms, cudaStream_t s);
int debug_tc_gemm(int M, int N, int K, const float* A_dev, const float* Bt_dev, float* C_dev, cudaStream_t s);
size_t cmp_image_words_fw(int ntypes);
size_t cmp_image_words_bw(int ntypes);
void cmp_build_images(const double* w_emb, int ntypes, uint32_t* img_fw, uint32_t* img_bw);
int compressed_forward(Model& m, const ForceArgs& a, int n_sms, cudaStream_t s);
int compressed_backward(Model& m, const ForceArgs& a, int n_sms, cudaStream_t s);

}  // namespace pimd
