// api.cu -- the C ABI of include/pimd.h: context, device-memory arena, model upload, the step driver.
// Host logic only; every step of the hot path runs in the kernels of integrator.cu, neighbor.cu,
// embedding.cu and fitting.cu.  No CPU fallback: CUDA errors are returned as PIMD_ECUDA.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include "common.cuh"

#include <mutex>
#include <unordered_map>

using namespace pimd;

namespace pimd {
void ensure_dyn_smem_impl(const void* kernel, int bytes) {
    static std::mutex mu;
    static std::unordered_map<const void*, unsigned long long> done;      // kernel -> bit per device ordinal
    int dev = 0;
    cudaGetDevice(&dev);
    std::lock_guard<std::mutex> lock(mu);
    unsigned long long& mask = done[kernel];
    if (dev < 64 && ((mask >> dev) & 1ull)) return;
    cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
    if (dev < 64) mask |= 1ull << dev;
}
}  // namespace pimd

struct pimd_ctx {
    int N = 0, P = 0, ntypes = 0;
    double box[3] = {0, 0, 0}, T = 0, dt = 0, gamma0 = 0;
    uint64_t seed = 0;
    int64_t step = 0;
    int64_t launches = 0;
    int integrator = PIMD_BAOAB;
    bool fixcom = false;
    int method = PIMD_NMPIMD;
    double* com = nullptr;        // [3] device: centroid COM momentum (fixcom)
    double inv_mtot = 0;
    bool baro = false;            // BZP barostat (Appendix E)
    bool baro_aniso = false;      // Eq. E2-E3: one cell velocity per component
    double p_ext = 0, baro_W = 0; // eV/A^3, eV ps^2
    double* baro_state = nullptr; // [BS_WIDTH] device
    std::vector<int32_t> types;
    std::vector<double> masses;
    std::string err;
    int n_sms = 148;

    // memory arena
    char* arena = nullptr; size_t arena_bytes = 0, arena_used = 0;    // caller-lent workspace (bump allocator)
    std::vector<void*> owned;                                          // cudaMalloc'ed buffers otherwise
    cudaStream_t stream = nullptr;

    // state
    bool have_state = false;
    int model_kind = 0;           // 0 none, 1 harmonic, 2 se_e2_a
    double k_spring = 0;
    double *x = nullptr, *vt = nullptr, *f = nullptr, *mass_atom = nullptr;
    double *scratch_a = nullptr, *scratch_b = nullptr;     // [P][N][3] each: momenta staging / timing outputs; inside
                                                           // pimd_step: the entry snapshot of x and v~ (rollback)
    double *snap_f = nullptr, *snap_small = nullptr;       // entry snapshot of f [P][N][3]; of U, Xi, barostat state
    int64_t evals_launched = 0;                            // force evaluations issued so far (mirrors model.overflow[2])
    // one captured launch sequence per step: {integrator, force evaluation} as a CUDA graph that is
    // replayed for the inner steps of a pimd_step call; step counter and estimator slot live on the device (ctl_dev)
    long long* ctl_dev = nullptr;                          // {step the next integrator launch opens, step of history slot 0}
    cudaGraphExec_t step_graph = nullptr;
    cudaStream_t graph_stream = nullptr;                   // the replayed loop runs here: the caller's stream may be the
    cudaEvent_t graph_ev = nullptr;                        // legacy default stream, which cannot be captured
    uint64_t graph_key = 0;
    int64_t graph_launches = 0;                            // kernels inside one replay
    bool graph_failed = false;
    int* types_d = nullptr;
    double *U = nullptr, *Xi = nullptr, *Eatom = nullptr;
    double* est = nullptr;        // [kEstCap + 2][kEstWidth]; slot kEstCap = "current", kEstCap+1 = scratch
    int est_hist_n = 0;           // valid history slots of the last pimd_step call
    int64_t est_hist_first_step = 0;
    ModeConsts mc;
    Model model;
    std::vector<double> emb_w_host;   // embedding weights as passed to pimd_set_model (the tables are built from them)

    // profiling
    bool profiling = false;
    cudaEvent_t ev[8] = {};
    double phase_ms[6] = {0, 0, 0, 0, 0, 0};
    int64_t phase_steps = 0;
};

namespace {

int fail(pimd_ctx* c, int code, const std::string& msg) {
    if (c) c->err = msg;
    return code;
}
#define CK(call)                                                                                   \
    do {                                                                                           \
        cudaError_t e__ = (call);                                                                  \
        if (e__ != cudaSuccess)                                                                    \
            return fail(ctx, PIMD_ECUDA, std::string(#call) + ": " + cudaGetErrorString(e__));   \
    } while (0)

size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

template <typename T>
int arena_alloc(pimd_ctx* ctx, T** out, size_t count) {
    const size_t bytes = align_up(count * sizeof(T), 256);
    if (!ctx->arena) {
        void* p = nullptr;
        CK(cudaMalloc(&p, bytes));
        ctx->owned.push_back(p);
        *out = reinterpret_cast<T*>(p);
        return PIMD_OK;
    }
    if (ctx->arena_used + bytes > ctx->arena_bytes)
        return fail(ctx, PIMD_ENOMEM, "device arena exhausted (workspace too small)");
    *out = reinterpret_cast<T*>(ctx->arena + ctx->arena_used);
    ctx->arena_used += bytes;
    return PIMD_OK;
}

size_t base_bytes(const pimd_ctx* c) {
    const size_t PN3 = (size_t)c->P * c->N * 3;
    size_t b = 0;
    b += 6 * align_up(PN3 * 8, 256);                          // x, vt, f, scratch_a, scratch_b, snap_f
    b += align_up(((size_t)c->P * 10 + BS_WIDTH) * 8, 256);   // snap_small
    b += 256 + align_up((size_t)3 * kMaxBeads * 8, 256);      // ctl_dev, com
    b += align_up((size_t)c->N * 8, 256) + align_up((size_t)c->N * 4, 256);
    b += align_up((size_t)c->P * 8, 256) + align_up((size_t)c->P * 72, 256) + align_up((size_t)c->P * c->N * 8, 256);
    b += align_up((size_t)(kEstCap + 2) * kEstWidth * 8, 256);
    b += align_up(barostat_state_doubles(3 * c->N) * 8, 256);
    return b + 4096 + 256;
}

void cell_grid(const double box[3], double rcut, int ncell[3], int R[3], int* ncells) {
    *ncells = 1;
    for (int a = 0; a < 3; ++a) {
        int nc = (int)std::floor(box[a] / (rcut * (1.0 + 1e-9)));
        if (nc < 1) nc = 1;
        ncell[a] = nc;
        const double w = box[a] / nc;
        R[a] = (int)std::ceil(rcut / w - 1e-12);
        if (R[a] < 1) R[a] = 1;
        *ncells *= nc;
    }
}

size_t model_bytes(const pimd_ctx* c, const pimd_model_desc* d) {
    if (!d) return 0;
    const size_t PN = (size_t)c->P * c->N;
    int nsel = 0;
    for (int t = 0; t < d->n_types; ++t) nsel += d->sel[t];
    const int M1 = d->embed[2], M2 = d->axis_neuron, NF = d->fit[0], ND = M1 * M2;
    int ncell[3], R[3], ncells;
    cell_grid(c->box, d->rcut, ncell, R, &ncells);
    size_t b = 0;
    b += align_up((size_t)d->n_types * d->n_types * 8192 * 4, 256);                     // embedding weights (padded)
    b += (size_t)d->n_types * (align_up(l1_wimg_bytes(ND), 256) + align_up(dd_wimg_bytes(ND) + 65536, 256));   // operand images of layer 1
    b += (size_t)d->n_types * 6 * (align_up((size_t)ND * NF * 4, 256) + 2 * align_up((size_t)NF * NF * 4, 256) + align_up(NF * 4, 256));
    b += (size_t)d->n_types * 4 * align_up((size_t)NF * 4, 256);
    b += (size_t)d->n_types * align_up(mid_wimg_bytes(), 256);
    b += 4 * align_up(PN * 4, 256);                                                    // cen_idx,row_of,cell_id,cell_tmp
    b += 3 * align_up((size_t)c->P * (ncells + 1) * 4, 256);
    b += align_up(PN * 24, 256) + align_up(PN * 32, 256);
    b += align_up(PN * d->n_types * 4, 256);
    b += 2 * align_up(PN * nsel * 16, 256);
    b += 256;
    b += 2 * align_up(PN * M1 * 16, 256);
    b += 2 * align_up(PN * ND * 4, 256);
    b += 7 * align_up(PN * NF * 4, 256);
    b += 2 * align_up((PN / 128 + d->n_types + 1) * mid_image_bytes(), 256) + 2 * align_up((PN / 128 + d->n_types + 1) * mid_scratch_bytes(), 256);
    b += 2 * align_up((size_t)d->n_types * d->n_types * emb_tc_image_h_bytes(), 256);
    b += align_up((size_t)d->n_types * (PN + 1) * 4, 256) + align_up(PN * nsel * 4, 256);
    b += align_up((size_t)d->n_types * ((PN + 1023) / 1024) * 4, 256) + align_up(PN * 72, 256);
    b += align_up(cmp_image_words_fw(d->n_types) * 4, 256) + align_up(cmp_image_words_bw(d->n_types) * 4, 256);
    b += align_up((PN / 8 + d->n_types + 1) * 4, 256);
    return b + 65536;
}

void mode_constants(pimd_ctx* c) {
    const int P = c->P;
    const double wP = P * kKB * c->T / kHbar;              // Eq. 2
    // BAOAB: A(dt/2) twice, O(dt) once; OBABO: A(dt) once, O(dt/2) twice (R-3)
    const bool obabo = c->integrator == PIMD_OBABO;
    const double h = obabo ? c->dt : 0.5 * c->dt;
    const double ho = obabo ? 0.5 * c->dt : c->dt;
    for (int k = 0; k < kMaxBeads; ++k) {
        c->mc.cosA[k] = 1; c->mc.sinA_w[k] = h; c->mc.msinA_w[k] = 0; c->mc.c1[k] = 1; c->mc.c2[k] = 0; c->mc.om2[k] = 0;
    }
    for (int k = 0; k < P; ++k) {
        const double sk = std::sin(k * M_PI / P);
        const double lam = 4.0 * sk * sk;                  // Eq. B2
        const double w = std::sqrt(lam) * wP;              // L469
        c->mc.om2[k] = w * w;
        if (k > 0) {
            c->mc.cosA[k] = std::cos(w * h);
            c->mc.sinA_w[k] = std::sin(w * h) / w;
            c->mc.msinA_w[k] = -w * std::sin(w * h);
        }
        double gam = (k == 0) ? c->gamma0 : 2.0 * w;  // Eq. D1; tau_0 = 1/gamma0 (L174)
        if (c->method == PIMD_CART) gam = 2.0 * wP;   // Eq. D3: tau = 1/(2 omega_n) for every bead (R-27)
        c->mc.c1[k] = std::exp(-ho * gam);
        c->mc.c2[k] = std::sqrt(1.0 - c->mc.c1[k] * c->mc.c1[k]);
    }
}

int alloc_base(pimd_ctx* ctx) {
    if (ctx->x) return PIMD_OK;
    const size_t PN3 = (size_t)ctx->P * ctx->N * 3;
    int rc;
    if ((rc = arena_alloc(ctx, &ctx->x, PN3))) return rc;
    if ((rc = arena_alloc(ctx, &ctx->vt, PN3))) return rc;
    if ((rc = arena_alloc(ctx, &ctx->f, PN3))) return rc;
    if ((rc = arena_alloc(ctx, &ctx->scratch_a, PN3))) return rc;
    if ((rc = arena_alloc(ctx, &ctx->scratch_b, PN3))) return rc;
    if ((rc = arena_alloc(ctx, &ctx->snap_f, PN3))) return rc;
    if ((rc = arena_alloc(ctx, &ctx->snap_small, (size_t)ctx->P * 10 + BS_WIDTH))) return rc;
    if ((rc = arena_alloc(ctx, &ctx->ctl_dev, (size_t)2))) return rc;
    CK(cudaMemsetAsync(ctx->ctl_dev, 0, 2 * sizeof(long long), ctx->stream));
    if ((rc = arena_alloc(ctx, &ctx->mass_atom, (size_t)ctx->N))) return rc;
    if ((rc = arena_alloc(ctx, &ctx->types_d, (size_t)ctx->N))) return rc;
    if ((rc = arena_alloc(ctx, &ctx->U, (size_t)ctx->P))) return rc;
    if ((rc = arena_alloc(ctx, &ctx->Xi, (size_t)ctx->P * 9))) return rc;
    if ((rc = arena_alloc(ctx, &ctx->Eatom, (size_t)ctx->P * ctx->N))) return rc;
    if ((rc = arena_alloc(ctx, &ctx->est, (size_t)(kEstCap + 2) * kEstWidth))) return rc;
    if ((rc = arena_alloc(ctx, &ctx->com, (size_t)3 * kMaxBeads))) return rc;      // nmpimd: [3]; Cartesian method: [P][3]
    std::vector<double> ma(ctx->N);
    double mtot = 0;
    for (int i = 0; i < ctx->N; ++i) { ma[i] = ctx->masses[ctx->types[i]]; mtot += ma[i]; }
    ctx->inv_mtot = 1.0 / mtot;
    CK(cudaMemcpyAsync(ctx->mass_atom, ma.data(), sizeof(double) * ctx->N, cudaMemcpyHostToDevice, ctx->stream));
    CK(cudaMemcpyAsync(ctx->types_d, ctx->types.data(), sizeof(int) * ctx->N, cudaMemcpyHostToDevice, ctx->stream));
    CK(cudaMemsetAsync(ctx->f, 0, PN3 * 8, ctx->stream));
    CK(cudaMemsetAsync(ctx->U, 0, sizeof(double) * ctx->P, ctx->stream));
    CK(cudaMemsetAsync(ctx->Xi, 0, sizeof(double) * 9 * ctx->P, ctx->stream));
    CK(cudaMemsetAsync(ctx->Eatom, 0, sizeof(double) * ctx->P * ctx->N, ctx->stream));
    CK(cudaMemsetAsync(ctx->est, 0, sizeof(double) * (kEstCap + 2) * kEstWidth, ctx->stream));
    CK(cudaStreamSynchronize(ctx->stream));
    return PIMD_OK;
}

void rec(pimd_ctx* ctx, int i) {
    if (ctx->profiling) cudaEventRecord(ctx->ev[i], ctx->stream);
}

// one force evaluation at the current x: f, U, Xi, Eatom
int eval_forces(pimd_ctx* ctx) {
    if (ctx->model_kind == 1) {
        ctx->launches += launch_harmonic(ctx->P, ctx->N, ctx->k_spring, ctx->x, ctx->f, ctx->U, ctx->Xi, ctx->Eatom, ctx->stream);
        return PIMD_OK;
    }
    ForceArgs a;
    a.P = ctx->P; a.N = ctx->N; a.ntypes = ctx->ntypes;
    for (int c = 0; c < 3; ++c) a.box[c] = ctx->box[c];
    a.box_dev = ctx->baro ? ctx->baro_state + BS_LX : nullptr;
    a.x = ctx->x; a.types = ctx->types_d; a.f = ctx->f; a.U = ctx->U; a.Xi = ctx->Xi; a.Eatom = ctx->Eatom;
    a.ctl = ctx->ctl_dev;
    const size_t PN3 = (size_t)ctx->P * ctx->N * 3;
    cudaMemsetAsync(ctx->f, 0, PN3 * 8, ctx->stream);
    cudaMemsetAsync(ctx->U, 0, sizeof(double) * ctx->P, ctx->stream);
    cudaMemsetAsync(ctx->Xi, 0, sizeof(double) * 9 * ctx->P, ctx->stream);
    rec(ctx, 1);
    ctx->evals_launched += 1;
    ctx->launches += neighbor_build(ctx->model, a, ctx->stream);
    if (ctx->model.compressed) {
        // tabulated embedding (NEXT-3): moments x table in tensor memory; no compact row index needed
        rec(ctx, 2);
        ctx->launches += compressed_forward(ctx->model, a, ctx->n_sms, ctx->stream);
        rec(ctx, 3);
        ctx->launches += fitting_forward_backward(ctx->model, a, ctx->stream);
        rec(ctx, 4);
        ctx->launches += compressed_backward(ctx->model, a, ctx->n_sms, ctx->stream);
        rec(ctx, 5);
        return PIMD_OK;
    }
    const bool tc_emb = ctx->model.use_tc_emb && ctx->model.tc_emb_ready;
    if (tc_emb) ctx->launches += emb_tc_row_index(ctx->model, a, ctx->stream);
    rec(ctx, 2);
    ctx->launches += tc_emb ? embedding_forward_tc(ctx->model, a, ctx->n_sms, ctx->stream)
                            : embedding_forward(ctx->model, a, ctx->n_sms, ctx->stream);
    rec(ctx, 3);
    ctx->launches += fitting_forward_backward(ctx->model, a, ctx->stream);
    rec(ctx, 4);
    ctx->launches += tc_emb ? embedding_backward_tc(ctx->model, a, ctx->n_sms, ctx->stream)
                            : embedding_backward(ctx->model, a, ctx->n_sms, ctx->stream);
    rec(ctx, 5);
    return PIMD_OK;
}

void fill_integrator_args(pimd_ctx* ctx, IntegratorArgs& a, int flags, int64_t step, double* est_slot) {
    a.N = ctx->N; a.n_dof = 3 * ctx->N; a.flags = flags;
    a.thermostat = (ctx->gamma0 != 0.0) ? 1 : 0;
    a.half_dt_mvv = 0.5 * ctx->dt / kMvv2e;
    a.PkT_mvv = ctx->P * kKB * ctx->T / kMvv2e;
    a.seed_lo = (uint32_t)ctx->seed; a.seed_hi = (uint32_t)(ctx->seed >> 32);
    a.step_lo = (uint32_t)(uint64_t)step; a.step_hi = (uint32_t)((uint64_t)step >> 32);
    { const uint64_t cs = (uint64_t)(step - 1); a.cstep_lo = (uint32_t)cs; a.cstep_hi = (uint32_t)(cs >> 32) | 0x80000000u; }
    if (ctx->integrator == PIMD_OBABO) a.flags |= I_OBABO;
    a.x_in = ctx->x; a.vt_in = ctx->vt; a.f = ctx->f; a.x_out = ctx->x; a.vt_out = ctx->vt;
    a.mass = ctx->mass_atom; a.U = ctx->U; a.est = est_slot;
    a.com = ctx->com; a.inv_mtot = ctx->inv_mtot;
    a.baro = ctx->baro ? ctx->baro_state : nullptr;
    { const double wP = ctx->P * kKB * ctx->T / kHbar; a.wP2 = wP * wP; }
    if (ctx->method == PIMD_CART) a.flags |= I_CART;
    a.ctl = nullptr;
    {
        static const char* pf = getenv("PIMD_INT_PREFETCH");          // blocks per SM ahead (measured best: 1)
        a.prefetch_ahead = (pf ? atoi(pf) : 1) * ctx->n_sms;
    }
    a.est_base = ctx->est;
    a.est_scratch = ctx->est + (size_t)(kEstCap + 1) * kEstWidth;
}

constexpr double kBarPerEvA3 = 1.602176634e6;    // DESIGN R-25

// the barostat's share of launch s (barostat.cu): closing E1 of the step that ends, opening E1 / E4-E7 of the next
int run_barostat(pimd_ctx* ctx, bool close, bool start, int64_t step, double* est_slot = nullptr) {
    BaroArgs b;
    b.P = ctx->P; b.N = ctx->N; b.n_dof = 3 * ctx->N;
    b.close = close; b.start = start; b.thermostat = (ctx->gamma0 != 0.0) ? 1 : 0;
    b.obabo = ctx->integrator == PIMD_OBABO; b.aniso = ctx->baro_aniso;
    b.h = 0.5 * ctx->dt; b.W = ctx->baro_W; b.p_ext = ctx->p_ext;
    b.nkT = ctx->P * kKB * ctx->T;
    b.c1 = std::exp(-(b.obabo ? 0.5 * ctx->dt : ctx->dt) * ctx->gamma0);
    b.c2 = std::sqrt(1.0 - b.c1 * b.c1);
    b.c2sig = b.c2 * std::sqrt(b.nkT / ctx->baro_W);
    b.half_dt_mvv = 0.5 * ctx->dt / kMvv2e;
    b.PkT_mvv = ctx->P * kKB * ctx->T / kMvv2e;
    b.seed_lo = (uint32_t)ctx->seed; b.seed_hi = (uint32_t)(ctx->seed >> 32);
    b.step_lo = (uint32_t)(uint64_t)step; b.step_hi = (uint32_t)((uint64_t)step >> 32);
    { const uint64_t cs = (uint64_t)(step - 1); b.cstep_lo = (uint32_t)cs; b.cstep_hi = (uint32_t)(cs >> 32) | 0x80000000u; }
    b.x = ctx->x; b.vt = ctx->vt; b.f = ctx->f; b.mass = ctx->mass_atom; b.Xi = ctx->Xi;
    b.state = ctx->baro_state; b.partial = ctx->baro_state + BS_WIDTH; b.est_slot = est_slot;
    return launch_barostat(b, ctx->stream);
}

// under a barostat the cell changes on the device: fetch it once per API call and refit the walk range of the
// (fixed) cell grid with a 3 % margin for the shrinkage inside the call (neighbor.cu flags a violation)
int sync_box(pimd_ctx* ctx) {
    if (!ctx->baro) return PIMD_OK;
    CK(cudaMemcpyAsync(ctx->box, ctx->baro_state + BS_LX, 3 * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
    CK(cudaStreamSynchronize(ctx->stream));
    if (ctx->model_kind == 2) {
        Model& m = ctx->model;
        for (int a = 0; a < 3; ++a) {
            const double w = ctx->box[a] / m.ncell[a];
            m.R[a] = std::max(1, (int)std::ceil(m.d.rcut * 1.03 / w - 1e-12));
            if (m.R[a] > 3) return fail(ctx, PIMD_EINVAL, "cell shrank below rcut/3 per grid cell");
        }
    }
    return PIMD_OK;
}

// model.overflow = {flag, first failing force evaluation (1-based count since pimd_set_model), evaluation counter, -}.
// Returns 0, or the error with *failed_eval = the 0-based index of the first evaluation that overflowed.
int check_overflow(pimd_ctx* ctx, int64_t* failed_eval = nullptr) {
    if (ctx->model_kind != 2) return PIMD_OK;
    unsigned flag[2] = {0u, 0u};
    CK(cudaMemcpyAsync(flag, ctx->model.overflow, sizeof(flag), cudaMemcpyDeviceToHost, ctx->stream));
    CK(cudaStreamSynchronize(ctx->stream));
    if (flag[0]) {
        const unsigned reset[2] = {0u, 0xFFFFFFFFu};
        cudaMemcpyAsync(ctx->model.overflow, reset, sizeof(reset), cudaMemcpyHostToDevice, ctx->stream);
        cudaStreamSynchronize(ctx->stream);
        if (failed_eval) *failed_eval = (int64_t)flag[1] - 1;
        if (flag[0] & 8u)
            return fail(ctx, PIMD_ECONTACT, "two atoms are closer than 0.01 A: s = 1/r leaves the range the FP16-split descriptor operands assume");
        if (flag[0] & 4u)
            return fail(ctx, PIMD_ETABLE_RANGE, "a neighbour row lies outside the compression table (s > 2, i.e. r < 0.5 A; DESIGN R-28)");
        if (flag[0] & 2u)
            return fail(ctx, PIMD_ESEL_OVERFLOW, "the cell shrank past the cell-grid margin inside one pimd_step call; use fewer steps per call");
        return fail(ctx, PIMD_ESEL_OVERFLOW, "an atom has more neighbours of one type than sel allows");
    }
    return PIMD_OK;
}

// forces + estimators of the current (x, v~): used after set_state / set_model
int refresh(pimd_ctx* ctx) {
    if (!ctx->have_state || ctx->model_kind == 0) return PIMD_OK;
    int rc = sync_box(ctx);
    if (rc) return rc;
    rc = eval_forces(ctx);
    if (rc) return rc;
    if (ctx->baro) ctx->launches += run_barostat(ctx, false, false, ctx->step);     // P_CV of the current state
    double* cur = ctx->est + (size_t)kEstCap * kEstWidth;
    CK(cudaMemsetAsync(cur, 0, sizeof(double) * kEstWidth, ctx->stream));
    IntegratorArgs a;
    fill_integrator_args(ctx, a, I_EST, ctx->step, cur);
    ctx->launches += launch_integrator(ctx->P, a, ctx->mc, ctx->stream);
    CK(cudaGetLastError());
    CK(cudaStreamSynchronize(ctx->stream));
    ctx->est_hist_n = 0;
    rc = check_overflow(ctx);
    if (rc) ctx->have_state = false;      // forces of a truncated neighbour list: nothing to integrate from (pimd.h)
    return rc;
}

void finalize_est(const pimd_ctx* c, const double raw[kEstWidth], int64_t step, pimd_estimators* e) {
    const double P = c->P, N = c->N;
    e->K_ring = raw[0]; e->S_ring = raw[1]; e->U_sum = raw[3];
    e->H = raw[0] + raw[1] + raw[3];
    e->K_PR = 1.5 * P * N * kKB * c->T - raw[1] / P;              // A7 with R-6
    e->K_CV = 1.5 * N * kKB * c->T - raw[2] / (2.0 * P);          // A9
    e->T_ring = 2.0 * raw[0] / (3.0 * P * N * kKB);
    e->step = step;
}

}  // namespace

extern "C" {

int pimd_create(pimd_ctx** out, int n_atoms, const int32_t* types, int n_types, const double* masses,
                const double box[3], int n_beads, double T, double dt, double gamma_centroid, uint64_t seed) {
    if (!out) return PIMD_EINVAL;
    *out = nullptr;
    if (n_atoms <= 0 || !types || n_types <= 0 || n_types > PIMD_MAX_TYPES || !masses || !box) return PIMD_EINVAL;
    if (!(n_beads == 1 || n_beads == 2 || n_beads == 4 || n_beads == 8 || n_beads == 16 || n_beads == 32 || n_beads == 64))
        return PIMD_EINVAL;
    if (!(T > 0) || !(dt > 0) || gamma_centroid < 0 || !(box[0] > 0 && box[1] > 0 && box[2] > 0)) return PIMD_EINVAL;
    for (int i = 0; i < n_atoms; ++i)
        if (types[i] < 0 || types[i] >= n_types) return PIMD_EINVAL;
    for (int t = 0; t < n_types; ++t)
        if (!(masses[t] > 0)) return PIMD_EINVAL;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) return PIMD_ECUDA;   // no CPU fallback
    pimd_ctx* ctx = new (std::nothrow) pimd_ctx();
    if (!ctx) return PIMD_ENOMEM;
    ctx->N = n_atoms; ctx->P = n_beads; ctx->ntypes = n_types;
    for (int c = 0; c < 3; ++c) ctx->box[c] = box[c];
    ctx->T = T; ctx->dt = dt; ctx->gamma0 = gamma_centroid; ctx->seed = seed;
    ctx->types.assign(types, types + n_atoms);
    ctx->masses.assign(masses, masses + n_types);
    int dev = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&ctx->n_sms, cudaDevAttrMultiProcessorCount, dev);
    mode_constants(ctx);
    for (int i = 0; i < 8; ++i) cudaEventCreate(&ctx->ev[i]);
    *out = ctx;
    return PIMD_OK;
}

void pimd_destroy(pimd_ctx* ctx) {
    if (!ctx) return;
    cudaStreamSynchronize(ctx->stream);
    if (ctx->step_graph) cudaGraphExecDestroy(ctx->step_graph);
    if (ctx->graph_stream) { cudaStreamDestroy(ctx->graph_stream); cudaEventDestroy(ctx->graph_ev); }
    if (ctx->model.aux_stream[0]) {
        for (int q = 0; q < Model::kChainStreams - 1; ++q) {
            cudaStreamSynchronize(ctx->model.aux_stream[q]);
            cudaStreamDestroy(ctx->model.aux_stream[q]);
            cudaEventDestroy(ctx->model.ev_join[q]);
        }
        cudaEventDestroy(ctx->model.ev_fork);
    }
    for (void* p : ctx->owned) cudaFree(p);
    for (int i = 0; i < 8; ++i)
        if (ctx->ev[i]) cudaEventDestroy(ctx->ev[i]);
    delete ctx;
}

const char* pimd_last_error(const pimd_ctx* ctx) { return ctx ? ctx->err.c_str() : "null context"; }

size_t pimd_workspace_bytes(const pimd_ctx* ctx, const pimd_model_desc* d) {
    if (!ctx) return 0;
    return base_bytes(ctx) + model_bytes(ctx, d);
}

int pimd_set_workspace(pimd_ctx* ctx, void* ws, size_t bytes, void* stream) {
    if (!ctx) return PIMD_EINVAL;
    if (ctx->arena || ctx->x) return fail(ctx, PIMD_EINVAL, "workspace must be set before any state or model call");
    ctx->stream = reinterpret_cast<cudaStream_t>(stream);
    if (ws) {
        if (((uintptr_t)ws & 255) != 0) return fail(ctx, PIMD_EINVAL, "workspace must be 256-byte aligned");
        ctx->arena = reinterpret_cast<char*>(ws);
        ctx->arena_bytes = bytes; ctx->arena_used = 0;
    }
    return PIMD_OK;
}

size_t pimd_model_n_weights(const pimd_model_desc* d) {
    if (!d) return 0;
    size_t ne = 0, nin = 1;
    for (int l = 0; l < 3; ++l) { ne += nin * d->embed[l] + d->embed[l]; nin = d->embed[l]; }
    size_t nf = 0;
    nin = (size_t)d->embed[2] * d->axis_neuron;
    for (int l = 0; l < 3; ++l) { nf += nin * d->fit[l] + d->fit[l]; nin = d->fit[l]; }
    nf += nin + 1;
    return (size_t)d->n_types * d->n_types * ne + (size_t)d->n_types * nf;
}

int pimd_set_state_dev(pimd_ctx* ctx, const double* x_dev, const double* p_dev) {
    if (!ctx || !x_dev || !p_dev) return fail(ctx, PIMD_EINVAL, "null argument");
    int rc;
    if ((rc = alloc_base(ctx))) return rc;
    const size_t PN3 = (size_t)ctx->P * ctx->N * 3;
    CK(cudaMemcpyAsync(ctx->x, x_dev, PN3 * 8, cudaMemcpyDeviceToDevice, ctx->stream));
    ctx->launches += ctx->method == PIMD_CART
        ? launch_cart_convert(ctx->P, ctx->N, p_dev, ctx->mass_atom, ctx->vt, 1, ctx->stream)
        : launch_to_nm_velocity(ctx->P, ctx->N, p_dev, ctx->mass_atom, ctx->vt, ctx->stream);
    CK(cudaGetLastError());
    ctx->have_state = true;
    ctx->step = 0;
    return refresh(ctx);
}

int pimd_set_state(pimd_ctx* ctx, const double* x, const double* p) {
    if (!ctx || !x || !p) return fail(ctx, PIMD_EINVAL, "null argument");
    int rc;
    if ((rc = alloc_base(ctx))) return rc;
    const size_t PN3 = (size_t)ctx->P * ctx->N * 3;
    CK(cudaMemcpyAsync(ctx->scratch_a, x, PN3 * 8, cudaMemcpyHostToDevice, ctx->stream));
    CK(cudaMemcpyAsync(ctx->scratch_b, p, PN3 * 8, cudaMemcpyHostToDevice, ctx->stream));
    return pimd_set_state_dev(ctx, ctx->scratch_a, ctx->scratch_b);
}

int pimd_restore(pimd_ctx* ctx, const double* x, const double* p, const double* f, const double* U, int64_t step) {
    if (!ctx || !x || !p || !f || !U || step < 0) return fail(ctx, PIMD_EINVAL, "bad argument");
    if (ctx->model_kind == 0) return fail(ctx, PIMD_ENOMODEL, "set the model before restoring a checkpoint");
    int rc;
    if ((rc = alloc_base(ctx))) return rc;
    const size_t PN3 = (size_t)ctx->P * ctx->N * 3;
    CK(cudaMemcpyAsync(ctx->x, x, PN3 * 8, cudaMemcpyHostToDevice, ctx->stream));
    CK(cudaMemcpyAsync(ctx->scratch_b, p, PN3 * 8, cudaMemcpyHostToDevice, ctx->stream));
    CK(cudaMemcpyAsync(ctx->f, f, PN3 * 8, cudaMemcpyHostToDevice, ctx->stream));
    CK(cudaMemcpyAsync(ctx->U, U, sizeof(double) * ctx->P, cudaMemcpyHostToDevice, ctx->stream));
    ctx->launches += ctx->method == PIMD_CART
        ? launch_cart_convert(ctx->P, ctx->N, ctx->scratch_b, ctx->mass_atom, ctx->vt, 1, ctx->stream)
        : launch_to_nm_velocity(ctx->P, ctx->N, ctx->scratch_b, ctx->mass_atom, ctx->vt, ctx->stream);
    ctx->have_state = true;
    ctx->step = step;
    if (ctx->baro) ctx->launches += run_barostat(ctx, false, false, ctx->step);     // P_CV of the restored state
    double* cur = ctx->est + (size_t)kEstCap * kEstWidth;
    CK(cudaMemsetAsync(cur, 0, sizeof(double) * kEstWidth, ctx->stream));
    IntegratorArgs a;
    fill_integrator_args(ctx, a, I_EST, ctx->step, cur);
    ctx->launches += launch_integrator(ctx->P, a, ctx->mc, ctx->stream);
    CK(cudaGetLastError());
    CK(cudaStreamSynchronize(ctx->stream));
    ctx->est_hist_n = 0;
    return PIMD_OK;
}

int pimd_get_neighbor_counts(pimd_ctx* ctx, int32_t* counts) {
    if (!ctx || !counts) return fail(ctx, PIMD_EINVAL, "null argument");
    if (ctx->model_kind != 2 || !ctx->have_state) return fail(ctx, PIMD_ENOMODEL, "needs an se_e2_a model and a state");
    CK(cudaMemcpyAsync(counts, ctx->model.ncount, sizeof(int32_t) * (size_t)ctx->P * ctx->N * ctx->ntypes,
                       cudaMemcpyDeviceToHost, ctx->stream));
    CK(cudaStreamSynchronize(ctx->stream));
    return PIMD_OK;
}

int64_t pimd_get_launch_count(const pimd_ctx* ctx) { return ctx ? ctx->launches : 0; }

int pimd_debug_get_row_index(pimd_ctx* ctx, int32_t* cen_idx, int32_t* rowstart) {
    if (!ctx || !cen_idx || !rowstart) return fail(ctx, PIMD_EINVAL, "null argument");
    if (ctx->model_kind != 2 || !ctx->have_state) return fail(ctx, PIMD_ENOMODEL, "needs an se_e2_a model and a state");
    const size_t PN = (size_t)ctx->P * ctx->N;
    CK(cudaMemcpyAsync(cen_idx, ctx->model.cen_idx, sizeof(int32_t) * PN, cudaMemcpyDeviceToHost, ctx->stream));
    CK(cudaMemcpyAsync(rowstart, ctx->model.rowstart, sizeof(int32_t) * (size_t)ctx->ntypes * (PN + 1),
                       cudaMemcpyDeviceToHost, ctx->stream));
    CK(cudaStreamSynchronize(ctx->stream));
    return PIMD_OK;
}

static int set_barostat(pimd_ctx* ctx, double p_ext_bar, double tau_p, bool aniso) {
    if (!ctx) return PIMD_EINVAL;
    if (!(tau_p > 0)) return fail(ctx, PIMD_EINVAL, "tau_p must be positive");
    if (ctx->fixcom) return fail(ctx, PIMD_EINVAL, "the barostat is not available with fixcom (DESIGN R-24)");
    if (ctx->method == PIMD_CART) return fail(ctx, PIMD_EINVAL, "the barostat needs the normal-mode method (DESIGN R-27)");
    if (!ctx->baro_state) {
        int rc = arena_alloc(ctx, &ctx->baro_state, barostat_state_doubles(3 * ctx->N));
        if (rc) return rc;
    }
    double st[BS_WIDTH] = {0};
    if (ctx->baro) { int rc = sync_box(ctx); if (rc) return rc; }     // keep the current cell
    for (int c = 0; c < 3; ++c) st[BS_LX + c] = ctx->box[c];
    CK(cudaMemcpyAsync(ctx->baro_state, st, sizeof(st), cudaMemcpyHostToDevice, ctx->stream));
    CK(cudaStreamSynchronize(ctx->stream));
    ctx->baro = true;
    ctx->baro_aniso = aniso;
    ctx->p_ext = p_ext_bar / kBarPerEvA3;
    // W = 3 n N k_B T tau_p^2, anisotropic n N k_B T tau_p^2 (L397)
    ctx->baro_W = (aniso ? 1.0 : 3.0) * ctx->P * ctx->N * kKB * ctx->T * tau_p * tau_p;
    return refresh(ctx);
}

int pimd_set_barostat(pimd_ctx* ctx, double p_ext_bar, double tau_p) { return set_barostat(ctx, p_ext_bar, tau_p, false); }
int pimd_set_barostat_aniso(pimd_ctx* ctx, double p_ext_bar, double tau_p) { return set_barostat(ctx, p_ext_bar, tau_p, true); }

int pimd_restore_cell(pimd_ctx* ctx, const double box[3], const double v_W[3], const double* xi) {
    if (!ctx || !box || !v_W || !xi) return fail(ctx, PIMD_EINVAL, "null argument");
    if (!ctx->baro) return fail(ctx, PIMD_EINVAL, "no barostat set");
    if (!(box[0] > 0 && box[1] > 0 && box[2] > 0)) return fail(ctx, PIMD_EINVAL, "cell lengths must be positive");
    int rc;
    if ((rc = alloc_base(ctx))) return rc;
    double st[6] = {v_W[0], v_W[1], v_W[2], box[0], box[1], box[2]};     // BS_VW .. BS_LZ
    CK(cudaMemcpyAsync(ctx->baro_state + BS_VW, st, sizeof(st), cudaMemcpyHostToDevice, ctx->stream));
    CK(cudaMemcpyAsync(ctx->Xi, xi, sizeof(double) * 9 * ctx->P, cudaMemcpyHostToDevice, ctx->stream));
    CK(cudaStreamSynchronize(ctx->stream));
    for (int c = 0; c < 3; ++c) ctx->box[c] = box[c];
    if (ctx->have_state && ctx->model_kind != 0) {
        ctx->launches += run_barostat(ctx, false, false, ctx->step);     // P_CV of the restored state
        CK(cudaStreamSynchronize(ctx->stream));
    }
    return PIMD_OK;
}

// Appendix A outputs 8-15 from the raw device record {v_W[3], L[3], diag P_CV[3], sum Tr Xi} and the estimator sums
static void finalize_baro(const pimd_ctx* ctx, const double* rec, const double* raw, pimd_barostat_state* b) {
    const double n = ctx->P, N = ctx->N;
    b->K_W = 0.0;
    for (int c = 0; c < 3; ++c) {
        b->v_W3[c] = rec[c];
        b->box[c] = rec[3 + c];
        b->P_CV3[c] = rec[6 + c] * kBarPerEvA3;                                            // E3 diagonal
        if (ctx->baro_aniso) b->K_W += 0.5 * ctx->baro_W * rec[c] * rec[c];                // A14
    }
    b->v_W = (rec[0] + rec[1] + rec[2]) / 3.0;
    if (!ctx->baro_aniso) b->K_W = 0.5 * ctx->baro_W * rec[0] * rec[0];                    // A13
    b->V = rec[3] * rec[4] * rec[5];
    b->P_CV = (rec[6] + rec[7] + rec[8]) / 3.0 * kBarPerEvA3;                              // A12 = the mean of E3's diagonal
    b->P_PR = (3.0 * n * N * kKB * ctx->T - 2.0 * raw[1] / n) / (3.0 * b->V) * kBarPerEvA3;  // A10 with R-6's 1/n: = 2 K_PR / (3V)
    b->P_MD = (2.0 * raw[0] + rec[9]) / (3.0 * b->V) * kBarPerEvA3;                        // A11
    b->U_W = n * ctx->p_ext * b->V;                                                        // A15
    b->J_W = -n * kKB * ctx->T * std::log(b->V);                                           // A16
    b->enthalpy = raw[0] + raw[1] + raw[3] + b->K_W + b->U_W + b->J_W;                     // A17
}

int pimd_get_barostat(pimd_ctx* ctx, pimd_barostat_state* b) {
    if (!ctx || !b) return fail(ctx, PIMD_EINVAL, "null argument");
    if (!ctx->baro) return fail(ctx, PIMD_EINVAL, "no barostat set");
    double st[BS_WIDTH], raw[kEstWidth];
    CK(cudaMemcpyAsync(st, ctx->baro_state, sizeof(st), cudaMemcpyDeviceToHost, ctx->stream));
    CK(cudaMemcpyAsync(raw, ctx->est + (size_t)kEstCap * kEstWidth, sizeof(raw), cudaMemcpyDeviceToHost, ctx->stream));
    CK(cudaStreamSynchronize(ctx->stream));
    const double rec[10] = {st[BS_VW], st[BS_VW + 1], st[BS_VW + 2], st[BS_LX], st[BS_LY], st[BS_LZ],
                            st[BS_PCV], st[BS_PCV + 1], st[BS_PCV + 2], st[BS_TRXI]};
    finalize_baro(ctx, rec, raw, b);
    return PIMD_OK;
}

int pimd_get_barostat_history(pimd_ctx* ctx, pimd_barostat_state* b, int cap) {
    if (!ctx || !b || cap < 0) return fail(ctx, PIMD_EINVAL, "bad argument");
    if (!ctx->baro) return fail(ctx, PIMD_EINVAL, "no barostat set");
    const int n = std::min(cap, ctx->est_hist_n);
    if (n == 0) return 0;
    std::vector<double> raw((size_t)ctx->est_hist_n * kEstWidth);
    CK(cudaMemcpyAsync(raw.data(), ctx->est, raw.size() * 8, cudaMemcpyDeviceToHost, ctx->stream));
    CK(cudaStreamSynchronize(ctx->stream));
    const int skip = ctx->est_hist_n - n;
    for (int q = 0; q < n; ++q) {
        const double* r = raw.data() + (size_t)(skip + q) * kEstWidth;
        finalize_baro(ctx, r + kEstBaro, r, b + q);
    }
    return n;
}

int pimd_set_method(pimd_ctx* ctx, int method) {
    if (!ctx) return PIMD_EINVAL;
    if (method != PIMD_NMPIMD && method != PIMD_CART) return fail(ctx, PIMD_EINVAL, "unknown method");
    if (method == PIMD_CART && ctx->baro)
        return fail(ctx, PIMD_EINVAL, "the Cartesian method is implemented without a barostat (DESIGN R-27)");
    if (method != ctx->method) ctx->have_state = false;      // the stored velocities change representation
    ctx->method = method;
    mode_constants(ctx);
    return PIMD_OK;
}

int pimd_set_fixcom(pimd_ctx* ctx, int on) {
    if (!ctx) return PIMD_EINVAL;
    if (on && ctx->baro) return fail(ctx, PIMD_EINVAL, "fixcom is not available with the barostat (DESIGN R-24)");
    ctx->fixcom = on != 0;
    return PIMD_OK;
}

int pimd_set_integrator(pimd_ctx* ctx, int kind) {
    if (!ctx) return PIMD_EINVAL;
    if (kind != PIMD_BAOAB && kind != PIMD_OBABO) return fail(ctx, PIMD_EINVAL, "unknown integrator kind");
    ctx->integrator = kind;
    mode_constants(ctx);
    return PIMD_OK;
}

int pimd_set_model_harmonic(pimd_ctx* ctx, double k_spring) {
    if (!ctx) return PIMD_EINVAL;
    int rc;
    if ((rc = alloc_base(ctx))) return rc;
    ctx->model_kind = 1;
    ctx->k_spring = k_spring;
    return refresh(ctx);
}

int pimd_set_model(pimd_ctx* ctx, const pimd_model_desc* d, const double* w, size_t n_weights) {
    if (!ctx || !d || !w) return fail(ctx, PIMD_EINVAL, "null argument");
    if (d->n_types != ctx->ntypes) return fail(ctx, PIMD_EINVAL, "model n_types differs from the context's");
    if (n_weights != pimd_model_n_weights(d)) return fail(ctx, PIMD_EINVAL, "weight vector has the wrong length");
    if (!(d->embed[0] == 25 && d->embed[1] == 50 && d->embed[2] == 100 && d->axis_neuron == 16))
        return fail(ctx, PIMD_EINVAL, "this build instantiates the embedding kernels for [25,50,100], axis 16 only");
    if (!(d->fit[0] == d->fit[1] && d->fit[1] == d->fit[2] && d->fit[0] % 16 == 0))
        return fail(ctx, PIMD_EINVAL, "fitting widths must be equal and a multiple of 16");
    if (!(d->rcut > d->rcut_smth && d->rcut_smth >= 0)) return fail(ctx, PIMD_EINVAL, "need rcut > rcut_smth >= 0");
    if (ctx->model.set) return fail(ctx, PIMD_EINVAL, "the model of a context can be set once");
    // The tensor-core kernels split every operand into FP16 hi / lo pairs with FIXED power-of-two scales (D x 256,
    // W1 x 64, unscaled embedding operands; DESIGN section 6 "Precision").  Those scales assume weights of order one;
    // a weight outside +-1000 (64 x 1000 is FP16's largest finite value) or a non-finite one is refused here rather
    // than turning into inf / NaN inside a kernel.
    for (size_t q = 0; q < n_weights; ++q)
        if (!(std::fabs(w[q]) <= 1000.0))
            return fail(ctx, PIMD_EINVAL, "weight " + std::to_string(q) + " is non-finite or exceeds 1000 in magnitude: outside the "
                                          "range of the FP16-split tensor-core operands");
    int rc;
    if ((rc = alloc_base(ctx))) return rc;
    Model& m = ctx->model;
    m.d = *d;
    const int nt = d->n_types;
    m.nsel = 0;
    for (int t = 0; t < nt; ++t) { m.seloff[t] = m.nsel; m.nsel += d->sel[t]; }
    for (int t = nt; t <= PIMD_MAX_TYPES; ++t) m.seloff[t] = m.nsel;
    m.E1 = d->embed[0]; m.E2 = d->embed[1]; m.M1 = d->embed[2]; m.M2 = d->axis_neuron; m.NF = d->fit[0];
    m.ND = m.M1 * m.M2;
    cell_grid(ctx->box, d->rcut, m.ncell, m.R, &m.ncells);
    for (int a = 0; a < 3; ++a)
        if (m.R[a] > 3) return fail(ctx, PIMD_EINVAL, "box shorter than rcut/3 is not supported");
    const size_t PN = (size_t)ctx->P * ctx->N;
    if (ctx->N >= (1 << 23)) return fail(ctx, PIMD_EINVAL, "at most 2^23 - 1 atoms");

    // ---- embedding weights, packed per (t_i, t_j): W1, b1, W2^T (k padded), b2, W3^T, b3 ----
    const int E1 = m.E1, E2 = m.E2, M1 = m.M1;
    const int E1p = (E1 + 3) / 4 * 4, E2p = (E2 + 3) / 4 * 4;
    const int oW1 = 0, ob1 = E1p, oW2t = 2 * E1p, ob2 = oW2t + E2 * E1p, oW3t = ob2 + E2p, ob3 = oW3t + M1 * E2p;
    m.emb_stride = (ob3 + M1 + 3) / 4 * 4;
    std::vector<float> ew((size_t)nt * nt * m.emb_stride, 0.f);
    size_t pos = 0;
    for (int ti = 0; ti < nt; ++ti)
        for (int tj = 0; tj < nt; ++tj) {
            float* o = ew.data() + (size_t)(ti * nt + tj) * m.emb_stride;
            for (int k = 0; k < E1; ++k) o[oW1 + k] = (float)w[pos + k];
            pos += E1;
            for (int k = 0; k < E1; ++k) o[ob1 + k] = (float)w[pos + k];
            pos += E1;
            for (int k = 0; k < E1; ++k)
                for (int n = 0; n < E2; ++n) o[oW2t + n * E1p + k] = (float)w[pos + (size_t)k * E2 + n];
            pos += (size_t)E1 * E2;
            for (int n = 0; n < E2; ++n) o[ob2 + n] = (float)w[pos + n];
            pos += E2;
            for (int k = 0; k < E2; ++k)
                for (int n = 0; n < M1; ++n) o[oW3t + n * E2p + k] = (float)w[pos + (size_t)k * M1 + n];
            pos += (size_t)E2 * M1;
            for (int n = 0; n < M1; ++n) o[ob3 + n] = (float)w[pos + n];
            pos += M1;
        }
    ctx->emb_w_host.assign(w, w + pos);          // the embedding part of the weight vector (all ordered pairs)
    if ((rc = arena_alloc(ctx, &m.emb_w, ew.size()))) return rc;
    CK(cudaMemcpyAsync(m.emb_w, ew.data(), ew.size() * 4, cudaMemcpyHostToDevice, ctx->stream));
    std::vector<uint8_t> img_h((size_t)nt * nt * emb_tc_image_h_bytes());
    {
        const size_t per_pair = (size_t)2 * E1 + (size_t)E1 * E2 + E2 + (size_t)E2 * M1 + M1;
        for (int q = 0; q < nt * nt; ++q) emb_tc_build_image_h(w + q * per_pair, img_h.data() + (size_t)q * emb_tc_image_h_bytes());
    }
    if ((rc = arena_alloc(ctx, &m.emb_img_h, img_h.size()))) return rc;
    CK(cudaMemcpyAsync(m.emb_img_h, img_h.data(), img_h.size(), cudaMemcpyHostToDevice, ctx->stream));
    std::vector<uint8_t> img_f(img_h.size());        // the forward kernel's copy: weights and biases x 2 log2(e) (tanh's exponent)
    {
        const size_t per_pair = (size_t)2 * E1 + (size_t)E1 * E2 + E2 + (size_t)E2 * M1 + M1;
        for (int q = 0; q < nt * nt; ++q)
            emb_tc_build_image_h(w + q * per_pair, img_f.data() + (size_t)q * emb_tc_image_h_bytes(), 2.8853900817779268);
    }
    if ((rc = arena_alloc(ctx, &m.emb_img_h_fwd, img_f.size()))) return rc;
    CK(cudaMemcpyAsync(m.emb_img_h_fwd, img_f.data(), img_f.size(), cudaMemcpyHostToDevice, ctx->stream));
    CK(cudaStreamSynchronize(ctx->stream));          // img_f leaves scope below

    // ---- fitting weights: W, W^T, b per layer ----
    std::vector<std::vector<float>> keep;
    std::vector<std::vector<uint8_t>> imgs;
    for (int t = 0; t < nt; ++t) {
        int nin = m.ND;
        for (int l = 0; l < 4; ++l) {
            const int nout = (l < 3) ? m.NF : 1;
            std::vector<float> W((size_t)nin * nout), WT((size_t)nin * nout), b(nout);
            for (int k = 0; k < nin; ++k)
                for (int n = 0; n < nout; ++n) {
                    const float v = (float)w[pos + (size_t)k * nout + n];
                    W[(size_t)k * nout + n] = v;
                    WT[(size_t)n * nin + k] = v;
                }
            pos += (size_t)nin * nout;
            for (int n = 0; n < nout; ++n) b[n] = (float)w[pos + n];
            pos += nout;
            if ((rc = arena_alloc(ctx, &m.fit_w[t][l], W.size()))) return rc;
            if ((rc = arena_alloc(ctx, &m.fit_wT[t][l], WT.size()))) return rc;
            if ((rc = arena_alloc(ctx, &m.fit_b[t][l], b.size()))) return rc;
            CK(cudaMemcpyAsync(m.fit_w[t][l], W.data(), W.size() * 4, cudaMemcpyHostToDevice, ctx->stream));
            CK(cudaMemcpyAsync(m.fit_wT[t][l], WT.data(), WT.size() * 4, cudaMemcpyHostToDevice, ctx->stream));
            CK(cudaMemcpyAsync(m.fit_b[t][l], b.data(), b.size() * 4, cudaMemcpyHostToDevice, ctx->stream));
            if (l < 3) {          // TF32 hi / lo images of W and W^T for the tensor-core GEMMs
                if ((rc = arena_alloc(ctx, &m.fit_w_hi[t][l], W.size()))) return rc;
                if ((rc = arena_alloc(ctx, &m.fit_w_lo[t][l], W.size()))) return rc;
                if ((rc = arena_alloc(ctx, &m.fit_wT_hi[t][l], W.size()))) return rc;
                if ((rc = arena_alloc(ctx, &m.fit_wT_lo[t][l], W.size()))) return rc;
                tc_split_weights(W.size(), m.fit_w[t][l], m.fit_w_hi[t][l], m.fit_w_lo[t][l], ctx->stream);
                tc_split_weights(W.size(), m.fit_wT[t][l], m.fit_wT_hi[t][l], m.fit_wT_lo[t][l], ctx->stream);
                if (l == 0) {     // operand images of layer 1 (fitting_tc.cu: l1_desc_kernel, dd_dt_kernel)
                    if (m.NF == 240 && nin % 160 == 0) {
                        std::vector<uint8_t> i1(l1_wimg_bytes(nin)), i2(dd_wimg_bytes(nin));
                        l1_build_wimg(WT.data(), nin, i1.data());
                        dd_build_wimg(W.data(), nin, i2.data());
                        if ((rc = arena_alloc(ctx, &m.l1_wimg[t], i1.size()))) return rc;
                        if ((rc = arena_alloc(ctx, &m.dd_wimg[t], i2.size()))) return rc;
                        CK(cudaMemcpyAsync(m.l1_wimg[t], i1.data(), i1.size(), cudaMemcpyHostToDevice, ctx->stream));
                        CK(cudaMemcpyAsync(m.dd_wimg[t], i2.data(), i2.size(), cudaMemcpyHostToDevice, ctx->stream));
                        imgs.push_back(std::move(i1)); imgs.push_back(std::move(i2));
                    }
                }
            }
            keep.push_back(std::move(W)); keep.push_back(std::move(WT)); keep.push_back(std::move(b));
            nin = nout;
        }
        if (m.NF == 240) {   // operand images of the fused middle of the chain (fitting_mid.cu)
            const size_t k0 = keep.size() - 12;              // W, WT, b of the four layers of this type
            std::vector<uint8_t> img(mid_wimg_bytes());
            mid_build_wimg(keep[k0 + 3].data(), keep[k0 + 4].data(), keep[k0 + 6].data(), keep[k0 + 7].data(), img.data());
            if ((rc = arena_alloc(ctx, &m.mid_wimg[t], img.size()))) return rc;
            CK(cudaMemcpyAsync(m.mid_wimg[t], img.data(), img.size(), cudaMemcpyHostToDevice, ctx->stream));
            imgs.push_back(std::move(img));
        }
    }

    {   // backward activations start at dy3 = w4: scale them by a power of two so that max |w4| lands in [8, 16)
        float wmax = 0.f;
        size_t q = (size_t)nt * nt * ((size_t)2 * E1 + (size_t)E1 * E2 + E2 + (size_t)E2 * M1 + M1);
        for (int t = 0; t < nt; ++t) {
            size_t nin = m.ND;
            for (int l = 0; l < 3; ++l) { q += nin * m.NF + m.NF; nin = m.NF; }
            for (int k = 0; k < m.NF; ++k) wmax = std::max(wmax, (float)std::fabs(w[q + k]));
            q += m.NF + 1;
        }
        int ex = 0;
        if (wmax > 0.f) std::frexp(wmax, &ex);            // wmax = f 2^ex, f in [0.5, 1)
        m.bwd_scale = std::ldexp(1.f, 4 - ex);
    }
    // ---- centre order [type][bead][atom of type] ----
    std::vector<int> cen(PN), rowof(PN);
    {
        size_t r = 0;
        for (int t = 0; t < nt; ++t) {
            m.type_row0[t] = (int)r;
            int cnt = 0;
            for (int k = 0; k < ctx->P; ++k)
                for (int i = 0; i < ctx->N; ++i)
                    if (ctx->types[i] == t) { cen[r] = k * ctx->N + i; rowof[(size_t)k * ctx->N + i] = (int)r; ++r; if (k == 0) ++cnt; }
            m.n_of_type[t] = cnt;
        }
        for (int t = nt; t <= PIMD_MAX_TYPES; ++t) m.type_row0[t] = (int)r;
    }
    if ((rc = arena_alloc(ctx, &m.cen_idx, PN))) return rc;
    if ((rc = arena_alloc(ctx, &m.row_of, PN))) return rc;
    CK(cudaMemcpyAsync(m.cen_idx, cen.data(), PN * 4, cudaMemcpyHostToDevice, ctx->stream));
    CK(cudaMemcpyAsync(m.row_of, rowof.data(), PN * 4, cudaMemcpyHostToDevice, ctx->stream));

    // ---- work buffers ----
    if ((rc = arena_alloc(ctx, &m.cell_count, (size_t)ctx->P * (m.ncells + 1)))) return rc;
    if ((rc = arena_alloc(ctx, &m.cell_start, (size_t)ctx->P * (m.ncells + 1)))) return rc;
    if ((rc = arena_alloc(ctx, &m.cell_fill, (size_t)ctx->P * (m.ncells + 1)))) return rc;
    if ((rc = arena_alloc(ctx, &m.cell_id, PN))) return rc;
    if ((rc = arena_alloc(ctx, &m.cell_tmp, PN))) return rc;
    if ((rc = arena_alloc(ctx, &m.wtmp, PN * 3))) return rc;
    if ((rc = arena_alloc(ctx, &m.wsorted, PN))) return rc;
    if ((rc = arena_alloc(ctx, &m.ncount, PN * nt))) return rc;
    if ((rc = arena_alloc(ctx, &m.slotA, PN * m.nsel))) return rc;
    if ((rc = arena_alloc(ctx, &m.slotB, PN * m.nsel))) return rc;
    if ((rc = arena_alloc(ctx, &m.overflow, (size_t)4))) return rc;
    if ((rc = arena_alloc(ctx, &m.Tm, PN * m.M1 * 4))) return rc;
    if ((rc = arena_alloc(ctx, &m.dTm, PN * m.M1 * 4))) return rc;
    if ((rc = arena_alloc(ctx, &m.D, PN * m.ND))) return rc;
    if ((rc = arena_alloc(ctx, &m.dD, PN * m.ND))) return rc;
    float** fb[7] = {&m.Y1, &m.T2, &m.Y2, &m.T3, &m.Y3, &m.G1, &m.G2};
    for (int q = 0; q < 7; ++q)
        if ((rc = arena_alloc(ctx, fb[q], PN * m.NF))) return rc;
    if (m.NF == 240) {   // hand-over images and scratch of the fused fitting chain, per 128-row tile
        const size_t tiles = PN / 128 + nt + 1;
        if ((rc = arena_alloc(ctx, &m.y1_img, tiles * mid_image_bytes()))) return rc;
        if ((rc = arena_alloc(ctx, &m.da1_img, tiles * mid_image_bytes()))) return rc;
        if ((rc = arena_alloc(ctx, &m.mid_t2, tiles * mid_scratch_bytes() / 16))) return rc;
        if ((rc = arena_alloc(ctx, &m.mid_g1, tiles * mid_scratch_bytes() / 16))) return rc;
    }
    if ((rc = arena_alloc(ctx, &m.rowstart, (size_t)nt * (PN + 1)))) return rc;
    if ((rc = arena_alloc(ctx, &m.rowaddr, PN * m.nsel))) return rc;
    if ((rc = arena_alloc(ctx, &m.row_bsum, (size_t)nt * ((PN + 1023) / 1024)))) return rc;
    if ((rc = arena_alloc(ctx, &m.cpart, PN * 9))) return rc;
    m.tc_emb_ready = true;
    {
        const unsigned ov0[4] = {0u, 0xFFFFFFFFu, (unsigned)ctx->evals_launched, 0u};
        CK(cudaMemcpyAsync(m.overflow, ov0, sizeof(ov0), cudaMemcpyHostToDevice, ctx->stream));
    }
    CK(cudaStreamSynchronize(ctx->stream));     // host staging vectors go out of scope below
    if (tc_setup_maps(m, nt))    // tensor-core fitting path (falls back to the CUDA-core GEMMs only if unsupported widths)
        fitting_mid_setup(m, nt);
    m.set = true;
    ctx->model_kind = 2;
    return refresh(ctx);
}

int pimd_set_embedding_compressed(pimd_ctx* ctx, int on) {
    if (!ctx) return PIMD_EINVAL;
    if (!ctx->model.set) return fail(ctx, PIMD_ENOMODEL, "set the se_e2_a model first: the tables are built from its weights");
    Model& m = ctx->model;
    if (on && ctx->ntypes > 2)
        return fail(ctx, PIMD_EINVAL, "the tensor-memory resident tables hold two neighbour types (2 x 40 intervals x 6 coefficients)");
    if (on && !m.cmp_img_fw) {
        int rc;
        std::vector<uint32_t> fw(cmp_image_words_fw(ctx->ntypes)), bw(cmp_image_words_bw(ctx->ntypes));
        cmp_build_images(ctx->emb_w_host.data(), ctx->ntypes, fw.data(), bw.data());     // FP64 on the host -> FP16 hi / lo
        if ((rc = arena_alloc(ctx, &m.cmp_img_fw, fw.size()))) return rc;
        if ((rc = arena_alloc(ctx, &m.cmp_img_bw, bw.size()))) return rc;
        if ((rc = arena_alloc(ctx, &m.cmp_need, (size_t)ctx->P * ctx->N / 8 + ctx->ntypes + 1))) return rc;
        CK(cudaMemcpyAsync(m.cmp_img_fw, fw.data(), fw.size() * 4, cudaMemcpyHostToDevice, ctx->stream));
        CK(cudaMemcpyAsync(m.cmp_img_bw, bw.data(), bw.size() * 4, cudaMemcpyHostToDevice, ctx->stream));
        CK(cudaStreamSynchronize(ctx->stream));
    }
    m.compressed = on != 0;
    return refresh(ctx);
}

int pimd_step(pimd_ctx* ctx, int64_t n_steps) {
    if (!ctx) return PIMD_EINVAL;
    if (n_steps < 0) return fail(ctx, PIMD_EINVAL, "n_steps < 0");
    if (!ctx->have_state) return fail(ctx, PIMD_ENOSTATE, "pimd_set_state has not been called");
    if (ctx->model_kind == 0) return fail(ctx, PIMD_ENOMODEL, "no force model set");
    if (n_steps == 0) return PIMD_OK;
    { int rc = sync_box(ctx); if (rc) return rc; }
    // Entry snapshot (se_e2_a model only: the harmonic model cannot fail): a sel overflow or a cell that outruns its
    // grid at step k leaves every later step of the call integrating truncated neighbour rows, so the call is then
    // undone as a whole -- x, v~, f, U, Xi, the barostat state and the step counter return to their entry values.
    const size_t PN3 = (size_t)ctx->P * ctx->N * 3;
    const bool snap = ctx->model_kind == 2;
    const int64_t evals0 = ctx->evals_launched;
    double box0[3] = {ctx->box[0], ctx->box[1], ctx->box[2]};
    if (snap) {
        CK(cudaMemcpyAsync(ctx->scratch_a, ctx->x, PN3 * 8, cudaMemcpyDeviceToDevice, ctx->stream));
        CK(cudaMemcpyAsync(ctx->scratch_b, ctx->vt, PN3 * 8, cudaMemcpyDeviceToDevice, ctx->stream));
        CK(cudaMemcpyAsync(ctx->snap_f, ctx->f, PN3 * 8, cudaMemcpyDeviceToDevice, ctx->stream));
        CK(cudaMemcpyAsync(ctx->snap_small, ctx->U, sizeof(double) * ctx->P, cudaMemcpyDeviceToDevice, ctx->stream));
        CK(cudaMemcpyAsync(ctx->snap_small + ctx->P, ctx->Xi, sizeof(double) * 9 * ctx->P, cudaMemcpyDeviceToDevice, ctx->stream));
        if (ctx->baro)
            CK(cudaMemcpyAsync(ctx->snap_small + 10 * (size_t)ctx->P, ctx->baro_state, sizeof(double) * BS_WIDTH,
                               cudaMemcpyDeviceToDevice, ctx->stream));
    }
    const int hist = (int)std::min<int64_t>(n_steps, kEstCap);
    const int64_t first_hist = n_steps - hist;            // steps before this index are not recorded
    CK(cudaMemsetAsync(ctx->est, 0, sizeof(double) * (size_t)hist * kEstWidth, ctx->stream));
    double* cur = ctx->est + (size_t)kEstCap * kEstWidth;
    double* scratch = ctx->est + (size_t)(kEstCap + 1) * kEstWidth;
    float ms_acc[6] = {0, 0, 0, 0, 0, 0};
    // launch s: closes step s-1 (B, estimators) and opens step s (B A O A).  ctl_mode: step counter and estimator slot
    // come from the device (graph replay), the host values are then ignored by the kernels.
    auto integ = [&](int64_t s, bool ctl_mode) {
        int flags = 0;
        double* slot = scratch;
        if (s > 0) {
            flags |= I_BCLOSE | I_EST;
            slot = (s - 1 >= first_hist) ? ctx->est + (size_t)(s - 1 - first_hist) * kEstWidth : scratch;
        }
        if (s < n_steps) flags |= I_START;
        IntegratorArgs a;
        rec(ctx, 0);
        if (ctx->baro) ctx->launches += run_barostat(ctx, s > 0, s < n_steps, ctx->step + s, s > 0 ? slot : nullptr);
        if (ctx->fixcom && s > 0) {
            // fixcom (R-19): the removal needs sum_i m_i v~_0,i over ALL atoms after the closing half,
            // so the launch splits: close + accumulate, then subtract + estimators (+ open)
            cudaMemsetAsync(ctx->com, 0, sizeof(double) * 3 * (ctx->method == PIMD_CART ? ctx->P : 1), ctx->stream);
            fill_integrator_args(ctx, a, I_BCLOSE | I_COMACC, ctx->step + s, scratch);
            if (ctl_mode) a.ctl = ctx->ctl_dev;
            ctx->launches += launch_integrator(ctx->P, a, ctx->mc, ctx->stream);
            flags = (flags & ~I_BCLOSE) | I_COMSUB;
        }
        fill_integrator_args(ctx, a, flags, ctx->step + s, slot);
        if (ctl_mode) a.ctl = ctx->ctl_dev;
        ctx->launches += launch_integrator(ctx->P, a, ctx->mc, ctx->stream);
    };
    const bool use_graph = ctx->model_kind == 2 && !ctx->baro && !ctx->profiling && n_steps >= 3 && !ctx->graph_failed &&
                           getenv("PIMD_NO_GRAPH") == nullptr;
    if (!use_graph) {
        for (int64_t s = 0; s <= n_steps; ++s) {
            integ(s, false);
            if (s < n_steps) {
                int rc = eval_forces(ctx);
                if (rc) return rc;
                if (ctx->profiling) {
                    rec(ctx, 6);
                    cudaEventSynchronize(ctx->ev[6]);
                    float t;
                    if (ctx->model_kind == 2) {
                        cudaEventElapsedTime(&t, ctx->ev[0], ctx->ev[1]); ms_acc[0] += t;
                        for (int q = 1; q < 5; ++q) { cudaEventElapsedTime(&t, ctx->ev[q], ctx->ev[q + 1]); ms_acc[q] += t; }
                    }
                }
            }
        }
    } else {
        // One captured launch sequence per step: {integrator launch of an inner step, force evaluation} becomes a CUDA
        // graph (the three streams of the fitting chain included) and is replayed n_steps - 1 times.
        if (!ctx->graph_stream) {
            CK(cudaStreamCreateWithFlags(&ctx->graph_stream, cudaStreamNonBlocking));
            CK(cudaEventCreateWithFlags(&ctx->graph_ev, cudaEventDisableTiming));
        }
        // hand over from the caller's stream: everything issued so far (snapshot copies, memsets) precedes the loop
        CK(cudaEventRecord(ctx->graph_ev, ctx->stream));
        CK(cudaStreamWaitEvent(ctx->graph_stream, ctx->graph_ev, 0));
        struct StreamSwap {
            pimd_ctx* c; cudaStream_t user;
            StreamSwap(pimd_ctx* c_) : c(c_), user(c_->stream) { c->stream = c->graph_stream; }
            ~StreamSwap() { cudaStreamSynchronize(c->graph_stream); c->stream = user; }
        } swap(ctx);
        const long long ctl_h[2] = {(long long)ctx->step, (long long)(ctx->step + first_hist)};
        CK(cudaMemcpyAsync(ctx->ctl_dev, ctl_h, sizeof(ctl_h), cudaMemcpyHostToDevice, ctx->stream));
        integ(0, true);
        { int rc = eval_forces(ctx); if (rc) return rc; }
        const Model& mm = ctx->model;
        const uint64_t key = 1ull | ((uint64_t)ctx->integrator << 1) | ((uint64_t)ctx->fixcom << 2) | ((uint64_t)ctx->method << 3) |
                             ((uint64_t)mm.compressed << 4) | ((uint64_t)mm.use_tc << 5) | ((uint64_t)mm.use_tc_emb << 6) |
                             ((uint64_t)(ctx->gamma0 != 0.0) << 7);
        if (ctx->step_graph && ctx->graph_key != key) { cudaGraphExecDestroy(ctx->step_graph); ctx->step_graph = nullptr; }
        if (!ctx->step_graph) {
            const int64_t l0 = ctx->launches, e0 = ctx->evals_launched;
            cudaGraph_t g = nullptr;
            bool ok = cudaStreamBeginCapture(ctx->stream, cudaStreamCaptureModeRelaxed) == cudaSuccess;
            if (ok) {
                integ(1, true);                         // an inner step: n_steps >= 3, so 0 < 1 < n_steps
                eval_forces(ctx);
                ok = cudaStreamEndCapture(ctx->stream, &g) == cudaSuccess && g != nullptr;
            }
            ctx->graph_launches = ctx->launches - l0;
            ctx->launches = l0; ctx->evals_launched = e0;     // a capture launches nothing
            if (ok) ok = cudaGraphInstantiate(&ctx->step_graph, g, 0) == cudaSuccess;
            if (g) cudaGraphDestroy(g);
            if (!ok) {
                ctx->step_graph = nullptr; ctx->graph_failed = true;
                ctx->err = std::string("graph capture failed, plain launches used: ") + cudaGetErrorString(cudaGetLastError());
            }
            ctx->graph_key = key;
        }
        for (int64_t s = 1; s < n_steps; ++s) {
            if (ctx->step_graph) {
                CK(cudaGraphLaunch(ctx->step_graph, ctx->stream));
                ctx->launches += ctx->graph_launches;
                ctx->evals_launched += 1;
            } else {
                integ(s, true);
                int rc = eval_forces(ctx);
                if (rc) return rc;
            }
        }
        integ(n_steps, true);
    }
    CK(cudaGetLastError());
    // the last slot is also "current"
    CK(cudaMemcpyAsync(cur, ctx->est + (size_t)(hist - 1) * kEstWidth, sizeof(double) * kEstWidth,
                       cudaMemcpyDeviceToDevice, ctx->stream));
    CK(cudaStreamSynchronize(ctx->stream));
    {
        int64_t failed_eval = -1;
        const int rc = check_overflow(ctx, &failed_eval);
        if (rc) {
            const std::string why = ctx->err;
            CK(cudaMemcpyAsync(ctx->x, ctx->scratch_a, PN3 * 8, cudaMemcpyDeviceToDevice, ctx->stream));
            CK(cudaMemcpyAsync(ctx->vt, ctx->scratch_b, PN3 * 8, cudaMemcpyDeviceToDevice, ctx->stream));
            CK(cudaMemcpyAsync(ctx->f, ctx->snap_f, PN3 * 8, cudaMemcpyDeviceToDevice, ctx->stream));
            CK(cudaMemcpyAsync(ctx->U, ctx->snap_small, sizeof(double) * ctx->P, cudaMemcpyDeviceToDevice, ctx->stream));
            CK(cudaMemcpyAsync(ctx->Xi, ctx->snap_small + ctx->P, sizeof(double) * 9 * ctx->P, cudaMemcpyDeviceToDevice, ctx->stream));
            if (ctx->baro) {
                CK(cudaMemcpyAsync(ctx->baro_state, ctx->snap_small + 10 * (size_t)ctx->P, sizeof(double) * BS_WIDTH,
                                   cudaMemcpyDeviceToDevice, ctx->stream));
                for (int c = 0; c < 3; ++c) ctx->box[c] = box0[c];
            }
            CK(cudaStreamSynchronize(ctx->stream));
            ctx->est_hist_n = 0;
            char where[256];
            snprintf(where, sizeof(where), " (first at step %lld of this call of %lld = absolute step %lld); the state has been "
                     "rolled back to the start of the call",
                     (long long)(failed_eval - evals0 + 1), (long long)n_steps, (long long)(ctx->step + failed_eval - evals0 + 1));
            return fail(ctx, rc, why + where);
        }
    }
    ctx->step += n_steps;
    ctx->est_hist_n = hist;
    ctx->est_hist_first_step = ctx->step - hist + 1;
    if (ctx->profiling) {
        for (int q = 0; q < 6; ++q) ctx->phase_ms[q] = ms_acc[q] / (double)n_steps;
        ctx->phase_steps = n_steps;
    }
    return PIMD_OK;
}

static int copy_out(pimd_ctx* ctx, const void* dev, void* host, size_t bytes) {
    if (!ctx || !host) return fail(ctx, PIMD_EINVAL, "null argument");
    if (!ctx->have_state) return fail(ctx, PIMD_ENOSTATE, "pimd_set_state has not been called");
    CK(cudaMemcpyAsync(host, dev, bytes, cudaMemcpyDeviceToHost, ctx->stream));
    CK(cudaStreamSynchronize(ctx->stream));
    return PIMD_OK;
}

int pimd_get_positions(pimd_ctx* ctx, double* x) {
    return copy_out(ctx, ctx ? ctx->x : nullptr, x, ctx ? (size_t)ctx->P * ctx->N * 24 : 0);
}
int pimd_get_momenta(pimd_ctx* ctx, double* p) {
    if (!ctx || !p) return fail(ctx, PIMD_EINVAL, "null argument");
    if (!ctx->have_state) return fail(ctx, PIMD_ENOSTATE, "pimd_set_state has not been called");
    ctx->launches += ctx->method == PIMD_CART
        ? launch_cart_convert(ctx->P, ctx->N, ctx->vt, ctx->mass_atom, ctx->scratch_a, 0, ctx->stream)
        : launch_from_nm_momenta(ctx->P, ctx->N, ctx->vt, ctx->mass_atom, ctx->scratch_a, ctx->stream);
    return copy_out(ctx, ctx->scratch_a, p, (size_t)ctx->P * ctx->N * 24);
}
int pimd_get_forces(pimd_ctx* ctx, double* f) {
    return copy_out(ctx, ctx ? ctx->f : nullptr, f, ctx ? (size_t)ctx->P * ctx->N * 24 : 0);
}
int pimd_get_virial(pimd_ctx* ctx, double* xi) {
    return copy_out(ctx, ctx ? ctx->Xi : nullptr, xi, ctx ? (size_t)ctx->P * 72 : 0);
}
int pimd_get_energies(pimd_ctx* ctx, double* U) {
    return copy_out(ctx, ctx ? ctx->U : nullptr, U, ctx ? (size_t)ctx->P * 8 : 0);
}
int pimd_get_atom_energies(pimd_ctx* ctx, double* E) {
    return copy_out(ctx, ctx ? ctx->Eatom : nullptr, E, ctx ? (size_t)ctx->P * ctx->N * 8 : 0);
}

int pimd_get_estimators(pimd_ctx* ctx, pimd_estimators* e) {
    if (!ctx || !e) return fail(ctx, PIMD_EINVAL, "null argument");
    if (!ctx->have_state) return fail(ctx, PIMD_ENOSTATE, "pimd_set_state has not been called");
    if (ctx->model_kind == 0) return fail(ctx, PIMD_ENOMODEL, "no force model set");
    double raw[kEstWidth];
    int rc = copy_out(ctx, ctx->est + (size_t)kEstCap * kEstWidth, raw, sizeof(raw));
    if (rc) return rc;
    finalize_est(ctx, raw, ctx->step, e);
    return PIMD_OK;
}

int pimd_get_estimator_history(pimd_ctx* ctx, pimd_estimators* e, int cap) {
    if (!ctx || !e || cap < 0) return fail(ctx, PIMD_EINVAL, "bad argument");
    const int n = std::min(cap, ctx->est_hist_n);
    if (n == 0) return 0;
    std::vector<double> raw((size_t)ctx->est_hist_n * kEstWidth);
    int rc = copy_out(ctx, ctx->est, raw.data(), raw.size() * 8);
    if (rc) return rc;
    const int skip = ctx->est_hist_n - n;
    for (int q = 0; q < n; ++q)
        finalize_est(ctx, raw.data() + (size_t)(skip + q) * kEstWidth, ctx->est_hist_first_step + skip + q, e + q);
    return n;
}

int pimd_get_positions_dev(pimd_ctx* ctx, double* x_dev) {
    if (!ctx || !x_dev) return fail(ctx, PIMD_EINVAL, "null argument");
    if (!ctx->have_state) return fail(ctx, PIMD_ENOSTATE, "pimd_set_state has not been called");
    CK(cudaMemcpyAsync(x_dev, ctx->x, (size_t)ctx->P * ctx->N * 24, cudaMemcpyDeviceToDevice, ctx->stream));
    CK(cudaStreamSynchronize(ctx->stream));
    return PIMD_OK;
}
int pimd_get_forces_dev(pimd_ctx* ctx, double* f_dev) {
    if (!ctx || !f_dev) return fail(ctx, PIMD_EINVAL, "null argument");
    if (!ctx->have_state) return fail(ctx, PIMD_ENOSTATE, "pimd_set_state has not been called");
    CK(cudaMemcpyAsync(f_dev, ctx->f, (size_t)ctx->P * ctx->N * 24, cudaMemcpyDeviceToDevice, ctx->stream));
    CK(cudaStreamSynchronize(ctx->stream));
    return PIMD_OK;
}

int64_t pimd_get_neighbors(pimd_ctx* ctx, int bead, int32_t* count, int32_t* jout, int8_t* shift, size_t cap) {
    if (!ctx || !count || !jout || !shift) return fail(ctx, PIMD_EINVAL, "null argument");
    if (ctx->model_kind != 2 || !ctx->have_state) return fail(ctx, PIMD_ENOMODEL, "needs an se_e2_a model and a state");
    if (bead < 0 || bead >= ctx->P) return fail(ctx, PIMD_EINVAL, "bead out of range");
    const Model& m = ctx->model;
    const int N = ctx->N, nt = ctx->ntypes;
    std::vector<int> cnt((size_t)N * nt);
    std::vector<NeighSlotB> sb((size_t)N * m.nsel);
    CK(cudaMemcpyAsync(cnt.data(), m.ncount + (size_t)bead * N * nt, cnt.size() * 4, cudaMemcpyDeviceToHost, ctx->stream));
    CK(cudaMemcpyAsync(sb.data(), m.slotB + (size_t)bead * N * m.nsel, sb.size() * sizeof(NeighSlotB),
                       cudaMemcpyDeviceToHost, ctx->stream));
    CK(cudaStreamSynchronize(ctx->stream));
    size_t total = 0;
    struct Row { int t, j, nx, ny, nz; };
    std::vector<Row> rows;
    for (int i = 0; i < N; ++i) {
        rows.clear();
        for (int t = 0; t < nt; ++t)
            for (int q = 0; q < cnt[(size_t)i * nt + t]; ++q) {
                const uint32_t jc = sb[(size_t)i * m.nsel + m.seloff[t] + q].jcode;
                const uint32_t code = jc >> 23;
                rows.push_back({t, (int)(jc & 0x7fffffu), (int)(code & 7) - 3, (int)((code >> 3) & 7) - 3, (int)((code >> 6) & 7) - 3});
            }
        std::sort(rows.begin(), rows.end(), [](const Row& a, const Row& b) {
            if (a.t != b.t) return a.t < b.t;
            if (a.j != b.j) return a.j < b.j;
            if (a.nx != b.nx) return a.nx < b.nx;
            if (a.ny != b.ny) return a.ny < b.ny;
            return a.nz < b.nz;
        });
        count[i] = (int32_t)rows.size();
        if (total + rows.size() > cap) return fail(ctx, PIMD_EINVAL, "cap too small for the neighbour rows");
        for (const Row& r : rows) {
            jout[total] = r.j;
            shift[3 * total] = (int8_t)r.nx; shift[3 * total + 1] = (int8_t)r.ny; shift[3 * total + 2] = (int8_t)r.nz;
            ++total;
        }
    }
    return (int64_t)total;
}

int pimd_debug_noise(pimd_ctx* ctx, int64_t step, int n, const int32_t* idx, uint32_t* words, double* eta) {
    if (!ctx || n <= 0 || !idx || !words || !eta) return fail(ctx, PIMD_EINVAL, "bad argument");
    int32_t* d_idx = nullptr; uint32_t* d_w = nullptr; double* d_e = nullptr;
    CK(cudaMalloc(&d_idx, sizeof(int32_t) * 3 * n));
    CK(cudaMalloc(&d_w, sizeof(uint32_t) * 4 * n));
    CK(cudaMalloc(&d_e, sizeof(double) * n));
    CK(cudaMemcpyAsync(d_idx, idx, sizeof(int32_t) * 3 * n, cudaMemcpyHostToDevice, ctx->stream));
    ctx->launches += launch_debug_noise(ctx->seed, (uint64_t)step, n, d_idx, d_w, d_e, ctx->stream);
    CK(cudaMemcpyAsync(words, d_w, sizeof(uint32_t) * 4 * n, cudaMemcpyDeviceToHost, ctx->stream));
    CK(cudaMemcpyAsync(eta, d_e, sizeof(double) * n, cudaMemcpyDeviceToHost, ctx->stream));
    CK(cudaStreamSynchronize(ctx->stream));
    cudaFree(d_idx); cudaFree(d_w); cudaFree(d_e);
    return PIMD_OK;
}

int pimd_time_kernel(pimd_ctx* ctx, int kind, int reps, double* ms) {
    if (!ctx || !ms || reps <= 0) return fail(ctx, PIMD_EINVAL, "bad argument");
    if (!ctx->have_state || ctx->model_kind == 0) return fail(ctx, PIMD_ENOSTATE, "needs a state and a model");
    if (kind != 0 && kind != 1) return fail(ctx, PIMD_EINVAL, "unknown kernel kind");
    IntegratorArgs a;
    double* scratch = ctx->est + (size_t)(kEstCap + 1) * kEstWidth;
    fill_integrator_args(ctx, a, I_BCLOSE | I_EST | I_START | (kind == 1 ? I_NOISE_PER_MODE : 0), ctx->step, scratch);
    a.x_out = ctx->scratch_a; a.vt_out = ctx->scratch_b;          // state is not advanced
    for (int w = 0; w < 3; ++w) ctx->launches += launch_integrator(ctx->P, a, ctx->mc, ctx->stream);
    CK(cudaEventRecord(ctx->ev[6], ctx->stream));
    for (int r = 0; r < reps; ++r) ctx->launches += launch_integrator(ctx->P, a, ctx->mc, ctx->stream);
    CK(cudaEventRecord(ctx->ev[7], ctx->stream));
    CK(cudaEventSynchronize(ctx->ev[7]));
    CK(cudaGetLastError());
    float t = 0;
    CK(cudaEventElapsedTime(&t, ctx->ev[6], ctx->ev[7]));
    *ms = (double)t / reps;
    return PIMD_OK;
}

int pimd_set_fitting_path(pimd_ctx* ctx, int use_tensor_cores) {
    if (!ctx) return PIMD_EINVAL;
    if (use_tensor_cores && ctx->model.set && !ctx->model.tc_ready)
        return fail(ctx, PIMD_EINVAL, "tensor-core path unavailable for this architecture (needs fit width 240)");
    ctx->model.use_tc = use_tensor_cores != 0;
    return PIMD_OK;
}

int pimd_set_embedding_path(pimd_ctx* ctx, int use_tensor_cores) {
    if (!ctx) return PIMD_EINVAL;
    ctx->model.use_tc_emb = use_tensor_cores != 0;
    return PIMD_OK;
}

int pimd_debug_gemm(pimd_ctx* ctx, int M, int N, int K, const float* A, const float* Bt, float* C) {
    if (!ctx || !A || !Bt || !C || M <= 0 || N <= 0 || K <= 0) return fail(ctx, PIMD_EINVAL, "bad argument");
    float *dA = nullptr, *dB = nullptr, *dC = nullptr;
    CK(cudaMalloc(&dA, sizeof(float) * (size_t)M * K));
    CK(cudaMalloc(&dB, sizeof(float) * (size_t)N * K));
    CK(cudaMalloc(&dC, sizeof(float) * (size_t)M * N));
    CK(cudaMemcpyAsync(dA, A, sizeof(float) * (size_t)M * K, cudaMemcpyHostToDevice, ctx->stream));
    CK(cudaMemcpyAsync(dB, Bt, sizeof(float) * (size_t)N * K, cudaMemcpyHostToDevice, ctx->stream));
    CK(cudaMemsetAsync(dC, 0xFF, sizeof(float) * (size_t)M * N, ctx->stream));
    const int rc = debug_tc_gemm(M, N, K, dA, dB, dC, ctx->stream);
    ctx->launches += 1;
    cudaError_t e = cudaStreamSynchronize(ctx->stream);
    if (rc == 0 && e == cudaSuccess) e = cudaMemcpy(C, dC, sizeof(float) * (size_t)M * N, cudaMemcpyDeviceToHost);
    cudaFree(dA); cudaFree(dB); cudaFree(dC);
    if (rc != 0) return fail(ctx, PIMD_EINVAL, "debug gemm: unsupported shape or tensor-map failure");
    if (e != cudaSuccess) return fail(ctx, PIMD_ECUDA, std::string("debug gemm: ") + cudaGetErrorString(e));
    return PIMD_OK;
}

int pimd_debug_graph_state(const pimd_ctx* ctx) {
    if (!ctx) return PIMD_EINVAL;
    return ctx->step_graph ? 1 : (ctx->graph_failed ? -100 : 0);
}

int pimd_set_profiling(pimd_ctx* ctx, int on) {
    if (!ctx) return PIMD_EINVAL;
    ctx->profiling = on != 0;
    return PIMD_OK;
}
int pimd_get_phase_ms(pimd_ctx* ctx, double ms[6]) {
    if (!ctx || !ms) return PIMD_EINVAL;
    for (int q = 0; q < 6; ++q) ms[q] = ctx->phase_ms[q];
    return PIMD_OK;
}

}  // extern "C"
