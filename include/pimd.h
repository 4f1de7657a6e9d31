/* pimd.h -- C ABI of libpimd_b200: one ring-polymer PIMD/Langevin BAOAB step for all P beads of an
 * N-atom system resident on one B200 (sm_100a), with a Deep-Potential se_e2_a force model.
 *
 * The calls follow the problem statement of arxiv/paper_2602_13553 ("fix pimd/langevin"), cited as
 * PAPER.md:Lnnn (= /root/reference/PAPER.md), and BASELINE.json's north_star
 * ("pimd_create with types, masses, box, P, T, dt, gamma and seed; pimd_set_model with the weights;
 * pimd_step(n); getters for positions, momenta, forces, virial and estimators").
 * Readings of garbled / silent passages are DESIGN.md section 3 (R-1 .. R-16).
 *
 * Conventions (all calls):
 *   - Units: Angstrom, ps, eV, g/mol, K (LAMMPS "metal"; the paper's worked constants PAPER.md:L458).
 *   - Unless a name ends in _dev, every array pointer is a HOST pointer owned by the caller; the
 *     library copies in / out and is synchronous on return.  _dev variants take DEVICE pointers that
 *     must stay valid until the call returns; work is issued on the context's stream and the call
 *     returns after that work is complete.
 *   - Layout of per-bead per-atom vectors: [P][N][3], C order, double.
 *   - Return value: 0 (PIMD_OK) or a negative code; the text of the last error of a context is
 *     available from pimd_last_error().  No C++ exception crosses this boundary.
 *   - A context is not thread-safe; use one context per host thread.
 *   - The library runs on the current CUDA device at pimd_create() time.  It has no CPU fallback:
 *     without a CUDA device pimd_create() returns PIMD_ECUDA.
 */
#ifndef PIMD_B200_H
#define PIMD_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define PIMD_OK              0
#define PIMD_EINVAL         -1   /* bad argument (null pointer, non-positive size, unsupported P, ...) */
#define PIMD_ENOSTATE       -2   /* pimd_set_state has not been called */
#define PIMD_ENOMODEL       -3   /* no force model has been set */
#define PIMD_ESEL_OVERFLOW  -4   /* an atom has more neighbours of one type than sel allows (R-11), or the cell outran
                                  * its cell grid inside one call.  From pimd_step: the call is undone as a whole (x, p, f,
                                  * U, Xi, cell and step counter are those at entry; the message names the failing step).
                                  * From pimd_set_state / pimd_set_model / pimd_set_barostat: the context is left WITHOUT
                                  * a state (the forces of a truncated neighbour list are not kept); set a new one. */
#define PIMD_ECUDA          -5   /* CUDA runtime error; see pimd_last_error */
#define PIMD_ENOMEM         -6   /* the caller-supplied workspace is too small */
#define PIMD_ECONTACT       -8   /* two atoms closer than 0.01 A (s = 1/r > 100): outside the range the fixed FP16 operand
                                  * scales of the descriptor / fitting kernels assume.  Reported like PIMD_ESEL_OVERFLOW. */
#define PIMD_ETABLE_RANGE   -7   /* compressed embedding: a neighbour row lies outside the table (s > 2, r < 0.5 A; R-28).
                                  * Reported like PIMD_ESEL_OVERFLOW (pimd_step rolls the call back). */

typedef struct pimd_ctx pimd_ctx;   /* opaque; owned by the library */

/* se_e2_a architecture (R-11..R-16; BASELINE.json configs[0]). */
#define PIMD_MAX_TYPES 4
typedef struct pimd_model_desc {
    double  rcut;                       /* cutoff radius r_c, Angstrom */
    double  rcut_smth;                  /* start of the smooth switch r_s */
    int32_t n_types;
    int32_t sel[PIMD_MAX_TYPES];        /* max neighbours per neighbour type; N_sel = sum */
    int32_t embed[3];                   /* embedding widths, each layer out = 2*in after the first: {25,50,100} */
    int32_t axis_neuron;                /* M2 (16) */
    int32_t fit[3];                     /* fitting hidden widths, all equal: {240,240,240} */
} pimd_model_desc;

/* Estimators of PAPER.md Appendix A (L319-365) after the last completed step, in eV (T_ring in K). */
typedef struct pimd_estimators {
    double  K_PR;     /* primitive kinetic-energy estimator, Eq. A7 (L354) with R-6 */
    double  K_CV;     /* centroid-virial kinetic-energy estimator, Eq. A9 (L365) */
    double  H;        /* total ring-polymer energy sum_k K+S+U, Eq. A6 (L350) */
    double  K_ring;   /* sum_k K^(k), Eq. A1 (L319) */
    double  S_ring;   /* sum_k S^(k), Eq. A3 (L330) */
    double  U_sum;    /* sum_k U^(k), Eq. A5 (L343) */
    double  T_ring;   /* 2 K_ring / (3 P N k_B); averages P*T (L194, L120) */
    int64_t step;     /* completed steps since pimd_set_state */
} pimd_estimators;

/* ---- lifetime ------------------------------------------------------------------------------- */

/* Creates a context for N atoms with P beads (Eq. 1: the ring-polymer Hamiltonian).
 *   types[N]         atom types 0..n_types-1            masses[n_types]  g/mol
 *   box[3]           orthorhombic periodic box lengths, Angstrom
 *   n_beads          P: 1, 2, 4, 8, 16, 32 or 64 (power of two; the transform is an in-register FFT)
 *   T                target temperature in K; the ring is sampled at P*T (L194)
 *   dt               time step in ps
 *   gamma_centroid   centroid friction 1/tau in 1/ps (keyword `tau`, L174); 0 = NVE, no O step (R-4)
 *   seed             Philox key (R-10)
 * On success *out holds the context.  Device memory is allocated with cudaMalloc unless
 * pimd_set_workspace() hands the library a buffer (e.g. from PyTorch's caching allocator). */
int pimd_create(pimd_ctx** out, int n_atoms, const int32_t* types, int n_types, const double* masses,
                const double box[3], int n_beads, double T, double dt, double gamma_centroid,
                uint64_t seed);
void pimd_destroy(pimd_ctx* ctx);
const char* pimd_last_error(const pimd_ctx* ctx);   /* never NULL; "" when there was no error */

/* Optional plumbing: the caller lends device memory and a stream (cudaStream_t as void*; NULL = the
 * legacy default stream).  pimd_workspace_bytes returns the bytes needed for this context including
 * the buffers of the se_e2_a model `d`.  Must be called before pimd_set_state / pimd_set_model*.  The buffer
 * (256-byte aligned) stays owned by the caller and must outlive the context. */
size_t pimd_workspace_bytes(const pimd_ctx* ctx, const pimd_model_desc* d /* NULL: harmonic model only */);
int pimd_set_workspace(pimd_ctx* ctx, void* workspace_dev, size_t bytes, void* cuda_stream);

/* ---- inputs --------------------------------------------------------------------------------- */

/* x[P][N][3] unwrapped Cartesian bead positions (L202); p[P][N][3] Cartesian bead momenta in
 * (g/mol) A/ps.  Resets the step counter to 0.  If a model is set, evaluates the initial forces
 * (BAOAB opens with a B that needs f(x0)). */
int pimd_set_state(pimd_ctx* ctx, const double* x, const double* p);

/* Resume from a checkpoint {x, p, f, U, step} (host arrays; SURVEY section 5 "checkpoint / resume"):
 * like pimd_set_state, but the forces f[P][N][3] and bead energies U[P] that belong to x are supplied,
 * so no force evaluation is run, and the step counter (which keys the Philox noise, R-10) is set to
 * `step`.  Because the noise is counter-based, restore + pimd_step(n) draws exactly the random numbers the
 * uninterrupted run would have drawn.  With the harmonic model the continued trajectory is bit-identical; with the
 * se_e2_a model the forces, U and the estimator sums are accumulated with floating-point atomics whose order is not
 * fixed, so two runs (restored or not) agree to rounding (~1e-16 relative per evaluation), not bit for bit.
 * A model must already be set. */
int pimd_restore(pimd_ctx* ctx, const double* x, const double* p, const double* f, const double* U, int64_t step);

/* The se_e2_a Deep-Potential model (PAPER.md:L47, L76 cite it; definition DESIGN.md R-11..R-16).
 * weights: n_weights doubles, row-major W[in][out] then bias[out] per layer, in the order
 *   for t_i: for t_j: embedding layers 1..3;  then for t_i: fitting layers 1..4 (last out = 1).
 * n_weights must equal pimd_model_n_weights(d).  The library converts to FP32 on the device.  Every weight must be
 * finite and at most 1000 in magnitude (the tensor-core kernels use FP16 hi / lo operand pairs with fixed scales):
 * PIMD_EINVAL otherwise. */
size_t pimd_model_n_weights(const pimd_model_desc* d);
int pimd_set_model(pimd_ctx* ctx, const pimd_model_desc* d, const double* weights, size_t n_weights);

/* Compressed ("tabulated") embedding net -- the model variant the paper's own runs use ("We use a
 * compressed DP model", L262; ref. 41 is only cited, so DESIGN R-28 fixes the table: per ordered type pair, G(s) on the
 * uniform grid s in [0, 2] with stride 0.05 is replaced by the quintic Hermite polynomial matching G, G', G'' at both
 * nodes of each interval; the backward pass differentiates the same polynomial, so forces remain the exact gradient of
 * the compressed energy).  on = 1 builds the tables from the weights given to pimd_set_model (FP64 on the host) and
 * switches the embedding steps F3 / F5 to them; on = 0 returns to the MLP.  The forces of the current state are
 * re-evaluated.  It is an APPROXIMATION of the MLP model (|G~ - G| <= 3e-8 at this stride) and is compared with the
 * oracle's compressed model.  PIMD_ENOMODEL before pimd_set_model; PIMD_EINVAL for more than two atom types.
 * A row with s > 2 (an atom pair closer than 0.5 A) is an error: PIMD_ETABLE_RANGE. */
int pimd_set_embedding_compressed(pimd_ctx* ctx, int on);

/* Test model: U = sum_i 1/2 k |r_i|^2 about the origin on the unwrapped coordinates (FP64), used to
 * check the integrator alone against closed forms (north_star's harmonic-oscillator check). */
int pimd_set_model_harmonic(pimd_ctx* ctx, double k_spring /* eV/A^2 */);

/* ---- the hot path --------------------------------------------------------------------------- */

/* n_steps BAOAB steps: B(dt/2) A(dt/2) O(dt) A(dt/2) [force] B(dt/2), with the three
 * normal-mode transforms of L192 and one force evaluation per step (R-7).  All work runs on the
 * GPU; there is no host round trip inside the loop.  Errors are detected when the call ends: on
 * PIMD_ESEL_OVERFLOW the whole call is rolled back (see the code's comment above), so the caller can retry with
 * a larger sel, fewer steps per call (barostat) or stop; the state is never left half-advanced. */
int pimd_step(pimd_ctx* ctx, int64_t n_steps);

/* ---- outputs -------------------------------------------------------------------------------- */
int pimd_get_positions(pimd_ctx* ctx, double* x /* [P][N][3] A, unwrapped */);
int pimd_get_momenta(pimd_ctx* ctx, double* p /* [P][N][3] Cartesian, (g/mol) A/ps */);
int pimd_get_forces(pimd_ctx* ctx, double* f /* [P][N][3] eV/A */);
int pimd_get_virial(pimd_ctx* ctx, double* xi /* [P][9] eV; Xi_ab = -sum_rows d_a dU/dd_b (L372, R-16) */);
int pimd_get_energies(pimd_ctx* ctx, double* U /* [P] eV, bead potential energies (A5, L343) */);
int pimd_get_atom_energies(pimd_ctx* ctx, double* E /* [P][N] eV, E_i of the fitting net */);
int pimd_get_estimators(pimd_ctx* ctx, pimd_estimators* e);
/* Estimators of each of the last `n` completed steps of the most recent pimd_step call, oldest first
 * (configs[1]: "estimators reported every step").  Returns the number written (<= cap) or < 0. */
int pimd_get_estimator_history(pimd_ctx* ctx, pimd_estimators* e, int cap);

/* Device-pointer variants for callers that keep the state in HBM (bench.py's resident-input leg). */
int pimd_set_state_dev(pimd_ctx* ctx, const double* x_dev, const double* p_dev);
int pimd_get_positions_dev(pimd_ctx* ctx, double* x_dev);
int pimd_get_forces_dev(pimd_ctx* ctx, double* f_dev);

/* ---- parity hooks (more of them, and the bench / bisecting switches, in pimd_debug.h) -------- */

/* Neighbour rows of one bead from the most recent force evaluation, in canonical order: for atom i
 * the rows sorted by (type_j, j, n_x, n_y, n_z).  count[N] receives the rows per atom; j[cap] and
 * shift[cap][3] (periodic image n of R-11) receive the concatenated rows.  Returns the total number
 * of rows, or PIMD_EINVAL when cap is too small. */
int64_t pimd_get_neighbors(pimd_ctx* ctx, int bead, int32_t* count, int32_t* j, int8_t* shift, size_t cap);

/* Neighbour rows per bead-atom and neighbour type from the most recent force evaluation:
 * counts[P][N][n_types] (host).  bench.py uses the total to state the algorithmic work. */
int pimd_get_neighbor_counts(pimd_ctx* ctx, int32_t* counts);

/* Number of kernels of this library launched on the context so far (the bench's gpu_launches). */
int64_t pimd_get_launch_count(const pimd_ctx* ctx);

/* Trotter splitting of the step ("integrator"): PIMD_BAOAB (default here; north_star's path) or
 * PIMD_OBABO (the fix's own default): O(dt/2) B(dt/2) A(dt) B(dt/2) O(dt/2), each O with c1 = exp(-gamma_k dt/2)
 * and its own normals (bit 31 of Philox counter word 1 marks the second half-step; DESIGN R-3, R-10).  Both run
 * in the same fused kernel, one launch per step.  Returns PIMD_EINVAL for an unknown kind.  May be changed
 * between pimd_step calls. */
#define PIMD_BAOAB 0
#define PIMD_OBABO 1
int pimd_set_integrator(pimd_ctx* ctx, int kind);

/* Coordinate system of the integration (keyword `method`).  PIMD_NMPIMD (default): normal modes, the
 * north_star path.  PIMD_CART (`method pimd`): Cartesian coordinates -- B kicks with the bead force plus the ring-spring
 * force of Eq. 1, A is the drift x += h v, and the thermostat is Eq. D3 (L478-484): the same tau = 1/(2 omega_n) on
 * every bead, normals keyed by the bead index (DESIGN R-27); both splittings; estimators as in Appendix A.  Call it
 * BEFORE pimd_set_state: a change of method drops the state (the stored velocities change representation).
 * PIMD_EINVAL for an unknown method, or for PIMD_CART with a barostat on (and the barostat refuses under PIMD_CART).
 * fixcom under PIMD_CART removes the centre-of-mass velocity of EACH BEAD. */
#define PIMD_NMPIMD 0
#define PIMD_CART 1
int pimd_set_method(pimd_ctx* ctx, int method);

/* `fixcom`: when on, the centre-of-mass velocity of the centroid mode (PIMD_NMPIMD) or of every bead
 * individually (PIMD_CART) is removed once per step,
 * after the step's last velocity update and before its estimators (DESIGN R-19).  Off by default (north_star's
 * create() list has no such argument).  The removal needs a reduction over all atoms between the closing and the
 * opening half of the fused integrator launch, so a step then costs two integrator launches instead of one. */
int pimd_set_fixcom(pimd_ctx* ctx, int on);

/* Isotropic BZP barostat (Appendix E Eq. E1, E4-E7, L488-522; keywords `iso`, `barostat BZP`, `taup`,
 * L176-179): the cell gets one velocity v_W with mass W = 3 n N k_B T tau_p^2 (L389), driven by the centroid-virial
 * pressure P_CV (Eq. A12) against p_ext_bar (bar; 1 eV/A^3 = 1.602176634e6 bar, DESIGN R-25).  With
 * gamma_centroid = 0 this is the NpH ensemble (the enthalpy of Eq. A17 is conserved); with gamma_centroid > 0 the
 * cell velocity is thermostatted by Eq. E7 next to PILE_L on the atoms: NpT.  Sub-step order DESIGN R-24; the
 * centroids scale with the cell, internal modes do not (R-21).  v_W starts at 0 and is reset by every call.  The
 * cell then lives on the device and is rescaled every step (Eq. E6); the neighbour list is rebuilt from the
 * current cell at every force evaluation.  Works with both splittings (PIMD_OBABO + npt is the paper's own example,
 * L82): the cell's sub-steps sit next to the atomic sub-steps of the same letter.  Returns PIMD_EINVAL with fixcom
 * on (and pimd_set_fixcom refuses while a barostat is on), and for tau_p <= 0.
 * If the cell shrinks by more than a few per cent inside ONE pimd_step call so that r_c no longer fits the cell
 * grid chosen at the start of the call, the call returns PIMD_ESEL_OVERFLOW (call with fewer steps). */
int pimd_set_barostat(pimd_ctx* ctx, double p_ext_bar, double tau_p);

/* Anisotropic variant (keyword `aniso`; Eq. E2-E3; Eq. A14): one cell velocity v_W,alpha
 * per Cartesian component, each driven by its own diagonal element of the centroid-virial stress tensor against the
 * same p_ext_bar, barostat mass W = n N k_B T tau_p^2 (L397), one thermostat normal per component (E7).  The cell
 * stays orthorhombic.  Same rules and errors as pimd_set_barostat; the later of the two calls wins. */
int pimd_set_barostat_aniso(pimd_ctx* ctx, double p_ext_bar, double tau_p);

/* Checkpoint / resume under a barostat: restores the cell lengths, the cell velocities (three equal values in
 * isotropic mode) and the bead virials xi[P][9] that belong to the checkpointed positions (the first E1 of the next
 * step needs them; pimd_restore carries x, p, f, U and the step counter).  Call after pimd_set_barostat[_aniso]
 * and around pimd_restore; restore + pimd_step(n) then continues the trajectory as the uninterrupted run would,
 * up to the rounding noted at pimd_step (a call boundary re-reads the kicked velocities).  PIMD_EINVAL without a
 * barostat or for a non-positive length. */
int pimd_restore_cell(pimd_ctx* ctx, const double box[3], const double v_W[3], const double* xi);

/* Barostat outputs after the last completed step (Appendix A outputs 8-15); pressures in bar,
 * energies in eV, lengths in Angstrom.  PIMD_EINVAL when no barostat is set. */
typedef struct pimd_barostat_state {
    double v_W;       /* cell velocity, 1/ps (output 11) */
    double box[3];    /* current cell lengths (Eq. E6) */
    double V;         /* box[0] box[1] box[2] */
    double P_CV;      /* centroid-virial pressure, Eq. A12 */
    double P_PR;      /* primitive pressure, Eq. A10 (omega_n squared as in A7, R-6) */
    double P_MD;      /* pressure of the extended classical system, Eq. A11 */
    double K_W;       /* W v_W^2 / 2, Eq. A13; anisotropic: sum over the three components, Eq. A14 */
    double U_W;       /* n P_ext V, Eq. A15 */
    double J_W;       /* -n k_B T ln V, Eq. A16 */
    double enthalpy;  /* H + K_W + U_W + J_W, Eq. A17 */
    double v_W3[3];   /* cell velocity per component (all equal to v_W in isotropic mode; v_W is their mean) */
    double P_CV3[3];  /* diagonal of the centroid-virial stress tensor, Eq. E3 (P_CV is its mean) */
} pimd_barostat_state;
int pimd_get_barostat(pimd_ctx* ctx, pimd_barostat_state* b);
/* The same outputs for each of the last `n` completed steps of the most recent pimd_step call, oldest first (the
 * barostat companion of pimd_get_estimator_history; at most 4096 steps per call are recorded).  Returns the number
 * written (<= cap) or < 0. */
int pimd_get_barostat_history(pimd_ctx* ctx, pimd_barostat_state* b, int cap);

/* Mean device milliseconds per step of each phase of the last pimd_step call, when profiling was
 * enabled with pimd_set_profiling(ctx, 1) (CUDA events on the context's stream):
 * ms[0] integrator, [1] neighbour+environment, [2] embedding fwd, [3] descriptor+fitting fwd/bwd,
 * [4] embedding bwd + force/virial, [5] reserved. */
int pimd_set_profiling(pimd_ctx* ctx, int on);
int pimd_get_phase_ms(pimd_ctx* ctx, double ms[6]);

#ifdef __cplusplus
}
#endif
#endif /* PIMD_B200_H */
