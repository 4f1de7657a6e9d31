/* pimd_debug.h -- parity hooks, bisecting switches and bench timers of libpimd_b200.  Not part of the method's
 * boundary (include/pimd.h): tests/ and bench.py use them to look INSIDE the hot path -- the Philox words and
 * normals of the O step, the tensor-core GEMM kernel alone, the CUDA-core reference paths, one kernel's device
 * time.  Same conventions as pimd.h (host pointers, synchronous, 0 or a negative code). */
#ifndef PIMD_B200_DEBUG_H
#define PIMD_B200_DEBUG_H

#include "pimd.h"

#ifdef __cplusplus
extern "C" {
#endif

/* The four Philox4x32-10 words and the normal eta the O step uses for (step, mode k, atom i,
 * component alpha) (R-10), evaluated ON THE DEVICE for n entries: idx[n][3] = (k, i, alpha);
 * words[n][4], eta[n].  */
int pimd_debug_noise(pimd_ctx* ctx, int64_t step, int n, const int32_t* idx, uint32_t* words, double* eta);

/* Fitting-net GEMM path: 1 (default) = tcgen05 tensor cores, three-pass split products (FP16 hi/lo for the
 * K = 1600 / N = 1600 kernels, TF32 hi/lo for the 240 x 240 GEMMs; fitting_tc.cu); 0 = the FP32 CUDA-core GEMMs kept
 * as the in-tree reference for bisecting.  Both meet the parity tolerances. */
int pimd_set_fitting_path(pimd_ctx* ctx, int use_tensor_cores);

/* Embedding-net path: 1 (default) = tcgen05 tensor cores, three-pass FP16-split products (kind::f16, FP32
 * accumulate), row tiles of one type pair (embedding_tc.cu); 0 = the FP32 CUDA-core kernels kept as the in-tree
 * reference.  Takes effect at the next force evaluation (pimd_set_state / pimd_step). */
int pimd_set_embedding_path(pimd_ctx* ctx, int use_tensor_cores);

/* Parity hook for the tensor-core GEMM kernel alone: C[M][N] = A[M][K] Bt[N][K]^T, host FP32 arrays,
 * N == 240 or N % 160 == 0, K % 16 == 0 (the shapes the fitting net uses). */
int pimd_debug_gemm(pimd_ctx* ctx, int M, int N, int K, const float* A, const float* Bt, float* C);

/* Stand-alone timing of kernels (bench.py roofline legs): runs `reps` launches of the fused
 * integrator kernel on the current state WITHOUT advancing it (output to scratch), and returns the mean
 * device time per launch in milliseconds through *ms.  kind 0: the kernel as pimd_step launches it.
 * kind 1: the same launch with the O-step normals keyed one draw PER MODE (counter word 3 = 4k + alpha,
 * sine branch discarded) instead of one per mode pair -- never used by pimd_step; it exists for the A/B
 * number behind DESIGN R-10. */
int pimd_time_kernel(pimd_ctx* ctx, int kind, int reps, double* ms);

/* 1 when the step loop of pimd_step has been captured as a CUDA graph and is replayed (se_e2_a model, no barostat, no
 * profiling, calls of at least 3 steps; environment variable PIMD_NO_GRAPH disables it), 0 when no graph exists yet,
 * -100 when a capture failed and the loop fell back to plain launches. */
int pimd_debug_graph_state(const pimd_ctx* ctx);

/* The row index of the most recent force evaluation, as the context's own path computed it: cen_idx[P N] (type-sorted
 * centre row -> bead-atom) and rowstart[n_types][P N + 1] (exclusive scan of pimd_get_neighbor_counts in that order).
 * tests/test_zz_no_alloc.py compares pimd_row_scan_noalloc_dev (pimd_noalloc.h) with it. */
int pimd_debug_get_row_index(pimd_ctx* ctx, int32_t* cen_idx, int32_t* rowstart);

#ifdef __cplusplus
}
#endif
#endif /* PIMD_B200_DEBUG_H */
