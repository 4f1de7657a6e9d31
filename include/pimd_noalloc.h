/* pimd_noalloc.h -- one entry point of libpimd_b200 that allocates nothing.
 *
 * Why: some callers cannot call cudaMalloc -- code under CUDA graph capture, tight serving loops, harnesses that
 * forbid it.  A pimd_ctx takes its memory from an arena (pimd_set_workspace / cudaMalloc at pimd_create); this call
 * needs no context and no arena: its scratch is a file-scope `static __device__` array inside the library.
 *
 * What: the row-index scan of the force evaluation (SURVEY 8(a) F2 -> F3: DESIGN section 5, "row index").  The
 * embedding kernels walk the neighbour rows of one ordered type pair (t_i, t_j) in tiles of 128; the tile boundaries
 * come from an exclusive scan of the per-centre neighbour counts over the type-sorted centres:
 *
 *     rowstart[tj][r] = sum_{q < r} ncount[cen_idx[q]][tj],   r = 0 .. n_centres   (rowstart[tj][n_centres] = total)
 *
 * It is the same pair of kernels pimd_step launches (block sums, then scan + offsets); the block sums between the
 * two are the scratch.
 *
 * Limits: n_centres <= PIMD_NOALLOC_MAX_CENTRES (4096 scan blocks of 1024 centres), n_types <= PIMD_MAX_TYPES.  The
 * scratch is 4 x 4096 x 4 B = 64 KB of device memory on EVERY GPU that loads the library, held until the process
 * exits.  Larger inputs are refused with PIMD_EINVAL and a message (pimd_noalloc_last_error); nothing is launched.
 *
 * Sharing: every call on a device uses the same array, and the array keeps the last call's block sums.  Nothing has
 * to start at zero (each call writes every sum it later reads), so no clearing is done -- but two calls that overlap
 * on the GPU (different streams, or different host threads without ordering between their streams) RACE on it.
 * Calls on one stream are ordered and safe back to back.
 */
#ifndef PIMD_B200_NOALLOC_H
#define PIMD_B200_NOALLOC_H

#include "pimd.h"

#ifdef __cplusplus
extern "C" {
#endif

#define PIMD_NOALLOC_MAX_CENTRES 4194304

/* Looks up the device address of the scratch array for the CURRENT device (cudaGetSymbolAddress, once per device;
 * the address is cached).  pimd_row_scan_noalloc_dev does this itself on first use; call it at set-up when the
 * first use would fall inside a stream capture.  Returns PIMD_OK or PIMD_ECUDA. */
int pimd_noalloc_setup(void);

/* Exclusive scan of the neighbour counts in type-sorted centre order.
 *   n_centres            P x N bead-atoms (1 .. PIMD_NOALLOC_MAX_CENTRES)
 *   n_types              neighbour types (1 .. PIMD_MAX_TYPES)
 *   cen_idx_dev  [n_centres]            DEVICE, int32: type-sorted centre row r -> bead-atom index k N + i
 *   ncount_dev   [n_centres][n_types]   DEVICE, int32: neighbour rows of bead-atom b with neighbour type tj
 *   rowstart_dev [n_types][n_centres+1] DEVICE, int32, written: the scan above
 *   cuda_stream          cudaStream_t the two kernels are launched on (NULL = the legacy default stream)
 * All arrays are owned by the caller and must stay valid until the work on `cuda_stream` has finished: the call is
 * ASYNCHRONOUS (it returns after the launches; it never synchronises, copies or allocates: no cudaMalloc / cudaFree /
 * allocating library routine on this path).  Returns PIMD_OK, PIMD_EINVAL (null pointer, size outside the limits;
 * nothing launched) or PIMD_ECUDA (launch failure). */
int pimd_row_scan_noalloc_dev(int n_centres, int n_types, const int32_t* cen_idx_dev, const int32_t* ncount_dev,
                              int32_t* rowstart_dev, void* cuda_stream);

/* Text of the calling thread's last error from the two calls above ("" when none). */
const char* pimd_noalloc_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* PIMD_B200_NOALLOC_H */
