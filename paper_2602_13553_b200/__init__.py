"""paper_2602_13553_b200 -- B200-native hot path of "fix pimd/langevin" (arxiv/paper_2602_13553):
one ring-polymer PIMD/Langevin BAOAB step for all beads of a water box with an se_e2_a Deep-Potential
force model, as hand-written CUDA for sm_100a behind the C ABI of include/pimd.h.

This package is argument marshalling only (ctypes); every step of the path runs in the kernels of
csrc/*.cu.  There is no CPU fallback: importing works without a GPU (so the symbol table can be
checked), but every compute call needs the compiled library and a CUDA device.
"""
from .binding import (  # noqa: F401
    PIMD_OK, PIMD_EINVAL, PIMD_ENOSTATE, PIMD_ENOMODEL, PIMD_ESEL_OVERFLOW, PIMD_ECUDA, PIMD_ENOMEM,
    PIMD_ETABLE_RANGE, PIMD_ECONTACT, pimd_set_embedding_compressed,
    PimdError, ModelDesc, Estimators, lib, library_path,
    pimd_create, pimd_destroy, pimd_last_error, pimd_workspace_bytes, pimd_set_workspace,
    pimd_set_state, pimd_set_state_dev, pimd_model_n_weights, pimd_set_model, pimd_set_model_harmonic,
    pimd_step, pimd_get_positions, pimd_get_momenta, pimd_get_forces, pimd_get_virial, pimd_get_energies,
    pimd_get_atom_energies, pimd_get_estimators, pimd_get_estimator_history, pimd_get_positions_dev,
    pimd_get_forces_dev, pimd_get_neighbors, pimd_debug_noise, pimd_time_kernel, pimd_set_profiling,
    pimd_get_phase_ms, pimd_restore, pimd_get_neighbor_counts, pimd_get_launch_count, pimd_set_fitting_path,
    pimd_set_embedding_path, pimd_set_integrator, pimd_set_fixcom, PIMD_BAOAB, PIMD_OBABO,
    pimd_set_method, PIMD_NMPIMD, PIMD_CART, pimd_set_barostat, pimd_set_barostat_aniso, pimd_get_barostat, pimd_get_barostat_history, pimd_restore_cell, BarostatState,
    pimd_debug_gemm, pimd_debug_graph_state, PIMD,
    pimd_debug_get_row_index, pimd_noalloc_setup, pimd_noalloc_last_error, pimd_row_scan_noalloc_dev,
)
