"""paper_2606_27086_b200 -- B200-native (sm_100a) superiorized simultaneous projection over hyperslabs + box.

The product is the C-ABI library libsup.so (include/sup.h; sources in csrc/).  This package is the thin Python
binding: argument marshalling only, every step of the path runs in the CUDA kernels.  PyTorch is used for device
memory and streams.  There is no CPU fallback: without the compiled library or without a CUDA device the calls fail.
"""
from .binding import (  # noqa: F401
    SupError,
    SupHandle,
    lib,
    sup_apply_update,
    sup_backproject_partial,
    sup_backproject_update,
    sup_block_iterative,
    sup_forward_violation,
    sup_create,
    sup_destroy,
    sup_get_state,
    sup_objective,
    sup_perturb_dose,
    sup_perturb_adaptive,
    sup_set_dose_mode,
    sup_set_perturb_mode,
    sup_perturb_mean,
    sup_project_drop,
    sup_project_emr,
    sup_perturb_tv,
    sup_project_simultaneous,
    sup_proximity,
    sup_set_blocks,
    sup_set_dose_matrix,
    sup_set_layout,
    sup_set_row_mode,
    sup_superiorize,
    sup_superiorize_host,
    sup_tv2d_value_static,
    sup_workspace_bytes,
    OBJ_NONE, OBJ_TV2D, OBJ_TV1D, OBJ_DOSE, OBJ_MEAN, OBJ_TV3D, PER_TRIAL, PER_SWEEP, F32, F64,
)
