"""B200-native (sm_100a) RPIM stiffness assembly + penalty BCs: thin binding over librpim.so.

The product is the C-ABI library declared in ``include/rpim.h`` (hand-written CUDA kernels);
this package only marshals arguments (``binding.py``).  PyTorch is used for device memory and
streams.  There is no CPU fallback: importing ``binding`` without the built library raises.
"""
from .binding import (  # noqa: F401
    Context,
    RpimError,
    library_path,
    rpim_create,
    rpim_destroy,
    rpim_build_pattern,
    rpim_get_pattern,
    rpim_assemble,
    rpim_add_point_loads,
    rpim_apply_penalty,
    rpim_apply_penalty_static,
    rpim_apply_penalty_static_max_nodes,
    rpim_get_shape,
    rpim_host_pattern,
    rpim_host_assemble,
    rpim_last_phase_ms,
    rpim_phase_totals,
    rpim_launch_count,
    rpim_matvec,
    rpim_set_panel_shape,
    rpim_solve_pcg,
    rpim_recover_stress,
    rpim_workspace_bytes,
    rpim_last_error,
    EXPORTED_SYMBOLS,
    RPIM_INDEX_MIXED,
)
