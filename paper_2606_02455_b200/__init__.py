"""B200-native (sm_100a) hot path of Langevin Speculative Dynamics: thin Python binding of liblsd_b200.so.

Every step of the path runs in the CUDA kernels behind the C ABI declared in include/lsd.h; this package only
marshals arguments.  There is no CPU fallback: importing works anywhere (the symbol table can be inspected),
but creating a context without the built library or without a CUDA device raises.
"""
from .api import (  # noqa: F401
    LsdError, Context, load_library, library_path, lsd_init, lsd_destroy, lsd_draft_rollout, lsd_verify_window,
    lsd_transport_accept, lsd_rollback, lsd_run, lsd_get_state, lsd_set_state, lsd_get_stats, lsd_get_window_state,
    lsd_get_window_debug, lsd_eval_forces, lsd_get_neighbors, lsd_set_skin, lsd_launch_count, lsd_version, lsd_profile, lsd_get_profile, lsd_get_edge_count, lsd_tc_enabled, lsd_tiny_rollout_enabled, lsd_set_window_slots,
    lsd_set_error_correction, lsd_get_ec_cache, lsd_set_ec_cache, lsd_plain_langevin, lsd_get_adaptive_k, lsd_get_window_obabo,
    lsd_get_edge_launch_info, lsd_measure_fma_peak, lsd_set_force_slack,
    lsd_transport_window_noalloc, LSD_NOALLOC_MAX_K, LSD_NOALLOC_MAX_ATOMS,
    context_from_workload, EXPORTED_SYMBOLS, LSD_FP32, LSD_BF16_TC, LSD_DRAFT, LSD_TARGET, LSD_HOST, LSD_DEVICE,
)
