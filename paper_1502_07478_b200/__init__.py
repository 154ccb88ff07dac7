"""B200-native (sm_100a) list-mode MLEM hot path for the two-strip J-PET detector (arXiv:1502.07478).

The product is the C-ABI library of include/jpet.h (CUDA kernels in csrc/); `binding` is its ctypes
front end with the same names, `synth` the seeded input generator, `build` the nvcc build step.
"""
from .binding import (  # noqa: F401
    JpetError,
    jpet_abi_version,
    jpet_count_evals,
    jpet_direct_histogram,
    jpet_generate_events,
    jpet_get_a3_coef,
    jpet_get_counters,
    jpet_get_gamma,
    jpet_get_option,
    jpet_get_sigma_z_edge,
    jpet_ipc_close,
    jpet_ipc_export,
    jpet_ipc_open,
    jpet_last_error,
    jpet_launch_count,
    jpet_plan_describe,
    jpet_mlem_accumulate,
    jpet_mlem_accumulator,
    jpet_mlem_begin,
    jpet_mlem_end,
    jpet_mlem_end_peers,
    jpet_mlem_iterate,
    jpet_mlem_iterate_host,
    jpet_reconstruct,
    jpet_reconstruct_host,
    jpet_release,
    jpet_sensitivity,
    jpet_set_a3_coef,
    jpet_set_gamma,
    jpet_set_option,
    jpet_set_sigma_z_edge,
    jpet_shape_name,
)
