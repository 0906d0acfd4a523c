"""B200-native CETRA hot path (arXiv 2503.20875): linear transit search + periodic search.

The product is the C-ABI library `libcetra_b200.so` (include/cetra.h, hand-written sm_100a CUDA
kernels under csrc/); this package is its thin ctypes binding.  PyTorch supplies device memory and
streams only.  There is no CPU fallback and nothing here imports the test oracle.
"""
from .binding import (  # noqa: F401
    CETRA_ERR_CUDA,
    CETRA_ERR_INVALID_ARG,
    CETRA_ERR_NONUNIFORM_TIMES,
    CETRA_ERR_UNSUPPORTED,
    CETRA_ERR_WORKSPACE,
    CETRA_F32,
    CETRA_F64,
    CETRA_OK,
    EXPORTED_SYMBOLS,
    PEAK_DTYPE,
    CetraError,
    LinearResult,
    cetra_device_info,
    cetra_kernel_launch_count,
    cetra_linear_search,
    cetra_linear_workspace_bytes,
    cetra_periodic_search,
    cetra_profile_enable,
    cetra_profile_read,
    cetra_periodic_search_stats,
    cetra_periodic_workspace_bytes,
    cetra_search_batched,
    cetra_search_batched_host,
    cetra_search_batched_host_workspace_bytes,
    cetra_search_batched_workspace_bytes,
    cetra_stats_pitch,
    load_library,
    peaks_to_numpy,
    status_string,
)
