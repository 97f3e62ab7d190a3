"""B200-native batched RBM local energy (jVMC hot path, arxiv 2108.03409).

Thin Python binding over the C-ABI library libnqs_b200.so (include/nqs.h): argument
marshalling only -- every step of the path runs in the CUDA kernels.  PyTorch is used for
device memory and streams.  There is no CPU fallback: without the built library or without a
CUDA device the calls raise.
"""
from .binding import (  # noqa: F401
    Hamiltonian,
    MICROBENCH_KINDS,
    NqsError,
    energy_stats,
    energy_stats_static,
    STATS_STATIC_MAX_B,
    A5_PATHS,
    PROFILE_SEGMENTS,
    connected_groups,
    debug_last_a5,
    enumerate_connected,
    enumerate_connected_h,
    fisher,
    get_option,
    set_option,
    forces,
    hamiltonian_info_host,
    last_error,
    launch_count,
    lib_path,
    load_library,
    local_energy,
    local_energy_host,
    log_psi,
    log_psi_host,
    metropolis,
    metropolis_shared,
    microbench,
    profile_enable,
    profile_last,
    release,
    version,
)
