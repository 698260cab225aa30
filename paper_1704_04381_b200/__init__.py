"""paper_1704_04381_b200 -- B200-native Rosenbluth chain generation (arXiv 1704.04381 hot path).

Public API = the C ABI of include/rosen.h, re-exported under the same names (binding.py).
"""
from .binding import (  # noqa: F401
    PER_CHAIN, ROSEN_ECUDA, ROSEN_EINVAL, ROSEN_ENOMEM, ROSEN_ERANGE, ROSEN_MEM_DEVICE, ROSEN_MEM_HOST, ROSEN_OK,
    RosenError, load_library, rosen_last_error, rosen_last_kernel_name, rosen_last_launch_count,
    rosen_lattice_dump, rosen_lattice_generate, rosen_lattice_generate_async, rosen_lattice_generate_noalloc,
    ROSEN_NOALLOC_MAX_N, ROSEN_NOALLOC_MAX_CHAINS, ROSEN_NOALLOC_SCRATCH_BYTES, rosen_realspace_generate_async,
    SUMMARY_BYTES, summary_from_device, rosen_realspace_dump, rosen_realspace_generate, rosen_strerror,
    rosen_summary_merge, rosen_fit_exponents, rosen_direction_eval, rosen_realspace_dump_probe, rosen_lattice_perm, rosen_lattice_generate_model, rosen_realspace_generate_model, rosen_version, rosen_debug_set, rosen_workspace_bytes, rosen_workspace_release,
)
from . import workloads  # noqa: F401
