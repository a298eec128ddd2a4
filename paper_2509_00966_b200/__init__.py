"""paper_2509_00966_b200 -- B200-native domain-batched real-time Kohn-Sham step (DC-MESH / LFD hot path).

Thin Python binding over the C-ABI library ``libmlmd.so`` (include/mlmd.h).  The binding only
marshals arguments: every step of the path runs in the library's CUDA kernels.  PyTorch is used
for device memory and streams.  There is no CPU fallback: without the built library or a B200
the calls raise.
"""
from .api import (  # noqa: F401
    Domain,
    MlmdError,
    lib,
    mlmd_workspace_bytes,
    mlmd_domain_create,
    mlmd_domain_destroy,
    mlmd_set_orbitals,
    mlmd_get_orbitals,
    mlmd_set_vloc,
    mlmd_set_projectors,
    mlmd_set_gemm_mode,
    mlmd_set_option,
    mlmd_propagate,
    mlmd_propagate_split,
    mlmd_density,
    mlmd_overlap,
    mlmd_orbital_norms_static,
    mlmd_occupations,
    mlmd_energy_nl,
    mlmd_current,
    mlmd_current_nl,
    mlmd_launch_count,
    mlmd_profile,
    mlmd_profile_read,
    KERNEL_CLASSES,
    mlmd_last_error,
    EXPORTED_SYMBOLS,
    HOST, DEVICE, BETA_REAL32, BETA_COMPLEX64,
    GEMM_FP32GRADE, GEMM_FP64, GEMM_LOWP_BF16, GEMM_TF32X1, GEMM_FP32_SIMT, GEMM_FP32GRADE_STAGED,
    KEEP_PSI0, CHECK_FINITE, BORROW_PSI,
    OPT_GRAPH, OPT_STENCIL, OPT_GEMM_PATH, OPT_KICK_NORM, OPT_FD_ORDER, OPT_LOCAL_SOLVER,
    OK, WARN_UNSTABLE,
)
