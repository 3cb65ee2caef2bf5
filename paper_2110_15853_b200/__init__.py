"""B200-native Chebyshev filter of ChFSI (TTDFT, arXiv 2110.15853, Algorithm 1 step 1).

Thin Python binding over the C-ABI library ``libttdft.so`` (``include/ttdft.h``).  PyTorch is used
for device memory and streams only; every step of the path runs in the library's CUDA kernels.
There is no CPU fallback: if the library is missing or no CUDA device is present, calls fail.
"""
from .api import (  # noqa: F401
    TTDFTError,
    Hamiltonian,
    h_storage_bytes,
    h_build,
    h_build_bsr,
    h_build_csr,
    spmm,
    cheb_step,
    cheb_scalars,
    cheb_filter,
    cheb_filter_work_bytes,
    cheb_filter_host,
    cheb_filter_host_work_bytes,
    probe_fp64_peak,
    launch_count,
    last_error,
    library_path,
    exported_symbols,
    CHECK_SORTED,
    CHECK_SYMMETRY,
    FORCE_GENERIC,
    NO_I8,
    MATH_AUTO,
    MATH_FP64,
    MATH_I8,
    MATH_I8X7,
    step_work_bytes,
    timing_enable,
    timing_read,
    KERNEL_IDS,
    gram,
    gram_work_bytes,
    project,
    project_work_bytes,
    rotate,
    rotate_work_bytes,
)
