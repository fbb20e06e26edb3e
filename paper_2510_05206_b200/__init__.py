"""B200-native particle-mesh force path of DISCO-DJ II (arXiv 2510.05206).

The product is ``libpmforce.so`` (hand-written CUDA for sm_100a behind the C ABI of
``include/pmforce.h``).  This package is the thin Python binding over it: the functions below have the
names of the C calls and only marshal arguments (torch tensors -> device pointers, the current CUDA stream
-> ``void*``).  PyTorch is used for device memory and streams, nothing else.  There is no CPU fallback:
if the library is missing or a call fails, a ``PMError`` / ``RuntimeError`` is raised.
"""
from .api import (  # noqa: F401
    PMError,
    PMParams,
    PMContext,
    pm_create,
    pm_destroy,
    pm_bin,
    pm_assign,
    pm_assign_vjp,
    pm_poisson_force,
    pm_poisson_force_vjp,
    pm_interp,
    pm_interp_vjp,
    nufft_spread,
    nufft_spread_vjp,
    nufft_poisson_force,
    nufft_poisson_force_vjp,
    nufft_interp,
    nufft_interp_vjp,
    pm_force,
    pm_force_vjp,
    pm_force_host,
    pm_force_host_async,
    pm_assign_jvp,
    pm_interp_jvp,
    pm_dkd_step,
    pm_dkd_step_adjoint,
    pm_power_spectrum,
    pm_sheet_resample,
    pm_mesh_power_noalloc,
    NOALLOC_MAX_BINS,
    pm_smem_peak,
    pm_set_profiling,
    pm_get_stage_ms,
    STAGE_NAMES,
    library_path,
    load_library,
    EXPORTED_SYMBOLS,
    FLAG_BIN_TWOPASS,
    FLAG_NO_XFUSE,
    FLAG_GRAD_REAL,
    FLAG_KERNEL_GRAD,
)
