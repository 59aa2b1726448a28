"""B200-native hot path of arxiv 2401.04865: spectral-Ewald evaluation of the
shell-regularized Coulomb operator, on-device induced-charge solve, forces and
torques.  The product is the CUDA library behind include/pce.h; this package is
its build script and a thin ctypes binding (argument marshalling only)."""
from .binding import (  # noqa: F401
    Context, PceError, PceParams, context_for, suggest_params, real_kernel_host, measure_fp64_peaks, poison_shared_memory, upload, load, lib_path, EXPORTS,
    radial_profile_static, PROFILE_STATIC_MAX_BINS,
)
from .build import build  # noqa: F401
