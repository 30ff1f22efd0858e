"""paper_2404_14401_b200 -- B200-native split-step Gross-Pitaevskii propagation (libgpe).

The product is the C-ABI shared library `libgpe.so` (include/gpe.h), built from the CUDA
sources under csrc/ for sm_100a.  This package is a thin ctypes binding with the same names:
argument marshalling only, every step of the path runs in the library's kernels.  There is
no CPU fallback: importing works without a GPU (so the build can be checked), every compute
call fails loudly with GPE_ECUDA when no device is present, and a missing library raises.
"""
from .binding import (  # noqa: F401
    GPE_C64, GPE_C128, GPE_REAL_TIME, GPE_IMAG_TIME, GPE_NREC, GpeError, Plan,
    gpe_plan_create, gpe_plan_set_stream, gpe_plan_destroy, gpe_set_potential, gpe_evolve,
    gpe_observables, gpe_populations, gpe_profile_passes, gpe_measure_roofs, gpe_norm_theta_noalloc, gpe_fft2_forward, gpe_get_step, gpe_set_step,
    gpe_last_error, gpe_version,
    gpe_potential_desc, gpe_obs, library_path, load_library,
    GPE3_NREC, OBS3_NAMES, Plan3, gpe3_plan_create, gpe3_plan_set_stream, gpe3_plan_destroy, gpe3_set_potential,
    gpe3_evolve, gpe3_observables, gpe3_synchronize, gpe3_get_step, gpe3_set_step,
)
