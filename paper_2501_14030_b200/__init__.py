"""B200-native hot path of the hyperbolic-relaxation puncture initial-data solver
(arxiv 2501.14030): a C-ABI CUDA library (include/hr.h, csrc/) and this thin binding.

Importing the package loads libhr_b200.so and raises if it has not been built -- there is no
CPU fallback (the CPU oracle under oracle/ is test infrastructure and is never imported here).
"""
from .binding import (HR_F32, HR_F64, HR_SINHSPHERICAL, HR_SINHSYMTP, HrError, Solver,  # noqa: F401
                      hr_host_setup, hr_measure_alu_peak, hr_measure_launch_floor, hr_params, hr_puncture, hr_step_many, hr_version, hr_workspace_bytes,
                      lib,
                      make_params)
