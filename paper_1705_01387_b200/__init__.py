"""B200-native GPUQT hot path (arXiv 1705.01387): C-ABI library libgpuqt.so + thin binding."""
from .binding import (DAMPING_JACKSON, DAMPING_LORENTZ, DAMPING_NONE, GpuQT, GpuqtError, MODE_MSD, MODE_PSI,  # noqa: F401
                      MODE_VAC, STATE_CHI, STATE_PSI, STATE_VAC_A, STATE_VAC_B, bessel_coeffs, default_options,
                      kpm_transform_static, load, plan_storage, validate)
