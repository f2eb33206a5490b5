"""B200-native GPUQT hot path (arXiv 1705.01387): C-ABI library libgpuqt.so + thin binding."""
from .binding import (GpuQT, GpuqtError, MODE_MSD, MODE_PSI, MODE_VAC, STATE_CHI, STATE_PSI,  # noqa: F401
                      STATE_VAC_A, STATE_VAC_B, bessel_coeffs, load, validate)
