"""B200-native Fourier-domain dedispersion hot path (arXiv:2110.03482): Python binding.

The product is the CUDA library behind include/fdd.h; this package only marshals arguments.
"""
from .binding import (FDD_KERNEL_AUTO, FDD_KERNEL_GENERIC, FDD_KERNEL_SYMMETRIC, FDD_KERNEL_SYMMETRIC2, FDD_KERNEL_MIXED, FDD_KERNEL_TENSOR,  # noqa: F401
                      FDD_MODE_FOURIER, FDD_MODE_TIME, FDD_INVERSE_CUFFT, FDD_INVERSE_TWO_PASS, FDD_INVERSE_AUTO, FddError, Plan, error_string,
                      load_library, measure_fp32_peak, tc_selftest, rotate_sum_static,
                      FDD_ERR_TOO_LARGE, FDD_STATIC_MAX_PHASES)
