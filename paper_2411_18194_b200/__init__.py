"""paper_2411_18194_b200 -- B200-native (sm_100a) hot path of the mumax+ method (arxiv 2411.18194):
finite-difference effective field, LLG torque and Runge-Kutta stepping behind a C-ABI library
(include/mmx.h, csrc/).  This package is the thin Python binding; it holds no arithmetic."""
from .binding import (BS23, CK45, DEVICE, DMI_INTER, DP45, F_M, F_M0, F_M1, F_M2, F_U, F_V, HEUN12, HOST, RK4, RKF45,  # noqa: F401
                      T_A0, T_A12, T_ALL, T_ANIS_C, T_ANIS_U, T_DEMAG, T_DMI, T_DMI_HOMO, T_DMI_INTER, T_EXCH,
                      T_MEL, T_ZEEMAN, STRAY_STATIC_MAX_CELLS, MmxError, World, kernel_spectrum_host, load, newell_tensor_host, rk_imag_stability_limit,
                      stray_field_static, stray_table_host)
