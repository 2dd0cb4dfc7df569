"""frb200: B200-native flux-reconstruction RHS and Runge-Kutta stage driver (C ABI in include/frb200.h)."""
from .binding import (Context, FrError, GemmPlan, gemm, load, probe_peaks)  # noqa: F401
