"""B200-native incoherent de-dispersion (hot path of Magro et al., arXiv 1107.2516).

The product is the C-ABI library built from ``csrc/`` (``include/dedisp.h``); this package holds
its build script, a ctypes binding with the same names, and the seeded input generators.
"""
from .binding import (Plan, Stream, Survey, power_corner_turn, bin_samples, fadd_microbench, detect_static, detect_static_max_slots, DedispError, ELIMIT, F32, U8, KERNEL_AUTO, KERNEL_NAIVE, KERNEL_DIRECT,
                      KERNEL_WINDOW, KERNEL_LONG, lib, version, EXPORTS, LIB_PATH)

__all__ = ["Plan", "Stream", "Survey", "power_corner_turn", "bin_samples", "fadd_microbench", "detect_static", "detect_static_max_slots", "DedispError", "ELIMIT", "F32", "U8", "KERNEL_AUTO", "KERNEL_NAIVE",
           "KERNEL_DIRECT", "KERNEL_WINDOW", "KERNEL_LONG", "lib", "version", "EXPORTS", "LIB_PATH"]
