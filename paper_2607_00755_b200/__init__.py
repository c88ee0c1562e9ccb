"""paper_2607_00755_b200 -- B200-native evaluation of the KineticXGPU 2->2 elastic self-collision
operator C[f] (arxiv/paper_2607_00755).  All arithmetic runs in hand-written CUDA kernels behind the
C ABI of include/kx.h (libkx.so); this package is the thin ctypes binding (argument marshalling only).
There is no CPU fallback: importing works anywhere, every call needs an sm_100 GPU.
"""
from .kx import (Handle, KxError, build_library, library_path, exported_symbols, plan_probe,
                 INTERP_LOG, INTERP_LINEAR, EXP_TABLE, EXP_LIBM, STORE_SYM_ROWS, STORE_TILED, STAT_CLASSICAL, STAT_BOSE, STAT_FERMI, PROJECT, DIAG,
                 EULER, HEUN, RK4, FP64, FP32)

__all__ = ["Handle", "KxError", "build_library", "library_path", "exported_symbols", "plan_probe",
           "INTERP_LOG", "INTERP_LINEAR", "EXP_TABLE", "EXP_LIBM", "STORE_SYM_ROWS", "STORE_TILED", "STAT_CLASSICAL", "STAT_BOSE", "STAT_FERMI", "PROJECT", "DIAG",
           "EULER", "HEUN", "RK4", "FP64", "FP32"]
