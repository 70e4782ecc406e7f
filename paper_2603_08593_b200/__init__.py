"""B200-native SFFT image differencing (hot path of arxiv/paper_2603_08593).

Public surface = thin ctypes binding over the C-ABI library `libsfft.so` (include/sfft.h).
Importing this package does not require a GPU; calling the hot path does, and fails loudly if
the CUDA library is missing (there is no CPU fallback).
"""
from . import synth  # noqa: F401
from .binding import (  # noqa: F401
    SfftError,
    SfftPlan,
    lib_path,
    load_library,
    EXPORTED_SYMBOLS,
    median_combine,
    aperture_stats,
    resample_affine,
    resample_mask_affine,
    cut_stamps,
    solve_static,
    SOLVE_STATIC_MAX_N,
)

__all__ = ["synth", "SfftPlan", "SfftError", "lib_path", "load_library", "EXPORTED_SYMBOLS",
           "median_combine", "aperture_stats", "resample_affine", "resample_mask_affine", "cut_stamps",
           "solve_static", "SOLVE_STATIC_MAX_N"]
