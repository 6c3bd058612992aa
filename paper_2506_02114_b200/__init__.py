"""paper_2506_02114_b200 -- B200-native microlensing magnification maps (arXiv 2506.02114 hot path).

Thin binding over the C ABI of include/mlens.h (libmlens.so, hand-written CUDA for sm_100a).
Every step of the path runs in the library's kernels; there is no CPU fallback.
"""
from .mlens import (  # noqa: F401
    MlensError, Field, ShootResult, lib, version, bench_dfma, bench_atomics, bench_shared_atomics, launch_count,
    SHAPE_DISC, SHAPE_RECT, MASS_EQUAL, MASS_POWER, EVAL_FMM, EVAL_DIRECT, EVAL_FMM_F32, MAP_IPM, MAP_IRS,
    BORDER_EQ16, BORDER_A6, BORDER_MARGIN, BORDER_EXPLICIT, MAX_ORDER, MAX_DIRECT,
    light_curve, histogram, INTERP_NEAREST, INTERP_BILINEAR, histogram_static, HIST_STATIC_MAXBINS,
)
from .starfile import read_star_file, write_star_file  # noqa: F401,E402
