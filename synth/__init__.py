"""Seeded synthetic inputs shared by tests, bench.py and smoke().

This package holds NO arithmetic of the method (no lens equation, no FMM, no
clipping, no star-field RNG of the library): only the parameter sets that stand
in for the paper's workloads (BASELINE.json `configs`) and plain numpy draws of
star positions / masses / sample points that are handed, as arrays, to BOTH the
CPU oracle and the CUDA library.
"""
from .configs import CONFIGS, LensConfig, get_config, salpeter_moments  # noqa: F401
from .stars import (  # noqa: F401
    clustered_stars, disc_stars, rect_stars, sample_points_window, sample_points_near_stars,
)
