"""CPU oracle (test infrastructure). See mlens_oracle.c for what it is and what pins it.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
may import this package.  It imports nothing from the CUDA package.
"""
from .oracle import (  # noqa: F401
    build, lib, Field, Geometry, alpha_star, alpha_smooth, lens_map, geometry, shoot,
    map_corners, map_centres, deposit_ipm, bin_irs, triangle_pixel_area, starfield, rng_draw,
    multipole_def, local_def, local_eval, num_threads, light_curve, histogram,
)
