"""Plain numpy draws of star fields and sample points (inputs only; see package docstring)."""
import numpy as np

from .configs import LensConfig, MASS_POWER, salpeter_moments


def _masses(rng, n, cfg: LensConfig | None):
    if cfg is None or cfg.mass_law != MASS_POWER:
        return np.ones(n)
    a, lo, hi = cfg.mass_a, cfg.mass_lo, cfg.mass_hi
    e = 1.0 - a
    u = rng.random(n)
    m = (lo ** e + u * (hi ** e - lo ** e)) ** (1.0 / e)
    return m / salpeter_moments(a, lo, hi)[0]


def disc_stars(n: int, R: float, seed: int, cfg: LensConfig | None = None):
    """n stars uniform in the disc |z| <= R; masses 1 or cfg's power law / <m>."""
    rng = np.random.default_rng(seed)
    r = R * np.sqrt(rng.random(n))
    phi = 2.0 * np.pi * rng.random(n)
    return r * np.cos(phi), r * np.sin(phi), _masses(rng, n, cfg)


def clustered_stars(n: int, R: float, seed: int, n_clumps: int = 6, clump_frac: float = 0.3, sigma: float = 3e-4,
                    cfg: LensConfig | None = None, r_clumps: float = 0.25):
    """Clustered star field ("spatial distributions including clustered or uniform random"): (1 - clump_frac) n
    stars uniform in the disc |z| <= R, the rest in n_clumps tight Gaussian clumps of width sigma R whose centres lie
    uniformly within r_clumps R of the origin.  The clumps force the quadtree many levels deeper than a uniform field
    of the same size (cell size ~ sigma R / sqrt(stars per clump / 32))."""
    rng = np.random.default_rng(seed)
    n_c = int(round(clump_frac * n / n_clumps)) * n_clumps
    n_u = n - n_c
    r = R * np.sqrt(rng.random(n_u))
    phi = 2.0 * np.pi * rng.random(n_u)
    x, y = r * np.cos(phi), r * np.sin(phi)
    rc = r_clumps * R * np.sqrt(rng.random(n_clumps))
    pc = 2.0 * np.pi * rng.random(n_clumps)
    cx = np.repeat(rc * np.cos(pc), n_c // n_clumps)
    cy = np.repeat(rc * np.sin(pc), n_c // n_clumps)
    x = np.concatenate([x, cx + sigma * R * rng.standard_normal(n_c)])
    y = np.concatenate([y, cy + sigma * R * rng.standard_normal(n_c)])
    return x, y, _masses(rng, n, cfg)


def rect_stars(n: int, c1: float, c2: float, seed: int, cfg: LensConfig | None = None):
    """n stars uniform in the rectangle |x1| <= c1, |x2| <= c2."""
    rng = np.random.default_rng(seed)
    x = c1 * (2.0 * rng.random(n) - 1.0)
    y = c2 * (2.0 * rng.random(n) - 1.0)
    return x, y, _masses(rng, n, cfg)


def sample_points_window(n: int, X1: float, X2: float, H1: float, H2: float, seed: int):
    """n points uniform in the shooting window [X-H, X+H]."""
    rng = np.random.default_rng(seed)
    return X1 + H1 * (2 * rng.random(n) - 1), X2 + H2 * (2 * rng.random(n) - 1)


def sample_points_near_stars(xs, ys, n: int, dist: float, seed: int, H1=None, H2=None):
    """n points at distance `dist` (random direction) from randomly chosen stars
    (restricted to stars inside |x|<=H1,|y|<=H2 when given)."""
    rng = np.random.default_rng(seed)
    idx = np.arange(len(xs))
    if H1 is not None:
        idx = idx[(np.abs(xs) <= H1) & (np.abs(ys) <= H2)]
        if len(idx) == 0:
            idx = np.arange(len(xs))
    pick = rng.choice(idx, size=n)
    ang = 2 * np.pi * rng.random(n)
    return xs[pick] + dist * np.cos(ang), ys[pick] + dist * np.sin(ang)
