"""The five synthetic workloads of BASELINE.json `configs` (0-based index = position there).

Each stands in for a parameter set the paper times:
seeded uniform-disc star fields, square maps centred at the origin, theta_star = 1.
Readings of what BASELINE.json leaves open are listed in DESIGN.md section 3.
"""
from dataclasses import dataclass, field
import math

# border modes (numeric values are the C-ABI's MLENS_BORDER_* and the oracle's ORC_BORDER_*)
BORDER_EQ16 = 0      # P:135 eq 16: dY + 10 theta sqrt(kappa_star)
BORDER_A6 = 1        # P:528 eq A6: dY + theta sqrt(kappa_star <m^2>/(f <m>)), param = f
BORDER_MARGIN = 2    # multiplicative margin on the macro preimage (BASELINE config 0), param = frac
BORDER_EXPLICIT = 3  # caller gives the window half-sizes

MASS_EQUAL = 0
MASS_POWER = 1       # dN/dm ~ m^-a on [m_lo, m_hi], divided by the theoretical mean


def salpeter_moments(a: float, lo: float, hi: float):
    """<m>, <m^2> of dN/dm ~ m^-a on [lo, hi] (closed-form integrals)."""
    def I(q):  # integral of m^q
        return (hi ** (q + 1) - lo ** (q + 1)) / (q + 1)
    n0 = I(-a)
    return I(1 - a) / n0, I(2 - a) / n0


@dataclass(frozen=True)
class LensConfig:
    name: str
    n_stars: int
    kappa_tot: float
    kappa_star: float
    gamma: float
    half_y: float            # source square half-length (theta_E)
    npix: int
    rays_per_pixel_length: float   # k; cell = pixel / k
    border_mode: int
    border_param: float
    mass_law: int = MASS_EQUAL
    mass_a: float = 2.35
    mass_lo: float = 0.08
    mass_hi: float = 1.0
    seed: int = 1000
    theta_star: float = 1.0

    @property
    def R_star(self) -> float:
        # eq 9 with A = pi R^2 and <m> = 1 after normalisation
        return self.theta_star * math.sqrt(self.n_stars / self.kappa_star)

    @property
    def m2_over_m(self) -> float:
        if self.mass_law == MASS_EQUAL:
            return 1.0
        m1, m2 = salpeter_moments(self.mass_a, self.mass_lo, self.mass_hi)
        return (m2 / m1) / m1   # masses are divided by <m>, so <m^2>/<m> -> <m^2>/<m>^2

    @property
    def mu_macro(self) -> float:
        return 1.0 / ((1 - self.kappa_tot) ** 2 - self.gamma ** 2)


CONFIGS = [
    # 0: tiny map; window = macro preimage + 10 % (BASELINE's wording), 8 rays per pixel AREA (~2M rays)
    LensConfig("cfg0_tiny", 200, 0.4, 0.2, 0.2, 5.0, 256, math.sqrt(8.0),
               BORDER_MARGIN, 0.1, seed=1001),
    # 1: typical quasar field (the bench workload); both IPM and IRS
    LensConfig("cfg1_quasar", 20000, 0.45, 0.45, 0.4, 25.0, 1000, 10.0,
               BORDER_EQ16, 0.0, seed=1002),
    # 2: Salpeter spectrum, saddle image
    LensConfig("cfg2_salpeter", 200000, 0.6, 0.3, 0.6, 50.0, 4000, 1.0,
               BORDER_EQ16, 0.0, mass_law=MASS_POWER, seed=1003),
    # 3: cluster caustic-crossing regime
    LensConfig("cfg3_cluster", 1000000, 0.7, 0.01, 0.29, 2.0, 2000, 1.0,
               BORDER_EQ16, 0.0, seed=1004),
    # 4: large production map
    LensConfig("cfg4_production", 10000000, 0.5, 0.4, 0.45, 100.0, 10000, 10.0,
               BORDER_EQ16, 0.0, mass_law=MASS_POWER, seed=1005),
]


def get_config(i: int) -> LensConfig:
    return CONFIGS[i]
