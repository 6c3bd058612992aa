"""Pins of the oracle's deflection, sheet terms and FMM-coefficient definitions (CPU only).

Each check is against something the paper or the mathematics fixes, not against the oracle's
own formula: hand values, symmetry, Gauss's law, 2-D quadrature of eq B1, finite differences.
"""
import math
import os

import numpy as np
import pytest

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def test_alpha_star_hand_values(orc):
    # eq 13 with one star m=2 at (1,1), ray at (4,5): d = (3,4), |d|^2 = 25 -> 2*(3,4)/25
    f = orc.Field.make(0, 0, 0, [1.0], [1.0], [2.0], R=10)
    ax, ay = orc.alpha_star(f, [4.0], [5.0])
    assert ax[0] == pytest.approx(0.24, abs=1e-16) and ay[0] == pytest.approx(0.32, abs=1e-16)
    # theta_star scales as theta^2
    f2 = orc.Field.make(0, 0, 0, [1.0], [1.0], [2.0], R=10, theta_star=3.0)
    ax2, ay2 = orc.alpha_star(f2, [4.0], [5.0])
    assert ax2[0] == pytest.approx(9 * 0.24, rel=1e-15)
    # two stars: m=1 at (0,0) and m=3 at (2,0), ray at (1,1): (1,1)/2 + 3*(-1,1)/2 = (-1, 2)
    f3 = orc.Field.make(0, 0, 0, [0.0, 2.0], [0.0, 0.0], [1.0, 3.0], R=10)
    ax3, ay3 = orc.alpha_star(f3, [1.0], [1.0])
    assert ax3[0] == pytest.approx(-1.0, abs=1e-15) and ay3[0] == pytest.approx(2.0, abs=1e-15)
    # a ray exactly on a star skips it (reading G11)
    ax4, ay4 = orc.alpha_star(f3, [2.0], [0.0])
    assert ax4[0] == pytest.approx(0.5, abs=1e-16) and ay4[0] == 0.0


def test_alpha_star_ring_and_gauss(orc):
    # a ring of n equal masses: deflection vanishes at its centre; outside, far away, it tends
    # to M/conj(z) (monopole), and Gauss's law gives the ring average exactly M/r outside.
    n = 64
    ang = 2 * np.pi * np.arange(n) / n
    f = orc.Field.make(0, 0, 0, 3 * np.cos(ang), 3 * np.sin(ang), np.ones(n), R=10)
    ax, ay = orc.alpha_star(f, [0.0], [0.0])
    assert abs(ax[0]) < 1e-13 and abs(ay[0]) < 1e-13
    # inside a ring of many equal masses the field is ~0 (shell theorem in 2-D), outside M/r
    ax, ay = orc.alpha_star(f, [1.0, 7.0], [0.5, 0.0])
    assert abs(ax[0]) < 1e-10 and abs(ay[0]) < 1e-10          # z^63 suppression
    assert ax[1] == pytest.approx(n / 7.0, rel=1e-10) and abs(ay[1]) < 1e-10


def test_alpha_star_is_gradient_of_log_potential(orc):
    # alpha = grad psi with psi = sum m ln|x - x_i| (eq 8): central differences of the
    # potential computed here with numpy, a different expression from the oracle's m d/|d|^2.
    rng = np.random.default_rng(5)
    xs, ys, ms = rng.normal(size=20) * 3, rng.normal(size=20) * 3, rng.uniform(0.1, 2, 20)
    f = orc.Field.make(0, 0, 0, xs, ys, ms, R=20)
    psi = lambda x, y: np.sum(ms * 0.5 * np.log((x - xs) ** 2 + (y - ys) ** 2))
    for (x, y) in [(0.3, -0.7), (5.1, 2.2), (-4.0, 4.5)]:
        e = 1e-5
        gx = (psi(x + e, y) - psi(x - e, y)) / (2 * e)
        gy = (psi(x, y + e) - psi(x, y - e)) / (2 * e)
        ax, ay = orc.alpha_star(f, [x], [y])
        assert ax[0] == pytest.approx(gx, rel=1e-7, abs=1e-8)
        assert ay[0] == pytest.approx(gy, rel=1e-7, abs=1e-8)


def test_disc_sheet(orc):
    # eq 19: -ks z inside; -ks R^2/conj(z) outside; continuous at |z| = R
    f = orc.Field.make(0.5, 0.3, 0.1, [0.0], [0.0], [0.0], R=2.0)
    ax, ay = orc.alpha_smooth(f, [1.0, 3.0, 2.0, 0.0], [-1.0, 4.0, 0.0, 0.0])
    assert (ax[0], ay[0]) == (pytest.approx(-0.3), pytest.approx(0.3))
    assert ax[1] == pytest.approx(-0.3 * 4 * 3 / 25) and ay[1] == pytest.approx(-0.3 * 4 * 4 / 25)
    assert ax[2] == pytest.approx(-0.6) and ay[2] == 0
    assert ax[3] == 0 and ay[3] == 0
    eps = 1e-9
    a_in, _ = orc.alpha_smooth(f, [2.0 - eps], [0.0])
    a_out, _ = orc.alpha_smooth(f, [2.0 + eps], [0.0])
    assert a_in[0] == pytest.approx(a_out[0], abs=1e-8)


def _rect_quadrature(ks, c1, c2, zx, zy):
    """conj(alpha_s) = (-ks/pi) int int dx' dy' /(z - z') (eq B1/B2) by scipy quadrature."""
    from scipy import integrate
    def re(yp, xp):
        dx, dy = zx - xp, zy - yp
        return dx / (dx * dx + dy * dy)
    def im(yp, xp):
        dx, dy = zx - xp, zy - yp
        return -dy / (dx * dx + dy * dy)
    R = integrate.dblquad(re, -c1, c1, -c2, c2, epsabs=1e-11, epsrel=1e-11)[0]
    I = integrate.dblquad(im, -c1, c1, -c2, c2, epsabs=1e-11, epsrel=1e-11)[0]
    # alpha = conj(that)
    return -ks / math.pi * R, +ks / math.pi * I


def test_rect_sheet_vs_quadrature_outside(orc):
    # eq B7 at points OUTSIDE the rectangle, all four sides and the corner regions,
    # incl. Re z > c1 with |Im z| <= c2 where both branch-cut terms are active.
    ks, c1, c2 = 0.37, 2.0, 1.25
    f = orc.Field.make(0.5, ks, 0.1, [0.0], [0.0], [0.0], shape=1, c1=c1, c2=c2)
    pts = [(3.1, 0.4), (-3.3, -0.6), (0.5, 2.2), (-0.7, -1.9), (2.9, 2.4), (-2.6, 1.8), (4.0, -3.0)]
    for (x, y) in pts:
        qx, qy = _rect_quadrature(ks, c1, c2, x, y)
        ax, ay = orc.alpha_smooth(f, [x], [y])
        assert ax[0] == pytest.approx(qx, abs=2e-9), (x, y)
        assert ay[0] == pytest.approx(qy, abs=2e-9), (x, y)


def test_rect_sheet_inside(orc):
    # Inside a uniform sheet of density -ks: div alpha = -2 ks, curl alpha = 0 (Poisson), alpha(0) = 0
    # by symmetry, odd parity, and far away alpha -> -ks (4 c1 c2/pi)/conj(z) (monopole of the sheet).
    ks, c1, c2 = 0.45, 3.0, 1.5
    f = orc.Field.make(0.5, ks, 0.1, [0.0], [0.0], [0.0], shape=1, c1=c1, c2=c2)
    a0 = orc.alpha_smooth(f, [0.0], [0.0])
    assert abs(a0[0][0]) < 1e-15 and abs(a0[1][0]) < 1e-15
    e = 1e-5
    for (x, y) in [(0.4, 0.3), (-2.5, 1.2), (2.9, -1.4), (0.0, 1.0), (-1.0, 0.0)]:
        axp, ayp = orc.alpha_smooth(f, [x + e, x - e, x, x], [y, y, y + e, y - e])
        div = (axp[0] - axp[1]) / (2 * e) + (ayp[2] - ayp[3]) / (2 * e)
        curl = (ayp[0] - ayp[1]) / (2 * e) - (axp[2] - axp[3]) / (2 * e)
        assert div == pytest.approx(-2 * ks, abs=1e-8)
        assert curl == pytest.approx(0.0, abs=1e-8)
        bx, by = orc.alpha_smooth(f, [-x], [-y])
        cx, cy = orc.alpha_smooth(f, [x], [y])
        assert bx[0] == pytest.approx(-cx[0], abs=1e-14) and by[0] == pytest.approx(-cy[0], abs=1e-14)
    # inside vs quadrature too (the integrand is singular but integrable; looser tolerance)
    qx, qy = _rect_quadrature(ks, c1, c2, 1.7, -0.8)
    ax, ay = orc.alpha_smooth(f, [1.7], [-0.8])
    assert ax[0] == pytest.approx(qx, abs=1e-5) and ay[0] == pytest.approx(qy, abs=1e-5)
    # far field
    zx, zy = 400.0, 300.0
    ax, ay = orc.alpha_smooth(f, [zx], [zy])
    M = ks * 4 * c1 * c2 / math.pi
    assert ax[0] == pytest.approx(-M * zx / (zx * zx + zy * zy), rel=1e-4)
    assert ay[0] == pytest.approx(-M * zy / (zx * zx + zy * zy), rel=1e-4)
    # continuity across every edge of the rectangle (branch-cut bookkeeping of eq B6/B7)
    for (x, y, nx, ny) in [(c1, 0.3, 1, 0), (-c1, -0.2, 1, 0), (0.5, c2, 0, 1), (-1.0, -c2, 0, 1)]:
        d = 1e-9
        p = orc.alpha_smooth(f, [x + d * nx, x - d * nx], [y + d * ny, y - d * ny])
        assert p[0][0] == pytest.approx(p[0][1], abs=1e-7) and p[1][0] == pytest.approx(p[1][1], abs=1e-7)


def test_lens_map_macro_terms(orc):
    # eq 7 / eq 12 with no stars: y = diag(1-k+g, 1-k-g) x
    f = orc.Field.make(0.45, 0.0, 0.4, [0.0], [0.0], [0.0], R=1e9)
    wx, wy = orc.lens_map(f, [2.0, -1.0], [3.0, 0.5])
    assert wx[0] == pytest.approx(0.95 * 2.0, rel=1e-15) and wy[0] == pytest.approx(0.15 * 3.0, rel=1e-14)
    # kappa_star compensates: stars + sheet; for one star at the origin of mass M inside a disc,
    # w = (1-k) z + g conj z - M/conj z + ks z
    f = orc.Field.make(0.6, 0.3, 0.1, [0.0], [0.0], [2.0], R=5.0)
    wx, wy = orc.lens_map(f, [1.0], [2.0])
    assert wx[0] == pytest.approx(0.4 * 1 + 0.1 * 1 - 2 * 1 / 5 + 0.3 * 1, rel=1e-15)
    assert wy[0] == pytest.approx(0.4 * 2 - 0.1 * 2 - 2 * 2 / 5 + 0.3 * 2, rel=1e-15)


def test_rect_over_circle_star_count_identity(orc):
    # eq 20-21: N_rect/N_circ = 2/(pi(1+2 g^2 |mu|)) follows from the areas of the
    # shooting rectangle (4 dX1 dX2) and its circumscribed circle (pi(dX1^2+dX2^2)) for a square
    # map; check the geometry helper reproduces it and the paper's worked value "~4x fewer".
    vals = {}
    for line in open(os.path.join(GOLD, "paper_values.txt")):
        if line.startswith("#") or not line.strip():
            continue
        name, v = line.split()[:2]
        vals[name] = float(v)
    k = g_ = 0.4
    geo = orc.geometry(k, 0.0, g_, 10.0, 100000, 1.0, 0)    # kappa_star=0: pure macro preimage (eq 15)
    ratio = (4 * geo.H1 * geo.H2) / (math.pi * (geo.H1 ** 2 + geo.H2 ** 2))
    mu = 1 / ((1 - k) ** 2 - g_ ** 2)
    assert ratio == pytest.approx(2 / (math.pi * (1 + 2 * g_ ** 2 * abs(mu))), rel=1e-4)   # whole-cell rounding
    assert ratio == pytest.approx(vals["rect_over_circ_kappa0.4_gamma0.4"], abs=0.02)
    assert ratio == pytest.approx(vals["fig7_rect_over_circ"], abs=0.02)


def test_multipole_and_local_definitions(orc):
    # eq C1/C2 and eq C4/C6: the expansions must reproduce the direct sum
    # (eq 13) where they converge.  alpha = theta^2 conj(dpsi/dz) (reading G1).
    rng = np.random.default_rng(11)
    n, p = 12, 40
    cx, cy, L = 3.0, -2.0, 0.5
    xs, ys = cx + L * rng.uniform(-1, 1, n), cy + L * rng.uniform(-1, 1, n)
    ms = rng.uniform(0.1, 1.0, n)
    f = orc.Field.make(0, 0, 0, xs, ys, ms, R=100)
    a = orc.multipole_def(xs, ys, ms, cx, cy, L, p)
    assert a[0] == pytest.approx(ms.sum(), rel=1e-15)
    # dipole: a_1 = -sum m zeta
    z1 = ((xs - cx) + 1j * (ys - cy)) / L
    assert a[1] == pytest.approx(-(ms * z1).sum(), rel=1e-14)
    zx, zy = cx + 4.1 * L, cy - 3.3 * L                       # well separated
    zeta = ((zx - cx) + 1j * (zy - cy)) / L
    dpsi = a[0] / zeta - sum(k * a[k] / zeta ** (k + 1) for k in range(1, p + 1))
    alpha = np.conj(dpsi) / L
    ax, ay = orc.alpha_star(f, [zx], [zy])
    assert alpha.real == pytest.approx(ax[0], rel=1e-12) and alpha.imag == pytest.approx(ay[0], rel=1e-12)
    # local expansion about a far centre
    tcx, tcy, TL = cx + 4 * 2 * L, cy + 2 * 2 * L, L
    c = orc.local_def(xs, ys, ms, tcx, tcy, TL, p)
    for (dx, dy) in [(0.9, -0.9), (-0.3, 0.2), (0.0, 0.0)]:
        px, py = tcx + dx * TL, tcy + dy * TL
        lx, ly = orc.local_eval(c, tcx, tcy, TL, px, py)
        ax, ay = orc.alpha_star(f, [px], [py])
        assert lx == pytest.approx(ax[0], rel=1e-11) and ly == pytest.approx(ay[0], rel=1e-11)
