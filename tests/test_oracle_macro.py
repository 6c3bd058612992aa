"""Pins of the oracle's macro model beyond linear (reading G23).

The paper prints no formula for this regime ("the chosen order to which the potential is Taylor expanded"), so the
reading is the textbook one: the macro deflection grad(psi) carries its second-order Taylor term, alpha_i += (1/2) psi_ijk x_j x_k
with the four third derivatives psi_111, psi_112, psi_122, psi_222 at the origin.  Pinned by what the mathematics fixes:
 - with psi_111 = g alone the map is the fold y1 = a x1 - g x1^2/2, y2 = b x2, whose inverse, magnification
   1/(|b| sqrt(a^2 - 2 g y1)) and pixel means are closed forms (a dropped 1/2, a wrong sign or a swapped axis fails);
 - the Jacobian by central differences must be symmetric (a potential exists) and equal A0 - (psi_ij1 x1 + psi_ij2 x2)
   (a transposed or misplaced coefficient among the four fails);
 - all four zero reproduces the paper's constant kappa, gamma to the last bit.
"""
import math

import numpy as np
import pytest


def _fold_field(orc, kt, gam, g, axis=0):
    z = np.zeros(0)
    quad = (g, 0.0, 0.0, 0.0) if axis == 0 else (0.0, 0.0, 0.0, g)
    return orc.Field.make(kt, 0.0, gam, z, z, z, R=1e9, macro_quad=quad)


def test_fold_image_positions(orc):
    kt, gam, g = 0.3, 0.1, 0.05
    a, b = 1 - kt + gam, 1 - kt - gam
    f = _fold_field(orc, kt, gam, g)
    x1 = np.linspace(-3.0, 3.0, 25); x2 = np.linspace(-2.0, 2.0, 25)
    wx, wy = orc.lens_map(f, x1, x2)
    assert np.allclose(wx, a * x1 - 0.5 * g * x1 ** 2, rtol=0, atol=1e-15)
    assert np.allclose(wy, b * x2, rtol=0, atol=1e-15)
    # hand value: a = 0.8, x1 = 2 -> 1.6 - 0.05 * 4 / 2 = 1.5
    wx, wy = orc.lens_map(f, np.array([2.0]), np.array([1.0]))
    assert wx[0] == pytest.approx(1.5, abs=1e-15) and wy[0] == pytest.approx(0.6, abs=1e-15)
    # the other axis
    f2 = _fold_field(orc, kt, gam, g, axis=1)
    wx, wy = orc.lens_map(f2, np.array([2.0]), np.array([2.0]))
    assert wx[0] == pytest.approx(1.6, abs=1e-15) and wy[0] == pytest.approx(0.6 * 2 - 0.05 * 4 / 2, abs=1e-15)


def test_jacobian_is_symmetric_and_linear_in_x(orc):
    kt, gam = 0.4, 0.15
    t = (0.03, -0.02, 0.05, 0.07)                          # psi_111, psi_112, psi_122, psi_222: all different
    z = np.zeros(0)
    f = orc.Field.make(kt, 0.0, gam, z, z, z, R=1e9, macro_quad=t)
    rng = np.random.default_rng(2)
    for x1, x2 in rng.uniform(-4, 4, (6, 2)):
        e = 1e-4
        w = lambda u, v: tuple(c[0] for c in orc.lens_map(f, np.array([u]), np.array([v])))
        d11 = (w(x1 + e, x2)[0] - w(x1 - e, x2)[0]) / (2 * e); d12 = (w(x1, x2 + e)[0] - w(x1, x2 - e)[0]) / (2 * e)
        d21 = (w(x1 + e, x2)[1] - w(x1 - e, x2)[1]) / (2 * e); d22 = (w(x1, x2 + e)[1] - w(x1, x2 - e)[1]) / (2 * e)
        assert d12 == pytest.approx(d21, abs=1e-9)                                        # grad of a potential
        assert d11 == pytest.approx(1 - kt + gam - (t[0] * x1 + t[1] * x2), abs=1e-9)     # 1 - psi_11(x)
        assert d22 == pytest.approx(1 - kt - gam - (t[2] * x1 + t[3] * x2), abs=1e-9)     # 1 - psi_22(x)
        assert d12 == pytest.approx(-(t[1] * x1 + t[2] * x2), abs=1e-9)                   # - psi_12(x)


def test_zero_coefficients_change_nothing(orc):
    import synth
    xs, ys, ms = synth.disc_stars(60, 20.0, 5)
    f0 = orc.Field.make(0.4, 0.15, 0.1, xs, ys, ms, R=20.0)
    f1 = orc.Field.make(0.4, 0.15, 0.1, xs, ys, ms, R=20.0, macro_quad=(0.0, 0.0, 0.0, 0.0))
    zx, zy = synth.sample_points_window(500, 0.0, 0.0, 10.0, 10.0, 1)
    a, b = orc.lens_map(f0, zx, zy), orc.lens_map(f1, zx, zy)
    assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1])


@pytest.mark.parametrize("k", [2.0, 8.0])
def test_fold_map_against_closed_form(orc, k):
    """No stars, psi_111 = g: one image of the map region inside an EXPLICIT window that stays on one side of the critical
    line x1 = a/g.  mu(y) = 1/(|b| sqrt(a^2 - 2 g y1)); its mean over a pixel [y, y + p] is
    (sqrt(a^2 - 2 g y) - sqrt(a^2 - 2 g (y + p)))/(g p |b|).  IPM spreads a cell's flux evenly over its image, so a pixel is
    off by at most the density variation across the one or two cells that straddle its edges: g h/(a - g x) of their share,
    <= 2/k of the pixel -- and the flux of a whole pixel COLUMN up to a pixel edge is exact to one cell (checked on the
    cumulative sum, which a wrong factor or sign in the quadratic term moves by many cells)."""
    kt, gam, g = 0.3, 0.1, 0.08
    a, b = 1 - kt + gam, 1 - kt - gam                      # 0.8, 0.6; critical line at x1 = 10
    f = _fold_field(orc, kt, gam, g)
    half, npix = 2.0, 32
    He = (4.0, 4.0)                                        # x1 in [-4, 4] -> y1 in [-3.84, 2.56]: covers [-2, 2]; x2 -> +-2.4
    geo = orc.geometry(kt, 0.0, gam, half, npix, k, 3, He=He)
    m = orc.shoot(f, geo, 0)
    p = geo.p1
    ylo = geo.ylo1 + p * np.arange(npix)
    want = (np.sqrt(a * a - 2 * g * ylo) - np.sqrt(a * a - 2 * g * (ylo + p))) / (g * p * abs(b))
    assert np.allclose(m, m[0][None, :], rtol=1e-12)       # nothing depends on y2
    row = m[npix // 2]
    xim = (a - np.sqrt(a * a - 2 * g * (ylo + 0.5 * p))) / g
    bound = (2.0 / k) * g * geo.h1 / (a - g * xim) * 1.5
    assert np.all(np.abs(row / want - 1) <= bound), np.max(np.abs(row / want - 1) / bound)
    assert np.max(np.abs(row / want - 1)) > 1e-9 or k > 4  # (it is not the affine case)
    # flux up to each pixel edge: sum_{pixels below} mu p = (x1(y_edge) - x1(y_lo)) / |b|, exact to one cell's width
    cum = np.cumsum(row) * p
    inv = lambda y: (a - np.sqrt(a * a - 2 * g * y)) / g
    exact = (inv(ylo + p) - inv(geo.ylo1)) / abs(b)
    assert np.all(np.abs(cum - exact) <= geo.h1 / abs(b) * 1.0001)
    assert cum[-1] == pytest.approx(exact[-1], abs=geo.h1 / abs(b))
    # the mean magnification of the strip differs from the linear model's 1/(a |b|): the term is really there
    assert abs(row.mean() * a * abs(b) - 1) > 1e-3
