"""Pins of the oracle's geometry, IPM apportioning and IRS binning (CPU only).

Closed forms (point lens, Chang-Refsdal cusps, affine maps), invariants (area conservation,
mean magnification) and brute force (Monte-Carlo / sub-sampling areas) -- see SURVEY.md 8(c).
"""
import math

import numpy as np
import pytest


# ----------------------------------------------------------------------------- geometry
def test_geometry_eq14_16(orc):
    # eq 16: dX = (dY + 10 theta sqrt(ks))/|1-k+-g|; grown to whole cells of size pixel/k
    g = orc.geometry(0.45, 0.45, 0.4, 25.0, 1000, 10.0, 0)
    assert g.p1 == pytest.approx(0.05) and g.h1 == pytest.approx(0.005)
    H1 = (25 + 10 * math.sqrt(0.45)) / 0.95
    H2 = (25 + 10 * math.sqrt(0.45)) / 0.15
    assert g.n1 == math.ceil(2 * H1 / g.h1) and g.n2 == math.ceil(2 * H2 / g.h2)
    assert 0 <= g.H1 - H1 < g.h1 and 0 <= g.H2 - H2 < g.h2
    assert g.X1 == 0 and g.X2 == 0 and g.x0_1 == -g.H1
    assert g.weight == pytest.approx(1 / 200.0)                  # 1/(2 k^2)
    # eq A6 with f = 1e-3 and <m^2>/<m> = 1.632
    g = orc.geometry(0.6, 0.3, 0.6, 50.0, 4000, 1.0, 1, 1e-3, m2_over_m=1.631996)
    r = math.sqrt(0.3 * 1.631996 / 1e-3)
    assert g.H1 >= (50 + r) / 1.0 and g.H1 - (50 + r) / 1.0 < g.h1
    assert g.H2 >= (50 + r) / 0.2 and g.H2 - (50 + r) / 0.2 < g.h2
    # eq 14: off-centre map
    g = orc.geometry(0.4, 0.2, 0.2, 5.0, 256, 1.0, 0, Y=(1.6, -0.8))
    assert g.X1 == pytest.approx(2.0) and g.X2 == pytest.approx(-2.0)
    # config 0 of BASELINE.json: "~2M rays" with 8 rays per pixel area and a 10 % margin
    g = orc.geometry(0.4, 0.2, 0.2, 5.0, 256, math.sqrt(8.0), 2, 0.1)
    assert 1.9e6 < (g.n1 + 1) * (g.n2 + 1) < 2.1e6


# ----------------------------------------------------------------------------- triangle / pixel areas
def _mc_area(tri, px, py, n=400):
    """Fraction of a fine n x n sub-grid of the pixel whose points lie inside the triangle."""
    s = (np.arange(n) + 0.5) / n
    X, Y = np.meshgrid(px + s, py + s)
    (x0, y0), (x1, y1), (x2, y2) = tri
    d1 = (x1 - x0) * (Y - y0) - (y1 - y0) * (X - x0)
    d2 = (x2 - x1) * (Y - y1) - (y2 - y1) * (X - x1)
    d3 = (x0 - x2) * (Y - y2) - (y0 - y2) * (X - x2)
    inside = ((d1 >= 0) & (d2 >= 0) & (d3 >= 0)) | ((d1 <= 0) & (d2 <= 0) & (d3 <= 0))
    return inside.mean()


def test_triangle_pixel_area_hand_and_subsampling(orc):
    # hand values: right triangle (0,0),(2,0),(0,2) has area 2; pixel [0,1]^2 is fully covered,
    # pixel [1,2]x[0,1] holds the triangle (1,0),(2,0),(1,1) of area 1/2, pixel [1,2]x[1,2] nothing.
    tri = [0, 0, 2, 0, 0, 2]
    assert orc.triangle_pixel_area(tri, 0, 0) == pytest.approx(1.0, abs=1e-15)
    assert orc.triangle_pixel_area(tri, 1, 0) == pytest.approx(0.5, abs=1e-15)
    assert orc.triangle_pixel_area(tri, 0, 1) == pytest.approx(0.5, abs=1e-15)
    assert orc.triangle_pixel_area(tri, 1, 1) == 0.0
    # orientation: clockwise triangle gives the negative (signed, reading G16)
    assert orc.triangle_pixel_area([0, 0, 0, 2, 2, 0], 1, 0) == pytest.approx(-0.5, abs=1e-15)
    # sub-sampling brute force on random triangles
    rng = np.random.default_rng(3)
    for _ in range(40):
        t = rng.uniform(-0.5, 3.5, 6)
        tri = [(t[0], t[1]), (t[2], t[3]), (t[4], t[5])]
        for px in range(-1, 4):
            for py in range(-1, 4):
                a = abs(orc.triangle_pixel_area(t, px, py))
                assert a == pytest.approx(_mc_area(tri, px, py), abs=6e-3)


def test_triangle_area_conservation(orc):
    # G16 (i): pieces over all pixels of the bounding box sum to the triangle's signed area (1e-10)
    rng = np.random.default_rng(4)
    for scale in (0.3, 2.0, 17.0):
        for _ in range(30):
            t = rng.uniform(0, scale, 6) + rng.uniform(0, 5)
            A = 0.5 * ((t[2] - t[0]) * (t[5] - t[1]) - (t[4] - t[0]) * (t[3] - t[1]))
            lo = int(math.floor(t.min())) - 1
            hi = int(math.ceil(t.max())) + 1
            s = sum(orc.triangle_pixel_area(t, px, py) for px in range(lo, hi) for py in range(lo, hi))
            assert s == pytest.approx(A, rel=1e-10, abs=1e-13)


# ----------------------------------------------------------------------------- IPM on affine maps
def test_ipm_exact_for_affine_maps(orc):
    # no stars, no sheet: w = diag(1-k+g, 1-k-g) z.  IPM is exact for affine maps, so every pixel
    # whose preimage lies inside the window holds 1/|(1-k)^2-g^2| (eq 21, eq 22).
    for (k, g_, kk) in [(0.0, 0.0, 1.0), (0.4, 0.2, 1.7), (0.6, 0.6, 2.0), (0.45, 0.4, 3.0)]:
        f = orc.Field.make(k, 0.0, g_, [0.0], [0.0], [0.0], R=1e9)
        geo = orc.geometry(k, 0.0, g_, 2.0, 32, kk, 2, 0.25)
        m = orc.shoot(f, geo, 0)
        mu = 1 / abs((1 - k) ** 2 - g_ ** 2)
        assert np.max(np.abs(m - mu)) < 2e-13 * mu, (k, g_)
    # identity lens on an aligned grid: exactly 1 in the interior
    f = orc.Field.make(0.0, 0.0, 0.0, [0.0], [0.0], [0.0], R=1e9)
    geo = orc.geometry(0.0, 0.0, 0.0, 2.0, 32, 2.0, 2, 0.25)
    assert np.all(orc.shoot(f, geo, 0) == 1.0)


def test_ipm_map_conservation(orc):
    # G16 (ii): sum(map) * pixel area = image-plane area of all triangles that land wholly inside
    # the map + the in-map fractions of the others; with a map that contains every mapped cell the
    # total is exactly the window area (1e-10).
    rng = np.random.default_rng(8)
    xs, ys = rng.uniform(-3, 3, 6), rng.uniform(-3, 3, 6)
    f = orc.Field.make(0.3, 0.0, 0.1, xs, ys, np.full(6, 0.05), R=1e9)
    # shoot a small window into a huge map so that nothing falls outside
    geo = orc.geometry(0.3, 0.0, 0.1, 400.0, 800, 1.0, 3, He=(2.0, 2.0))
    # make the window fine: override by using a separate geometry with explicit window and k
    geo = orc.geometry(0.3, 0.0, 0.1, 40.0, 160, 25.0, 3, He=(2.0, 2.0))
    m = orc.shoot(f, geo, 0)
    window_area = (geo.n1 * geo.h1) * (geo.n2 * geo.h2)
    assert m.sum() * geo.p1 * geo.p2 == pytest.approx(window_area, rel=1e-10)


# ----------------------------------------------------------------------------- point lens
def _point_lens_pixel_mean(x0, x1, y0, y1, n=64):
    """Mean over a pixel of mu(u) = (u^2+2)/(u sqrt(u^2+4)) by Gauss-Legendre quadrature."""
    gx, gw = np.polynomial.legendre.leggauss(n)
    X = 0.5 * (x1 + x0) + 0.5 * (x1 - x0) * gx
    Y = 0.5 * (y1 + y0) + 0.5 * (y1 - y0) * gx
    XX, YY = np.meshgrid(X, Y)
    W = np.outer(gw, gw) / 4.0
    u2 = XX ** 2 + YY ** 2
    return float(np.sum(W * (u2 + 2) / np.sqrt(u2 * (u2 + 4))))


def test_point_lens_magnification(orc):
    # one star m=1, kappa = gamma = 0: total magnification (u^2+2)/(u sqrt(u^2+4)) (BASELINE north_star).
    # Window must hold both images of every source point: |x| <= (u + sqrt(u^2+4))/2.
    f = orc.Field.make(0.0, 0.0, 0.0, [0.0], [0.0], [1.0], R=1e9)
    half, npix, k = 1.5, 30, 8.0
    umax = half * math.sqrt(2)
    Hw = 0.5 * (umax + math.sqrt(umax ** 2 + 4)) + 0.2
    geo = orc.geometry(0.0, 0.0, 0.0, half, npix, k, 3, He=(Hw, Hw))
    m = orc.shoot(f, geo, 0)
    worst = 0.0
    for iy in range(npix):
        for ix in range(npix):
            x0, y0 = geo.ylo1 + ix * geo.p1, geo.ylo2 + iy * geo.p2
            uc = math.hypot(x0 + geo.p1 / 2, y0 + geo.p2 / 2)
            if uc < 0.2:
                continue                     # the pixels touching the point caustic at u = 0
            ref = _point_lens_pixel_mean(x0, x0 + geo.p1, y0, y0 + geo.p2)
            worst = max(worst, abs(m[iy, ix] / ref - 1))
    assert worst < 2e-3
    # IRS on the same field converges to the same numbers within Poisson noise
    geo = orc.geometry(0.0, 0.0, 0.0, half, npix, 12.0, 3, He=(Hw, Hw))
    c = orc.shoot(f, geo, 1).astype(float) / 144.0
    ix = iy = 25
    x0, y0 = geo.ylo1 + ix * geo.p1, geo.ylo2 + iy * geo.p2
    ref = _point_lens_pixel_mean(x0, x0 + geo.p1, y0, y0 + geo.p2)
    assert c[iy, ix] == pytest.approx(ref, rel=4 / math.sqrt(144 * ref))


# ----------------------------------------------------------------------------- Chang-Refsdal
def _cr_images(w, a, g):
    """Images of source w for the lens w = a z + g conj(z) - 1/conj(z) (point mass + shear),
    from the quartic obtained by eliminating conj(z):  with q(z) = conj(w) z - g z^2 + 1 (so that
    conj(z) = q/(a z)),  g q^2 - a^2 z^2 - a z (w - a z) q = 0.  Returns (roots, magnifications)."""
    P = np.polynomial.polynomial
    q = np.array([1.0, np.conj(w), -g])                       # ascending powers
    poly = g * P.polymul(q, q)
    poly = P.polysub(poly, np.array([0, 0, a * a]))
    poly = P.polysub(poly, a * P.polymul(np.array([0, w, -a]), q))
    roots = np.roots(poly[::-1])
    good = [z for z in roots if abs(a * z + g * np.conj(z) - 1 / np.conj(z) - w) < 1e-8]
    mus = [1 / abs(a * a - abs(g + 1 / np.conj(z) ** 2) ** 2) for z in good]
    return good, mus


def test_chang_refsdal_caustic(orc):
    # point mass + shear (+ smooth convergence), kappa_star = 0.  With g' = g/(1-k) < 1 the caustic
    # is a single astroid with cusps on the axes at
    #   y1 = +- sqrt(1-k) 2g'/sqrt(1-g'),   y2 = +- sqrt(1-k) 2g'/sqrt(1+g')
    # (Chang & Refsdal 1984 in the paper's sign convention, +gamma on x1).
    k, g_ = 0.2, 0.2
    a = 1 - k
    gp = g_ / a
    cusp1 = math.sqrt(a) * 2 * gp / math.sqrt(1 - gp)
    cusp2 = math.sqrt(a) * 2 * gp / math.sqrt(1 + gp)
    # (1) the analytic image solver changes from 4 to 2 images exactly at the closed-form cusps
    for (w_in, w_out) in [(cusp1 - 1e-3, cusp1 + 1e-3), (1j * (cusp2 - 1e-3), 1j * (cusp2 + 1e-3)),
                          (-cusp1 + 1e-3, -cusp1 - 1e-3)]:
        assert len(_cr_images(w_in, a, g_)[0]) == 4 and len(_cr_images(w_out, a, g_)[0]) == 2
    # (2) the oracle's IPM map equals the summed image magnifications away from the caustic, and
    # so reproduces the 4 <-> 2 image jump where the closed form puts it
    f = orc.Field.make(k, 0.0, g_, [0.0], [0.0], [1.0], R=1e9)
    half, npix = 1.0, 50
    geo = orc.geometry(k, 0.0, g_, half, npix, 8.0, 3, He=(3.5, 5.0))
    m = orc.shoot(f, geo, 0)
    pix = geo.p1
    n_in = n_out = 0
    for iy in range(npix):
        for ix in range(npix):
            xc, yc = geo.ylo1 + (ix + 0.5) * pix, geo.ylo2 + (iy + 0.5) * pix
            # image counts at the pixel's centre and corners: skip pixels the caustic crosses or nears
            cnt = {len(_cr_images(complex(xc + dx * pix, yc + dy * pix), a, g_)[0])
                   for dx in (-2.4, -1.2, 0, 1.2, 2.4) for dy in (-2.4, -1.2, 0, 1.2, 2.4)}
            near_cusp = min(math.hypot(abs(xc) - cusp1, yc), math.hypot(xc, abs(yc) - cusp2)) < 5 * pix
            if len(cnt) != 1 or near_cusp:       # (the 3x3 quadrature below is not adequate at a cusp)
                continue
            # pixel mean of the point-source magnification by 3x3 Gauss-Legendre
            gx = np.array([-math.sqrt(0.6), 0, math.sqrt(0.6)]) * 0.5 * pix
            gw = np.array([5, 8, 5]) / 18.0
            ref = sum(gw[i] * gw[j] * sum(_cr_images(complex(xc + gx[i], yc + gx[j]), a, g_)[1])
                      for i in range(3) for j in range(3))
            tol = 0.02 if cnt == {2} else 0.06           # inside: steep 1/sqrt(d) fold wings
            assert m[iy, ix] == pytest.approx(ref, rel=tol), (ix, iy, cnt)
            n_in += cnt == {4}
            n_out += cnt == {2}
    assert n_in >= 20 and n_out > 1000
    assert cusp1 > cusp2 + 2 * pix            # a flipped shear sign would swap the two axes


# ----------------------------------------------------------------------------- mean magnification
def test_mean_magnification(orc):
    # <mu> over the map = 1/|(1-k)^2-g^2| (eq A4) up to the flux lost outside the
    # eq-16 border (~1 %) and the sampling error over seeds.
    import synth
    k, ks, g_ = 0.4, 0.2, 0.2
    mu = 1 / abs((1 - k) ** 2 - g_ ** 2)
    means = []
    for seed in range(8):
        R = math.sqrt(200 / ks)
        xs, ys, ms = synth.disc_stars(200, R, 500 + seed)
        f = orc.Field.make(k, ks, g_, xs, ys, ms, R=R)
        geo = orc.geometry(k, ks, g_, 5.0, 64, 2.0, 0)
        assert math.hypot(geo.H1, geo.H2) < R
        means.append(orc.shoot(f, geo, 0).mean())
    means = np.array(means)
    sem = means.std(ddof=1) / math.sqrt(len(means))
    assert abs(means.mean() - mu) < 3 * sem + 0.02 * mu
    assert means.mean() < mu * 1.01 + 3 * sem            # flux can only be lost, not gained


# ----------------------------------------------------------------------------- IRS / IPM consistency
def test_irs_binning_rules(orc):
    geo = orc.geometry(0.0, 0.0, 0.0, 1.0, 4, 1.0, 2, 0.0)        # pixels of size 0.5 on [-1,1]
    # lower edge inclusive, upper exclusive (G15); outside dropped
    wx = np.array([-1.0, -0.5, 0.999999, 1.0, 0.0, -1.0000001])
    wy = np.array([-1.0, -0.5, 0.999999, 0.0, 1.0, 0.0])
    c = orc.bin_irs(wx, wy, geo)
    exp = np.zeros((4, 4), dtype=np.uint64)
    exp[0, 0] = 1; exp[1, 1] = 1; exp[3, 3] = 1
    assert np.array_equal(c, exp)


def test_ipm_vs_irs_agree(orc):
    # P:288 "We do not find any differences": IRS at high ray density converges to IPM within Poisson noise
    rng = np.random.default_rng(21)
    xs, ys = rng.uniform(-6, 6, 12), rng.uniform(-6, 6, 12)
    f = orc.Field.make(0.3, 0.0, 0.1, xs, ys, np.ones(12), R=1e9)
    g_ipm = orc.geometry(0.3, 0.0, 0.1, 2.0, 16, 4.0, 3, He=(8.0, 8.0))
    g_irs = orc.geometry(0.3, 0.0, 0.1, 2.0, 16, 24.0, 3, He=(8.0, 8.0))
    ipm = orc.shoot(f, g_ipm, 0)
    irs = orc.shoot(f, g_irs, 1).astype(float) / 24.0 ** 2
    z = (irs - ipm) / np.sqrt(np.maximum(ipm, 0.05) / 24.0 ** 2)
    assert np.mean(np.abs(z) < 5) > 0.95
    assert ipm.mean() == pytest.approx(irs.mean(), rel=5e-3)


def test_subrange_shoot_adds_up(orc):
    # shooting the window in slabs accumulates to the whole (the C-ABI's sub-range contract)
    rng = np.random.default_rng(2)
    xs, ys = rng.uniform(-3, 3, 5), rng.uniform(-3, 3, 5)
    f = orc.Field.make(0.3, 0.0, 0.1, xs, ys, np.ones(5), R=1e9)
    geo = orc.geometry(0.3, 0.0, 0.1, 1.5, 12, 3.0, 3, He=(4.0, 4.0))
    whole = orc.shoot(f, geo, 0)
    acc = np.zeros_like(whole)
    jm = geo.n2 // 3
    orc.shoot(f, geo, 0, sub=(0, geo.n1, 0, jm), out=acc)
    orc.shoot(f, geo, 0, sub=(0, geo.n1, jm, geo.n2), out=acc)
    assert np.allclose(acc, whole, rtol=1e-12, atol=1e-14)


def test_degenerate_triangle_rule_G12(orc):
    """Reading G12: a mapped triangle whose signed area is exactly 0 puts its whole
    weight into the pixel that holds vertex 0, if that pixel is in the map, and nothing anywhere else; no division.
    Hand-built corner grids (2 x 2 corners = one cell = T1 (a, b, c) + T2 (a, c, d)) whose images are collinear."""
    g = orc.geometry(0.0, 0.0, 0.0, 4.0, 8, 1.0, 3, He=(1.0, 1.0))      # 8 x 8 pixels of size 1, lower-left (-4, -4)
    assert (g.p1, g.p2, g.ylo1, g.ylo2) == (1.0, 1.0, -4.0, -4.0)
    w = g.weight

    def cell(a, b, c, d):
        wx = np.array([[a[0], b[0]], [d[0], c[0]]]) + g.ylo1          # row 0 = corners (i, j), (i+1, j); row 1 = (i, j+1), (i+1, j+1)
        wy = np.array([[a[1], b[1]], [d[1], c[1]]]) + g.ylo2
        return orc.deposit_ipm(wx, wy, g)

    # the cell collapsed onto a horizontal segment spanning three pixels: both triangles go to vertex a's pixel (2, 1)
    m = cell((2.3, 1.4), (3.3, 1.4), (4.3, 1.4), (2.8, 1.4))
    assert m[1, 2] == 2 * w and m.sum() == 2 * w
    # onto a diagonal segment (exactly representable, A = 0 exactly): vertex a in pixel (0, 0)
    m = cell((0.5, 0.5), (1.5, 1.5), (2.5, 2.5), (3.5, 3.5))
    assert m[0, 0] == 2 * w and m.sum() == 2 * w
    # onto a single point
    m = cell((5.25, 6.75), (5.25, 6.75), (5.25, 6.75), (5.25, 6.75))
    assert m[6, 5] == 2 * w and m.sum() == 2 * w
    # only T1 degenerate (a, b, c collinear), T2 = (a, c, d) a proper triangle inside pixel (1, 1): 2 w in all, one of them by G12
    m = cell((1.25, 1.25), (1.5, 1.5), (1.75, 1.75), (1.25, 1.75))
    assert m[1, 1] == pytest.approx(2 * w, rel=1e-15) and m.sum() == pytest.approx(2 * w, rel=1e-15)
    # T1 degenerate with vertex a in pixel (1, 1) but b, c elsewhere; T2 proper over pixels of row 1..2: the degenerate
    # weight goes to a's pixel, not to where the segment's other end lies
    m = cell((1.5, 1.5), (2.5, 1.5), (3.5, 1.5), (1.5, 2.5))
    t2 = np.zeros_like(m)
    for qy in range(8):
        for qx in range(8):
            t2[qy, qx] = w * orc.triangle_pixel_area([1.5, 1.5, 3.5, 1.5, 1.5, 2.5], qx, qy) / 1.0   # |A| = 1
    assert np.allclose(m - t2, np.where((np.arange(8)[:, None] == 1) & (np.arange(8)[None, :] == 1), w, 0.0), atol=1e-16)
    # vertex 0 outside the map (the segment itself crosses the map): nothing is deposited
    m = cell((-0.5, 3.5), (2.5, 3.5), (5.5, 3.5), (1.5, 3.5))
    assert m.sum() == 0.0
    # ... and the conservation of a whole map is unchanged by degenerate cells: a grid folded flat along x2 = const
    # (every cell degenerate) carries exactly 2 w per cell whose vertex a lies in the map
    xs = np.linspace(-3.9, 3.9, 14)
    wx = np.tile(xs, (5, 1)); wy = np.full((5, 14), 0.3)
    m = orc.deposit_ipm(wx, wy, g)
    assert m.sum() == pytest.approx(2 * w * 4 * 13, rel=1e-14) and np.count_nonzero(m[:4]) == 0 and np.count_nonzero(m[5:]) == 0
