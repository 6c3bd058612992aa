"""Pins of the oracle's map consumers (light curve Fig 4 P:212 / Fig 8, histogram Fig 5 P:216 / Fig 10)
against what the definitions fix: hand values, exactness of bilinear interpolation on affine maps, numpy's own
histogram on the same edges, counts that add up."""
import numpy as np
import pytest


def test_light_curve_nearest_hand_values(orc):
    m = np.arange(12, dtype=float).reshape(3, 4)          # 3 rows (y2), 4 columns (y1); pixel 0.5 x 2, lower left (-1, -3)
    lc = orc.light_curve(m, -1.0, -3.0, 0.5, 2.0, (-1.0, -3.0), (0.99, 2.99), 5, mode=0)
    # samples: (-1,-3) -> pixel (0,0)=0; (-0.5025,-1.5025) -> (0,0)... computed by hand below
    pts = [(-1.0 + (0.99 + 1.0) * t, -3.0 + (2.99 + 3.0) * t) for t in (0, 0.25, 0.5, 0.75, 1.0)]
    want = [m[int(np.floor((y2 + 3.0) / 2.0)), int(np.floor((y1 + 1.0) / 0.5))] for y1, y2 in pts]
    assert list(lc) == want == [0.0, 0.0, 5.0, 10.0, 11.0]   # pixels (0,0), (0,0), (1,1), (2,2), (3,2) worked out by hand
    # lower edge inclusive, upper edge outside; outside the map -> NaN
    lc = orc.light_curve(m, -1.0, -3.0, 0.5, 2.0, (-0.5, -1.0), (1.0, 3.0), 2, mode=0)
    assert lc[0] == m[1, 1] and np.isnan(lc[1])
    assert np.isnan(orc.light_curve(m, -1.0, -3.0, 0.5, 2.0, (-1.1, 0.0), (-1.1, 0.0), 1, mode=0)[0])


def test_light_curve_bilinear_exact_on_affine_maps(orc):
    # mu(y) = a + b y1 + c y2 sampled at pixel centres: bilinear interpolation between centres reproduces it exactly
    npix1, npix2, p1, p2, ylo1, ylo2 = 40, 30, 0.25, 0.5, -3.0, 1.0
    c1 = ylo1 + (np.arange(npix1) + 0.5) * p1
    c2 = ylo2 + (np.arange(npix2) + 0.5) * p2
    m = 2.0 + 0.7 * c1[None, :] - 1.3 * c2[:, None]
    ya, yb, n = (ylo1 + 0.5 * p1, ylo2 + 0.5 * p2), (ylo1 + (npix1 - 0.5) * p1, ylo2 + (npix2 - 0.5) * p2), 257
    lc = orc.light_curve(m, ylo1, ylo2, p1, p2, ya, yb, n, mode=1)
    t = np.arange(n) / (n - 1)
    want = 2.0 + 0.7 * (ya[0] + (yb[0] - ya[0]) * t) - 1.3 * (ya[1] + (yb[1] - ya[1]) * t)
    assert np.max(np.abs(lc - want)) <= 1e-12
    # within half a pixel of the border the indices are clamped: the value of the border pixel along that axis
    lc = orc.light_curve(m, ylo1, ylo2, p1, p2, (ylo1 + 1e-3, c2[7]), (ylo1 + 1e-3, c2[7]), 1, mode=1)
    assert lc[0] == pytest.approx(m[7, 0], abs=1e-12)
    # on a pixel centre both modes give the pixel
    a = orc.light_curve(m, ylo1, ylo2, p1, p2, (c1[5], c2[9]), (c1[5], c2[9]), 1, mode=0)[0]
    b = orc.light_curve(m, ylo1, ylo2, p1, p2, (c1[5], c2[9]), (c1[5], c2[9]), 1, mode=1)[0]
    assert a == m[9, 5] and b == pytest.approx(m[9, 5], abs=1e-13)


def test_histogram_against_numpy_and_hand_values(orc):
    # hand values: edges at 0.1, 1, 10 (mu_ref 1, [-1, 1), 2 bins)
    m = np.array([0.05, 0.1, 0.5, 1.0, 9.999, 10.0, 50.0, -3.0, 0.0, np.nan])
    h = orc.histogram(m, 1.0, -1.0, 1.0, 2)
    assert list(h) == [4, 2, 2, 2]          # below: 0.05, -3, 0, NaN; [0.1,1): 0.1, 0.5; [1,10): 1, 9.999; above: 10, 50
    rng = np.random.default_rng(5)
    mu = 3.0 * 10.0 ** rng.normal(0.0, 0.6, 200000)
    nb, lo, hi = 64, -1.5, 1.5
    h = orc.histogram(mu, 3.0, lo, hi, nb)
    assert int(h.sum()) == mu.size
    edges = 3.0 * np.power(10.0, lo + np.arange(nb + 1) * (hi - lo) / nb)
    ref, _ = np.histogram(mu, bins=edges)     # numpy closes the last bin on the right: no value sits exactly there here
    assert np.array_equal(h[1:-1].astype(np.int64), ref)
    assert h[0] == np.sum(mu < edges[0]) and h[-1] == np.sum(mu >= edges[-1])
    # a log-normal peaks at its median: the two central bins hold the most
    assert abs(int(np.argmax(h[1:-1])) - nb // 2) <= 1
