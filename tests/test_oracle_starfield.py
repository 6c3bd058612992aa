"""Pins of the oracle's seeded star-field generator."""
import math
import os

import numpy as np
import pytest
from scipy import stats

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def test_splitmix64_known_answers(orc):
    want = [int(l, 16) for l in open(os.path.join(GOLD, "splitmix64_seed0.txt"))
            if l.strip() and not l.startswith("#")]
    assert [orc.rng_draw(0, n) for n in range(3)] == want


def test_disc_field_statistics(orc):
    n, R = 200000, 37.5
    x, y, m = orc.starfield(1234, n, shape=0, a1=R)
    assert np.all(m == 1.0)
    r2 = (x * x + y * y) / (R * R)
    assert r2.max() <= 1.0
    # uniform in area: r^2/R^2 ~ U(0,1), angle ~ U(-pi, pi), independent
    assert stats.kstest(r2, "uniform").pvalue > 1e-3
    assert stats.kstest((np.arctan2(y, x) + math.pi) / (2 * math.pi), "uniform").pvalue > 1e-3
    assert abs(np.corrcoef(r2, np.arctan2(y, x))[0, 1]) < 0.01
    # eq 9: kappa_star = pi theta^2 N <m> / (pi R^2)
    assert n * m.mean() / R ** 2 == pytest.approx(n / R ** 2)
    # different seeds give different fields; same seed the same field; prefix property (counter based)
    x2, _, _ = orc.starfield(1235, 100, shape=0, a1=R)
    x3, _, _ = orc.starfield(1234, 100, shape=0, a1=R)
    assert not np.array_equal(x2, x[:100]) and np.array_equal(x3, x[:100])


def test_unit_vector_accuracy(orc):
    # positions on the unit circle to ~1 ulp: |(x,y)| = r exactly up to rounding, and the angle
    # matches 2 pi u2 of the same counter stream
    n = 5000
    x, y, _ = orc.starfield(77, n, shape=0, a1=1.0)
    u1 = np.array([(orc.rng_draw(77, 3 * i) >> 11) * 2.0 ** -53 for i in range(n)])
    u2 = np.array([(orc.rng_draw(77, 3 * i + 1) >> 11) * 2.0 ** -53 for i in range(n)])
    r = np.sqrt(u1)
    assert np.max(np.abs(x - r * np.cos(2 * math.pi * u2))) < 1e-15
    assert np.max(np.abs(y - r * np.sin(2 * math.pi * u2))) < 1e-15


def test_rect_field(orc):
    n = 100000
    x, y, m = orc.starfield(9, n, shape=1, a1=4.0, a2=0.5)
    assert np.abs(x).max() <= 4.0 and np.abs(y).max() <= 0.5
    assert stats.kstest((x + 4) / 8, "uniform").pvalue > 1e-3
    assert stats.kstest((y + 0.5), "uniform").pvalue > 1e-3


def test_salpeter_masses(orc):
    import synth
    n = 400000
    a, lo, hi = 2.35, 0.08, 1.0
    _, _, m = orc.starfield(5, n, shape=0, a1=1.0, mass_law=1, a=a, lo=lo, hi=hi)
    m1, m2 = synth.salpeter_moments(a, lo, hi)
    # <m> = 0.187283, <m^2> = 0.057242 (closed-form integrals)
    assert m1 == pytest.approx(0.187283, abs=1e-6) and m2 == pytest.approx(0.057242, abs=1e-6)
    assert m.min() >= lo / m1 * (1 - 1e-12) and m.max() <= hi / m1 * (1 + 1e-12)
    assert m.mean() == pytest.approx(1.0, abs=4 * math.sqrt(m2 / m1 ** 2 - 1) / math.sqrt(n))
    assert (m ** 2).mean() == pytest.approx(m2 / m1 ** 2, rel=0.01)
    # CDF of the power law: F(m) = (m^(1-a) - lo^(1-a))/(hi^(1-a) - lo^(1-a))
    e = 1 - a
    F = ((m * m1) ** e - lo ** e) / (hi ** e - lo ** e)
    assert stats.kstest(F, "uniform").pvalue > 1e-3
