"""The seeded generators: reproducible, in range, and distributed like the model they stand for."""
import math

import numpy as np
from scipy import integrate

import mf_datagen as dg
import oracle


def test_reproducible_and_prefix_stable():
    a = dg.gen_mass(5000, seed=3)
    assert np.array_equal(a, dg.gen_mass(5000, seed=3))
    assert not np.array_equal(a, dg.gen_mass(5000, seed=4))
    toys = dg.gen_mass_toys(3, 1000, first_seed=7)
    assert np.array_equal(toys[1], dg.gen_mass(1000, seed=8))
    ang = dg.gen_angular(3000, seed=2)
    assert np.array_equal(ang[:, :1000], dg.gen_angular(1000, seed=2))
    assert np.array_equal(dg.gen_4d(2000, seed=3), dg.gen_4d(2000, seed=3))


def test_ranges():
    m = dg.gen_mass(20000, seed=0)
    assert m.min() >= dg.MASS_LO and m.max() <= dg.MASS_HI and m.dtype == np.float64
    a = dg.gen_angular(20000, seed=2)
    assert a.shape == (3, 20000) and np.all(np.abs(a[:2]) < 1) and np.all(np.abs(a[2]) <= math.pi)
    d = dg.gen_4d(20000, seed=3)
    assert d.shape == (4, 20000) and d[0].min() >= dg.MASS_LO and d[0].max() <= dg.MASS_HI
    assert np.all(np.abs(d[1:3]) < 1) and np.all(np.abs(d[3]) <= math.pi)


def test_mass_moments_follow_the_model():
    n = 200_000
    m = dg.gen_mass(n, seed=11)
    P = lambda x: oracle.pdf(oracle.MASS, np.array([x]), dg.MASS_TRUTH, dg.MASS_LO, dg.MASS_HI, want_grad=False)[0][0]
    pts = [5.22, 5.26, 5.28, 5.30, 5.34]
    mean = integrate.quad(lambda x: x * P(x), dg.MASS_LO, dg.MASS_HI, points=pts, limit=200)[0]
    var = integrate.quad(lambda x: (x - mean) ** 2 * P(x), dg.MASS_LO, dg.MASS_HI, points=pts, limit=200)[0]
    assert abs(m.mean() - mean) < 5 * math.sqrt(var / n)
    frac = np.mean(np.abs(m - 5.28) < 0.04)
    want = integrate.quad(P, 5.24, 5.32, points=[5.28], limit=200)[0]
    assert abs(frac - want) < 5 * math.sqrt(want * (1 - want) / n)


def test_angular_moments_follow_the_model():
    n = 200_000
    a = dg.gen_angular(n, seed=12)
    FL, S3, S4, S5, AFB, S7, S8, S9 = dg.ANG_TRUTH
    # forward-backward asymmetry in cos(theta_l) is AFB; <cos^2 thK> = (1 + 2 FL)/5 ... from the marginals
    afb = (np.sum(a[0] > 0) - np.sum(a[0] < 0)) / n
    assert abs(afb - AFB) < 5 / math.sqrt(n)
    ck2 = np.mean(a[1] ** 2)
    want = 0.75 * (1 - FL) * (2 / 3 - 2 / 5) + 1.5 * FL * (2 / 5)
    assert abs(ck2 - want) < 5 * 0.3 / math.sqrt(n)
    assert abs(np.mean(np.cos(2 * a[2])) - S3 / 2) < 5 / math.sqrt(2 * n)


def test_lambda_points():
    p = dg.gen_lambda_points(1000, 1001, dg.MASS_TRUTH, 3 * dg.mass_sigma_stat(1_000_000))
    assert p.shape == (1000, 4)
    assert np.all(np.abs(p - np.array(dg.MASS_TRUTH)) <= 3 * dg.mass_sigma_stat(1_000_000))
    assert np.array_equal(p, dg.gen_lambda_points(1000, 1001, dg.MASS_TRUTH, 3 * dg.mass_sigma_stat(1_000_000)))
