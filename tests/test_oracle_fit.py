"""Pins for the oracle's fit iteration (SURVEY.md §8(c) "Fit"): the closed-form maximum-likelihood
estimate of a pure Gaussian, convergence from the BASELINE start point, covariance scale."""
import math

import numpy as np

import mf_datagen as dg
import oracle


def test_pure_gaussian_closed_form_mle():
    """f fixed at 1, range +-40 sigma (N1 = 1): mu_hat = sample mean, sigma_hat^2 = biased sample
    variance, -ln L_min = (N/2)(1 + ln(2 pi sigma_hat^2)); cov = diag(s^2/N, s^2/(2N))."""
    rng = np.random.default_rng(1)
    n = 5000
    x = rng.normal(5.3, 0.01, n)
    lo, hi = 5.3 - 0.4, 5.3 + 0.4
    r = oracle.fit(oracle.MASS, x, (1.0, 5.301, 0.012, -1.0), fixed=(True, False, False, True), lo=lo, hi=hi)
    assert r.converged
    mean = math.fsum(x) / n
    var = math.fsum((xi - mean) ** 2 for xi in x) / n
    s = math.sqrt(var)
    assert abs(r.lam[1] - mean) < 1e-9 * s / math.sqrt(n) * 1e3   # 1e-6 of its statistical error
    assert abs(r.lam[2] - s) < 1e-6 * s / math.sqrt(2 * n)
    assert abs(r.nll - 0.5 * n * (1 + math.log(2 * math.pi * var))) < 1e-9 * abs(r.nll)
    assert r.lam[0] == 1.0 and r.lam[3] == -1.0
    assert abs(r.cov[1, 1] / (var / n) - 1) < 1e-5
    assert abs(r.cov[2, 2] / (var / (2 * n)) - 1) < 1e-5
    assert abs(r.cov[1, 2]) < 1e-4 * math.sqrt(r.cov[1, 1] * r.cov[2, 2])
    assert np.all(r.cov[0] == 0) and np.all(r.cov[:, 3] == 0)


def test_c0_fit_from_the_baseline_start_point():
    m = dg.gen_mass(10_000, seed=0)
    r = oracle.fit(oracle.MASS, m, dg.MASS_START, lo=dg.MASS_LO, hi=dg.MASS_HI)
    assert r.converged
    _, g, _ = oracle.nll_grad(oracle.MASS, m, r.lam, dg.MASS_LO, dg.MASS_HI)
    # stationary: Newton step below 1e-8 sigma
    assert np.max(np.abs(r.cov @ g) / r.sigma) < 1e-8
    pulls = (r.lam - np.array(dg.MASS_TRUTH)) / r.sigma
    assert np.all(np.abs(pulls) < 4.5)
    # HESSE errors agree with the expected Fisher information (SURVEY.md §8(c) scales) within 10 %
    np.testing.assert_allclose(r.sigma * 100.0, dg.MASS_SQRTN_SIGMA, rtol=0.1)
    # a second start point reaches the same minimum to 1e-6 sigma
    r2 = oracle.fit(oracle.MASS, m, dg.MASS_TRUTH, lo=dg.MASS_LO, hi=dg.MASS_HI)
    assert r2.converged and np.max(np.abs(r2.lam - r.lam) / r.sigma) < 1e-6


def test_angular_fit_is_the_unique_minimum():
    ev = dg.gen_angular(20_000, seed=2)
    r = oracle.fit(oracle.ANGULAR, ev, dg.ANG_TRUTH)
    assert r.converged
    r2 = oracle.fit(oracle.ANGULAR, ev, (0.5, 0, 0, 0, 0, 0, 0, 0))
    assert r2.converged and np.max(np.abs(r2.lam - r.lam) / r.sigma) < 1e-6
    expected = np.array([0.6887, 0.9464, 1.0409, 1.0319, 0.6709, 1.0858, 1.1068, 0.9489])
    np.testing.assert_allclose(r.sigma * math.sqrt(20_000), expected, rtol=0.05)
    assert np.all(np.abs((r.lam - np.array(dg.ANG_TRUTH)) / r.sigma) < 4.5)
