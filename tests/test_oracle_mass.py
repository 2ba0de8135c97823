"""Pins for the oracle's mass model (Eq. 2) against things other than itself:
scipy's truncated-normal / truncated-exponential densities, unit integral by adaptive
quadrature, the score identity, Richardson finite differences, mpmath closed forms of the
normalisations, and brute-force sums on tiny inputs."""
import math

import mpmath as mp
import numpy as np
import pytest
from scipy import integrate, stats

import oracle

LO, HI = 5.0, 5.6
POINTS = [
    (0.3, 5.28, 0.02, -1.5),     # BASELINE.json truth
    (0.5, 5.27, 0.03, -1.0),     # BASELINE.json start point
    (0.4, 5.05, 0.1, 0.7),       # off-config: N1 = 0.6915, exercises the erf normalisation
    (0.7, 5.58, 0.05, 2.5),      # peak near the upper edge, rising background
    (0.2, 5.3, 0.15, 0.0),       # tau == 0 branch
    (0.6, 5.2, 0.04, 1e-7),      # tiny tau: cancellation region of N2 and dlnN2/dtau
]


def breakpoints(lam, lo=LO, hi=HI):
    _, mu, s, _ = lam
    pts = [mu + k * s for k in (-8, -3, -1, 0, 1, 3, 8)]
    return [p for p in pts if lo < p < hi]


def P_of(lam, lo=LO, hi=HI):
    return lambda m: oracle.pdf(oracle.MASS, np.array([m]), lam, lo, hi, want_grad=False)[0][0]


def scipy_mixture(m, lam, lo, hi):
    f, mu, s, tau = lam
    sig = stats.truncnorm.pdf(m, (lo - mu) / s, (hi - mu) / s, loc=mu, scale=s)
    w = hi - lo
    if tau == 0.0:
        bkg = np.full_like(m, 1.0 / w)
    elif tau < 0:
        bkg = stats.truncexpon.pdf(m, b=w * -tau, loc=lo, scale=1.0 / -tau)
    else:  # rising exponential = falling exponential in (hi - m)
        bkg = stats.truncexpon.pdf(hi - m, b=w * tau, loc=0.0, scale=1.0 / tau)
    return f * sig + (1.0 - f) * bkg


@pytest.mark.parametrize("lam", POINTS)
def test_pdf_equals_scipy_truncated_mixture(lam):
    m_all = np.linspace(LO, HI, 1201)
    assert np.all(oracle.pdf(oracle.MASS, m_all, lam, LO, HI, want_grad=False)[0] > 0)
    m = m_all[1:-1]  # scipy's truncexpon support test is rounding-sensitive exactly on the edge
    p, _ = oracle.pdf(oracle.MASS, m, lam, LO, HI, want_grad=False)
    ref = scipy_mixture(m, lam, LO, HI)
    np.testing.assert_allclose(p, ref, rtol=2e-12, atol=0)


def test_pdf_paper_table1_values_range_5_7():
    # PAPER.md:158-165 Table 1 and the [5,7] range of PAPER.md:173: N1 = 1 - 1.5e-6 there
    lam = (0.3, 5.28, 0.06, -1.0)
    m = np.linspace(5.0, 7.0, 801)[1:-1]
    p, _ = oracle.pdf(oracle.MASS, m, lam, 5.0, 7.0, want_grad=False)
    np.testing.assert_allclose(p, scipy_mixture(m, lam, 5.0, 7.0), rtol=2e-12)
    n1 = oracle.mass_norms(lam, 5.0, 7.0)["N1"]
    assert abs((1.0 - n1) - float(mp.erfc(mp.mpf("0.28") / (mp.sqrt(2) * mp.mpf("0.06"))) / 2)) < 1e-12


@pytest.mark.parametrize("lam", POINTS)
def test_unit_integral(lam):
    val, err = integrate.quad(P_of(lam), LO, HI, points=breakpoints(lam), epsabs=1e-13, epsrel=1e-13, limit=400)
    assert abs(val - 1.0) < 5e-12


@pytest.mark.parametrize("lam", POINTS)
def test_score_identity(lam):
    """int P dlnP/dlambda_k dm = d/dlambda_k int P dm = 0: catches wrong normalisation derivatives."""
    def integrand(k):
        def fn(m):
            p, d = oracle.pdf(oracle.MASS, np.array([m]), lam, LO, HI)
            return p[0] * d[k, 0]
        return fn
    for k in range(4):
        # scale of the integrand: int P |dlnP_k| dm
        val, _ = integrate.quad(integrand(k), LO, HI, points=breakpoints(lam), epsabs=1e-13, epsrel=1e-13, limit=400)
        scale, _ = integrate.quad(lambda m: abs(integrand(k)(m)), LO, HI, points=breakpoints(lam), limit=400)
        assert abs(val) < 1e-10 * max(scale, 1.0), (k, val, scale)


def richardson(fn, x, h):
    d1 = (fn(x + h) - fn(x - h)) / (2 * h)
    d2 = (fn(x + h / 2) - fn(x - h / 2)) / h
    return (4 * d2 - d1) / 3


@pytest.mark.parametrize("lam", POINTS[:5])
def test_gradient_vs_finite_differences(lam):
    ms = np.array([5.0, 5.013, 5.13, 5.27, 5.28, 5.31, 5.45, 5.6])
    _, d = oracle.pdf(oracle.MASS, ms, lam, LO, HI)
    steps = (1e-3, 1e-3, 2e-4, 1e-3)
    for k in range(4):
        if k == 0 and not (steps[0] < lam[0] < 1 - steps[0]):
            continue
        for j, m in enumerate(ms):
            def lnp(v):
                l = list(lam); l[k] = v
                return math.log(oracle.pdf(oracle.MASS, np.array([m]), l, LO, HI, want_grad=False)[0][0])
            fd = richardson(lnp, lam[k], steps[k])
            assert abs(fd - d[k, j]) < 2e-7 * (1 + abs(d[k, j])), (k, m, fd, d[k, j])


@pytest.mark.parametrize("tau", [-10.0, -1.5, -1e-3, -1e-6, -1e-9, 0.0, 1e-12, 1e-7, 1e-4, 9e-3, 1.1e-2, 0.05, 0.7, 10.0])
def test_exponential_normalisation_against_mpmath(tau):
    mp.mp.dps = 50
    a, b, t = mp.mpf(LO), mp.mpf(HI), mp.mpf(tau)
    if tau == 0.0:
        n2, mean = b - a, (a + b) / 2
    else:
        n2 = (mp.exp(t * b) - mp.exp(t * a)) / t
        mean = ((b * mp.exp(t * b) - a * mp.exp(t * a)) / t - n2 / t) / n2
    got = oracle.mass_norms((0.3, 5.28, 0.02, tau), LO, HI)
    assert abs(got["N2"] / float(n2) - 1) < 4e-16
    assert abs(got["dlnN2_dtau"] / float(mean) - 1) < 4e-16


@pytest.mark.parametrize("mu,s", [(5.28, 0.02), (5.05, 0.1), (5.58, 0.05), (4.9, 0.2), (5.3, 1.0)])
def test_gaussian_normalisation_against_scipy_and_fd(mu, s):
    got = oracle.mass_norms((0.3, mu, s, -1.5), LO, HI)
    ref = stats.norm.cdf(HI, mu, s) - stats.norm.cdf(LO, mu, s)
    assert abs(got["N1"] - ref) < 1e-15
    mp.mp.dps = 40
    N1 = lambda m_, s_: (mp.erf((m_ - LO) / (mp.sqrt(2) * s_)) - mp.erf((m_ - HI) / (mp.sqrt(2) * s_))) / 2
    dmu = mp.diff(lambda v: N1(v, mp.mpf(s)), mp.mpf(mu))
    ds = mp.diff(lambda v: N1(mp.mpf(mu), v), mp.mpf(s))
    assert abs(got["dN1_dmu"] - float(dmu)) < 1e-13 * (1 + abs(float(dmu)))
    assert abs(got["dN1_dsigma"] - float(ds)) < 1e-13 * (1 + abs(float(ds)))


def test_closed_form_special_cases():
    # one event at m = mu, pure Gaussian, range +-40 sigma: -ln L = ln(sqrt(2 pi) sigma)
    mu, s = 5.3, 0.01
    v, g, nb = oracle.nll_grad(oracle.MASS, np.array([mu]), (1.0, mu, s, -1.0), mu - 40 * s, mu + 40 * s)
    assert nb == 0
    assert abs(v - math.log(math.sqrt(2 * math.pi) * s)) < 1e-15
    assert abs(g[1]) < 1e-12 and abs(g[2] - 1.0 / s) < 1e-10  # d(-lnL)/dsigma = +1/sigma at m = mu
    # pure uniform background: f = 0, tau = 0: -ln L = N ln(hi - lo)
    m = np.linspace(LO, HI, 7)
    v, g, _ = oracle.nll_grad(oracle.MASS, m, (0.0, 5.28, 0.02, 0.0), LO, HI)
    assert abs(v - 7 * math.log(HI - LO)) < 1e-14
    # d(-lnL)/dtau at tau = 0 for a uniform background: -(sum m - N (a+b)/2) = 0 for a symmetric grid
    assert abs(g[3]) < 1e-12


def test_sum_is_brute_force_sum_of_log_pdf():
    rng = np.random.default_rng(5)
    m = rng.uniform(LO, HI, 8)
    lam = POINTS[2]
    p, d = oracle.pdf(oracle.MASS, m, lam, LO, HI)
    v, g, nb = oracle.nll_grad(oracle.MASS, m, lam, LO, HI)
    assert nb == 0
    assert abs(v + math.fsum(math.log(x) for x in p)) < 1e-14
    for k in range(4):
        assert abs(g[k] + math.fsum(d[k])) < 1e-13
    # empty input: the empty sum
    v, g, nb = oracle.nll_grad(oracle.MASS, np.empty(0), lam, LO, HI)
    assert v == 0.0 and np.all(g == 0.0) and nb == 0


def test_threads_do_not_change_the_result():
    rng = np.random.default_rng(6)
    m = rng.uniform(LO, HI, 10007)
    lam = POINTS[0]
    v1, g1, _ = oracle.nll_grad(oracle.MASS, m, lam, LO, HI, nthreads=1)
    v3, g3, _ = oracle.nll_grad(oracle.MASS, m, lam, LO, HI, nthreads=3)
    assert abs(v1 - v3) <= 1e-15 * abs(v1)
    np.testing.assert_allclose(g1, g3, rtol=0, atol=1e-12 * np.max(np.abs(g1)))


def test_domain_errors():
    m = np.array([5.1, 5.2])
    for bad in [(-0.1, 5.28, 0.02, -1.5), (1.1, 5.28, 0.02, -1.5), (0.3, 5.28, 0.0, -1.5),
                (0.3, 5.28, -0.02, -1.5), (0.3, float("nan"), 0.02, -1.5), (0.3, 5.28, 0.02, float("inf"))]:
        with pytest.raises(ValueError):
            oracle.nll_grad(oracle.MASS, m, bad, LO, HI)
