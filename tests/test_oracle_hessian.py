"""Pins for the oracle's analytic Hessian, independent of its own formulas:
  * Richardson-extrapolated central differences of the oracle GRADIENT (already pinned by test_oracle_mass.py);
  * the information identity  E[d2 ln P/da db + (d ln P/da)(d ln P/db)] = 0  by quadrature over the mass range —
    it involves the second derivatives of both normalisations, which the configs' truth point cannot see;
  * angular: the Hessian of a PDF that is linear in its coefficients is minus the outer product of the scores."""
import numpy as np
import pytest
from scipy import integrate

import mf_datagen as dg
import oracle

LO, HI = dg.MASS_LO, dg.MASS_HI
POINTS = [dg.MASS_TRUTH, dg.MASS_START, (0.4, 5.05, 0.1, 0.7), (0.3, 5.28, 0.02, 0.0), (0.3, 5.28, 0.02, 1e-7),
          (0.7, 5.58, 0.05, 3.0)]


def fd_hessian(kind, ev, lam, lo, hi, rel=1e-4):
    lam = np.asarray(lam, dtype=np.float64)
    K = lam.size
    H = np.zeros((K, K))
    for k in range(K):
        h = rel * max(abs(lam[k]), 0.05)

        def g(step):
            x = lam.copy()
            x[k] += step
            return oracle.nll_grad(kind, ev, x, lo, hi)[1]
        d1 = (g(h) - g(-h)) / (2 * h)
        d2 = (g(h / 2) - g(-h / 2)) / h
        H[k] = (4 * d2 - d1) / 3          # Richardson: O(h^4)
    return 0.5 * (H + H.T)


@pytest.mark.parametrize("lam", POINTS)
def test_mass_hessian_vs_finite_differences(lam):
    m = dg.gen_mass(400, seed=11)
    nll, g, H, bad = oracle.nll_grad_hess(oracle.MASS, m, lam, LO, HI)
    assert bad == 0
    n0, g0, _ = oracle.nll_grad(oracle.MASS, m, lam, LO, HI)
    assert abs(nll - n0) <= 1e-13 * abs(n0) and np.allclose(g, g0, rtol=1e-11, atol=1e-9)   # two algebraic routes
    assert np.allclose(H, H.T, rtol=0, atol=0)
    F = fd_hessian(oracle.MASS, m, lam, LO, HI)
    scale = np.sqrt(np.outer(np.abs(np.diag(F)), np.abs(np.diag(F)))) + 1e-9
    assert np.max(np.abs(H - F) / scale) < 2e-7, (H, F)


@pytest.mark.parametrize("lam", [(0.4, 5.05, 0.1, 0.7), (0.3, 5.28, 0.02, -1.5), (0.6, 5.5, 0.08, 0.0), (0.2, 5.1, 0.05, 1e-6)])
def test_mass_information_identity(lam):
    """int P (l_ab + l_a l_b) dm = 0 for the ten (a, b): wrong second derivatives of N1 or N2 fail this."""
    idx = [(i, j) for i in range(4) for j in range(i, 4)]
    mu, sg = lam[1], lam[2]
    brk = sorted({min(max(mu + k * sg, LO), HI) for k in (-8, -3, 0, 3, 8)})
    for q, (i, j) in enumerate(idx):
        def f(x):
            P, g, h = oracle.mass_hess_points(np.array([x]), lam, LO, HI)
            return P[0] * (h[0, q] + g[0, i] * g[0, j])
        val, _ = integrate.quad(f, LO, HI, points=brk, epsabs=1e-11, epsrel=1e-11, limit=400)
        def fa(x):
            P, g, h = oracle.mass_hess_points(np.array([x]), lam, LO, HI)
            return P[0] * abs(g[0, i] * g[0, j])
        ref, _ = integrate.quad(fa, LO, HI, points=brk, limit=400)
        assert abs(val) < 1e-8 * (1 + ref), ((i, j), val, ref)


def test_angular_hessian():
    ev = dg.gen_angular(300, seed=12)
    lam = dg.ANG_TRUTH
    nll, g, H, bad = oracle.nll_grad_hess(oracle.ANGULAR, ev, lam)
    assert bad == 0
    P, dl = oracle.pdf(oracle.ANGULAR, ev, lam)          # d ln P / d a_k per event, [8][n]
    assert np.allclose(H, dl @ dl.T, rtol=1e-12, atol=0)  # -sum(-s s^T)
    F = fd_hessian(oracle.ANGULAR, ev, lam, 0.0, 0.0, rel=1e-3)
    assert np.max(np.abs(H - F)) < 1e-6 * np.max(np.abs(H))


# ---- 4D model (the model is BASELINE.json configs[3]) ----------------------------------------
FOURD_POINTS = [
    dg.FOURD_TRUTH,
    (0.45, 5.2, 0.12, 0.8, 0.35, 0.11, -0.07, 0.21, 0.3, -0.13, 0.05, 0.09, -0.3, 0.2, 0.25, -0.15),   # N1 != 1, tau > 0
]


@pytest.mark.parametrize("lam", FOURD_POINTS)
def test_4d_hessian_vs_finite_differences(lam):
    ev = dg.gen_4d(150, seed=13)
    nll, g, H, bad = oracle.nll_grad_hess(oracle.FOURD, ev, lam, LO, HI)
    assert bad == 0
    n0, g0, _ = oracle.nll_grad(oracle.FOURD, ev, lam, LO, HI)
    assert abs(nll - n0) <= 1e-13 * abs(n0) and np.allclose(g, g0, rtol=1e-10, atol=1e-9)   # two algebraic routes
    assert np.array_equal(H, H.T)
    F = fd_hessian(oracle.FOURD, ev, lam, LO, HI)
    scale = np.sqrt(np.outer(np.abs(np.diag(F)), np.abs(np.diag(F)))) + 1e-9
    assert np.max(np.abs(H - F) / scale) < 5e-7, np.max(np.abs(H - F) / scale)


@pytest.mark.parametrize("lam", FOURD_POINTS)
def test_4d_information_identity(lam):
    """int P (l_xy + l_x l_y) dm dOmega = 0 for all 136 pairs, on the quadrature grid of test_oracle_4d.py: a wrong or
    missing second derivative of P (any of the seven non-zero families) fails its pair."""
    from test_oracle_4d import mass_nodes, omega_grid
    m, wm = mass_nodes(lam, n=16)
    cl, ck, ph, wo = omega_grid(n=12)
    acc = np.zeros((16, 16))
    ref = np.zeros((16, 16))
    for mi, wi in zip(m, wm):
        ev = np.stack([np.full(cl.size, mi), cl, ck, ph])
        P, g, Hh = oracle.hess_points(oracle.FOURD, ev, lam, LO, HI)
        pw = P * wo * wi
        gg = g[:, :, None] * g[:, None, :]
        acc += np.einsum("e,eij->ij", pw, Hh + gg)
        ref += np.einsum("e,eij->ij", pw, np.abs(gg))
    assert np.max(np.abs(acc) / (1 + ref)) < 1e-8, np.max(np.abs(acc) / (1 + ref))


def test_4d_hessian_structural_zeros():
    """Pairs whose second derivative of P vanishes: l_xy = -l_x l_y exactly (e.g. (mu, tau), (a_k, a_l), (a_k, c))."""
    ev = dg.gen_4d(20, seed=14)
    P, g, H = oracle.hess_points(oracle.FOURD, ev, FOURD_POINTS[1], LO, HI)
    zero_pairs = [(1, 3), (2, 3), (1, 12), (2, 15), (3, 4), (3, 11), (4, 5), (6, 11), (4, 12), (11, 15), (12, 13), (14, 15),
                  (0, 0), (5, 5), (12, 12)]
    for i, j in zero_pairs:
        np.testing.assert_allclose(H[:, i, j], -g[:, i] * g[:, j], rtol=1e-15, atol=0)


# ---- weighted sums and the Fisher matrix of weighted fits (reading R23) ------------
KINDS = [(oracle.MASS, lambda n, s: dg.gen_mass(n, seed=s), dg.MASS_START, LO, HI),
         (oracle.ANGULAR, lambda n, s: dg.gen_angular(n, seed=s), dg.ANG_TRUTH, 0.0, 0.0),
         (oracle.FOURD, lambda n, s: dg.gen_4d(n, seed=s), dg.FOURD_TRUTH, LO, HI)]


@pytest.mark.parametrize("kind,gen,lam,lo,hi", KINDS)
def test_unit_weights_reproduce_the_unweighted_sums_bit_for_bit(kind, gen, lam, lo, hi):
    ev = gen(333, 21)
    n = np.atleast_2d(ev).shape[1]
    ones = np.ones(n)
    for nt in (1, 3):
        a = oracle.nll_grad(kind, ev, lam, lo, hi, nthreads=nt)
        b = oracle.nll_grad(kind, ev, lam, lo, hi, nthreads=nt, weights=ones)
        assert a[0] == b[0] and np.array_equal(a[1], b[1])
    h0 = oracle.nll_grad_hess(kind, ev, lam, lo, hi)
    h1 = oracle.nll_grad_hess(kind, ev, lam, lo, hi, weights=ones)
    assert h0[0] == h1[0] and np.array_equal(h0[1], h1[1]) and np.array_equal(h0[2], h1[2])
    if kind != oracle.FOURD:   # the routine as first written (pinned above) and the weighted one with w = NULL
        h2 = oracle.nll_grad_hess_unweighted_c(kind, ev, lam, lo, hi)
        assert h0[0] == h2[0] and np.array_equal(h0[1], h2[1]) and np.array_equal(h0[2], h2[2])


@pytest.mark.parametrize("kind,gen,lam,lo,hi", KINDS)
def test_integer_weights_equal_event_duplication(kind, gen, lam, lo, hi):
    ev = np.atleast_2d(gen(60, 22))
    rng = np.random.default_rng(5)
    w = rng.integers(0, 4, ev.shape[1]).astype(np.float64)          # 0 drops the event
    dup = np.repeat(ev, w.astype(int), axis=1)
    a = oracle.nll_grad_hess(kind, ev if kind != oracle.MASS else ev[0], lam, lo, hi, weights=w, want_fisher=True)
    b = oracle.nll_grad_hess(kind, dup if kind != oracle.MASS else dup[0], lam, lo, hi, want_fisher=True)
    assert abs(a[0] - b[0]) <= 1e-15 * abs(b[0])
    np.testing.assert_allclose(a[1], b[1], rtol=1e-14, atol=1e-12)
    np.testing.assert_allclose(a[2], b[2], rtol=1e-13, atol=1e-10)
    # the Fisher sum carries w^2, duplication carries w: they agree only where w is 0 or 1
    w01 = (w > 0).astype(np.float64)
    dup01 = ev[:, w > 0]
    c = oracle.nll_grad_hess(kind, ev if kind != oracle.MASS else ev[0], lam, lo, hi, weights=w01, want_fisher=True)
    d = oracle.nll_grad_hess(kind, dup01 if kind != oracle.MASS else dup01[0], lam, lo, hi, want_fisher=True)
    np.testing.assert_allclose(c[3], d[3], rtol=1e-13, atol=1e-10)
    v, g, _ = oracle.nll_grad(kind, ev if kind != oracle.MASS else ev[0], lam, lo, hi, nthreads=2, weights=w)
    assert abs(v - b[0]) <= 1e-15 * abs(b[0])
    np.testing.assert_allclose(g, b[1], rtol=1e-14, atol=1e-12)


@pytest.mark.parametrize("kind,gen,lam,lo,hi", KINDS)
def test_weighted_sums_are_the_per_event_quantities_times_the_weights(kind, gen, lam, lo, hi):
    """The per-event P and scores are pinned elsewhere (test_oracle_mass / angular / 4d); here the sums are rebuilt
    from them in numpy with real, partly negative weights (sWeights are signed)."""
    ev = gen(200, 23)
    n = np.atleast_2d(ev).shape[1]
    w = np.random.default_rng(6).normal(0.8, 0.9, n)
    P, d = oracle.pdf(kind, ev, lam, lo, hi)                       # d ln P / d lambda [K][n]
    _, _, Hh = oracle.hess_points(kind, ev, lam, lo, hi)
    nll, g, H, F, bad = oracle.nll_grad_hess(kind, ev, lam, lo, hi, weights=w, want_fisher=True)
    assert bad == 0
    assert abs(nll + np.sum(w * np.log(P))) < 1e-12 * np.sum(np.abs(w * np.log(P)))
    np.testing.assert_allclose(g, -(d * w).sum(axis=1), rtol=1e-10, atol=1e-9)
    np.testing.assert_allclose(H, -np.einsum("e,eij->ij", w, Hh), rtol=1e-11, atol=1e-8)
    np.testing.assert_allclose(F, (d * w * w) @ d.T, rtol=1e-10, atol=1e-8)
    assert np.all(np.linalg.eigvalsh(F) > -1e-9 * np.max(np.abs(F)))   # a sum of w^2 s s^T is positive semi-definite


def test_weighted_gaussian_closed_form_and_sandwich():
    """Pure Gaussian (f fixed at 1, wide range so N1 = 1): the weighted MLE is the weighted mean / weighted biased
    variance, and H, F and the sandwich H^-1 F H^-1 have closed forms in the weighted moments."""
    rng = np.random.default_rng(7)
    n = 4000
    x = rng.normal(5.3, 0.05, n)
    w = rng.choice([0.2, 1.8], n)
    lo, hi = 5.3 - 40 * 0.05, 5.3 + 40 * 0.05
    r = oracle.fit(oracle.MASS, x, (1.0, 5.29, 0.06, 0.0), fixed=[True, False, False, True], lo=lo, hi=hi, weights=w)
    assert r.converged
    W = w.sum()
    mu = (w * x).sum() / W
    var = (w * (x - mu) ** 2).sum() / W
    sg = np.sqrt(var)
    assert abs(r.lam[1] - mu) < 1e-9 * sg and abs(r.lam[2] - sg) < 1e-9 * sg
    assert abs(r.nll - 0.5 * W * (1 + np.log(2 * np.pi * var))) < 1e-9 * abs(r.nll)
    d = x - mu
    H = np.array([[W / var, 0.0], [0.0, 2 * W / var]])                        # sum w d = 0, sum w d^2 = W var
    s_mu, s_sg = d / var, d * d / sg ** 3 - 1 / sg
    F = np.array([[(w * w * s_mu * s_mu).sum(), (w * w * s_mu * s_sg).sum()],
                  [(w * w * s_mu * s_sg).sum(), (w * w * s_sg * s_sg).sum()]])
    Hi = np.linalg.inv(H)
    np.testing.assert_allclose(r.cov_hesse[1:3, 1:3], Hi, rtol=2e-6, atol=1e-12 * Hi[0, 0])
    np.testing.assert_allclose(r.cov[1:3, 1:3], Hi @ F @ Hi, rtol=2e-6, atol=1e-12 * Hi[0, 0])
    # the analytic weighted Hessian at the minimum against the same closed form
    _, _, Ha, Fa, _ = oracle.nll_grad_hess(oracle.MASS, x, r.lam, lo, hi, weights=w, want_fisher=True)
    np.testing.assert_allclose(Ha[1:3, 1:3], H, rtol=1e-7, atol=1e-6 * H[0, 0])
    np.testing.assert_allclose(Fa[1:3, 1:3], F, rtol=1e-7)


def test_weight_scale_leaves_estimate_and_sandwich_unchanged():
    m = dg.gen_mass(3000, seed=24)
    w = np.random.default_rng(8).uniform(0.3, 1.7, m.size)
    a = oracle.fit(oracle.MASS, m, dg.MASS_TRUTH, lo=LO, hi=HI, weights=w)
    b = oracle.fit(oracle.MASS, m, dg.MASS_TRUTH, lo=LO, hi=HI, weights=7.0 * w)
    assert a.converged and b.converged
    assert np.max(np.abs(a.lam - b.lam) / a.sigma) < 1e-6
    sc = np.sqrt(np.outer(np.diag(a.cov), np.diag(a.cov)))                     # finite-difference Hessians: 1e-5 of sigma_i sigma_j
    assert np.max(np.abs(a.cov - b.cov) / sc) < 1e-5                           # H scales by 7, F by 49
    assert np.max(np.abs(7.0 * b.cov_hesse - a.cov_hesse) / sc) < 1e-5         # H^-1 alone is NOT invariant


def test_sandwich_covariance_gives_unit_pulls_where_the_inverse_hessian_does_not():
    """Toy study with two-valued weights independent of the observable (E[w^2]/E[w] = 1.64): pulls of the mean of a
    pure Gaussian computed with the sandwich errors have unit width, those with H^-1 are too wide by sqrt(1.64)."""
    rng = np.random.default_rng(9)
    pulls_s, pulls_h = [], []
    for t in range(120):
        x = rng.normal(5.3, 0.05, 600)
        w = rng.choice([0.2, 1.8], 600)
        r = oracle.fit(oracle.MASS, x, (1.0, 5.3, 0.05, 0.0), fixed=[True, False, False, True], lo=3.3, hi=7.3, weights=w)
        assert r.converged
        pulls_s.append((r.lam[1] - 5.3) / np.sqrt(r.cov[1, 1]))
        pulls_h.append((r.lam[1] - 5.3) / np.sqrt(r.cov_hesse[1, 1]))
    ws, wh = np.std(pulls_s), np.std(pulls_h)
    assert 0.82 < ws < 1.18, ws                       # 1 +- 3 x 0.065
    assert 1.05 < wh / ws < 1.55, (wh, ws)            # sqrt(1.64) = 1.28 toy by toy up to fluctuations of sum w^2
