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


def test_hessian_not_defined_for_4d():
    ev = dg.gen_4d(50, seed=3)
    with pytest.raises(ValueError):
        oracle.nll_grad_hess(oracle.FOURD, ev, dg.FOURD_TRUTH, LO, HI)
