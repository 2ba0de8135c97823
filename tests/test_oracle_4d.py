"""Pins for the oracle's 4D model (BASELINE.json configs[3]):
P = f (G/N1) A(Omega) + (1-f) (E/N2) L(Omega)."""
import math

import numpy as np
import pytest

import oracle

LO, HI = 5.0, 5.6
ANG = (0.6, -0.02, -0.15, -0.2, -0.05, 0.0, -0.02, -0.01)
LAMS = [
    (0.2, 5.28, 0.02, -1.5) + ANG + (0.1, -0.05, 0.1, -0.05),                       # BASELINE truth
    (0.45, 5.2, 0.12, 0.8, 0.35, 0.11, -0.07, 0.21, 0.3, -0.13, 0.05, 0.09, -0.3, 0.2, 0.25, -0.15),  # N1 != 1
]


def gl(n, a, b):
    x, w = np.polynomial.legendre.leggauss(n)
    return 0.5 * (b - a) * x + 0.5 * (a + b), 0.5 * (b - a) * w


def mass_nodes(lam, n=24):
    mu, s = lam[1], lam[2]
    edges = sorted({LO, HI, *[min(max(mu + k * s, LO), HI) for k in (-8, -4, -2, -1, 0, 1, 2, 4, 8)]})
    xs, ws = [], []
    for a, b in zip(edges[:-1], edges[1:]):
        x, w = gl(n, a, b)
        xs.append(x); ws.append(w)
    return np.concatenate(xs), np.concatenate(ws)


def omega_grid(n=20):
    x, wx = gl(n, -1.0, 1.0)
    p, wp = gl(n, -math.pi, math.pi)
    CL, CK, PH = np.meshgrid(x, x, p, indexing="ij")
    W = (wx[:, None, None] * wx[None, :, None] * wp[None, None, :]).ravel()
    return CL.ravel(), CK.ravel(), PH.ravel(), W


@pytest.mark.parametrize("lam", LAMS)
def test_unit_integral_and_score_identity(lam):
    m, wm = mass_nodes(lam)
    cl, ck, ph, wo = omega_grid()
    tot = 0.0
    score = np.zeros(16)
    for mi, wi in zip(m, wm):
        ev = np.stack([np.full(cl.size, mi), cl, ck, ph])
        p, d = oracle.pdf(oracle.FOURD, ev, lam, LO, HI)
        tot += wi * np.sum(p * wo)
        score += wi * (d @ (p * wo))
    assert abs(tot - 1.0) < 1e-11
    assert np.max(np.abs(score)) < 2e-9, score


@pytest.mark.parametrize("lam", LAMS)
def test_marginal_over_angles_is_the_mass_model(lam):
    cl, ck, ph, wo = omega_grid()
    for mi in (5.01, 5.2, 5.27, 5.29, 5.5):
        ev = np.stack([np.full(cl.size, mi), cl, ck, ph])
        p, _ = oracle.pdf(oracle.FOURD, ev, lam, LO, HI, want_grad=False)
        pm, _ = oracle.pdf(oracle.MASS, np.array([mi]), lam[:4], LO, HI, want_grad=False)
        assert abs(np.sum(p * wo) / pm[0] - 1) < 1e-12


def test_factorisation_at_f_0_and_1():
    rng = np.random.default_rng(2)
    n = 100
    ev = np.stack([rng.uniform(LO, HI, n), rng.uniform(-1, 1, n), rng.uniform(-1, 1, n), rng.uniform(-math.pi, math.pi, n)])
    lam = list(LAMS[1])
    lam[0] = 1.0
    p, _ = oracle.pdf(oracle.FOURD, ev, lam, LO, HI, want_grad=False)
    pm, _ = oracle.pdf(oracle.MASS, ev[0], lam[:4], LO, HI, want_grad=False)
    pa, _ = oracle.pdf(oracle.ANGULAR, ev[1:], lam[4:12], want_grad=False)
    np.testing.assert_allclose(p, pm * pa, rtol=1e-14)
    lam[0] = 0.0
    p, _ = oracle.pdf(oracle.FOURD, ev, lam, LO, HI, want_grad=False)
    pm, _ = oracle.pdf(oracle.MASS, ev[0], lam[:4], LO, HI, want_grad=False)
    leg = np.polynomial.legendre.legval
    L = (0.5 * leg(ev[1], [1, lam[12], lam[13]])) * (0.5 * leg(ev[2], [1, lam[14], lam[15]])) / (2 * math.pi)
    np.testing.assert_allclose(p, pm * L, rtol=1e-14)


@pytest.mark.parametrize("lam", LAMS)
def test_gradient_vs_finite_differences(lam):
    rng = np.random.default_rng(9)
    n = 12
    ev = np.stack([rng.uniform(LO, HI, n), rng.uniform(-1, 1, n), rng.uniform(-1, 1, n), rng.uniform(-math.pi, math.pi, n)])
    ev[0, :4] = lam[1] + lam[2] * np.array([-1.5, -0.3, 0.4, 2.0])  # some events under the peak
    _, d = oracle.pdf(oracle.FOURD, ev, lam, LO, HI)
    lam = np.array(lam)
    for k in range(16):
        h = 2e-4 if k == 2 else 1e-3

        def lnp(v):
            l = lam.copy(); l[k] = v
            return np.log(oracle.pdf(oracle.FOURD, ev, l, LO, HI, want_grad=False)[0])
        d1 = (lnp(lam[k] + h) - lnp(lam[k] - h)) / (2 * h)
        d2 = (lnp(lam[k] + h / 2) - lnp(lam[k] - h / 2)) / h
        fd = (4 * d2 - d1) / 3
        np.testing.assert_allclose(fd, d[k], rtol=0, atol=3e-7 * (1 + np.max(np.abs(d[k]))))


def test_sum_is_brute_force():
    rng = np.random.default_rng(10)
    n = 6
    ev = np.stack([rng.uniform(LO, HI, n), rng.uniform(-1, 1, n), rng.uniform(-1, 1, n), rng.uniform(-math.pi, math.pi, n)])
    p, d = oracle.pdf(oracle.FOURD, ev, LAMS[0], LO, HI)
    v, g, nb = oracle.nll_grad(oracle.FOURD, ev, LAMS[0], LO, HI, nthreads=2)
    assert nb == 0 and abs(v + math.fsum(math.log(x) for x in p)) < 1e-13
    for k in range(16):
        assert abs(g[k] + math.fsum(d[k])) < 1e-12 * (1 + abs(g[k]))
