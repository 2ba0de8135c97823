"""Pins for the oracle's angular model (Eq. 4): the constants printed in
Listing 4, hand-evaluated points of Eq. 4, unit integral, the closed-form 1D marginals,
the score identity, finite differences and linearity in the coefficients."""
import math
from fractions import Fraction  # noqa: F401  (fixtures use plain python arithmetic)

import numpy as np
import pytest

import oracle

C = 9.0 / (32.0 * math.pi)
TRUTH = (0.6, -0.02, -0.15, -0.2, -0.05, 0.0, -0.02, -0.01)
COEFFS = [
    TRUTH,
    (0.6, 0, 0, 0, 0, 0, 0, 0),                       # the paper's generation values
    (0.35, 0.11, -0.07, 0.21, 0.3, -0.13, 0.05, 0.09),
    (0.8, -0.05, 0.2, -0.1, -0.1, 0.08, -0.12, -0.03),
]
# term index (printed order of Eq. 4) paired with each fitted coefficient FL,S3..S9
TERM_OF_COEFF = {1: 4, 2: 5, 3: 6, 4: 7, 5: 8, 6: 9, 7: 10}


def gl(n, a, b):
    x, w = np.polynomial.legendre.leggauss(n)
    return 0.5 * (b - a) * x + 0.5 * (a + b), 0.5 * (b - a) * w


def grid3(n=48):
    x, wx = gl(n, -1.0, 1.0)
    p, wp = gl(n, -math.pi, math.pi)
    CL, CK, PH = np.meshgrid(x, x, p, indexing="ij")
    W = wx[:, None, None] * wx[None, :, None] * wp[None, None, :]
    return CL, CK, PH, W


def test_listing4_printed_constants(golden_dir):
    """oracle c*term == printed constant * printed expression, for every intact line of Listing 4."""
    col_to_terms = {3: [10], 4: [9], 6: [7], 9: [4], 12: [0], 13: [1]}
    scale = {12: 1.0, 13: 1.0}
    rng = np.random.default_rng(11)
    env = {"sin": math.sin, "cos": math.cos, "sqrt": math.sqrt}
    rows = [l for l in open(f"{golden_dir}/listing4_constants.txt") if l.strip() and not l.startswith("#")]
    assert len(rows) == 6
    for line in rows:
        col, const, expr, _coef = [s.strip() for s in line.split("|")]
        col, const = int(col), float(const)
        for _ in range(20):
            ctl, ctk, phi = rng.uniform(-1, 1), rng.uniform(-1, 1), rng.uniform(-math.pi, math.pi)
            printed = const * eval(expr, {"__builtins__": {}}, dict(env, ctl=ctl, ctk=ctk, phi=phi))
            t = oracle.angular_terms(ctl, ctk, phi)
            got = sum(t[j] for j in col_to_terms[col]) * scale.get(col, 1.0)
            assert abs(got - printed) < 4e-16 + 1e-14 * abs(printed), (col, got, printed)
    # the four distinct printed numbers are c, 4c, 4c/3, 3c/4 with c = 9/(32 pi)
    for printed, mult in [(8.952465548919113e-02, 1.0), (3.580986219567645e-01, 4.0),
                          (1.193662073189215e-01, 4.0 / 3.0), (6.714349161689334e-02, 0.75)]:
        assert abs(printed - mult * C) < 1e-16 * 4


def test_hand_evaluated_points_of_eq4(golden_dir):
    env = {"sqrt": math.sqrt, "pi": math.pi}
    rows = [l for l in open(f"{golden_dir}/eq4_points.txt") if l.strip() and not l.startswith("#")]
    assert len(rows) == 4
    for line in rows:
        thl, thk, phi, terms = [s.strip() for s in line.split("|")]
        thl, thk, phi = (eval(s, {"__builtins__": {}}, env) for s in (thl, thk, phi))
        want = np.array([eval(s, {"__builtins__": {}}, env) for s in terms.split(";")])
        assert want.size == 11
        got = oracle.angular_terms(math.cos(thl), math.cos(thk), phi) / C
        np.testing.assert_allclose(got, want, rtol=0, atol=5e-16)
        # and the PDF assembles them with the coefficients of Eq. 4
        for a in COEFFS:
            FL = a[0]
            p_want = C * ((1 - FL) * want[0] + FL * want[1] + (1 - FL) * want[2] - FL * want[3]
                          + sum(a[k] * want[TERM_OF_COEFF[k]] for k in range(1, 8)))
            ev = np.array([[math.cos(thl)], [math.cos(thk)], [phi]])
            p, d = oracle.pdf(oracle.ANGULAR, ev, a)
            assert abs(p[0] - p_want) < 1e-15
            # d ln P / d S_k = c t_k / P ; d ln P / d FL = c (-t0 + t1 - t2 - t3) / P
            assert abs(d[0, 0] * p[0] - C * (-want[0] + want[1] - want[2] - want[3])) < 1e-15
            for k in range(1, 8):
                assert abs(d[k, 0] * p[0] - C * want[TERM_OF_COEFF[k]]) < 1e-15


@pytest.mark.parametrize("a", COEFFS)
def test_unit_integral_and_term_integrals(a):
    """norm() = 1 for any coefficients: every S_i term integrates to zero."""
    CL, CK, PH, W = grid3()
    ev = np.stack([CL.ravel(), CK.ravel(), PH.ravel()])
    p, d = oracle.pdf(oracle.ANGULAR, ev, a)
    assert abs(np.sum(p * W.ravel()) - 1.0) < 1e-13
    # score identity: int P dlnP/da_k = int dP/da_k = 0 for all eight coefficients
    for k in range(8):
        assert abs(np.sum(p * d[k] * W.ravel())) < 1e-13


@pytest.mark.parametrize("a", COEFFS)
def test_closed_form_marginals(a):
    """dG/dcos(thl) = 3/4 FL (1-cl^2) + 3/8 (1-FL)(1+cl^2) + AFB cl;
    dG/dcos(thK) = 3/4 (1-FL)(1-ck^2) + 3/2 FL ck^2;  dG/dphi = [1 + S3 cos 2phi + S9 sin 2phi]/(2 pi)
    (the standard one-dimensional projections of Eq. 4)."""
    FL, S3, _, _, AFB, _, _, S9 = a
    n = 40
    x, wx = gl(n, -1.0, 1.0)
    ph, wp = gl(n, -math.pi, math.pi)
    for fixed in (-0.83, -0.2, 0.0, 0.41, 0.97):
        CK, PH = np.meshgrid(x, ph, indexing="ij")
        W = (wx[:, None] * wp[None, :]).ravel()
        ev = np.stack([np.full(CK.size, fixed), CK.ravel(), PH.ravel()])
        got = np.sum(oracle.pdf(oracle.ANGULAR, ev, a, want_grad=False)[0] * W)
        want = 0.75 * FL * (1 - fixed**2) + 0.375 * (1 - FL) * (1 + fixed**2) + AFB * fixed
        assert abs(got - want) < 1e-13
        CL, PH = np.meshgrid(x, ph, indexing="ij")
        ev = np.stack([CL.ravel(), np.full(CL.size, fixed), PH.ravel()])
        got = np.sum(oracle.pdf(oracle.ANGULAR, ev, a, want_grad=False)[0] * W)
        want = 0.75 * (1 - FL) * (1 - fixed**2) + 1.5 * FL * fixed**2
        assert abs(got - want) < 1e-13
    for fixed in (-3.0, -1.1, 0.0, 0.6, 2.9):
        CL, CK = np.meshgrid(x, x, indexing="ij")
        W = (wx[:, None] * wx[None, :]).ravel()
        ev = np.stack([CL.ravel(), CK.ravel(), np.full(CL.size, fixed)])
        got = np.sum(oracle.pdf(oracle.ANGULAR, ev, a, want_grad=False)[0] * W)
        want = (1 + S3 * math.cos(2 * fixed) + S9 * math.sin(2 * fixed)) / (2 * math.pi)
        assert abs(got - want) < 1e-13


def test_positive_at_truth_and_zero_on_the_corners():
    rng = np.random.default_rng(3)
    ev = np.stack([rng.uniform(-0.999, 0.999, 200000), rng.uniform(-0.999, 0.999, 200000),
                   rng.uniform(-math.pi, math.pi, 200000)])
    p, _ = oracle.pdf(oracle.ANGULAR, ev, TRUTH, want_grad=False)
    assert p.min() > 0 and p.max() < 0.1111
    for cl in (-1.0, 1.0):
        for ck in (-1.0, 1.0):
            p, _ = oracle.pdf(oracle.ANGULAR, np.array([[cl], [ck], [0.3]]), TRUTH, want_grad=False)
            assert p[0] == 0.0


def test_gradient_vs_finite_differences_and_linearity():
    rng = np.random.default_rng(4)
    ev = np.stack([rng.uniform(-1, 1, 50), rng.uniform(-1, 1, 50), rng.uniform(-math.pi, math.pi, 50)])
    a = np.array(COEFFS[2])
    p, d = oracle.pdf(oracle.ANGULAR, ev, a)
    for k in range(8):
        e = np.zeros(8); e[k] = 1e-3
        pp, _ = oracle.pdf(oracle.ANGULAR, ev, a + e, want_grad=False)
        pm, _ = oracle.pdf(oracle.ANGULAR, ev, a - e, want_grad=False)
        # P is linear in every coefficient: the central difference is exact up to rounding
        np.testing.assert_allclose((pp - pm) / 2e-3, d[k] * p, rtol=0, atol=2e-13)
        np.testing.assert_allclose(pp + pm, 2 * p, rtol=0, atol=1e-15)


def test_nonpositive_pdf_is_flagged():
    ev = np.array([[0.1, 0.2], [0.0, 0.3], [0.5, -0.4]])
    bad = (0.5, 0, 0, 0, -3.0, 0, 0, 0)  # a huge AFB makes P negative for cos(thl) > 0
    p, _ = oracle.pdf(oracle.ANGULAR, ev, bad, want_grad=False)
    assert (p <= 0).sum() == 2
    v, g, nbad = oracle.nll_grad(oracle.ANGULAR, ev, bad)
    assert nbad == 2 and v == math.inf and np.all(np.isnan(g))


def test_sum_is_brute_force():
    rng = np.random.default_rng(8)
    ev = np.stack([rng.uniform(-1, 1, 7), rng.uniform(-1, 1, 7), rng.uniform(-math.pi, math.pi, 7)])
    p, d = oracle.pdf(oracle.ANGULAR, ev, TRUTH)
    v, g, nb = oracle.nll_grad(oracle.ANGULAR, ev, TRUTH)
    assert nb == 0 and abs(v + math.fsum(math.log(x) for x in p)) < 1e-14
    for k in range(8):
        assert abs(g[k] + math.fsum(d[k])) < 1e-13
