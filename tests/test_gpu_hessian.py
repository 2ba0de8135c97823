"""GPU parity of the analytic Hessian (mf_nll_grad_hess, mf_nll_grad_hess_batch) against the oracle's
(oracle.nll_grad_hess, pinned in tests/test_oracle_hessian.py).  Tolerance: value and gradient as everywhere;
Hessian |dH_ab| <= 1e-9 (1 + sqrt(|H_aa H_bb|)) — the entries are sums of terms of that magnitude that partly cancel."""
import math

import numpy as np
import pytest

import mf_datagen as dg
import oracle

pytestmark = pytest.mark.gpu
LO, HI = dg.MASS_LO, dg.MASS_HI


@pytest.fixture(scope="module")
def mf():
    import paper_2505_12414_b200 as mf
    from paper_2505_12414_b200 import build
    build.build()          # no-op when lib/libmorefit_b200.so is newer than its sources (nvcc, sm_100a)
    return mf


@pytest.fixture(scope="module")
def ctx(mf):
    c = mf.Context(0)
    yield c
    c.close()


def check(nll, g, H, o_nll, o_g, o_H, what):
    assert abs(nll - o_nll) <= 1e-11 * abs(o_nll), what
    assert np.all(np.abs(g - o_g) <= 1e-9 * (1 + np.abs(o_g))), what
    scale = 1.0 + np.sqrt(np.abs(np.outer(np.diag(o_H), np.diag(o_H))))
    assert np.all(np.abs(H - o_H) <= 1e-9 * scale), (what, H - o_H, scale)
    assert np.array_equal(H, H.T)


POINTS = [dg.MASS_TRUTH, dg.MASS_START, (0.4, 5.05, 0.1, 0.7), (0.3, 5.28, 0.02, 0.0), (0.3, 5.28, 0.02, 1e-7),
          (0.7, 5.58, 0.05, 3.0), (0.3, 5.28, 0.02, -40.0)]


@pytest.mark.parametrize("n", [10_000, 10_007, 1, 65, 300_001])
def test_mass_hessian_parity(mf, ctx, n):
    m = dg.gen_mass(n, seed=21)
    model = ctx.model_create(mf.MF_MASS_GAUSS_EXP, ctx.dataset_upload(m, LO, HI))
    assert model.has_hessian
    for lam in POINTS:
        nll, g, H = model.nll_grad_hess(lam)
        o_nll, o_g, o_H, bad = oracle.nll_grad_hess(oracle.MASS, m, lam, LO, HI)
        assert bad == 0
        check(nll, g, H, o_nll, o_g, o_H, f"n={n} lam={lam}")
        n2, g2 = model.nll_grad(lam)           # the value+gradient kernel agrees with the Hessian kernel
        assert abs(n2 - nll) <= 1e-13 * abs(nll) + 1e-300 and np.all(np.abs(g2 - g) <= 1e-11 * (1 + np.abs(g)))


def test_mass_hessian_batch_parity(mf, ctx):
    T, n = 6, 5003
    toys = dg.gen_mass_toys(T, n, first_seed=500)
    model = ctx.model_create(mf.MF_MASS_GAUSS_EXP, ctx.dataset_upload(toys, LO, HI, n_toys=T))
    lams = dg.gen_lambda_points(T, 8, dg.MASS_TRUTH, 3 * dg.mass_sigma_stat(n))
    lams[1] = (0.4, 5.05, 0.1, 0.7)
    active = np.ones(T, dtype=np.uint8)
    active[4] = 0
    nll, g, H = model.nll_grad_hess_batch(lams, active)
    assert math.isnan(nll[4]) and np.all(np.isnan(H[4]))
    for t in range(T):
        if active[t]:
            o_nll, o_g, o_H, _ = oracle.nll_grad_hess(oracle.MASS, toys[t], lams[t], LO, HI)
            check(nll[t], g[t], H[t], o_nll, o_g, o_H, f"toy {t}")


def test_hessian_status(mf, ctx):
    ev = dg.gen_4d(1000, seed=3)
    amodel = ctx.model_create(mf.MF_MASS_X_ANGULAR, ctx.dataset_upload(ev, LO, HI))
    assert amodel.has_hessian                     # single dataset: every family (4D through the second-order kernel)
    assert amodel.fit(dg.FOURD_TRUTH).converged
    ofd = mf.default_fit_opts()
    ofd.analytic_hessian = 0                      # the finite-difference mode stays available (register kernel, n_pad < 1024)
    assert amodel.fit(dg.FOURD_TRUTH, opts=ofd).converged
    toys4 = np.stack([dg.gen_4d(500, seed=s) for s in (1, 2)], axis=1)      # [4][2][500]
    bmodel = ctx.model_create(mf.MF_MASS_X_ANGULAR, ctx.dataset_upload(toys4, LO, HI, n_toys=2))
    assert bmodel.has_hessian                     # batched 4D toys: the second-order kernel toy by toy
    m = dg.gen_mass(1000, seed=0)
    model = ctx.model_create(mf.MF_MASS_GAUSS_EXP, ctx.dataset_upload(m, LO, HI))
    with pytest.raises(mf.MoreFitError) as e:
        model.nll_grad_hess((0.3, 5.28, -1.0, -1.5))
    assert e.value.status == mf.MF_ERR_PARAM_DOMAIN


def test_fit_analytic_vs_finite_difference_vs_oracle(mf, ctx):
    """The Newton fit on the analytic Hessian, the BFGS + finite-difference fit and the oracle's own fit reach the same
    minimum (1e-6 sigma) and the same covariance; the analytic mode needs far fewer evaluations."""
    m = dg.gen_mass(10_000, seed=0)
    model = ctx.model_create(mf.MF_MASS_GAUSS_EXP, ctx.dataset_upload(m, LO, HI))
    oa, of = mf.default_fit_opts(), mf.default_fit_opts()
    assert oa.analytic_hessian == 1
    of.analytic_hessian = 0
    ra, rf = model.fit(dg.MASS_START, opts=oa), model.fit(dg.MASS_START, opts=of)
    o = oracle.fit(oracle.MASS, m, dg.MASS_START, lo=LO, hi=HI)
    assert ra.converged and rf.converged
    assert np.max(np.abs(ra.lam - o.lam) / o.sigma) < 1e-6 and np.max(np.abs(rf.lam - o.lam) / o.sigma) < 1e-6
    assert np.max(np.abs(ra.sigma / o.sigma - 1)) < 1e-6      # analytic covariance vs the oracle's FD covariance
    assert np.max(np.abs(ra.cov - rf.cov) / np.outer(ra.sigma, ra.sigma)) < 1e-5   # FD Hessian error of the other fit
    assert ra.n_calls <= 15 < rf.n_calls
    # fixed parameters work in the analytic mode too
    fx = np.array([0, 0, 0, 1], dtype=np.uint8)
    r2 = model.fit(dg.MASS_START, fixed=fx, opts=oa)
    assert r2.converged and r2.lam[3] == dg.MASS_START[3] and r2.cov[3, 3] == 0.0
    o2 = oracle.fit(oracle.MASS, m, dg.MASS_START, lo=LO, hi=HI, fixed=fx)
    assert np.max(np.abs(r2.lam[:3] - o2.lam[:3]) / o2.sigma[:3]) < 1e-6


def test_fit_batch_analytic(mf, ctx):
    T, n = 64, 2000
    toys = dg.gen_mass_toys(T, n, first_seed=900)
    model = ctx.model_create(mf.MF_MASS_GAUSS_EXP, ctx.dataset_upload(toys, LO, HI, n_toys=T))
    oa, of = mf.default_fit_opts(), mf.default_fit_opts()
    of.analytic_hessian = 0
    ra, rf = model.fit_batch(np.array(dg.MASS_TRUTH), opts=oa), model.fit_batch(np.array(dg.MASS_TRUTH), opts=of)
    assert ra.converged.all() and rf.converged.all()
    assert np.max(np.abs(ra.lam - rf.lam) / rf.sigma) < 1e-6
    # the other fit's covariance is a finite-difference Hessian taken up to 1e-3 sigma from the minimum: loose bound
    assert np.max(np.abs(ra.cov - rf.cov) / (ra.sigma[:, :, None] * ra.sigma[:, None, :])) < 2e-3
    assert ra.n_calls.mean() < 0.5 * rf.n_calls.mean()
    for t in (0, 63):
        o = oracle.fit(oracle.MASS, toys[t], dg.MASS_TRUTH, lo=LO, hi=HI)
        assert np.max(np.abs(ra[t].lam - o.lam) / o.sigma) < 1e-6
        # HESSE: the returned covariance is the inverse of the (oracle's) analytic Hessian at the fitted point
        _, _, H, _ = oracle.nll_grad_hess(oracle.MASS, toys[t], ra[t].lam, LO, HI)
        c = np.linalg.inv(H)
        assert np.max(np.abs(ra[t].cov - c) / np.outer(ra[t].sigma, ra[t].sigma)) < 1e-7


@pytest.mark.parametrize("n", [20_000, 20_011, 37])
def test_angular_hessian_parity(mf, ctx, n):
    ev = dg.gen_angular(n, seed=31)
    model = ctx.model_create(mf.MF_ANGULAR_KSTMUMU, ctx.dataset_upload(ev))
    assert model.has_hessian
    for lam in (dg.ANG_TRUTH, (0.55, 0.03, -0.1, -0.25, 0.02, 0.04, -0.05, 0.03)):
        nll, g, H = model.nll_grad_hess(lam)
        o_nll, o_g, o_H, bad = oracle.nll_grad_hess(oracle.ANGULAR, ev, lam)
        assert bad == 0
        check(nll, g, H, o_nll, o_g, o_H, f"angular n={n}")


def test_angular_hessian_batch_and_fit(mf, ctx):
    T, n = 3, 4000
    ev = np.stack([dg.gen_angular(n, seed=60 + t) for t in range(T)], axis=1)  # [3][T][n]
    model = ctx.model_create(mf.MF_ANGULAR_KSTMUMU, ctx.dataset_upload(ev, n_toys=T))
    lams = np.tile(np.array(dg.ANG_TRUTH), (T, 1))
    lams[1, 0] = 0.5
    nll, g, H = model.nll_grad_hess_batch(lams)
    for t in range(T):
        o_nll, o_g, o_H, _ = oracle.nll_grad_hess(oracle.ANGULAR, ev[:, t, :], lams[t])
        check(nll[t], g[t], H[t], o_nll, o_g, o_H, f"angular toy {t}")
    # the analytic-mode fit of one dataset against the oracle's fit
    one = dg.gen_angular(50_000, seed=2)
    m1 = ctx.model_create(mf.MF_ANGULAR_KSTMUMU, ctx.dataset_upload(one))
    r = m1.fit(dg.ANG_TRUTH)
    o = oracle.fit(oracle.ANGULAR, one, dg.ANG_TRUTH)
    assert r.converged and np.max(np.abs(r.lam - o.lam) / o.sigma) < 1e-6
    assert np.max(np.abs(r.sigma / o.sigma - 1)) < 1e-5
    assert r.n_calls <= 12


def test_fourd_hessian_batch_and_toy_fits(mf, ctx):
    """mf_nll_grad_hess_batch for 4D toys (second-order kernel toy by toy) against the oracle, with an inactive toy and a toy
    whose lambda is outside the parameter domain; then all toys fitted concurrently by Newton steps on that Hessian."""
    T, n = 5, 3_001
    toys = np.stack([dg.gen_4d(n, seed=70 + t) for t in range(T)], axis=1)          # [4][T][n]
    model = ctx.model_create(mf.MF_MASS_X_ANGULAR, ctx.dataset_upload(toys, LO, HI, n_toys=T))
    lams = np.tile(np.array(dg.FOURD_TRUTH), (T, 1))
    lams[1, 4:12] += 0.02
    lams[3, 2] = -0.01                            # sigma < 0
    active = np.ones(T, dtype=np.uint8)
    active[2] = 0
    nll, g, H = model.nll_grad_hess_batch(lams, active)
    assert math.isnan(nll[2]) and np.all(np.isnan(H[2]))
    assert nll[3] == math.inf and np.all(np.isnan(g[3])) and np.all(np.isnan(H[3]))
    for t in (0, 1, 4):
        o_nll, o_g, o_H, bad = oracle.nll_grad_hess(oracle.FOURD, toys[:, t, :], lams[t], LO, HI)
        assert bad == 0
        check(nll[t], g[t], H[t], o_nll, o_g, o_H, f"4D toy {t}")
    fr = model.fit_batch(np.array(dg.FOURD_TRUTH))
    assert np.all(fr.converged) and np.all(fr.n_calls <= 12), fr.n_calls
    for t in (0, 4):
        o = oracle.fit(oracle.FOURD, toys[:, t, :], dg.FOURD_TRUTH, lo=LO, hi=HI)
        assert np.max(np.abs(fr.lam[t] - o.lam) / o.sigma) < 1e-6
