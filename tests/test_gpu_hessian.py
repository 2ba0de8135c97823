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
    ev = dg.gen_angular(1000, seed=2)
    amodel = ctx.model_create(mf.MF_ANGULAR_KSTMUMU, ctx.dataset_upload(ev))
    assert not amodel.has_hessian
    with pytest.raises(mf.MoreFitError) as e:
        amodel.nll_grad_hess(dg.ANG_TRUTH)
    assert e.value.status == mf.MF_ERR_ARG
    m = dg.gen_mass(1000, seed=0)
    model = ctx.model_create(mf.MF_MASS_GAUSS_EXP, ctx.dataset_upload(m, LO, HI))
    with pytest.raises(mf.MoreFitError) as e:
        model.nll_grad_hess((0.3, 5.28, -1.0, -1.5))
    assert e.value.status == mf.MF_ERR_PARAM_DOMAIN
