"""GPU parity of the second-order kernels (mf_second.cuh: fp64 tensor-core contraction over the event index) against the
oracle: the 4D analytic Hessian, weighted value / gradient / Hessian and the Fisher matrix of weighted
fits (reading R23) for all three families, and weighted fits.
Tolerances: value 1e-11 relative, gradient 1e-9 (1 + |g_k|), second-order matrices 1e-9 (1 + sqrt(|M_aa M_bb|)),
fitted parameters 1e-6 sigma."""
import math

import numpy as np
import pytest

import mf_datagen as dg
import oracle

pytestmark = pytest.mark.gpu
LO, HI = dg.MASS_LO, dg.MASS_HI
FOURD_OFF = (0.45, 5.2, 0.12, 0.8, 0.35, 0.11, -0.07, 0.21, 0.3, -0.13, 0.05, 0.09, -0.3, 0.2, 0.25, -0.15)


@pytest.fixture(scope="module")
def mf():
    import paper_2505_12414_b200 as mf
    from paper_2505_12414_b200 import build
    build.build()
    return mf


@pytest.fixture(scope="module")
def ctx(mf):
    c = mf.Context(0)
    yield c
    c.close()


def mat_close(A, B, what):
    scale = 1.0 + np.sqrt(np.abs(np.outer(np.diag(B), np.diag(B))))
    assert np.all(np.abs(A - B) <= 1e-9 * scale), (what, np.max(np.abs(A - B) / scale))
    assert np.array_equal(A, A.T), what


def val_close(nll, g, o_nll, o_g, what, scale=None):
    ref = abs(o_nll) if scale is None else scale
    assert abs(nll - o_nll) <= 1e-11 * ref, (what, nll, o_nll)
    assert np.all(np.abs(g - o_g) <= 1e-9 * (1 + np.abs(o_g))), (what, g - o_g)


def families(mf):
    return [
        (mf.MF_MASS_GAUSS_EXP, oracle.MASS, lambda n, s: dg.gen_mass(n, seed=s), [dg.MASS_TRUTH, dg.MASS_START, (0.4, 5.05, 0.1, 0.7)], LO, HI),
        (mf.MF_ANGULAR_KSTMUMU, oracle.ANGULAR, lambda n, s: dg.gen_angular(n, seed=s), [dg.ANG_TRUTH], None, None),
        (mf.MF_MASS_X_ANGULAR, oracle.FOURD, lambda n, s: dg.gen_4d(n, seed=s), [dg.FOURD_TRUTH, FOURD_OFF], LO, HI),
    ]


@pytest.mark.parametrize("n", [37, 256, 30_001])
def test_4d_hessian_parity(mf, ctx, n):
    ev = dg.gen_4d(n, seed=31)
    model = ctx.model_create(mf.MF_MASS_X_ANGULAR, ctx.dataset_upload(ev, LO, HI))
    assert model.has_hessian and not model.weighted
    for lam in (dg.FOURD_TRUTH, FOURD_OFF):
        nll, g, H = model.nll_grad_hess(lam)
        o_nll, o_g, o_H, bad = oracle.nll_grad_hess(oracle.FOURD, ev, lam, LO, HI)
        assert bad == 0
        val_close(nll, g, o_nll, o_g, f"n={n}")
        mat_close(H, o_H, f"4D Hessian n={n}")
        n2, g2 = model.nll_grad(lam)           # the value+gradient kernel agrees with the second-order kernel
        assert abs(n2 - nll) <= 1e-12 * abs(nll) and np.all(np.abs(g2 - g) <= 1e-10 * (1 + np.abs(g)))


@pytest.mark.parametrize("fam", [0, 1, 2])
@pytest.mark.parametrize("n", [1, 63, 5_003])
def test_fisher_and_hessian_unweighted(mf, ctx, fam, n):
    kind, okind, gen, lams, lo, hi = families(mf)[fam]
    ev = gen(n, 32)
    model = ctx.model_create(kind, ctx.dataset_upload(ev, lo, hi))
    for lam in lams:
        nll, g, H, F = model.nll_grad_hess_fisher(lam)
        o = oracle.nll_grad_hess(okind, ev, lam, lo or 0.0, hi or 0.0, want_fisher=True)
        val_close(nll, g, o[0], o[1], f"fam {fam} n={n}", scale=max(abs(o[0]), 1.0))
        mat_close(H, o[2], f"Hessian fam {fam} n={n}")
        mat_close(F, o[3], f"Fisher fam {fam} n={n}")
        if fam != 2:                            # the register-accumulator Hessian kernels agree with the contraction
            _, _, H2 = model.nll_grad_hess(lam)
            mat_close(H2, H, "two Hessian kernels")


@pytest.mark.parametrize("fam", [0, 1, 2])
@pytest.mark.parametrize("n", [129, 20_011])
def test_weighted_parity(mf, ctx, fam, n):
    kind, okind, gen, lams, lo, hi = families(mf)[fam]
    ev = gen(n, 33)
    w = np.random.default_rng(40 + fam).normal(0.9, 0.7, n)          # partly negative, like sWeights
    ds = ctx.dataset_upload(ev, lo, hi)
    ds.set_weights(w)
    model = ctx.model_create(kind, ds)
    assert model.weighted
    for lam in lams:
        o = oracle.nll_grad_hess(okind, ev, lam, lo or 0.0, hi or 0.0, weights=w, want_fisher=True)
        P, _ = oracle.pdf(okind, ev, lam, lo or 0.0, hi or 0.0, want_grad=False)
        mag = float(np.sum(np.abs(w * np.log(P))))                   # signed weights: the value can cancel
        nll, g = model.nll_grad(lam)
        val_close(nll, g, o[0], o[1], f"weighted fam {fam}", scale=mag)
        nll, g, H = model.nll_grad_hess(lam)
        val_close(nll, g, o[0], o[1], f"weighted fam {fam}", scale=mag)
        mat_close(H, o[2], f"weighted Hessian fam {fam}")
        nll, g, H, F = model.nll_grad_hess_fisher(lam)
        mat_close(H, o[2], f"weighted Hessian fam {fam}")
        mat_close(F, o[3], f"weighted Fisher fam {fam}")
    # an unweighted model on the same dataset object created BEFORE set_weights would be unaffected; after resetting:
    ds.set_weights(None)
    plain = ctx.model_create(kind, ds)
    assert not plain.weighted
    nll, g = plain.nll_grad(lams[0])
    o_nll, o_g, _ = oracle.nll_grad(okind, ev, lams[0], lo or 0.0, hi or 0.0)
    val_close(nll, g, o_nll, o_g, "unweighted after reset")
    nll, g = model.nll_grad(lams[0])                                  # the weighted model keeps its weights
    o = oracle.nll_grad(okind, ev, lams[0], lo or 0.0, hi or 0.0, weights=w)
    val_close(nll, g, o[0], o[1], "weighted model after reset", scale=mag)


def test_weighted_points_and_async(mf, ctx):
    import torch
    m = dg.gen_mass(7_001, seed=34)
    w = np.random.default_rng(44).uniform(0.2, 1.8, m.size)
    ds = ctx.dataset_upload(m, LO, HI)
    ds.set_weights(w)
    model = ctx.model_create(mf.MF_MASS_GAUSS_EXP, ds)
    pts = dg.gen_lambda_points(20, 5, dg.MASS_TRUTH, 3 * dg.mass_sigma_stat(m.size))
    d_out = torch.zeros((20, 6), dtype=torch.float64, device="cuda")
    model.nll_grad_points(pts, d_out.data_ptr())
    torch.cuda.synchronize()
    res = d_out.cpu().numpy()
    for p in range(20):
        o = oracle.nll_grad(oracle.MASS, m, pts[p], LO, HI, weights=w)
        val_close(res[p, 0], res[p, 1:5], o[0], o[1], f"point {p}")
        assert res[p, 5] == 0.0


def test_weight_errors(mf, ctx):
    m = dg.gen_mass(100, seed=35)
    ds = ctx.dataset_upload(m, LO, HI)
    w = np.ones(100)
    w[17] = np.nan
    with pytest.raises(mf.MoreFitError) as e:
        ds.set_weights(w)
    assert e.value.status == mf.MF_ERR_DATA_RANGE
    toys = dg.gen_mass_toys(2, 100, first_seed=1)
    dst = ctx.dataset_upload(toys, LO, HI, n_toys=2)
    with pytest.raises(mf.MoreFitError) as e:
        dst.set_weights(np.ones(100))
    assert e.value.status == mf.MF_ERR_ARG


def test_second_order_nonpositive_pdf(mf, ctx):
    ev = dg.gen_angular(500, seed=36)
    model = ctx.model_create(mf.MF_ANGULAR_KSTMUMU, ctx.dataset_upload(ev))
    bad = np.array(dg.ANG_TRUTH)
    bad[1] = 5.0                                   # S3 = 5: the PDF goes negative for many events
    with pytest.raises(mf.MoreFitError) as e:
        model.nll_grad_hess_fisher(bad)
    assert e.value.status == mf.MF_NONPOSITIVE_PDF
    _, _, _, nbad = oracle.nll_grad_hess(oracle.ANGULAR, ev, bad)
    assert nbad > 0
    with pytest.raises(mf.MoreFitError) as e:      # domain error through the second-order path
        ctx.model_create(mf.MF_MASS_X_ANGULAR, ctx.dataset_upload(dg.gen_4d(100, seed=3), LO, HI)).nll_grad_hess(
            (0.2, 5.28, -0.02, -1.5) + dg.ANG_TRUTH + dg.BKG_TRUTH)
    assert e.value.status == mf.MF_ERR_PARAM_DOMAIN


def test_bitwise_reproducible(mf, ctx):
    ev = dg.gen_4d(50_000, seed=37)
    model = ctx.model_create(mf.MF_MASS_X_ANGULAR, ctx.dataset_upload(ev, LO, HI))
    a = model.nll_grad_hess_fisher(dg.FOURD_TRUTH)
    for _ in range(3):
        b = model.nll_grad_hess_fisher(dg.FOURD_TRUTH)
        assert a[0] == b[0] and all(np.array_equal(x, y) for x, y in zip(a[1:], b[1:]))


def test_4d_fit_uses_the_analytic_hessian(mf, ctx):
    ev = dg.gen_4d(40_000, seed=38)
    model = ctx.model_create(mf.MF_MASS_X_ANGULAR, ctx.dataset_upload(ev, LO, HI))
    r = model.fit(dg.FOURD_TRUTH)
    o = oracle.fit(oracle.FOURD, ev, dg.FOURD_TRUTH, lo=LO, hi=HI, nthreads=oracle.max_threads())
    assert r.converged and o.converged
    assert np.max(np.abs(r.lam - o.lam) / o.sigma) < 1e-6
    assert r.n_calls <= 12, r.n_calls                       # Newton on the analytic Hessian (finite differences: ~100)
    sc = np.sqrt(np.outer(np.diag(o.cov), np.diag(o.cov)))
    assert np.max(np.abs(r.cov - o.cov) / sc) < 1e-4         # the oracle's covariance is a finite-difference one


@pytest.mark.parametrize("fam", [0, 1])
def test_weighted_fit(mf, ctx, fam):
    kind, okind, gen, lams, lo, hi = families(mf)[fam]
    n = 20_000
    ev = gen(n, 39)
    w = np.random.default_rng(50 + fam).choice([0.2, 1.8], n)
    ds = ctx.dataset_upload(ev, lo, hi)
    ds.set_weights(w)
    model = ctx.model_create(kind, ds)
    start = lams[0]
    r = model.fit(start)
    o = oracle.fit(okind, ev, start, lo=lo or 0.0, hi=hi or 0.0, weights=w, nthreads=oracle.max_threads())
    assert r.converged and o.converged
    assert np.max(np.abs(r.lam - o.lam) / o.sigma) < 1e-6
    sc = np.sqrt(np.outer(np.diag(o.cov), np.diag(o.cov)))
    assert np.max(np.abs(r.cov - o.cov) / sc) < 1e-4         # sandwich covariance H^-1 F H^-1
    assert np.max(np.abs(r.cov - o.cov_hesse) / sc) > 0.1    # ... which is not H^-1 for these weights (E[w^2]/E[w] = 1.64)
