"""The resident evaluation kernel (mf_model_serve, mf_server.cuh): parity with the oracle through the mailbox path, restart
after the idle time-out, coexistence with launches on the same model, status codes, clean shutdown."""
import math
import time

import numpy as np
import pytest

import mf_datagen as dg
import oracle

pytestmark = pytest.mark.gpu
LO, HI = dg.MASS_LO, dg.MASS_HI
POINTS = [dg.MASS_TRUTH, dg.MASS_START, (0.4, 5.05, 0.1, 0.7), (0.3, 5.28, 0.02, 0.0), (0.9, 5.5, 0.05, 3.0)]


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


def check(nll, g, o_nll, o_g, what):
    assert abs(nll - o_nll) <= 1e-11 * abs(o_nll), (what, nll, o_nll)
    assert np.all(np.abs(g - o_g) <= 1e-9 * (1 + np.abs(o_g))), (what, g - o_g)


@pytest.mark.parametrize("n", [1, 63, 10_000, 300_001])
def test_served_evaluations_match_the_oracle(mf, ctx, n):
    m = dg.gen_mass(n, seed=41)
    model = ctx.model_create(mf.MF_MASS_GAUSS_EXP, ctx.dataset_upload(m, LO, HI))
    model.serve(True)
    for rep in range(2):
        for lam in POINTS:
            nll, g = model.nll_grad(lam)
            o_nll, o_g, _ = oracle.nll_grad(oracle.MASS, m, lam, LO, HI)
            check(nll, g, o_nll, o_g, f"n={n} {lam}")
            nll2, g2, H = model.nll_grad_hess(lam)
            o = oracle.nll_grad_hess(oracle.MASS, m, lam, LO, HI)
            check(nll2, g2, o[0], o[1], f"hess n={n} {lam}")
            scale = 1.0 + np.sqrt(np.abs(np.outer(np.diag(o[2]), np.diag(o[2]))))
            assert np.all(np.abs(H - o[2]) <= 1e-9 * scale)
    a = model.nll_grad(dg.MASS_START)
    for _ in range(5):
        b = model.nll_grad(dg.MASS_START)
        assert a[0] == b[0] and np.array_equal(a[1], b[1])          # bit-reproducible
    model.serve(False)
    nll, g = model.nll_grad(dg.MASS_START)                           # back on the launch path
    o_nll, o_g, _ = oracle.nll_grad(oracle.MASS, m, dg.MASS_START, LO, HI)
    check(nll, g, o_nll, o_g, "after serve(False)")
    model.close()


def test_restart_after_idle_timeout_and_coexistence(mf, ctx):
    import torch
    m = dg.gen_mass(20_000, seed=42)
    model = ctx.model_create(mf.MF_MASS_GAUSS_EXP, ctx.dataset_upload(m, LO, HI))
    model.serve(True)
    o_nll, o_g, _ = oracle.nll_grad(oracle.MASS, m, dg.MASS_TRUTH, LO, HI)
    for pause in (0.0, 0.03, 0.0, 0.05):                             # the kernel leaves after 5 ms without a request
        time.sleep(pause)
        nll, g = model.nll_grad(dg.MASS_TRUTH)
        check(nll, g, o_nll, o_g, f"pause {pause}")
    # launches on the same model and context run beside the resident kernel
    pts = dg.gen_lambda_points(32, 9, dg.MASS_TRUTH, 3 * dg.mass_sigma_stat(m.size))
    out = torch.zeros((32, 6), dtype=torch.float64, device="cuda")
    model.nll_grad_points(pts, out.data_ptr())
    nll, g = model.nll_grad(dg.MASS_START)
    torch.cuda.synchronize()
    res = out.cpu().numpy()
    for p in (0, 31):
        o = oracle.nll_grad(oracle.MASS, m, pts[p], LO, HI)
        check(res[p, 0], res[p, 1:5], o[0], o[1], f"points row {p}")
    o = oracle.nll_grad(oracle.MASS, m, dg.MASS_START, LO, HI)
    check(nll, g, o[0], o[1], "served beside a launch")
    other = ctx.model_create(mf.MF_MASS_GAUSS_EXP, ctx.dataset_upload(m[:5000], LO, HI))   # a second served model
    other.serve(True)
    o2 = oracle.nll_grad(oracle.MASS, m[:5000], dg.MASS_TRUTH, LO, HI)
    for _ in range(3):
        check(*other.nll_grad(dg.MASS_TRUTH), o2[0], o2[1], "second served model")
        check(*model.nll_grad(dg.MASS_TRUTH), o_nll, o_g, "first served model")
    other.close()                                                     # destroyed while serving
    model.close()


def test_served_status_codes(mf, ctx):
    m = dg.gen_mass(2_000, seed=43)
    model = ctx.model_create(mf.MF_MASS_GAUSS_EXP, ctx.dataset_upload(m, LO, HI))
    model.serve(True)
    with pytest.raises(mf.MoreFitError) as e:
        model.nll_grad((0.3, 5.28, -0.02, -1.5))
    assert e.value.status == mf.MF_ERR_PARAM_DOMAIN
    with pytest.raises(mf.MoreFitError) as e:                        # exp(-b0 d^2) underflows for every background-free event
        model.nll_grad((1.0, 5.0, 1e-3, -1.5))
    assert e.value.status == mf.MF_NONPOSITIVE_PDF
    nll, g = model.nll_grad(dg.MASS_TRUTH)                           # still alive afterwards
    o = oracle.nll_grad(oracle.MASS, m, dg.MASS_TRUTH, LO, HI)
    check(nll, g, o[0], o[1], "after errors")
    ang = ctx.model_create(mf.MF_ANGULAR_KSTMUMU, ctx.dataset_upload(dg.gen_angular(1000, seed=2)))
    with pytest.raises(mf.MoreFitError) as e:
        ang.serve(True)
    assert e.value.status == mf.MF_ERR_ARG


def test_fit_is_served_and_agrees_with_the_oracle(mf, ctx):
    m = dg.gen_mass(10_000, seed=0)
    model = ctx.model_create(mf.MF_MASS_GAUSS_EXP, ctx.dataset_upload(m, LO, HI))
    l0 = ctx.kernel_launches
    r = model.fit(dg.MASS_START)                                     # serves itself for the duration of the fit
    assert ctx.kernel_launches - l0 <= 2, "the fit's evaluations must not be kernel launches"
    o = oracle.fit(oracle.MASS, m, dg.MASS_START, lo=LO, hi=HI)
    assert r.converged and np.max(np.abs(r.lam - o.lam) / o.sigma) < 1e-6
    assert np.max(np.abs(r.sigma / o.sigma - 1)) < 1e-6
    ofd = mf.default_fit_opts()
    ofd.analytic_hessian = 0
    rf = model.fit(dg.MASS_START, opts=ofd)
    assert rf.converged and np.max(np.abs(rf.lam - o.lam) / o.sigma) < 1e-6
