"""GPU parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times (500 lambda points per
mf_nll_grad_points call for C1, single evaluations for C2/C3, one batched launch over 4096 toys for C4).
The oracle (OpenMP over event chunks) is called on a SAMPLE of the outputs: it needs ~0.1-3 s per evaluation at
these sizes.  Tolerances are north_star's, as in test_gpu_parity.py."""
import math

import numpy as np
import pytest

import mf_datagen as dg
import oracle

pytestmark = pytest.mark.gpu

NLL_RTOL = 1e-11
GRAD_TOL = 1e-9


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


def check(nll, grad, o_nll, o_grad, what):
    assert abs(nll - o_nll) <= NLL_RTOL * abs(o_nll), f"{what}: nll {nll!r} vs oracle {o_nll!r}"
    err = np.abs(grad - o_grad)
    tol = GRAD_TOL * (1.0 + np.abs(o_grad))
    assert np.all(err <= tol), f"{what}: grad err {err} tol {tol}"


def test_c1_points_mode_full_size(mf, ctx):
    """C1: N = 1e6, the 1,000 seeded lambda points, evaluated 500 per call exactly as bench.py does."""
    import torch
    n = 1_000_000
    m = dg.gen_mass(n, seed=1)
    model = ctx.model_create(mf.MF_MASS_GAUSS_EXP, ctx.dataset_upload(m, dg.MASS_LO, dg.MASS_HI))
    pts = dg.gen_lambda_points(1000, 1001, dg.MASS_TRUTH, 3 * dg.mass_sigma_stat(n))
    out = torch.full((1000, 6), float("nan"), dtype=torch.float64, device="cuda")
    for c in (0, 500):
        model.nll_grad_points(pts[c:c + 500], out[c].data_ptr())
    torch.cuda.synchronize()
    res = out.cpu().numpy()
    assert np.all(np.isfinite(res)) and np.all(res[:, 5] == 0)
    for p in range(1000):                  # every output of both calls (the oracle needs ~12 s for the 1e9 event evaluations)
        o_nll, o_g, _ = oracle.nll_grad(oracle.MASS, m, pts[p], dg.MASS_LO, dg.MASS_HI, nthreads=oracle.max_threads())
        check(res[p, 0], res[p, 1:5], o_nll, o_g, f"C1 point {p}")
    # properties that hold for every point: the lone-call kernel agrees with the points-mode kernel
    for p in (3, 750):
        nll, g = model.nll_grad(pts[p])
        assert abs(nll - res[p, 0]) <= 1e-12 * abs(nll)
        assert np.all(np.abs(g - res[p, 1:5]) <= 1e-10 * (1 + np.abs(g)))


def test_c1_full_fit(mf, ctx):
    """C1's full fit from the BASELINE start point; the GPU fit must satisfy the oracle's gradient = 0 condition."""
    n = 1_000_000
    m = dg.gen_mass(n, seed=1)
    model = ctx.model_create(mf.MF_MASS_GAUSS_EXP, ctx.dataset_upload(m, dg.MASS_LO, dg.MASS_HI))
    r = model.fit(dg.MASS_START)
    assert r.converged
    o_nll, o_g, _ = oracle.nll_grad(oracle.MASS, m, r.lam, dg.MASS_LO, dg.MASS_HI, nthreads=oracle.max_threads())
    assert abs(r.nll - o_nll) <= NLL_RTOL * abs(o_nll)
    # a Newton step from the fitted point, with the oracle's gradient and the fit's covariance, is < 1e-6 sigma
    step = r.cov @ o_g
    assert np.max(np.abs(step) / r.sigma) < 1e-6, (step, r.sigma)
    pull = (r.lam - np.array(dg.MASS_TRUTH)) / r.sigma
    assert np.all(np.abs(pull) < 5)


def test_c2_full_size(mf, ctx):
    ev = dg.gen_angular(1_000_000, seed=2)
    model = ctx.model_create(mf.MF_ANGULAR_KSTMUMU, ctx.dataset_upload(ev))
    for lam in (dg.ANG_TRUTH, (0.55, 0.03, -0.1, -0.25, 0.02, 0.04, -0.05, 0.03)):
        nll, g = model.nll_grad(lam)
        o_nll, o_g, _ = oracle.nll_grad(oracle.ANGULAR, ev, lam, nthreads=oracle.max_threads())
        check(nll, g, o_nll, o_g, "C2")


def _check_full_size_fit(r, o_nll, o_g, truth, what):
    """The fitted point satisfies the ORACLE's stationarity condition: a Newton step from it, taken with the oracle's
    gradient and the fit's covariance, is below 1e-6 sigma in every parameter (north_star's fit tolerance)."""
    assert r.converged, what
    assert abs(r.nll - o_nll) <= NLL_RTOL * abs(o_nll), what
    step = r.cov @ o_g
    assert np.max(np.abs(step) / r.sigma) < 1e-6, (what, step, r.sigma)
    pull = (r.lam - np.array(truth)) / r.sigma
    assert np.all(np.abs(pull) < 5), (what, pull)


def test_c2_full_fit(mf, ctx):
    """C2's full fit (N = 1e6, all 8 coefficients free, from the truth) checked at full size like C1's."""
    ev = dg.gen_angular(1_000_000, seed=2)
    model = ctx.model_create(mf.MF_ANGULAR_KSTMUMU, ctx.dataset_upload(ev))
    r = model.fit(dg.ANG_TRUTH)
    o_nll, o_g, _ = oracle.nll_grad(oracle.ANGULAR, ev, r.lam, nthreads=oracle.max_threads())
    _check_full_size_fit(r, o_nll, o_g, dg.ANG_TRUTH, "C2 fit")


def test_c3_full_size(mf, ctx):
    ev = dg.gen_4d(2_000_000, seed=3)
    model = ctx.model_create(mf.MF_MASS_X_ANGULAR, ctx.dataset_upload(ev, dg.MASS_LO, dg.MASS_HI))
    nll, g = model.nll_grad(dg.FOURD_TRUTH)
    o_nll, o_g, _ = oracle.nll_grad(oracle.FOURD, ev, dg.FOURD_TRUTH, dg.MASS_LO, dg.MASS_HI, nthreads=oracle.max_threads())
    check(nll, g, o_nll, o_g, "C3")
    # C3's full fit (16 free parameters, from the truth) at full size
    r = model.fit(dg.FOURD_TRUTH)
    o_nll, o_g, _ = oracle.nll_grad(oracle.FOURD, ev, r.lam, dg.MASS_LO, dg.MASS_HI, nthreads=oracle.max_threads())
    _check_full_size_fit(r, o_nll, o_g, dg.FOURD_TRUTH, "C3 fit")
    assert r.n_calls <= 12, r.n_calls           # Newton on the analytic Hessian (round 1: 100 evaluations by finite differences)
    # the 136-entry analytic Hessian and the Fisher matrix at full size (second-order kernel) against the oracle
    nll, g, H, F = model.nll_grad_hess_fisher(dg.FOURD_TRUTH)
    o = oracle.nll_grad_hess(oracle.FOURD, ev, dg.FOURD_TRUTH, dg.MASS_LO, dg.MASS_HI, want_fisher=True)
    check(nll, g, o[0], o[1], "C3 second-order")
    for A, B, what in ((H, o[2], "Hessian"), (F, o[3], "Fisher")):
        scale = 1.0 + np.sqrt(np.abs(np.outer(np.diag(B), np.diag(B))))
        assert np.all(np.abs(A - B) <= 1e-9 * scale), (what, np.max(np.abs(A - B) / scale))


def test_c2_many_points_full_size(mf, ctx):
    """Every point of a 64-point call on C2 (1e6 events, one pass over the data: mf_points.cuh) against the oracle."""
    import torch
    ev = dg.gen_angular(1_000_000, seed=2)
    model = ctx.model_create(mf.MF_ANGULAR_KSTMUMU, ctx.dataset_upload(ev))
    pts = np.tile(np.array(dg.ANG_TRUTH), (64, 1)) + np.random.default_rng(5).uniform(-0.03, 0.03, (64, 8))
    out = torch.full((64, 10), float("nan"), dtype=torch.float64, device="cuda")
    model.nll_grad_points(pts, out.data_ptr())
    torch.cuda.synchronize()
    res = out.cpu().numpy()
    assert np.all(res[:, 9] == 0)
    for p in range(64):
        o_nll, o_g, _ = oracle.nll_grad(oracle.ANGULAR, ev, pts[p], nthreads=oracle.max_threads())
        check(res[p, 0], res[p, 1:9], o_nll, o_g, f"C2 point {p}")


def test_c1_weighted_full_size(mf, ctx):
    """C1's events with weights: value, gradient, Hessian and Fisher matrix at N = 1e6, and the weighted fit."""
    m = dg.gen_mass(1_000_000, seed=1)
    w = np.random.default_rng(91).choice([0.2, 1.8], m.size)
    ds = ctx.dataset_upload(m, dg.MASS_LO, dg.MASS_HI)
    ds.set_weights(w)
    model = ctx.model_create(mf.MF_MASS_GAUSS_EXP, ds)
    nll, g, H, F = model.nll_grad_hess_fisher(dg.MASS_START)
    o = oracle.nll_grad_hess(oracle.MASS, m, dg.MASS_START, dg.MASS_LO, dg.MASS_HI, weights=w, want_fisher=True)
    check(nll, g, o[0], o[1], "C1 weighted")
    for A, B, what in ((H, o[2], "Hessian"), (F, o[3], "Fisher")):
        scale = 1.0 + np.sqrt(np.abs(np.outer(np.diag(B), np.diag(B))))
        assert np.all(np.abs(A - B) <= 1e-9 * scale), (what, np.max(np.abs(A - B) / scale))
    r = model.fit(dg.MASS_START)
    assert r.converged
    o_nll, o_g, o_H, o_F, _ = oracle.nll_grad_hess(oracle.MASS, m, r.lam, dg.MASS_LO, dg.MASS_HI, weights=w, want_fisher=True)
    Hi = np.linalg.inv(o_H)
    sand = Hi @ o_F @ Hi                          # the oracle's sandwich covariance at the fitted point
    sig = np.sqrt(np.diag(sand))
    assert np.max(np.abs(Hi @ o_g) / sig) < 1e-6  # the oracle's Newton step from the fitted point
    assert np.max(np.abs(r.cov - sand) / np.sqrt(np.outer(np.diag(sand), np.diag(sand)))) < 1e-6


def test_c4_full_size(mf, ctx):
    """C4: 4096 toys x 1e4 events in one launch, every toy at its own lambda_t; sampled toys against the oracle,
    every toy against the invariants; then all toys fitted concurrently and the pulls checked."""
    T, n = 4096, 10_000
    toys = dg.gen_mass_toys(T, n, first_seed=0)
    model = ctx.model_create(mf.MF_MASS_GAUSS_EXP, ctx.dataset_upload(toys, dg.MASS_LO, dg.MASS_HI, n_toys=T))
    lams = dg.gen_lambda_points(T, 4242, dg.MASS_TRUTH, 3 * dg.mass_sigma_stat(n))
    nll, g = model.nll_grad_batch(lams)
    assert np.all(np.isfinite(nll)) and np.all(np.isfinite(g))
    for t in range(T):                     # every toy (4.1e7 oracle event evaluations, a few seconds)
        o_nll, o_g, _ = oracle.nll_grad(oracle.MASS, toys[t], lams[t], dg.MASS_LO, dg.MASS_HI)
        check(nll[t], g[t], o_nll, o_g, f"C4 toy {t}")
    # a 1-toy model of the same events gives the same numbers (same kernel arithmetic, different tiling)
    one = ctx.model_create(mf.MF_MASS_GAUSS_EXP, ctx.dataset_upload(toys[123], dg.MASS_LO, dg.MASS_HI))
    n1, g1 = one.nll_grad(lams[123])
    assert abs(n1 - nll[123]) <= 1e-12 * abs(n1) and np.all(np.abs(g1 - g[123]) <= 1e-10 * (1 + np.abs(g1)))
    res = model.fit_batch(np.array(dg.MASS_TRUTH))
    assert sum(r.converged for r in res) == T
    pulls = np.array([(r.lam - np.array(dg.MASS_TRUTH)) / r.sigma for r in res])
    # mean 0 +- 1/sqrt(T) = 0.016 (plus O(1/N) bias), width 1 +- 0.011
    assert np.all(np.abs(pulls.mean(0)) < 0.08), pulls.mean(0)
    assert np.all(np.abs(pulls.std(0) - 1.0) < 0.05), pulls.std(0)
    # sampled toys: the batched fit agrees with the oracle's own fit to 1e-6 sigma
    for t in (5, 3000):
        o = oracle.fit(oracle.MASS, toys[t], dg.MASS_TRUTH, lo=dg.MASS_LO, hi=dg.MASS_HI)
        assert np.max(np.abs(res[t].lam - o.lam) / o.sigma) < 1e-6


def test_beyond_4gib_of_events(mf, ctx):
    """Maximum sizes: one dataset of 5.5e8 events (4.4 GB: element and byte offsets beyond 2^32), generated on the device,
    evaluated by the lone kernel and the points-mode kernel, and checked against the oracle on the downloaded events."""
    import torch
    n = 550_000_000
    ds = ctx.generate_mass(31, 1, n, dg.MASS_TRUTH, dg.MASS_LO, dg.MASS_HI)
    model = ctx.model_create(mf.MF_MASS_GAUSS_EXP, ds)
    lam = (0.31, 5.2801, 0.0201, -1.45)
    nll, g = model.nll_grad(lam)
    x = ds.download()[0, 0]
    assert x.size == n and np.all((x >= dg.MASS_LO) & (x <= dg.MASS_HI))
    o_nll, o_g, bad = oracle.nll_grad(oracle.MASS, x, lam, dg.MASS_LO, dg.MASS_HI, nthreads=oracle.max_threads())
    assert bad == 0
    check(nll, g, o_nll, o_g, "5.5e8 events")
    pts = np.tile(np.array(lam), (16, 1))
    out = torch.zeros((16, 6), dtype=torch.float64, device="cuda")
    model.nll_grad_points(pts, out.data_ptr())
    torch.cuda.synchronize()
    r = out.cpu().numpy()
    check(r[15, 0], r[15, 1:5], o_nll, o_g, "5.5e8 events, points mode")
