"""GPU parity: the CUDA path (through the C-ABI library) against the CPU oracle, element by
element on the same seeded inputs.  Tolerances are BASELINE.json's north_star:
|d(-lnL)| / |-lnL| <= 1e-11, |d g_k| <= 1e-9 (1 + |g_k|), fitted lambda within 1e-6 sigma_stat."""
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


def assert_parity(nll, grad, o_nll, o_grad, what=""):
    assert abs(nll - o_nll) <= NLL_RTOL * abs(o_nll) + 1e-300, f"{what}: nll {nll!r} vs oracle {o_nll!r}"
    err = np.abs(grad - o_grad)
    tol = GRAD_TOL * (1.0 + np.abs(o_grad))
    assert np.all(err <= tol), f"{what}: grad err {err} tol {tol}"


MASS_POINTS = [
    dg.MASS_TRUTH,
    dg.MASS_START,
    (0.4, 5.05, 0.1, 0.7),      # N1 = 0.69: the erf normalisation and its derivatives matter
    (0.3, 5.28, 0.02, 0.0),     # tau == 0 branch of N2
    (0.3, 5.28, 0.02, 1e-9),    # tiny tau: cancellation-free forms
    (0.0, 5.28, 0.02, -1.5),    # f = 0
    (1.0, 5.3, 0.2, -1.5),      # f = 1
    (0.7, 5.58, 0.05, 3.0),     # peak at the range edge
]


@pytest.mark.parametrize("n", [10_000, 10_007, 1, 63, 64, 65, 129])
def test_mass_parity_sizes(mf, ctx, n):
    m = dg.gen_mass(n, seed=0)
    ds = ctx.dataset_upload(m, dg.MASS_LO, dg.MASS_HI)
    model = ctx.model_create(mf.MF_MASS_GAUSS_EXP, ds)
    for lam in MASS_POINTS:
        o_nll, o_g, nbad = oracle.nll_grad(oracle.MASS, m, lam, dg.MASS_LO, dg.MASS_HI)
        assert nbad == 0
        nll, g = model.nll_grad(lam)
        assert_parity(nll, g, o_nll, o_g, f"mass n={n} lam={lam}")


def test_mass_empty_dataset(mf, ctx):
    ds = ctx.dataset_upload(np.zeros(0), dg.MASS_LO, dg.MASS_HI)
    model = ctx.model_create(mf.MF_MASS_GAUSS_EXP, ds)
    nll, g = model.nll_grad(dg.MASS_TRUTH)
    assert nll == 0.0 and np.all(g == 0.0)


def test_mass_paper_range_point(mf, ctx):
    """The paper's own benchmark values: range [5,7], sigma 0.06, alpha -1."""
    lam = (0.3, 5.28, 0.06, -1.0)
    m = dg.gen_mass(20_000, seed=11, lam=lam, lo=5.0, hi=7.0)
    ds = ctx.dataset_upload(m, 5.0, 7.0)
    model = ctx.model_create(mf.MF_MASS_GAUSS_EXP, ds)
    for pt in [lam, (0.35, 5.3, 0.07, -0.8)]:
        o_nll, o_g, _ = oracle.nll_grad(oracle.MASS, m, pt, 5.0, 7.0)
        nll, g = model.nll_grad(pt)
        assert_parity(nll, g, o_nll, o_g, f"paper range {pt}")


def test_mass_device_columns(mf, ctx):
    import torch
    m = dg.gen_mass(5000, seed=3)
    t = torch.from_numpy(m).cuda()
    ds = ctx.dataset_upload([t], dg.MASS_LO, dg.MASS_HI)
    model = ctx.model_create(mf.MF_MASS_GAUSS_EXP, ds)
    ds.close()  # the model keeps its own reference
    o_nll, o_g, _ = oracle.nll_grad(oracle.MASS, m, dg.MASS_TRUTH, dg.MASS_LO, dg.MASS_HI)
    nll, g = model.nll_grad(dg.MASS_TRUTH)
    assert_parity(nll, g, o_nll, o_g, "device columns")


ANG_POINTS = [
    dg.ANG_TRUTH,
    (0.5, 0, 0, 0, 0, 0, 0, 0),
    (0.7, 0.05, -0.1, 0.1, 0.1, 0.03, 0.04, -0.05),
]


@pytest.mark.parametrize("n", [20_000, 20_011, 37])
def test_angular_parity(mf, ctx, n):
    ev = dg.gen_angular(n, seed=2)
    ds = ctx.dataset_upload(ev)
    model = ctx.model_create(mf.MF_ANGULAR_KSTMUMU, ds)
    for lam in ANG_POINTS:
        o_nll, o_g, nbad = oracle.nll_grad(oracle.ANGULAR, ev, lam)
        assert nbad == 0
        nll, g = model.nll_grad(lam)
        assert_parity(nll, g, o_nll, o_g, f"angular n={n} lam={lam}")


FOURD_POINTS = [
    dg.FOURD_TRUTH,
    (0.25, 5.27, 0.025, -1.2, 0.55, 0.01, -0.1, -0.15, -0.02, 0.02, 0.0, 0.03, 0.15, -0.1, 0.05, 0.02),
    (0.4, 5.05, 0.1, 0.7) + dg.ANG_TRUTH + (-0.2, 0.1, 0.3, 0.2),
]


@pytest.mark.parametrize("n", [30_000, 30_001])
def test_fourd_parity(mf, ctx, n):
    ev = dg.gen_4d(n, seed=3)
    ds = ctx.dataset_upload(ev, dg.MASS_LO, dg.MASS_HI)
    model = ctx.model_create(mf.MF_MASS_X_ANGULAR, ds)
    for lam in FOURD_POINTS:
        o_nll, o_g, nbad = oracle.nll_grad(oracle.FOURD, ev, lam, dg.MASS_LO, dg.MASS_HI)
        assert nbad == 0
        nll, g = model.nll_grad(lam)
        assert_parity(nll, g, o_nll, o_g, f"4d n={n}")


def test_bitwise_reproducible(mf, ctx):
    ev = dg.gen_4d(50_000, seed=5)
    ds = ctx.dataset_upload(ev, dg.MASS_LO, dg.MASS_HI)
    model = ctx.model_create(mf.MF_MASS_X_ANGULAR, ds)
    ref = model.nll_grad(dg.FOURD_TRUTH)
    for _ in range(20):
        nll, g = model.nll_grad(dg.FOURD_TRUTH)
        assert nll == ref[0] and np.array_equal(g, ref[1])


def test_status_codes(mf, ctx):
    m = dg.gen_mass(1000, seed=0)
    ds = ctx.dataset_upload(m, dg.MASS_LO, dg.MASS_HI)
    model = ctx.model_create(mf.MF_MASS_GAUSS_EXP, ds)
    for bad in [(1.2, 5.28, 0.02, -1.5), (0.3, 5.28, -0.02, -1.5), (0.3, 5.28, 0.0, -1.5), (0.3, math.nan, 0.02, -1.5)]:
        st, nll, g = model.nll_grad_status(bad)
        assert st == mf.MF_ERR_PARAM_DOMAIN
        assert math.isnan(nll) and np.all(np.isnan(g))  # outputs untouched
        assert not oracle.check_domain(oracle.MASS, bad)
    # angular coefficients that make P negative for some events
    ev = dg.gen_angular(5000, seed=2)
    ads = ctx.dataset_upload(ev)
    amodel = ctx.model_create(mf.MF_ANGULAR_KSTMUMU, ads)
    lam = (0.6, 0.9, 0.9, -0.9, 0.9, 0.9, 0.9, 0.9)
    _, _, nbad = oracle.nll_grad(oracle.ANGULAR, ev, lam)
    assert nbad > 0
    st, nll, g = amodel.nll_grad_status(lam)
    assert st == mf.MF_NONPOSITIVE_PDF and nll == math.inf and np.all(np.isnan(g))
    # next call is clean again
    nll, g = amodel.nll_grad(dg.ANG_TRUTH)
    o_nll, o_g, _ = oracle.nll_grad(oracle.ANGULAR, ev, dg.ANG_TRUTH)
    assert_parity(nll, g, o_nll, o_g, "after a P<=0 call")
    # data outside the range
    with pytest.raises(mf.MoreFitError) as e:
        ctx.dataset_upload(np.array([5.1, 5.7, 5.2]), dg.MASS_LO, dg.MASS_HI)
    assert e.value.status == mf.MF_ERR_DATA_RANGE
    with pytest.raises(mf.MoreFitError) as e:
        ctx.dataset_upload(np.array([5.1, math.nan]), dg.MASS_LO, dg.MASS_HI)
    assert e.value.status == mf.MF_ERR_DATA_RANGE
    with pytest.raises(mf.MoreFitError) as e:
        ctx.model_create(mf.MF_ANGULAR_KSTMUMU, ds)  # ndim mismatch
    assert e.value.status == mf.MF_ERR_ARG


@pytest.mark.parametrize("n_events", [1000, 1003, 70_001])
def test_batch_parity(mf, ctx, n_events):
    """mf_nll_grad_batch: every toy at its own lambda_t in one launch (70,001 events: several CTAs per toy)."""
    T = 7
    toys = dg.gen_mass_toys(T, n_events, first_seed=100)
    ds = ctx.dataset_upload(toys, dg.MASS_LO, dg.MASS_HI, n_toys=T)
    model = ctx.model_create(mf.MF_MASS_GAUSS_EXP, ds)
    lams = dg.gen_lambda_points(T, 5, dg.MASS_TRUTH, 3 * dg.mass_sigma_stat(n_events))
    lams[1] = (0.4, 5.05, 0.1, 0.7)
    lams[2] = (0.3, 5.28, 0.02, 0.0)
    active = np.ones(T, dtype=np.uint8)
    active[3] = 0
    nll, g = model.nll_grad_batch(lams, active)
    assert math.isnan(nll[3]) and np.all(np.isnan(g[3]))   # untouched
    for t in range(T):
        if not active[t]:
            continue
        o_nll, o_g, _ = oracle.nll_grad(oracle.MASS, toys[t], lams[t], dg.MASS_LO, dg.MASS_HI)
        assert_parity(nll[t], g[t], o_nll, o_g, f"toy {t}")
    # a toy outside the domain gets +inf / NaN, the others are unaffected
    lams2 = lams.copy()
    lams2[0] = (0.3, 5.28, -1.0, -1.5)
    nll2, g2 = model.nll_grad_batch(lams2)
    assert nll2[0] == math.inf and np.all(np.isnan(g2[0]))
    assert nll2[1] == nll[1] and np.array_equal(g2[1], g[1])


def test_batch_many_toys_active_subset(mf, ctx):
    """More toys than CTAs resident at once (the kernel then requests the events of the toy `ahead` slots further on while it
    evaluates its own, through the list of active toys), ragged toy length (not a multiple of the 256-event group), an active
    subset: EVERY active toy against the oracle; inactive rows untouched; a second call with all toys active."""
    T, n = 700, 1337
    toys = dg.gen_mass_toys(T, n, first_seed=4000)
    model = ctx.model_create(mf.MF_MASS_GAUSS_EXP, ctx.dataset_upload(toys, dg.MASS_LO, dg.MASS_HI, n_toys=T))
    lams = dg.gen_lambda_points(T, 6, dg.MASS_TRUTH, 3 * dg.mass_sigma_stat(n))
    active = (np.random.default_rng(8).uniform(size=T) < 0.6).astype(np.uint8)
    active[0] = 0
    active[T - 1] = 1
    nll, g = model.nll_grad_batch(lams, active)
    for t in range(T):
        if not active[t]:
            assert math.isnan(nll[t]) and np.all(np.isnan(g[t]))
            continue
        o_nll, o_g, _ = oracle.nll_grad(oracle.MASS, toys[t], lams[t], dg.MASS_LO, dg.MASS_HI)
        assert_parity(nll[t], g[t], o_nll, o_g, f"toy {t} (subset)")
    nll_all, g_all = model.nll_grad_batch(lams)
    for t in range(T):
        if active[t]:  # the same toy at the same point: the same bits, whatever its slot and neighbours
            assert nll_all[t] == nll[t] and np.array_equal(g_all[t], g[t])
        else:
            o_nll, o_g, _ = oracle.nll_grad(oracle.MASS, toys[t], lams[t], dg.MASS_LO, dg.MASS_HI)
            assert_parity(nll_all[t], g_all[t], o_nll, o_g, f"toy {t} (all)")


def test_batch_cta_size_by_number_of_toys(mf, ctx):
    """The library picks the toy kernel's CTA size from the number of active toys (4 warps, 2 warps from 24 toys per SM, 1 warp
    from 40 per SM on: 3552 / 5920 on a B200): 6000 toys of 300 events cross both thresholds when evaluated in full and as
    subsets of 4000 and 1000; sampled toys against the oracle, and a toy's result must not depend on which CTA size ran it
    beyond the summation order (same tolerance)."""
    T, n = 6000, 300
    toys = dg.gen_mass_toys(T, n, first_seed=7000)
    model = ctx.model_create(mf.MF_MASS_GAUSS_EXP, ctx.dataset_upload(toys, dg.MASS_LO, dg.MASS_HI, n_toys=T))
    lams = dg.gen_lambda_points(T, 12, dg.MASS_TRUTH, 0.5 * dg.mass_sigma_stat(n))
    results = []
    for n_act in (T, 4000, 1000):
        active = np.zeros(T, dtype=np.uint8)
        active[np.random.default_rng(n_act).choice(T, n_act, replace=False)] = 1
        active[0] = active[T - 1] = 1
        nll, g = model.nll_grad_batch(lams, active)
        results.append((active, nll, g))
        for t in list(range(0, T, 397)) + [T - 1]:
            if not active[t]:
                continue
            o_nll, o_g, _ = oracle.nll_grad(oracle.MASS, toys[t], lams[t], dg.MASS_LO, dg.MASS_HI)
            assert_parity(nll[t], g[t], o_nll, o_g, f"{n_act} active, toy {t}")
    (a0, n0, g0), (a1, n1, g1), (a2, n2, g2) = results
    both = np.flatnonzero(a1 & a2)
    assert len(both) > 100
    assert np.all(np.abs(n0[both] - n2[both]) <= 1e-12 * np.abs(n0[both]))
    assert np.all(np.abs(g1[both] - g2[both]) <= 1e-9 * (1 + np.abs(g2[both])))


def test_batch_angular_parity(mf, ctx):
    T, n = 3, 4000
    ev = np.stack([dg.gen_angular(n, seed=40 + t) for t in range(T)], axis=1)  # [3][T][n]
    ds = ctx.dataset_upload(ev, n_toys=T)
    model = ctx.model_create(mf.MF_ANGULAR_KSTMUMU, ds)
    lams = np.array(ANG_POINTS)
    nll, g = model.nll_grad_batch(lams)
    for t in range(T):
        o_nll, o_g, _ = oracle.nll_grad(oracle.ANGULAR, ev[:, t, :], lams[t])
        assert_parity(nll[t], g[t], o_nll, o_g, f"angular toy {t}")


def _assert_fit_agrees(r, o):
    assert r.converged and o.converged
    assert np.max(np.abs(r.lam - o.lam) / o.sigma) < 1e-6, (r.lam, o.lam, o.sigma)
    np.testing.assert_allclose(r.sigma, o.sigma, rtol=1e-4)
    assert abs(r.nll - o.nll) <= 1e-11 * abs(o.nll)


def test_fit_c0(mf, ctx):
    """BASELINE.json configs[0]: full fit from (0.5, 5.27, 0.03, -1.0)."""
    m = dg.gen_mass(10_000, seed=0)
    ds = ctx.dataset_upload(m, dg.MASS_LO, dg.MASS_HI)
    model = ctx.model_create(mf.MF_MASS_GAUSS_EXP, ds)
    r = model.fit(dg.MASS_START)
    o = oracle.fit(oracle.MASS, m, dg.MASS_START, lo=dg.MASS_LO, hi=dg.MASS_HI)
    _assert_fit_agrees(r, o)
    # fixed parameters stay put and get zero covariance
    r2 = model.fit(dg.MASS_START, fixed=[0, 0, 0, 1])
    o2 = oracle.fit(oracle.MASS, m, dg.MASS_START, fixed=[0, 0, 0, 1], lo=dg.MASS_LO, hi=dg.MASS_HI)
    assert r2.lam[3] == dg.MASS_START[3] and np.all(r2.cov[3] == 0)
    assert np.max(np.abs(r2.lam[:3] - o2.lam[:3]) / o2.sigma[:3]) < 1e-6


def test_fit_angular(mf, ctx):
    ev = dg.gen_angular(20_000, seed=2)
    ds = ctx.dataset_upload(ev)
    model = ctx.model_create(mf.MF_ANGULAR_KSTMUMU, ds)
    r = model.fit(dg.ANG_TRUTH)
    o = oracle.fit(oracle.ANGULAR, ev, dg.ANG_TRUTH)
    _assert_fit_agrees(r, o)


def test_fit_fourd(mf, ctx):
    ev = dg.gen_4d(20_000, seed=3)
    ds = ctx.dataset_upload(ev, dg.MASS_LO, dg.MASS_HI)
    model = ctx.model_create(mf.MF_MASS_X_ANGULAR, ds)
    r = model.fit(dg.FOURD_TRUTH)
    o = oracle.fit(oracle.FOURD, ev, dg.FOURD_TRUTH, lo=dg.MASS_LO, hi=dg.MASS_HI, nthreads=oracle.max_threads())
    _assert_fit_agrees(r, o)


def test_fit_batch_small(mf, ctx):
    """mf_fit_batch: concurrent toy fits agree with one oracle fit per toy."""
    T, n = 6, 2000
    toys = dg.gen_mass_toys(T, n, first_seed=0)
    ds = ctx.dataset_upload(toys, dg.MASS_LO, dg.MASS_HI, n_toys=T)
    model = ctx.model_create(mf.MF_MASS_GAUSS_EXP, ds)
    res = model.fit_batch(np.array(dg.MASS_TRUTH))
    for t in range(T):
        o = oracle.fit(oracle.MASS, toys[t], dg.MASS_TRUTH, lo=dg.MASS_LO, hi=dg.MASS_HI)
        _assert_fit_agrees(res[t], o)


def _ulp_err(y, ref):
    return np.abs(y - ref) / np.spacing(np.abs(ref))


def test_device_math_accuracy(mf, ctx):
    """The kernels' own exp / log / reciprocal (mf_math.cuh) against numpy's libm: a few ulp at most."""
    from paper_2505_12414_b200 import probe
    rng = np.random.default_rng(0)
    x = np.concatenate([rng.uniform(-707.9, 700.0, 200_000), rng.uniform(-5, 5, 200_000), [0.0, -0.0, 1e-300, -1e-300]])
    y = probe.math("exp", x)
    assert np.max(_ulp_err(y, np.exp(x))) <= 2.0
    assert np.all(probe.math("exp", np.array([-708.0, -750.0, -1e4, -1e300])) == 0.0)
    y32 = probe.math("exp32", x)   # the table-by-shuffle variant used inside the event loops
    assert np.max(_ulp_err(y32, np.exp(x))) <= 2.0
    tiny = probe.math("exp32", np.array([-709.5, -750.0, -1e4, -9e11]))   # clamped, not flushed: callers treat < 2^-1000 as 0
    assert np.all((tiny >= 2.0 ** -1022) & (tiny <= 2.0 ** -1021))
    assert probe.math("exp32", np.array([0.0]))[0] == 1.0
    v = np.concatenate([np.exp(rng.uniform(-700, 700, 200_000)), rng.uniform(0.5, 2.0, 200_000),
                        1.0 + rng.uniform(-1e-3, 1e-3, 100_000), [1.0, 2.0, 0.5, 2.2250738585072014e-308]])
    lg = probe.math("log", v)
    ref = np.log(v)
    # absolute error matters for sums of ln P: <= 2 ulp of max(|ln v|, ~0.35) (log is exact at 1)
    assert np.max(np.abs(lg - ref) / np.spacing(np.maximum(np.abs(ref), 0.35))) <= 2.0
    assert probe.math("log", np.array([1.0]))[0] == 0.0
    r = probe.math("rcp", v)
    assert np.max(_ulp_err(r, 1.0 / v)) <= 2.0


def test_points_and_pipelining(mf, ctx):
    """mf_nll_grad_points: 40 back-to-back evaluations (more than the scratch ring holds, programmatic dependent
    launch between them) give, point by point, exactly what mf_nll_grad gives, and match the oracle."""
    import torch
    n = 100_003
    m = dg.gen_mass(n, seed=5)
    model = ctx.model_create(mf.MF_MASS_GAUSS_EXP, ctx.dataset_upload(m, dg.MASS_LO, dg.MASS_HI))
    pts = dg.gen_lambda_points(40, 77, dg.MASS_TRUTH, 3 * dg.mass_sigma_stat(n))
    out = torch.full((40, 6), float("nan"), dtype=torch.float64, device="cuda")
    for _ in range(3):                      # repeated: the ring wraps many times
        model.nll_grad_points(pts, out.data_ptr())
    out2 = torch.full((40, 6), float("nan"), dtype=torch.float64, device="cuda")
    model.nll_grad_points(pts, out2.data_ptr())
    torch.cuda.synchronize()
    res = out.cpu().numpy()
    assert np.array_equal(res, out2.cpu().numpy())      # a series is bit-reproducible
    assert np.all(res[:, 5] == 0)
    for p in (0, 1, 7, 39):
        nll, g = model.nll_grad(pts[p])   # the lone call uses a larger grid: same value up to summation order
        assert abs(res[p, 0] - nll) <= 1e-13 * abs(nll) and np.all(np.abs(res[p, 1:5] - g) <= 1e-11 * (1 + np.abs(g)))
        o_nll, o_g, _ = oracle.nll_grad(oracle.MASS, m, pts[p], dg.MASS_LO, dg.MASS_HI)
        assert_parity(res[p, 0], res[p, 1:5], o_nll, o_g, f"point {p}")
    # a point outside the domain stops the series with MF_ERR_PARAM_DOMAIN
    bad = pts.copy()
    bad[3, 2] = -1.0
    with pytest.raises(mf.MoreFitError):
        model.nll_grad_points(bad, out.data_ptr())
    torch.cuda.synchronize()


def test_overlapping_points_calls(mf, ctx):
    """Back-to-back mf_nll_grad_points calls overlap on the GPU (constants read in place, the wait only before the shared
    scratch is written): 60 calls of varying size on two models, more than the staging ring holds, the same output rows
    written again and again — every call gives bit for bit what the same call gives when the stream is drained first, all
    rows match the oracle at sampled points, and a sweep (sub-calls of 128 points) agrees with them."""
    import torch
    n1, n2 = 300_007, 70_001
    m1, m2 = dg.gen_mass(n1, seed=21), dg.gen_mass(n2, seed=22)
    mod1 = ctx.model_create(mf.MF_MASS_GAUSS_EXP, ctx.dataset_upload(m1, dg.MASS_LO, dg.MASS_HI))
    mod2 = ctx.model_create(mf.MF_MASS_GAUSS_EXP, ctx.dataset_upload(m2, dg.MASS_LO, dg.MASS_HI))
    pts = dg.gen_lambda_points(350, 9, dg.MASS_TRUTH, 3 * dg.mass_sigma_stat(n2))   # offsets < 50, sizes <= 300
    sizes = [16, 200, 33, 128, 64, 17, 300, 50, 20, 100]
    calls = [((mod1, m1) if i % 3 else (mod2, m2), sizes[i % len(sizes)], (7 * i) % 50) for i in range(60)]
    # reference: each call alone, the stream drained before and after
    ref = []
    for (mod, _), k, off in calls:
        o = torch.full((k, 6), float("nan"), dtype=torch.float64, device="cuda")
        torch.cuda.synchronize()
        mod.nll_grad_points(pts[off:off + k], o.data_ptr())
        torch.cuda.synchronize()
        ref.append(o.cpu().numpy())
    # the same calls back to back; calls i and i + 2 write the same rows of one buffer (stream order must hold)
    bufs = [torch.full((300, 6), float("nan"), dtype=torch.float64, device="cuda") for _ in range(2)]
    got = []
    for i, ((mod, _), k, off) in enumerate(calls):
        mod.nll_grad_points(pts[off:off + k], bufs[i % 2].data_ptr())
        if i % 7 == 6:                      # read some results back mid-series (asynchronously ordered copy)
            got.append((i, bufs[i % 2][:k].clone()))
    torch.cuda.synchronize()
    for i, t in got:
        assert np.array_equal(t.cpu().numpy(), ref[i]), f"call {i}"
    for i in (58, 59):                      # the last writers of the two buffers
        k = calls[i][1]
        assert np.array_equal(bufs[i % 2][:k].cpu().numpy(), ref[i]), f"call {i}"
    for i in (0, 6, 13, 59):
        (mod, ev), k, off = calls[i]
        for p in (0, k - 1):
            o_nll, o_g, _ = oracle.nll_grad(oracle.MASS, ev, pts[off + p], dg.MASS_LO, dg.MASS_HI)
            assert_parity(ref[i][p, 0], ref[i][p, 1:5], o_nll, o_g, f"call {i} point {p}")
    pts = pts[:300]
    nll, g, nbad = mod1.nll_grad_sweep(pts)   # 300 points: three sub-calls
    assert not nbad
    for p in (0, 127, 128, 299):
        o_nll, o_g, _ = oracle.nll_grad(oracle.MASS, m1, pts[p], dg.MASS_LO, dg.MASS_HI)
        assert_parity(nll[p], g[p], o_nll, o_g, f"sweep point {p}")
    bad = pts.copy()
    bad[290, 2] = -1.0                        # in the last sub-call: the caller's arrays are not touched
    with pytest.raises(mf.MoreFitError) as e:
        mod1.nll_grad_sweep(bad)
    assert e.value.status == mf.MF_ERR_PARAM_DOMAIN
    torch.cuda.synchronize()


def test_batch_async_parity(mf, ctx):
    """mf_nll_grad_batch_async (device pointers, no host copies) equals mf_nll_grad_batch bit for bit."""
    import torch
    T, n = 9, 3000
    toys = dg.gen_mass_toys(T, n, first_seed=300)
    model = ctx.model_create(mf.MF_MASS_GAUSS_EXP, ctx.dataset_upload(toys, dg.MASS_LO, dg.MASS_HI, n_toys=T))
    lams = dg.gen_lambda_points(T, 6, dg.MASS_TRUTH, 3 * dg.mass_sigma_stat(n))
    lams[4] = (0.3, 5.28, -2.0, -1.5)       # outside the domain: +inf / NaN / n_bad = -1
    nll, g = model.nll_grad_batch(lams)
    d_lam = torch.from_numpy(lams).cuda()
    d_out = torch.zeros((T, 6), dtype=torch.float64, device="cuda")
    model.nll_grad_batch_async(d_lam.data_ptr(), d_out.data_ptr())
    torch.cuda.synchronize()
    res = d_out.cpu().numpy()
    ok = np.arange(T) != 4
    assert np.array_equal(res[ok, 0], nll[ok]) and np.array_equal(res[ok, 1:5], g[ok])
    assert res[4, 0] == math.inf and np.all(np.isnan(res[4, 1:5])) and res[4, 5] == -1.0
    o_nll, o_g, _ = oracle.nll_grad(oracle.MASS, toys[2], lams[2], dg.MASS_LO, dg.MASS_HI)
    assert_parity(res[2, 0], res[2, 1:5], o_nll, o_g, "toy 2")


def test_underflowed_pdf_is_flagged(mf, ctx):
    """f = 1 and an event 60 sigma from the peak: P underflows to 0 in fp64 (oracle: P <= 0 -> +inf); the CUDA
    path's exponential is clamped, not flushed, and LogProd flags the event instead (reading R15)."""
    m = np.array([5.10, 5.28, 5.29, 5.27])
    model = ctx.model_create(mf.MF_MASS_GAUSS_EXP, ctx.dataset_upload(m, dg.MASS_LO, dg.MASS_HI))
    lam = (1.0, 5.28, 0.003, -1.5)
    o_nll, o_g, o_bad = oracle.nll_grad(oracle.MASS, m, lam, dg.MASS_LO, dg.MASS_HI)
    assert o_bad == 1 and o_nll == math.inf
    st, nll, g = model.nll_grad_status(lam)
    assert st == mf.MF_NONPOSITIVE_PDF and nll == math.inf and np.all(np.isnan(g))
    # with a background component the same event is fine on both sides
    lam2 = (0.9, 5.28, 0.003, -1.5)
    nll, g = model.nll_grad(lam2)
    o_nll, o_g, o_bad = oracle.nll_grad(oracle.MASS, m, lam2, dg.MASS_LO, dg.MASS_HI)
    assert o_bad == 0
    assert_parity(nll, g, o_nll, o_g, "f = 0.9")


def test_edge_cases_batch_and_points(mf, ctx):
    """Empty toys, a single toy through the batch entries, and a bad point in a many-point call (nothing is enqueued)."""
    import torch
    # toys with zero events: every sum is 0
    empty = ctx.model_create(mf.MF_MASS_GAUSS_EXP, ctx.dataset_upload(np.zeros((3, 0)), dg.MASS_LO, dg.MASS_HI, n_toys=3))
    nll, g = empty.nll_grad_batch(np.tile(np.array(dg.MASS_TRUTH), (3, 1)))
    assert np.all(nll == 0.0) and np.all(g == 0.0)
    # many points, one outside the domain: MF_ERR_PARAM_DOMAIN and the output buffer is untouched
    m = dg.gen_mass(5000, seed=8)
    model = ctx.model_create(mf.MF_MASS_GAUSS_EXP, ctx.dataset_upload(m, dg.MASS_LO, dg.MASS_HI))
    pts = dg.gen_lambda_points(32, 3, dg.MASS_TRUTH, 3 * dg.mass_sigma_stat(5000))
    pts[20, 0] = 1.5
    out = torch.full((32, 6), -7.0, dtype=torch.float64, device="cuda")
    with pytest.raises(mf.MoreFitError) as e:
        model.nll_grad_points(pts, out.data_ptr())
    assert e.value.status == mf.MF_ERR_PARAM_DOMAIN
    torch.cuda.synchronize()
    assert torch.all(out == -7.0)
    # a point with P <= 0 for some event inside a many-point call: that row is +inf / NaN / n_bad > 0, the others are fine
    am = ctx.model_create(mf.MF_ANGULAR_KSTMUMU, ctx.dataset_upload(dg.gen_angular(3000, seed=4)))
    apts = np.tile(np.array(dg.ANG_TRUTH), (16, 1))
    apts[5, 0] = 3.0          # FL = 3: the PDF goes negative for many events
    aout = torch.zeros((16, 10), dtype=torch.float64, device="cuda")
    am.nll_grad_points(apts, aout.data_ptr())
    torch.cuda.synchronize()
    r = aout.cpu().numpy()
    assert r[5, 0] == math.inf and np.all(np.isnan(r[5, 1:9])) and r[5, 9] > 0
    n0, g0 = am.nll_grad(dg.ANG_TRUTH)
    assert abs(r[4, 0] - n0) <= 1e-12 * abs(n0) and r[4, 9] == 0
    # the 1-toy model through the batch entry points
    n1, g1 = model.nll_grad_batch(np.array([dg.MASS_TRUTH]))
    n2, g2 = model.nll_grad(dg.MASS_TRUTH)
    assert n1[0] == n2 and np.array_equal(g1[0], g2)
