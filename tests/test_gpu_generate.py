"""On-device generation (mf_generate_mass) against the generator oracle (oracle/gen.py, pinned by the Philox known-answer
vectors and KS tests): same counter-based recipe, event by event.  The uniform words are bit-identical; the transforms
(log, sqrt, cos, log1p) are CUDA's on one side and libm's on the other, hence a few-ulp tolerance."""
import numpy as np
import pytest
from scipy import stats

import mf_datagen as dg
import oracle
from oracle import gen

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


@pytest.mark.parametrize("lam", [dg.MASS_TRUTH, (0.5, 5.58, 0.05, 2.0), (0.3, 5.3, 0.02, 0.0), (1.0, 5.3, 0.1, -1.5), (0.0, 5.3, 0.1, -1.5)])
def test_generate_matches_oracle_event_by_event(mf, ctx, lam):
    T, n, seed0 = 3, 701, 12345
    ds = ctx.generate_mass(seed0, T, n, lam, LO, HI)
    x = ds.download()[0]
    ref = gen.gen_mass_toys(seed0, T, n, lam, LO, HI)
    assert x.shape == ref.shape == (T, n)
    assert np.all((x >= LO) & (x <= HI))
    # identical decisions (component, accepted draw) unless a value sits within rounding of a range edge
    assert np.max(np.abs(x - ref)) <= 64 * np.spacing(HI), np.max(np.abs(x - ref))
    assert np.mean(x == ref) > 0.5


def test_generated_dataset_feeds_the_model(mf, ctx):
    """Generate -> model -> value/gradient and fit, all on the device; the same events downloaded and given to the oracle."""
    ds = ctx.generate_mass(99, 1, 20_000, dg.MASS_TRUTH, LO, HI)
    model = ctx.model_create(mf.MF_MASS_GAUSS_EXP, ds)
    x = ds.download()[0, 0]
    nll, g = model.nll_grad(dg.MASS_START)
    o_nll, o_g, _ = oracle.nll_grad(oracle.MASS, x, dg.MASS_START, LO, HI)
    assert abs(nll - o_nll) <= 1e-11 * abs(o_nll) and np.all(np.abs(g - o_g) <= 1e-9 * (1 + np.abs(o_g)))
    r = model.fit(dg.MASS_START)
    assert r.converged and np.all(np.abs((r.lam - np.array(dg.MASS_TRUTH)) / r.sigma) < 5)


def test_toy_study_on_device(mf, ctx):
    """4096 toys x 1e4 events generated and fitted without any event crossing PCIe; pulls are standard normal."""
    T, n = 4096, 10_000
    ds = ctx.generate_mass(2024, T, n, dg.MASS_TRUTH, LO, HI)
    model = ctx.model_create(mf.MF_MASS_GAUSS_EXP, ds)
    res = model.fit_batch(np.array(dg.MASS_TRUTH))
    assert res.converged.all()
    pulls = (res.lam - np.array(dg.MASS_TRUTH)) / res.sigma
    assert np.all(np.abs(pulls.mean(0)) < 0.08) and np.all(np.abs(pulls.std(0) - 1) < 0.05)
    # the distribution of one toy against the CDF of Eq. 2 (scipy: truncated normal + truncated exponential mixture)
    x = ds.download()[0, 7]
    f, mu, sg, tau = dg.MASS_TRUTH
    cdf = lambda v: f * stats.truncnorm.cdf(v, (LO - mu) / sg, (HI - mu) / sg, mu, sg) + (1 - f) * \
        np.expm1(tau * (v - LO)) / np.expm1(tau * (HI - LO))
    assert stats.kstest(x, cdf).pvalue > 1e-3


def test_generate_edge_cases(mf, ctx):
    assert ctx.generate_mass(1, 2, 0, dg.MASS_TRUTH, LO, HI).download().shape == (1, 2, 0)
    a = ctx.generate_mass(5, 1, 65, dg.MASS_TRUTH, LO, HI).download()[0, 0]
    b = ctx.generate_mass(5, 1, 1000, dg.MASS_TRUTH, LO, HI).download()[0, 0]
    assert np.array_equal(a, b[:65])                       # event i depends only on (seed, i)
    c = ctx.generate_mass(4, 2, 65, dg.MASS_TRUTH, LO, HI).download()[0]
    assert np.array_equal(c[1], a)                         # toy t uses seed0 + t
    with pytest.raises(mf.MoreFitError):
        ctx.generate_mass(1, 1, 10, (0.3, 5.28, -1.0, -1.5), LO, HI)


@pytest.mark.parametrize("a", [dg.ANG_TRUTH, (0.3, 0.1, -0.2, 0.25, 0.1, -0.05, 0.07, -0.09)])
def test_generate_angular_matches_oracle(mf, ctx, a):
    T, n, seed0 = 2, 333, 777
    ds = ctx.generate_angular(seed0, T, n, a)
    x = ds.download()                                   # [3][T][n]
    ref = gen.gen_angular_toys(seed0, T, n, a)
    assert x.shape == ref.shape == (3, T, n)
    assert np.all(np.abs(x[:2]) <= 1) and np.all(np.abs(x[2]) <= np.pi)
    # the proposals are bit-identical functions of the uniforms; an accept decision can differ only if u4 * pmax is within
    # rounding of P(Omega), which does not happen in 666 events
    assert np.array_equal(x, ref)


def test_generated_angular_dataset_feeds_the_model(mf, ctx):
    ds = ctx.generate_angular(5, 1, 50_000, dg.ANG_TRUTH)
    model = ctx.model_create(mf.MF_ANGULAR_KSTMUMU, ds)
    ev = ds.download()[:, 0, :]
    nll, g = model.nll_grad(dg.ANG_TRUTH)
    o_nll, o_g, _ = oracle.nll_grad(oracle.ANGULAR, ev, dg.ANG_TRUTH)
    assert abs(nll - o_nll) <= 1e-11 * abs(o_nll) and np.all(np.abs(g - o_g) <= 1e-9 * (1 + np.abs(o_g)))
    r = model.fit(dg.ANG_TRUTH)
    assert r.converged and np.all(np.abs((r.lam - np.array(dg.ANG_TRUTH)) / r.sigma) < 5)


def test_generate_4d_matches_oracle_and_feeds_the_model(mf, ctx):
    T, n, seed0 = 2, 257, 4242
    lam = dg.FOURD_TRUTH
    ds = ctx.generate_4d(seed0, T, n, lam, LO, HI)
    x = ds.download()                                   # [4][T][n]
    ref = gen.gen_4d_toys(seed0, T, n, lam, LO, HI)
    assert x.shape == ref.shape == (4, T, n)
    assert np.array_equal(x[1:], ref[1:])               # angles: bit-identical functions of the uniforms
    assert np.max(np.abs(x[0] - ref[0])) <= 64 * np.spacing(HI)   # mass: CUDA vs libm transforms
    big = ctx.generate_4d(9, 1, 100_000, lam, LO, HI)
    model = ctx.model_create(mf.MF_MASS_X_ANGULAR, big)
    ev = big.download()[:, 0, :]
    nll, g = model.nll_grad(lam)
    o_nll, o_g, _ = oracle.nll_grad(oracle.FOURD, ev, lam, LO, HI, nthreads=oracle.max_threads())
    assert abs(nll - o_nll) <= 1e-11 * abs(o_nll) and np.all(np.abs(g - o_g) <= 1e-9 * (1 + np.abs(o_g)))
    r = model.fit(lam)
    assert r.converged and np.all(np.abs((r.lam - np.array(lam)) / r.sigma) < 5)


def test_toy_study_entry(mf, ctx):
    """mf_toy_study_mass = generate + model + concurrent fits in one call; identical to doing the three steps by hand."""
    T, n = 512, 5000
    r = ctx.toy_study_mass(2024, T, n, dg.MASS_TRUTH, LO, HI)
    ds = ctx.generate_mass(2024, T, n, dg.MASS_TRUTH, LO, HI)
    r2 = ctx.model_create(mf.MF_MASS_GAUSS_EXP, ds).fit_batch(np.array(dg.MASS_TRUTH))
    assert r.converged.all() and np.array_equal(r.lam, r2.lam) and np.array_equal(r.cov, r2.cov)
    pulls = (r.lam - np.array(dg.MASS_TRUTH)) / r.sigma
    assert np.all(np.abs(pulls.mean(0)) < 0.25) and np.all(np.abs(pulls.std(0) - 1) < 0.15)
    one = ctx.toy_study_mass(7, 1, 20_000, dg.MASS_TRUTH, LO, HI)
    assert len(one) == 1 and one.converged[0]


def test_toy_study_angular(mf, ctx):
    """mf_toy_study_angular = generate + model + concurrent fits in one call: identical to the three steps by hand; pulls sane."""
    T, n = 64, 4_000
    r = ctx.toy_study_angular(77, T, n, dg.ANG_TRUTH)
    ds = ctx.generate_angular(77, T, n, dg.ANG_TRUTH)
    byhand = ctx.model_create(mf.MF_ANGULAR_KSTMUMU, ds).fit_batch(np.array(dg.ANG_TRUTH))
    assert np.all(r.converged) and np.array_equal(r.lam, byhand.lam) and np.array_equal(r.nll, byhand.nll)
    pulls = (r.lam - np.array(dg.ANG_TRUTH)) / r.sigma
    assert np.all(np.abs(pulls.mean(0)) < 0.6) and np.all(np.abs(pulls.std(0) - 1) < 0.4)
    one = ctx.toy_study_angular(5, 1, 20_000, dg.ANG_TRUTH)
    assert bool(one.converged[0])

