"""mf_nll_grad_mass_noalloc (include/morefit_b200.h): the evaluation that allocates nothing — scratch in a fixed
`static __device__` array of the library image — against the existing path (mf_dataset_upload + mf_model_create + mf_nll_grad)
and the oracle, within the tolerances of the other parity tests, on calls in a row that share the scratch.

This file is named so that pytest collects it LAST: the suite runs with `pytest -x`, a failure here must not hide other tests.
It passes alone in a fresh process (`pytest tests/test_zz_no_alloc.py -m gpu`) and after the rest of the suite."""
import numpy as np
import pytest

import mf_datagen as dg
import oracle

pytestmark = pytest.mark.gpu

NLL_RTOL = 1e-11   # as tests/test_gpu_parity.py
GRAD_TOL = 1e-9


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


def close(row, nll, g, what):
    assert row[5] == 0.0, f"{what}: n_bad {row[5]}"
    assert abs(row[0] - nll) <= NLL_RTOL * abs(nll) + 1e-300, f"{what}: nll {row[0]!r} vs {nll!r}"
    err = np.abs(row[1:5] - g)
    assert np.all(err <= GRAD_TOL * (1.0 + np.abs(g))), f"{what}: gradient error {err}"


@pytest.mark.parametrize("n", [100, 8192, 100_003, 1_000_000])
def test_noalloc_matches_existing_path_two_calls_in_a_row(mf, ctx, n):
    """n = 100: only the ragged tail; 8192: exactly one chunk; 100,003: 13 chunks + a tail of 163 events; 1e6: C1's size."""
    import torch
    m = dg.gen_mass(n, seed=11)
    model = ctx.model_create(mf.MF_MASS_GAUSS_EXP, ctx.dataset_upload(m, dg.MASS_LO, dg.MASS_HI))
    d_m = torch.from_numpy(m).cuda()
    assert d_m.data_ptr() % 16 == 0
    out = torch.full((3, 6), float("nan"), dtype=torch.float64, device="cuda")
    lam_a = np.array(dg.MASS_TRUTH)
    lam_b = np.array(dg.MASS_START)
    # three calls back to back on the context's stream, sharing the static scratch: point a, point b, point a again
    for row, lam in enumerate((lam_a, lam_b, lam_a)):
        ctx.nll_grad_mass_noalloc(d_m.data_ptr(), n, dg.MASS_LO, dg.MASS_HI, lam, out[row].data_ptr())
    model.nll_grad(lam_a)             # synchronises the context's stream (same stream: ordered after the three kernels)
    torch.cuda.synchronize()
    r = out.cpu().numpy()
    for row, lam in enumerate((lam_a, lam_b, lam_a)):
        nll, g = model.nll_grad(lam)
        close(r[row], nll, g, f"n={n} call {row} vs mf_nll_grad")
        o_nll, o_g, _ = oracle.nll_grad(oracle.MASS, m, lam, dg.MASS_LO, dg.MASS_HI)
        close(r[row], o_nll, o_g, f"n={n} call {row} vs oracle")
    assert np.array_equal(r[0], r[2])  # what the call in between left in the scratch does not matter: same bits
    model.close()


def test_noalloc_general_parameter_point_and_bad_events(mf, ctx):
    """A point outside the fast range of the other kernels (f close to 1, steep slope) and a dataset with an event the PDF
    cannot describe to a positive normal number: n_bad > 0, +inf / NaN — as mf_nll_grad reports it."""
    import torch
    n = 30_001
    m = dg.gen_mass(n, seed=12)
    model = ctx.model_create(mf.MF_MASS_GAUSS_EXP, ctx.dataset_upload(m, dg.MASS_LO, dg.MASS_HI))
    d_m = torch.from_numpy(m).cuda()
    out = torch.zeros(6, dtype=torch.float64, device="cuda")
    lam = np.array([0.9, 5.3, 0.05, -2.5])
    ctx.nll_grad_mass_noalloc(d_m.data_ptr(), n, dg.MASS_LO, dg.MASS_HI, lam, out.data_ptr())
    torch.cuda.synchronize()
    nll, g = model.nll_grad(lam)
    close(out.cpu().numpy(), nll, g, "general point")
    # f = 1 and a narrow Gaussian far from the events: P underflows for most events
    lam_bad = np.array([1.0, 5.0, 0.002, 0.0])
    ctx.nll_grad_mass_noalloc(d_m.data_ptr(), n, dg.MASS_LO, dg.MASS_HI, lam_bad, out.data_ptr())
    torch.cuda.synchronize()
    r = out.cpu().numpy()
    with pytest.raises(mf.MoreFitError):
        model.nll_grad(lam_bad)
    assert r[5] > 0 and r[0] == np.inf and np.all(np.isnan(r[1:5]))
    # and the next call is unaffected by it
    ctx.nll_grad_mass_noalloc(d_m.data_ptr(), n, dg.MASS_LO, dg.MASS_HI, lam, out.data_ptr())
    torch.cuda.synchronize()
    close(out.cpu().numpy(), nll, g, "after a bad call")
    model.close()


def test_noalloc_on_a_caller_stream_and_empty(mf, ctx):
    import torch
    n = 50_000
    m = dg.gen_mass(n, seed=13)
    d_m = torch.from_numpy(m).cuda()
    out = torch.zeros(6, dtype=torch.float64, device="cuda")
    s = torch.cuda.Stream()
    torch.cuda.synchronize()
    lam = np.array(dg.MASS_TRUTH)
    ctx.nll_grad_mass_noalloc(d_m.data_ptr(), n, dg.MASS_LO, dg.MASS_HI, lam, out.data_ptr(), stream=s.cuda_stream)
    s.synchronize()
    o_nll, o_g, _ = oracle.nll_grad(oracle.MASS, m, lam, dg.MASS_LO, dg.MASS_HI)
    close(out.cpu().numpy(), o_nll, o_g, "caller's stream")
    ctx.nll_grad_mass_noalloc(0, 0, dg.MASS_LO, dg.MASS_HI, lam, out.data_ptr())   # no events: -ln L = 0, gradient 0
    torch.cuda.synchronize()
    assert np.all(out.cpu().numpy() == 0.0)


def test_noalloc_rejects_what_it_cannot_hold(mf, ctx):
    import torch
    out = torch.zeros(6, dtype=torch.float64, device="cuda")
    buf = torch.zeros(64, dtype=torch.float64, device="cuda")
    lam = np.array(dg.MASS_TRUTH)
    with pytest.raises(mf.MoreFitError) as e:   # beyond the scratch: rejected before anything is enqueued or read
        ctx.nll_grad_mass_noalloc(buf.data_ptr(), mf.MF_NOALLOC_MAX_EVENTS + 1, dg.MASS_LO, dg.MASS_HI, lam, out.data_ptr())
    assert e.value.status == mf.MF_ERR_ARG and "MF_NOALLOC_MAX_EVENTS" in str(e.value)
    with pytest.raises(mf.MoreFitError) as e:   # misaligned events
        ctx.nll_grad_mass_noalloc(buf.data_ptr() + 8, 16, dg.MASS_LO, dg.MASS_HI, lam, out.data_ptr())
    assert e.value.status == mf.MF_ERR_ARG
    with pytest.raises(mf.MoreFitError) as e:   # sigma <= 0
        ctx.nll_grad_mass_noalloc(buf.data_ptr(), 16, dg.MASS_LO, dg.MASS_HI, [0.3, 5.28, -1.0, -1.5], out.data_ptr())
    assert e.value.status == mf.MF_ERR_PARAM_DOMAIN
    torch.cuda.synchronize()
    assert np.all(out.cpu().numpy() == 0.0)     # outputs untouched
