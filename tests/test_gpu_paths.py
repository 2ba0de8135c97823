"""GPU parity for every code path that is not the default single-evaluation one: many-point launches of the angular and
4D models, batched toys of the 4D model, the register-buffer 4D kernel (n < 1024), the host-result sweep, the
MF_NO_TMA / MF_NO_PDL ablation paths (subprocess: the switches are read once per process) and the sharded evaluation of
paper_2505_12414_b200.dist with the CUDA path supplying the shard sums.  Every comparison is against the oracle."""
import math
import os
import subprocess
import sys
import textwrap

import numpy as np
import pytest

import mf_datagen as dg
import oracle

pytestmark = pytest.mark.gpu

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
NLL_RTOL = 1e-11
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


def check(nll, grad, o_nll, o_grad, what):
    assert abs(nll - o_nll) <= NLL_RTOL * abs(o_nll), f"{what}: nll {nll!r} vs oracle {o_nll!r}"
    err = np.abs(grad - o_grad)
    tol = GRAD_TOL * (1.0 + np.abs(o_grad))
    assert np.all(err <= tol), f"{what}: grad err {err} tol {tol}"


def _ang_points(n_pts, seed):
    rng = np.random.default_rng(seed)
    pts = np.tile(np.array(dg.ANG_TRUTH), (n_pts, 1)) + rng.uniform(-0.03, 0.03, (n_pts, 8))
    pts[0] = dg.ANG_TRUTH
    return pts


def _fourd_points(n_pts, seed):
    rng = np.random.default_rng(seed)
    pts = np.tile(np.array(dg.FOURD_TRUTH), (n_pts, 1))
    scale = np.array([0.02, 0.002, 0.001, 0.2] + [0.03] * 8 + [0.05] * 4)
    pts += rng.uniform(-1, 1, (n_pts, 16)) * scale
    pts[0] = dg.FOURD_TRUTH
    return pts


@pytest.mark.parametrize("n,n_pts", [(20_011, 16), (150_000, 64), (1, 16), (10_007, 17), (20_011, 40), (5_000, 100), (20_011, 6),
                                     (20_011, 9)])
def test_points_mode_angular_vs_oracle(mf, ctx, n, n_pts):
    """The angular many-points kernel (two tensor-core contractions, mf_points.cuh): every row of a >= 16-point call
    against the oracle, with ragged event counts, partly filled point blocks and more than one 64-point pass."""
    import torch
    ev = dg.gen_angular(n, seed=21)
    model = ctx.model_create(mf.MF_ANGULAR_KSTMUMU, ctx.dataset_upload(ev))
    pts = _ang_points(n_pts, 5)
    out = torch.full((n_pts, 10), float("nan"), dtype=torch.float64, device="cuda")
    model.nll_grad_points(pts, out.data_ptr())
    torch.cuda.synchronize()
    res = out.cpu().numpy()
    assert np.all(res[:, 9] == 0)
    for p in range(n_pts):
        o_nll, o_g, _ = oracle.nll_grad(oracle.ANGULAR, ev, pts[p], nthreads=oracle.max_threads())
        check(res[p, 0], res[p, 1:9], o_nll, o_g, f"angular points row {p}")


def test_points_mode_angular_bad_point(mf, ctx):
    """A point at which the PDF goes negative for some events gets +inf / NaN and the count; its neighbours are unaffected."""
    import torch
    ev = dg.gen_angular(4_000, seed=22)
    model = ctx.model_create(mf.MF_ANGULAR_KSTMUMU, ctx.dataset_upload(ev))
    pts = _ang_points(20, 7)
    pts[11, 1] = 5.0
    out = torch.full((20, 10), float("nan"), dtype=torch.float64, device="cuda")
    model.nll_grad_points(pts, out.data_ptr())
    torch.cuda.synchronize()
    res = out.cpu().numpy()
    _, _, nbad = oracle.nll_grad(oracle.ANGULAR, ev, pts[11])
    assert nbad > 0 and res[11, 9] == nbad and res[11, 0] == math.inf and np.all(np.isnan(res[11, 1:9]))
    for p in (10, 12):
        o_nll, o_g, _ = oracle.nll_grad(oracle.ANGULAR, ev, pts[p])
        check(res[p, 0], res[p, 1:9], o_nll, o_g, f"row {p}")
    pts[3, 2] = np.nan
    with pytest.raises(mf.MoreFitError) as e:
        model.nll_grad_points(pts, out.data_ptr())
    assert e.value.status == mf.MF_ERR_PARAM_DOMAIN


@pytest.mark.parametrize("n,n_pts", [(30_001, 16), (100_000, 64), (1, 16), (10_007, 17), (5_000, 41), (30_001, 10), (30_001, 13)])
def test_points_mode_fourd_vs_oracle(mf, ctx, n, n_pts):
    """The 4D many-points kernel (mf_points4d.cuh: one pass over the data per 16 points, tensor-core contractions around
    the per-pair exponential): every row against the oracle, ragged event counts, partly filled point blocks."""
    import torch
    ev = dg.gen_4d(n, seed=23)
    model = ctx.model_create(mf.MF_MASS_X_ANGULAR, ctx.dataset_upload(ev, dg.MASS_LO, dg.MASS_HI))
    pts = _fourd_points(n_pts, 6)
    out = torch.full((n_pts, 18), float("nan"), dtype=torch.float64, device="cuda")
    model.nll_grad_points(pts, out.data_ptr())
    torch.cuda.synchronize()
    res = out.cpu().numpy()
    assert np.all(res[:, 17] == 0)
    for p in range(n_pts):
        o_nll, o_g, _ = oracle.nll_grad(oracle.FOURD, ev, pts[p], dg.MASS_LO, dg.MASS_HI, nthreads=oracle.max_threads())
        check(res[p, 0], res[p, 1:17], o_nll, o_g, f"4D points row {p}")


def test_points_mode_fourd_edge_points(mf, ctx):
    """Points with f = 0 or f = 1 exactly go through the (point, chunk) kernel (the one-pass kernel folds ln f, 1/f and
    1/(1-f) into its constants); a point outside the parameter domain is refused; a point with P <= 0 events is flagged."""
    import torch
    ev = dg.gen_4d(6_000, seed=24)
    model = ctx.model_create(mf.MF_MASS_X_ANGULAR, ctx.dataset_upload(ev, dg.MASS_LO, dg.MASS_HI))
    pts = _fourd_points(20, 8)
    pts[5, 0] = 0.0
    pts[9, 0] = 1.0
    out = torch.full((20, 18), float("nan"), dtype=torch.float64, device="cuda")
    model.nll_grad_points(pts, out.data_ptr())
    torch.cuda.synchronize()
    res = out.cpu().numpy()
    for p in (4, 5, 9, 19):
        o_nll, o_g, nbad = oracle.nll_grad(oracle.FOURD, ev, pts[p], dg.MASS_LO, dg.MASS_HI)
        assert nbad == 0 and res[p, 17] == 0
        check(res[p, 0], res[p, 1:17], o_nll, o_g, f"4D edge row {p}")
    pts = _fourd_points(20, 8)
    pts[7, 5] = 5.0                       # S3 = 5: the signal's angular PDF goes negative for many events
    model.nll_grad_points(pts, out.data_ptr())
    torch.cuda.synchronize()
    res = out.cpu().numpy()
    _, _, nbad = oracle.nll_grad(oracle.FOURD, ev, pts[7], dg.MASS_LO, dg.MASS_HI)
    assert nbad > 0 and res[7, 17] == nbad and res[7, 0] == math.inf and np.all(np.isnan(res[7, 1:17]))
    o_nll, o_g, _ = oracle.nll_grad(oracle.FOURD, ev, pts[8], dg.MASS_LO, dg.MASS_HI)
    check(res[8, 0], res[8, 1:17], o_nll, o_g, "row beside a bad point")
    pts[3, 2] = -0.01                     # sigma < 0
    with pytest.raises(mf.MoreFitError) as e:
        model.nll_grad_points(pts, out.data_ptr())
    assert e.value.status == mf.MF_ERR_PARAM_DOMAIN


@pytest.mark.parametrize("n", [3000, 40_001])
def test_batch_fourd_vs_oracle(mf, ctx, n):
    """launch_batch<FourDModel>: T toys of the 4D model at their own lambda_t (40,001 events: two CTAs per toy)."""
    T = 5
    ev = np.stack([dg.gen_4d(n, seed=60 + t) for t in range(T)], axis=1)  # [4][T][n]
    model = ctx.model_create(mf.MF_MASS_X_ANGULAR, ctx.dataset_upload(ev, dg.MASS_LO, dg.MASS_HI, n_toys=T))
    lams = _fourd_points(T, 9)
    nll, g = model.nll_grad_batch(lams)
    for t in range(T):
        o_nll, o_g, _ = oracle.nll_grad(oracle.FOURD, ev[:, t, :], lams[t], dg.MASS_LO, dg.MASS_HI)
        check(nll[t], g[t], o_nll, o_g, f"4D toy {t}")


@pytest.mark.parametrize("n", [1, 37, 640, 1023])
def test_small_fourd_register_kernel_vs_oracle(mf, ctx, n):
    """n_pad < 1024: nll_grad_kernel<FourDModel> (register buffers) instead of the shared-memory-staged kernel."""
    ev = dg.gen_4d(n, seed=70 + n)
    model = ctx.model_create(mf.MF_MASS_X_ANGULAR, ctx.dataset_upload(ev, dg.MASS_LO, dg.MASS_HI))
    for lam in _fourd_points(3, n):
        nll, g = model.nll_grad(lam)
        o_nll, o_g, _ = oracle.nll_grad(oracle.FOURD, ev, lam, dg.MASS_LO, dg.MASS_HI)
        check(nll, g, o_nll, o_g, f"4D n={n}")


@pytest.mark.parametrize("n", [37, 640])
def test_small_angular_register_kernel_vs_oracle(mf, ctx, n):
    ev = dg.gen_angular(n, seed=80 + n)
    model = ctx.model_create(mf.MF_ANGULAR_KSTMUMU, ctx.dataset_upload(ev))
    for lam in _ang_points(3, n):
        nll, g = model.nll_grad(lam)
        o_nll, o_g, _ = oracle.nll_grad(oracle.ANGULAR, ev, lam)
        check(nll, g, o_nll, o_g, f"angular n={n}")


def test_sweep_host_results_vs_oracle(mf, ctx):
    """mf_nll_grad_sweep: host lambda points in, host results out; both branches (< 16 and >= 16 points)."""
    n = 50_003
    m = dg.gen_mass(n, seed=9)
    model = ctx.model_create(mf.MF_MASS_GAUSS_EXP, ctx.dataset_upload(m, dg.MASS_LO, dg.MASS_HI))
    for n_pts in (5, 40):
        pts = dg.gen_lambda_points(n_pts, 31, dg.MASS_TRUTH, 3 * dg.mass_sigma_stat(n))
        nll, g, nbad = model.nll_grad_sweep(pts)
        assert nbad == 0
        for p in range(n_pts):
            o_nll, o_g, _ = oracle.nll_grad(oracle.MASS, m, pts[p], dg.MASS_LO, dg.MASS_HI)
            check(nll[p], g[p], o_nll, o_g, f"sweep {n_pts} row {p}")
    # repeated calls reuse the model's scratch; a larger call grows it
    pts = dg.gen_lambda_points(200, 32, dg.MASS_TRUTH, 3 * dg.mass_sigma_stat(n))
    a = model.nll_grad_sweep(pts)
    b = model.nll_grad_sweep(pts)
    assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1])
    o_nll, o_g, _ = oracle.nll_grad(oracle.MASS, m, pts[199], dg.MASS_LO, dg.MASS_HI)
    check(a[0][199], a[1][199], o_nll, o_g, "sweep 200 row 199")
    # a point with P <= 0 is counted, not an error
    am = ctx.model_create(mf.MF_ANGULAR_KSTMUMU, ctx.dataset_upload(dg.gen_angular(3000, seed=4)))
    apts = np.tile(np.array(dg.ANG_TRUTH), (20, 1))
    apts[7, 0] = 3.0
    nll, g, nbad = am.nll_grad_sweep(apts)
    assert nbad == 1 and nll[7] == np.inf and np.all(np.isnan(g[7])) and np.isfinite(nll[6])


def test_first_evaluation_after_create_is_ordered(mf, ctx):
    """mf_model_create no longer synchronises: the first launch on a fresh model must still see the S0/S1 kernels' output
    (padding, basis columns, sum_i m_i).  Create-then-evaluate immediately, many times, for every entry point."""
    import torch
    ev = dg.gen_4d(200_003, seed=12)
    o_nll, o_g, _ = oracle.nll_grad(oracle.FOURD, ev, dg.FOURD_TRUTH, dg.MASS_LO, dg.MASS_HI, nthreads=oracle.max_threads())
    d_ev = [torch.from_numpy(np.ascontiguousarray(ev[j])).cuda() for j in range(4)]
    pts = np.tile(np.array(dg.FOURD_TRUTH), (16, 1))
    for rep in range(6):
        ds = ctx.dataset_upload(d_ev, dg.MASS_LO, dg.MASS_HI)
        model = ctx.model_create(mf.MF_MASS_X_ANGULAR, ds)
        if rep % 2 == 0:
            nll, g = model.nll_grad(dg.FOURD_TRUTH)
            check(nll, g, o_nll, o_g, f"fresh model rep {rep}")
        else:
            nll, g, _ = model.nll_grad_sweep(pts)
            check(nll[15], g[15], o_nll, o_g, f"fresh model sweep rep {rep}")
        model.close()
        ds.close()


def test_overlapping_angular_points_calls(mf, ctx):
    """Angular many-points calls of up to 256 points carry their coefficients in the kernel parameters and overlap on the GPU:
    40 back-to-back calls of varying size on two models, writing the same rows again and again, give bit for bit what each
    call gives alone; sampled rows against the oracle; a 300-point call (copy path) in between."""
    import torch
    ev1, ev2 = dg.gen_angular(120_011, seed=31), dg.gen_angular(30_001, seed=32)
    mod1 = ctx.model_create(mf.MF_ANGULAR_KSTMUMU, ctx.dataset_upload(ev1))
    mod2 = ctx.model_create(mf.MF_ANGULAR_KSTMUMU, ctx.dataset_upload(ev2))
    pts = _ang_points(350, 12)
    sizes = [6, 64, 17, 256, 33, 300, 16, 100]
    calls = [((mod1, ev1) if i % 3 else (mod2, ev2), sizes[i % len(sizes)], (5 * i) % 50) for i in range(40)]
    ref = []
    for (mod, _), k, off in calls:
        o = torch.full((k, 10), float("nan"), dtype=torch.float64, device="cuda")
        torch.cuda.synchronize()
        mod.nll_grad_points(pts[off:off + k], o.data_ptr())
        torch.cuda.synchronize()
        ref.append(o.cpu().numpy())
    bufs = [torch.full((300, 10), float("nan"), dtype=torch.float64, device="cuda") for _ in range(2)]
    got = []
    for i, ((mod, _), k, off) in enumerate(calls):
        mod.nll_grad_points(pts[off:off + k], bufs[i % 2].data_ptr())
        if i % 5 == 4:
            got.append((i, bufs[i % 2][:k].clone()))
    torch.cuda.synchronize()
    for i, t in got:
        assert np.array_equal(t.cpu().numpy(), ref[i]), f"call {i}"
    for i in (38, 39):
        k = calls[i][1]
        assert np.array_equal(bufs[i % 2][:k].cpu().numpy(), ref[i]), f"call {i}"
    for i in (0, 3, 5, 39):
        (mod, ev), k, off = calls[i]
        for p in (0, k - 1):
            o_nll, o_g, _ = oracle.nll_grad(oracle.ANGULAR, ev, pts[off + p])
            assert abs(ref[i][p, 0] - o_nll) <= 1e-11 * abs(o_nll), (i, p)
            assert np.all(np.abs(ref[i][p, 1:9] - o_g) <= 1e-9 * (1 + np.abs(o_g))), (i, p)


def test_overlapping_fourd_points_calls(mf, ctx):
    """4D many-points calls of up to 96 points carry their per-point data in the kernel parameters and overlap on the GPU:
    back-to-back calls of varying size, writing the same rows again and again, give bit for bit what each call gives alone;
    sampled rows against the oracle; a 120-point call (copy path) in between."""
    import torch
    ev = dg.gen_4d(60_013, seed=41)
    mod = ctx.model_create(mf.MF_MASS_X_ANGULAR, ctx.dataset_upload(ev, dg.MASS_LO, dg.MASS_HI))
    pts = _fourd_points(170, 14)
    sizes = [10, 64, 17, 96, 33, 120, 16]
    calls = [(sizes[i % len(sizes)], (5 * i) % 50) for i in range(21)]
    ref = []
    for k, off in calls:
        o = torch.full((k, 18), float("nan"), dtype=torch.float64, device="cuda")
        torch.cuda.synchronize()
        mod.nll_grad_points(pts[off:off + k], o.data_ptr())
        torch.cuda.synchronize()
        ref.append(o.cpu().numpy())
    bufs = [torch.full((120, 18), float("nan"), dtype=torch.float64, device="cuda") for _ in range(2)]
    got = []
    for i, (k, off) in enumerate(calls):
        mod.nll_grad_points(pts[off:off + k], bufs[i % 2].data_ptr())
        if i % 4 == 3:
            got.append((i, bufs[i % 2][:k].clone()))
    torch.cuda.synchronize()
    for i, t in got:
        assert np.array_equal(t.cpu().numpy(), ref[i]), f"call {i}"
    for i in (19, 20):
        k = calls[i][0]
        assert np.array_equal(bufs[i % 2][:k].cpu().numpy(), ref[i]), f"call {i}"
    for i in (0, 3, 5, 20):
        k, off = calls[i]
        for p in (0, k - 1):
            o_nll, o_g, _ = oracle.nll_grad(oracle.FOURD, ev, pts[off + p], dg.MASS_LO, dg.MASS_HI)
            assert abs(ref[i][p, 0] - o_nll) <= 1e-11 * abs(o_nll), (i, p)
            assert np.all(np.abs(ref[i][p, 1:17] - o_g) <= 1e-9 * (1 + np.abs(o_g))), (i, p)


_ABLATION = textwrap.dedent("""
    import numpy as np, sys
    sys.path.insert(0, {root!r})
    import mf_datagen as dg, oracle, paper_2505_12414_b200 as mf
    import torch
    ctx = mf.Context(0)
    def check(nll, g, o):
        assert abs(nll - o[0]) <= 1e-11 * abs(o[0]), (nll, o[0])
        assert np.all(np.abs(g - o[1]) <= 1e-9 * (1 + np.abs(o[1]))), (g, o[1])
    ev = dg.gen_angular(50_021, seed=2)
    am = ctx.model_create(mf.MF_ANGULAR_KSTMUMU, ctx.dataset_upload(ev))
    for _ in range(3):
        nll, g = am.nll_grad(dg.ANG_TRUTH)
    check(nll, g, oracle.nll_grad(oracle.ANGULAR, ev, dg.ANG_TRUTH))
    apts = np.tile(np.array(dg.ANG_TRUTH), (20, 1)) + np.random.default_rng(3).uniform(-0.03, 0.03, (20, 8))
    aout = torch.zeros((20, 10), dtype=torch.float64, device="cuda")
    am.nll_grad_points(apts, aout.data_ptr())      # >= 16 points: the many-points kernel of the angular model
    torch.cuda.synchronize()
    ar = aout.cpu().numpy()
    for p in (0, 7, 19):
        check(ar[p, 0], ar[p, 1:9], oracle.nll_grad(oracle.ANGULAR, ev, apts[p]))
    ev4 = dg.gen_4d(50_021, seed=3)
    fm = ctx.model_create(mf.MF_MASS_X_ANGULAR, ctx.dataset_upload(ev4, dg.MASS_LO, dg.MASS_HI))
    nll, g = fm.nll_grad(dg.FOURD_TRUTH)
    check(nll, g, oracle.nll_grad(oracle.FOURD, ev4, dg.FOURD_TRUTH, dg.MASS_LO, dg.MASS_HI))
    m = dg.gen_mass(100_003, seed=5)
    mm = ctx.model_create(mf.MF_MASS_GAUSS_EXP, ctx.dataset_upload(m, dg.MASS_LO, dg.MASS_HI))
    pts = dg.gen_lambda_points(40, 77, dg.MASS_TRUTH, 3 * dg.mass_sigma_stat(100_003))
    out = torch.zeros((40, 6), dtype=torch.float64, device="cuda")
    for p in range(0, 39, 3):                       # pipelined single launches (< 4 points per call at this size)
        mm.nll_grad_points(pts[p:p + 3], out[p].data_ptr())
    mm.nll_grad_points(pts[39:40], out[39].data_ptr())
    for p in range(0, 40, 5):                       # the smallest many-point calls
        mm.nll_grad_points(pts[p:p + 5], out[p].data_ptr())
    for p in range(0, 40, 10):                      # small many-point calls (8 .. 15 points: one launch each)
        mm.nll_grad_points(pts[p:p + 10], out[p].data_ptr())
    torch.cuda.synchronize()
    r = out.cpu().numpy()
    for p in (0, 13, 39):
        check(r[p, 0], r[p, 1:5], oracle.nll_grad(oracle.MASS, m, pts[p], dg.MASS_LO, dg.MASS_HI))
    nllb, gb, _ = mm.nll_grad_sweep(pts)            # one many-point launch
    check(nllb[17], gb[17], oracle.nll_grad(oracle.MASS, m, pts[17], dg.MASS_LO, dg.MASS_HI))
    toys = dg.gen_mass_toys(6, 3000, first_seed=9)
    bm = ctx.model_create(mf.MF_MASS_GAUSS_EXP, ctx.dataset_upload(toys, dg.MASS_LO, dg.MASS_HI, n_toys=6))
    lam = np.tile(np.array(dg.MASS_TRUTH), (6, 1))
    bn, bg = bm.nll_grad_batch(lam)
    check(bn[5], bg[5], oracle.nll_grad(oracle.MASS, toys[5], lam[5], dg.MASS_LO, dg.MASS_HI))
    toys = dg.gen_mass_toys(400, 700, first_seed=20)     # more toys than resident CTAs of a small grid, ragged groups
    bm2 = ctx.model_create(mf.MF_MASS_GAUSS_EXP, ctx.dataset_upload(toys, dg.MASS_LO, dg.MASS_HI, n_toys=400))
    lam = np.tile(np.array(dg.MASS_TRUTH), (400, 1))
    bn, bg = bm2.nll_grad_batch(lam)
    for t in (0, 147, 148, 399):
        check(bn[t], bg[t], oracle.nll_grad(oracle.MASS, toys[t], lam[t], dg.MASS_LO, dg.MASS_HI))
    r = mm.fit(dg.MASS_START)
    assert r.converged
    print("ablation ok")
""")


@pytest.mark.parametrize("switch", ["MF_NO_TMA", "MF_NO_PDL", "MF_NO_POINTS_MMA", "MF_BATCH_STAGES=0", "MF_BATCH_STAGES=2",
                                    "MF_BATCH_BLOCK=32", "MF_BATCH_BLOCK=64", "MF_POINTS_COPY", "MF_BATCH_COPY"])
def test_ablation_switches_vs_oracle(mf, switch):
    """The MF_NO_TMA=1 (register-buffer kernels for the angular / 4D models), MF_NO_PDL=1 (plain stream order),
    MF_NO_POINTS_MMA=1, MF_BATCH_STAGES=0 (batched toys with direct loads) and MF_BATCH_BLOCK=32 / 64 (the one- and two-warp
    CTAs that the library picks by itself from 5920 / 3552 active toys on), MF_POINTS_COPY=1 (many-points calls fed by a
    stream-ordered copy: no overlap of consecutive calls) and MF_BATCH_COPY=1 (batch calls with copies of lambda and the rows)
    paths that DESIGN.md quotes numbers for,
    against the oracle."""
    env = dict(os.environ)
    name, _, value = switch.partition("=")
    env[name] = value or "1"
    p = subprocess.run([sys.executable, "-c", _ABLATION.format(root=ROOT)], env=env, capture_output=True, text=True, timeout=600)
    assert p.returncode == 0 and "ablation ok" in p.stdout, p.stdout[-2000:] + p.stderr[-4000:]


_DIST_WORKER = textwrap.dedent("""
    import os, sys
    import numpy as np
    sys.path.insert(0, {root!r})
    import torch.distributed as dist
    import mf_datagen as dg, oracle
    import paper_2505_12414_b200 as mf
    from paper_2505_12414_b200 import dist as mfd
    rank, world = int(sys.argv[1]), int(sys.argv[2])
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=sys.argv[3], RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ctx = mf.Context(0)
    # (a) one dataset, events sharded over the ranks: each rank's CUDA evaluation of its shard, rank-ordered combine
    n = 100_037
    ev = dg.gen_4d(n, seed=33)
    first, count = mfd.shard_events(n, rank, world)
    model = ctx.model_create(mf.MF_MASS_X_ANGULAR, ctx.dataset_upload(ev[:, first:first + count], dg.MASS_LO, dg.MASS_HI))
    nll, g = model.nll_grad(dg.FOURD_TRUTH)
    tot = mfd.combine_partials(np.concatenate([[nll], g]))
    o_nll, o_g, _ = oracle.nll_grad(oracle.FOURD, ev, dg.FOURD_TRUTH, dg.MASS_LO, dg.MASS_HI)
    assert abs(tot[0] - o_nll) <= 1e-11 * abs(o_nll), (tot[0], o_nll)
    assert np.all(np.abs(tot[1:] - o_g) <= 1e-9 * (1 + np.abs(o_g)))
    # (b) toys dealt to the ranks in contiguous blocks, per-toy rows gathered in toy order
    T, ne = 11, 2000
    toys = dg.gen_mass_toys(T, ne, first_seed=500)
    t0, tc = mfd.shard_toys(T, rank, world)
    bm = ctx.model_create(mf.MF_MASS_GAUSS_EXP, ctx.dataset_upload(toys[t0:t0 + tc], dg.MASS_LO, dg.MASS_HI, n_toys=tc))
    lam = np.tile(np.array(dg.MASS_TRUTH), (tc, 1))
    bn, bg = bm.nll_grad_batch(lam)
    rows = mfd.gather_toy_rows(np.concatenate([bn[:, None], bg], axis=1), T)
    for t in range(T):
        o_nll, o_g, _ = oracle.nll_grad(oracle.MASS, toys[t], dg.MASS_TRUTH, dg.MASS_LO, dg.MASS_HI)
        assert abs(rows[t, 0] - o_nll) <= 1e-11 * abs(o_nll)
        assert np.all(np.abs(rows[t, 1:] - o_g) <= 1e-9 * (1 + np.abs(o_g)))
    dist.barrier()
    dist.destroy_process_group()
    print("dist ok", rank)
""")


def test_dist_with_cuda_shard_sums(mf):
    """paper_2505_12414_b200.dist over gloo, world_size 2, both ranks on cuda:0 (independent kernels: no rank waits for
    another on the device): the shard sums come from the CUDA path, the totals are compared with the oracle."""
    import socket
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = str(s.getsockname()[1])
    s.close()
    code = _DIST_WORKER.format(root=ROOT)
    procs = [subprocess.Popen([sys.executable, "-c", code, str(r), "2", port], stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True)
             for r in range(2)]
    outs = [p.communicate(timeout=600) for p in procs]
    for r, (p, (so, se)) in enumerate(zip(procs, outs)):
        assert p.returncode == 0 and f"dist ok {r}" in so, so[-2000:] + se[-4000:]
