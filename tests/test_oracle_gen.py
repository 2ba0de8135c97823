"""Pins for the generator oracle (oracle/gen.py): the published Philox4x32-10 known-answer vectors (Random123
kat_vectors) and the distribution of the generated events against the closed-form CDF of Eq. 2."""
import math

import numpy as np
from scipy import special, stats

import mf_datagen as dg
from oracle import gen

LO, HI = dg.MASS_LO, dg.MASS_HI


def test_philox_known_answers():
    assert gen.philox4x32_10((0, 0, 0, 0), (0, 0)) == (0x6627e8d5, 0xe169c58d, 0xbc57ac4c, 0x9b00dbd8)
    assert gen.philox4x32_10((0xffffffff,) * 4, (0xffffffff,) * 2) == (0x408f276d, 0x41c83b0e, 0xa20bc7c6, 0x6d5451fd)
    assert gen.philox4x32_10((0x243f6a88, 0x85a308d3, 0x13198a2e, 0x03707344), (0xa4093822, 0x299f31d0)) == \
        (0xd16cfe09, 0x94fdcceb, 0x5001e420, 0x24126ea1)


def test_uniforms_are_open_interval_and_distinct():
    u = [gen.uniforms(7, i, d) for i in range(200) for d in range(3)]
    flat = np.array(u).ravel()
    assert np.all((flat > 0) & (flat < 1)) and len(set(flat)) == flat.size
    assert abs(flat.mean() - 0.5) < 0.03
    assert gen.uniforms(7, 5, 1) != gen.uniforms(8, 5, 1) != gen.uniforms(7, 6, 1)


def mass_cdf(x, lam):
    f, mu, sigma, tau = lam
    s2 = math.sqrt(2) * sigma
    n1 = 0.5 * (special.erf((mu - LO) / s2) - special.erf((mu - HI) / s2))
    sig = 0.5 * (special.erf((x - mu) / s2) - special.erf((LO - mu) / s2)) / n1
    bkg = (x - LO) / (HI - LO) if tau == 0 else np.expm1(tau * (x - LO)) / math.expm1(tau * (HI - LO))
    return f * sig + (1 - f) * bkg


def test_generated_events_follow_eq2():
    for lam, seed in ((dg.MASS_TRUTH, 3), ((0.5, 5.55, 0.08, 2.0), 4), ((0.2, 5.3, 0.05, 0.0), 5)):
        x = gen.gen_mass_toys(seed, 1, 6000, lam, LO, HI)[0]
        assert np.all((x >= LO) & (x <= HI))
        d, p = stats.kstest(x, lambda v: mass_cdf(v, lam))
        assert p > 1e-3, (lam, d, p)


def test_signal_fraction_and_redraws():
    lam = (0.5, 5.58, 0.05, -1.5)         # peak near the upper edge: ~35 % of the Gaussian draws are rejected
    r = [gen.gen_mass_event(11, i, lam, LO, HI) for i in range(4000)]
    sig = np.array([s for _, s, _ in r])
    draws = np.array([k for _, s, k in r if s])
    assert abs(sig.mean() - 0.5) < 0.03
    assert 1.3 < draws.mean() < 1.8         # expected 1 / P(accept) = 1 / 0.655 = 1.53 Gaussian draws per signal event (draw 0 is the first)


def test_angular_generator_pdf_is_the_pinned_oracle_pdf():
    """oracle/gen.py's Eq. 4 (used for the accept decision) equals the pinned likelihood oracle's PDF (mf_oracle.c)."""
    import oracle
    rng = np.random.default_rng(1)
    ev = np.stack([rng.uniform(-1, 1, 200), rng.uniform(-1, 1, 200), rng.uniform(-np.pi, np.pi, 200)])
    for a in (dg.ANG_TRUTH, (0.3, 0.1, -0.2, 0.25, 0.1, -0.05, 0.07, -0.09)):
        P, _ = oracle.pdf(oracle.ANGULAR, ev, a)
        mine = np.array([gen.angular_pdf(*ev[:, i], a) for i in range(200)])
        assert np.allclose(mine, P, rtol=1e-13, atol=1e-16)
        assert np.all(P <= gen.angular_pmax(a))


def test_angular_generated_marginals():
    """Closed-form marginals of Eq. 4: dG/dcos(theta_l) = 3/4 FL (1-cl^2) + 3/8 (1-FL)(1+cl^2) + AFB cl,
    dG/dcos(theta_K) = 3/4 (1-FL)(1-ck^2) + 3/2 FL ck^2, dG/dphi = [1 + S3 cos 2phi + S9 sin 2phi] / (2 pi)."""
    a = (0.6, -0.1, -0.15, -0.2, 0.2, 0.0, -0.02, 0.15)
    FL, S3, AFB, S9 = a[0], a[1], a[4], a[7]
    x = gen.gen_angular_toys(21, 1, 5000, a)[:, 0, :]
    cdf_l = lambda c: 0.75 * FL * (c - c ** 3 / 3 + 2 / 3) + 0.375 * (1 - FL) * (c + c ** 3 / 3 + 4 / 3) + AFB * (c * c - 1) / 2
    cdf_k = lambda c: 0.75 * (1 - FL) * (c - c ** 3 / 3 + 2 / 3) + 0.5 * FL * (c ** 3 + 1)
    cdf_p = lambda p: (p + np.pi + S3 * np.sin(2 * p) / 2 + S9 * (1 - np.cos(2 * p)) / 2) / (2 * np.pi)
    for col, cdf in ((x[0], cdf_l), (x[1], cdf_k), (x[2], cdf_p)):
        assert stats.kstest(col, cdf).pvalue > 1e-3
    eff = np.mean([1.0 / gen.gen_angular_event(5, i, a)[1] for i in range(500)])
    assert 0.05 < eff < 0.9


def test_4d_generated_sample_is_consistent_with_the_4d_pdf():
    """The generated 4D sample maximises its own likelihood near the generating values: the pinned oracle's gradient at
    the truth, in units of its statistical spread, is O(1) (score test), and the signal fraction and the marginals match."""
    import oracle
    lam = dg.FOURD_TRUTH
    n = 4000
    ev = gen.gen_4d_toys(77, 1, n, lam, LO, HI)[:, 0, :]
    assert np.all((ev[0] >= LO) & (ev[0] <= HI)) and np.all(np.abs(ev[1:3]) <= 1) and np.all(np.abs(ev[3]) <= np.pi)
    sig = np.array([gen.gen_4d_event(77, i, lam, LO, HI)[1] for i in range(n)])
    assert abs(sig.mean() - lam[0]) < 4 * math.sqrt(lam[0] * (1 - lam[0]) / n)
    # score test: g_k / sqrt(sum of squared per-event scores) ~ N(0, 1) at the generating point
    nll, g, bad = oracle.nll_grad(oracle.FOURD, ev, lam, LO, HI)
    P, dl = oracle.pdf(oracle.FOURD, ev, lam, LO, HI)
    z = -g / np.sqrt((dl ** 2).sum(axis=1))
    assert bad == 0 and np.all(np.abs(z) < 4.5), z
    # background angles: Legendre marginal in cos theta_l of the background events
    x = ev[1][~sig]
    c1, c2 = lam[12], lam[13]
    cdf = lambda v: 0.5 * ((v + 1) + c1 * (v * v - 1) / 2 + c2 * 0.5 * (v ** 3 - v))
    assert stats.kstest(x, cdf).pvalue > 1e-3
