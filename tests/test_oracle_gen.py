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
    assert 1.3 < (draws - 1).mean() < 1.8   # expected 1 / P(accept) = 1 / 0.655 = 1.53 Gaussian draws per signal event
