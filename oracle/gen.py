"""CPU ORACLE of the on-device pseudo-data generator (accept-reject /
inverse-CDF generation with a counter-based per-work-item RNG) — TEST INFRASTRUCTURE ONLY, like the rest of oracle/.

The recipe, followed step by step, one event at a time:

  RNG     Philox4x32-10 (Salmon et al., "Parallel random numbers: as easy as 1, 2, 3", SC'11), written out below.
          key = (seed mod 2^32, seed >> 32) with seed = seed0 + toy; counter = (event mod 2^32, event >> 32, draw, 0).
          One call gives four 32-bit words w0..w3 = two uniforms  u = ((w_hi * 2^32 + w_lo) >> 11 + 1/2) * 2^-53  in (0, 1).
  event   (mass model; round 2: ONE Philox block per event in the common case, all four words used)
          draw k gives  s = (w0 + 1/2) 2^-32,  u = ((w1 2^32 + w2) >> 11 + 1/2) 2^-53,  v = (w3 + 1/2) 2^-32.
          draw 0: signal if s < f, else background.
          background:  m = lo + log1p(u * expm1(tau w)) / tau   (tau != 0),  lo + u w  (tau == 0),  w = hi - lo; clamped to [lo, hi].
          signal: z = sqrt(-2 ln u) cos(2 pi v), m = mu + sigma z, with (u, v) of draw 0; if m is outside [lo, hi], (u, v) of
          draws 1, 2, ... until it is inside (after 64 rejected draws the last m is clamped into the range).
          (The angular and 4D recipes below keep two 53-bit uniforms per draw.)

The CUDA path implements the same recipe in its own code (mf_generate.cu); uniform words are bit-identical, the
floating-point transforms agree to a few ulp.  Pins (tests/test_oracle_gen.py): the published Philox4x32-10 known-answer
vectors; Kolmogorov-Smirnov distance of generated samples to the closed-form CDF of Eq. 2.
"""
from __future__ import annotations

import math

import numpy as np

_M0, _M1 = 0xD2511F53, 0xCD9E8D57
_W0, _W1 = 0x9E3779B9, 0xBB67AE85
_MASK = 0xFFFFFFFF


def philox4x32_10(counter, key):
    """counter: 4 ints, key: 2 ints (32-bit each) -> 4 ints."""
    c0, c1, c2, c3 = [int(x) & _MASK for x in counter]
    k0, k1 = [int(x) & _MASK for x in key]
    for _ in range(10):
        p0 = _M0 * c0
        p1 = _M1 * c2
        hi0, lo0 = p0 >> 32, p0 & _MASK
        hi1, lo1 = p1 >> 32, p1 & _MASK
        c0, c1, c2, c3 = (hi1 ^ c1 ^ k0) & _MASK, lo1, (hi0 ^ c3 ^ k1) & _MASK, lo0
        k0, k1 = (k0 + _W0) & _MASK, (k1 + _W1) & _MASK
    return c0, c1, c2, c3


def _uniform(w_hi: int, w_lo: int) -> float:
    return (((w_hi << 32) | w_lo) >> 11) * 2.0 ** -53 + 2.0 ** -54


def uniforms(seed: int, event: int, draw: int):
    w = philox4x32_10((event & _MASK, event >> 32, draw, 0), (seed & _MASK, seed >> 32))
    return _uniform(w[0], w[1]), _uniform(w[2], w[3])


def mass_draw(seed: int, event: int, draw: int):
    """(s, u, v) of one Philox block: s, v with 32 bits, u with 53 bits, all in (0, 1)."""
    w = philox4x32_10((event & _MASK, event >> 32, draw, 0), (seed & _MASK, seed >> 32))
    return (w[0] + 0.5) * 2.0 ** -32, _uniform(w[1], w[2]), (w[3] + 0.5) * 2.0 ** -32


def gen_mass_event(seed: int, event: int, lam, lo: float, hi: float):
    """(m, is_signal, number of draws used) of one event."""
    f, mu, sigma, tau = [float(x) for x in lam]
    s, u, v = mass_draw(seed, event, 0)
    if s < f:
        m = mu
        for k in range(0, 65):
            if k:
                _, u, v = mass_draw(seed, event, k)
            z = math.sqrt(-2.0 * math.log(u)) * math.cos(2.0 * math.pi * v)
            m = mu + sigma * z
            if lo <= m <= hi:
                return m, True, k + 1
        return min(max(m, lo), hi), True, 65
    w = hi - lo
    m = lo + u * w if tau == 0.0 else lo + math.log1p(u * math.expm1(tau * w)) / tau
    return min(max(m, lo), hi), False, 1


def gen_mass_toys(seed0: int, n_toys: int, n_events: int, lam, lo: float, hi: float) -> np.ndarray:
    """[n_toys][n_events]: toy t uses seed0 + t."""
    out = np.empty((n_toys, n_events))
    for t in range(n_toys):
        for i in range(n_events):
            out[t, i] = gen_mass_event(seed0 + t, i, lam, lo, hi)[0]
    return out


# ---------------------------------------------------------------- angular model (Eq. 4), accept-reject
#
#   proposal k = 0, 1, ... of event i uses draws 2k and 2k+1:  (u1, u2) -> cos theta_l = 2 u1 - 1, cos theta_K = 2 u2 - 1;
#   (u3, u4) -> phi = pi (2 u3 - 1), accepted if u4 * pmax < P(Omega), pmax = the paper's get_max() bound
#   9/(32 pi) (4 + sum |S_i| + 4/3 |AFB|).  The first accepted proposal is the event (after 4096
#   rejected proposals the last one is taken: unreachable in practice, the efficiency is >= 10 %).
#   P(Omega) is Eq. 4 written out term by term, here in Python, in the CUDA path in mf_generate.cu.

def angular_pdf(cl: float, ck: float, phi: float, a) -> float:
    FL, S3, S4, S5, AFB, S7, S8, S9 = [float(x) for x in a]
    cos2_l, cos2_k = cl * cl, ck * ck
    sin2_l, sin2_k = 1.0 - cos2_l, 1.0 - cos2_k
    sin_l, sin_k = math.sqrt(sin2_l), math.sqrt(sin2_k)
    cos2theta_l = 2.0 * cos2_l - 1.0
    sin2theta_l, sin2theta_k = 2.0 * sin_l * cl, 2.0 * sin_k * ck
    return 9.0 / (32.0 * math.pi) * (
        0.75 * (1.0 - FL) * sin2_k + FL * cos2_k + 0.25 * (1.0 - FL) * sin2_k * cos2theta_l - FL * cos2_k * cos2theta_l
        + S3 * sin2_k * sin2_l * math.cos(2.0 * phi) + S4 * sin2theta_k * sin2theta_l * math.cos(phi)
        + S5 * sin2theta_k * sin_l * math.cos(phi) + (4.0 / 3.0) * AFB * sin2_k * cl
        + S7 * sin2theta_k * sin_l * math.sin(phi) + S8 * sin2theta_k * sin2theta_l * math.sin(phi)
        + S9 * sin2_k * sin2_l * math.sin(2.0 * phi))


def angular_pmax(a) -> float:
    FL, S3, S4, S5, AFB, S7, S8, S9 = [float(x) for x in a]
    return 9.0 / (32.0 * math.pi) * (4.0 + abs(S3) + abs(S4) + abs(S5) + 4.0 / 3.0 * abs(AFB) + abs(S7) + abs(S8) + abs(S9))


def gen_angular_event(seed: int, event: int, a):
    """((cos theta_l, cos theta_K, phi), number of proposals) of one event."""
    pmax = angular_pmax(a)
    cl = ck = phi = 0.0
    for k in range(4096):
        u1, u2 = uniforms(seed, event, 2 * k)
        u3, u4 = uniforms(seed, event, 2 * k + 1)
        cl, ck, phi = 2.0 * u1 - 1.0, 2.0 * u2 - 1.0, math.pi * (2.0 * u3 - 1.0)
        if u4 * pmax < angular_pdf(cl, ck, phi, a):
            return (cl, ck, phi), k + 1
    return (cl, ck, phi), 4096


def gen_angular_toys(seed0: int, n_toys: int, n_events: int, a) -> np.ndarray:
    """[3][n_toys][n_events]"""
    out = np.empty((3, n_toys, n_events))
    for t in range(n_toys):
        for i in range(n_events):
            out[:, t, i] = gen_angular_event(seed0 + t, i, a)[0]
    return out


# ---------------------------------------------------------------- 4D model (BASELINE.json configs[3])
#
#   draw 0: (uA, uB).  Signal if uA < f.
#   signal:      mass from draws k = 1..64: (u1, u2) -> mu + sigma sqrt(-2 ln u1) cos(2 pi u2), the first inside [lo, hi]; angles by
#                the angular accept-reject above with the proposals taken from draws 100 + 2k, 101 + 2k.
#   background:  mass from uB by the inverse CDF; draw 1: (u1, -) -> phi = pi (2 u1 - 1);
#                (cos theta_l, cos theta_K) by accept-reject of the Legendre product l(x; cl1, cl2) l(y; ck1, ck2),
#                l(x; c1, c2) = 1/2 [1 + c1 x + c2 (3 x^2 - 1)/2], under the bound lmax(c1, c2) = 1/2 (1 + |c1| + |c2|) per factor:
#                proposal k uses draws 100 + 2k -> (x, y) = (2 u1 - 1, 2 u2 - 1) and 101 + 2k -> (u3, -), accepted if
#                u3 lmax_l lmax_k < l(x) l(y).

def _legendre2(x: float, c1: float, c2: float) -> float:
    return 0.5 * (1.0 + c1 * x + c2 * 0.5 * (3.0 * x * x - 1.0))


def gen_4d_event(seed: int, event: int, lam, lo: float, hi: float):
    """((m, cos theta_l, cos theta_K, phi), is_signal)."""
    lam = [float(x) for x in lam]
    f, mu, sigma, tau = lam[:4]
    a = lam[4:12]
    cl1, cl2, ck1, ck2 = lam[12:16]
    ua, ub = uniforms(seed, event, 0)
    if ua < f:
        m = mu
        for k in range(1, 65):
            u1, u2 = uniforms(seed, event, k)
            m = mu + sigma * (math.sqrt(-2.0 * math.log(u1)) * math.cos(2.0 * math.pi * u2))
            if lo <= m <= hi:
                break
        else:
            m = min(max(m, lo), hi)
        pmax = angular_pmax(a)
        cl = ck = phi = 0.0
        for k in range(4096):
            u1, u2 = uniforms(seed, event, 100 + 2 * k)
            u3, u4 = uniforms(seed, event, 101 + 2 * k)
            cl, ck, phi = 2.0 * u1 - 1.0, 2.0 * u2 - 1.0, math.pi * (2.0 * u3 - 1.0)
            if u4 * pmax < angular_pdf(cl, ck, phi, a):
                break
        return (m, cl, ck, phi), True
    w = hi - lo
    m = lo + ub * w if tau == 0.0 else lo + math.log1p(ub * math.expm1(tau * w)) / tau
    m = min(max(m, lo), hi)
    phi = math.pi * (2.0 * uniforms(seed, event, 1)[0] - 1.0)
    bound = 0.5 * (1.0 + abs(cl1) + abs(cl2)) * 0.5 * (1.0 + abs(ck1) + abs(ck2))
    x = y = 0.0
    for k in range(4096):
        u1, u2 = uniforms(seed, event, 100 + 2 * k)
        u3, _ = uniforms(seed, event, 101 + 2 * k)
        x, y = 2.0 * u1 - 1.0, 2.0 * u2 - 1.0
        if u3 * bound < _legendre2(x, cl1, cl2) * _legendre2(y, ck1, ck2):
            break
    return (m, x, y, phi), False


def gen_4d_toys(seed0: int, n_toys: int, n_events: int, lam, lo: float, hi: float) -> np.ndarray:
    """[4][n_toys][n_events]"""
    out = np.empty((4, n_toys, n_events))
    for t in range(n_toys):
        for i in range(n_events):
            out[:, t, i] = gen_4d_event(seed0 + t, i, lam, lo, hi)[0]
    return out
