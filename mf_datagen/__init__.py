"""Seeded synthetic event generators for the five BASELINE.json configs.

This module only PRODUCES INPUT ARRAYS.  It holds none of the method's
arithmetic (no likelihood, no gradient, no normalisation constants used by
either evaluation path) and imports neither ``oracle/`` nor the CUDA package;
both of them are fed the arrays made here.  The arrays, not the RNG stream,
are the parity contract (PAPER.md:132,146 — the paper's own
Xoshiro stream cannot be reproduced from the text).

RNG: numpy's counter-based ``Philox`` bit generator, keyed by
``(seed, stream)``; uniforms are the top 53 bits of each raw 64-bit word.
Only ``random_raw`` is used (numpy guarantees bit-generator stream stability;
it does not guarantee it for ``Generator`` distributions).

Recipes:

* mass (C0, C1, C4; Eq. 2 shapes with BASELINE.json values):
  per event one uniform picks the component (signal with probability f);
  signal = Box-Muller normal(mu, sigma) re-drawn until inside [lo, hi];
  background = inverse CDF of exp(tau*m) truncated to [lo, hi].
* angular (C2; Eq. 4): accept-reject of uniform proposals in
  (cos theta_l, cos theta_K, phi) against the paper's ``get_max()`` envelope
  9/(32 pi) (4 + sum|S_i| + 4/3 |AFB|), flat acceptance.
* 4D (C3; BASELINE.json): signal with probability f = mass Gaussian x angular
  PDF, background = exponential x Legendre(2) product in the two cosines x
  flat phi (accept-reject against the product of the two 1D maxima).
"""
from __future__ import annotations

import math

import numpy as np

MASS_LO, MASS_HI = 5.0, 5.6
MASS_TRUTH = (0.3, 5.28, 0.02, -1.5)            # f, mu, sigma, tau (BASELINE.json C0)
MASS_START = (0.5, 5.27, 0.03, -1.0)            # BASELINE.json C0 start point
ANG_TRUTH = (0.6, -0.02, -0.15, -0.2, -0.05, 0.0, -0.02, -0.01)  # FL,S3,S4,S5,AFB,S7,S8,S9
BKG_TRUTH = (0.1, -0.05, 0.1, -0.05)            # cl1, cl2, ck1, ck2 (BASELINE.json C3)
FOURD_TRUTH = (0.2, 5.28, 0.02, -1.5) + ANG_TRUTH + BKG_TRUTH
# sqrt(N)*sigma_stat at the mass truth (quadrature of the Fisher matrix)
MASS_SQRTN_SIGMA = (0.61094, 0.049350, 0.044491, 7.0731)

_TWO_M53 = 2.0 ** -53


class _Stream:
    """Sequential reader of uniforms from one Philox(key=(seed, stream))."""

    def __init__(self, seed: int, stream: int):
        self._bg = np.random.Philox(key=[int(seed), int(stream)])

    def take(self, n: int) -> np.ndarray:
        raw = self._bg.random_raw(int(n))
        return (raw >> np.uint64(11)).astype(np.float64) * _TWO_M53


def _box_muller(u1: np.ndarray, u2: np.ndarray) -> np.ndarray:
    # u1 in [0,1): use 1-u1 in (0,1] so the log is finite
    return np.sqrt(-2.0 * np.log1p(-u1)) * np.cos(2.0 * math.pi * u2)


def _exp_inverse_cdf(u: np.ndarray, tau: float, lo: float, hi: float) -> np.ndarray:
    if tau == 0.0:
        return lo + (hi - lo) * u
    # F(m) = expm1(tau (m-lo)) / expm1(tau (hi-lo))
    return lo + np.log1p(u * math.expm1(tau * (hi - lo))) / tau


def _mass_from_streams(n, f, mu, sigma, tau, lo, hi, s_main: _Stream, s_redo: _Stream):
    u = s_main.take(3 * n).reshape(n, 3)
    is_sig = u[:, 0] < f
    m = np.where(is_sig,
                 mu + sigma * _box_muller(u[:, 1], u[:, 2]),
                 _exp_inverse_cdf(u[:, 1], tau, lo, hi))
    # re-draw Gaussian events that fell outside the range (never at the C0 truth: +-14 sigma)
    bad = np.flatnonzero(is_sig & ((m < lo) | (m > hi)))
    while bad.size:
        v = s_redo.take(2 * bad.size).reshape(bad.size, 2)
        m[bad] = mu + sigma * _box_muller(v[:, 0], v[:, 1])
        bad = bad[(m[bad] < lo) | (m[bad] > hi)]
    # the inverse CDF can round to just outside; clamp (closed range)
    np.clip(m, lo, hi, out=m)
    return m, is_sig


def gen_mass(n: int, seed: int, lam=MASS_TRUTH, lo: float = MASS_LO, hi: float = MASS_HI) -> np.ndarray:
    """C0/C1/C4 events: n doubles m in [lo, hi] from the Gaussian+exponential mixture."""
    f, mu, sigma, tau = (float(x) for x in lam)
    m, _ = _mass_from_streams(int(n), f, mu, sigma, tau, lo, hi, _Stream(seed, 0), _Stream(seed, 1))
    return np.ascontiguousarray(m)


def gen_mass_toys(n_toys: int, n_events: int, first_seed: int = 0, lam=MASS_TRUTH,
                  lo: float = MASS_LO, hi: float = MASS_HI) -> np.ndarray:
    """C4: [n_toys][n_events] array, toy t = gen_mass(n_events, seed=first_seed+t)."""
    out = np.empty((int(n_toys), int(n_events)), dtype=np.float64)
    for t in range(int(n_toys)):
        out[t] = gen_mass(n_events, first_seed + t, lam, lo, hi)
    return out


def _angular_shape(cl, ck, phi, a):
    """Shape of Eq. 4 used ONLY for the accept-reject decision."""
    FL, S3, S4, S5, AFB, S7, S8, S9 = a
    cl2, ck2 = cl * cl, ck * ck
    sl2, sk2 = 1.0 - cl2, 1.0 - ck2
    sl, sk = np.sqrt(sl2), np.sqrt(sk2)
    c2l = 2.0 * cl2 - 1.0
    s2l, s2k = 2.0 * sl * cl, 2.0 * sk * ck
    cp, sp = np.cos(phi), np.sin(phi)
    c2p, s2p = np.cos(2.0 * phi), np.sin(2.0 * phi)
    return (9.0 / (32.0 * math.pi)) * (
        0.75 * (1.0 - FL) * sk2 + FL * ck2 + 0.25 * (1.0 - FL) * sk2 * c2l - FL * ck2 * c2l
        + S3 * sk2 * sl2 * c2p + S4 * s2k * s2l * cp + S5 * s2k * sl * cp
        + (4.0 / 3.0) * AFB * sk2 * cl + S7 * s2k * sl * sp + S8 * s2k * s2l * sp + S9 * sk2 * sl2 * s2p)


def angular_envelope(a) -> float:
    """The paper's get_max() bound."""
    FL, S3, S4, S5, AFB, S7, S8, S9 = a
    return 9.0 / (32.0 * math.pi) * (4.0 + abs(S3) + abs(S4) + abs(S5) + 4.0 / 3.0 * abs(AFB)
                                     + abs(S7) + abs(S8) + abs(S9))


def _accept_reject_angular(n, a, stream: _Stream, block: int = 1 << 20):
    pmax = angular_envelope(a)
    got, parts = 0, []
    while got < n:
        u = stream.take(4 * block).reshape(block, 4)
        cl = 2.0 * u[:, 0] - 1.0
        ck = 2.0 * u[:, 1] - 1.0
        phi = math.pi * (2.0 * u[:, 2] - 1.0)
        keep = u[:, 3] * pmax < _angular_shape(cl, ck, phi, a)
        parts.append(np.stack([cl[keep], ck[keep], phi[keep]]))
        got += int(keep.sum())
    return np.concatenate(parts, axis=1)[:, :n]


def gen_angular(n: int, seed: int, a=ANG_TRUTH) -> np.ndarray:
    """C2 events: array [3][n] = (cos theta_l, cos theta_K, phi), first n accepted proposals."""
    return np.ascontiguousarray(_accept_reject_angular(int(n), tuple(float(x) for x in a), _Stream(seed, 0)))


def _legendre2(x, c1, c2):
    return 0.5 * (1.0 + c1 * x + c2 * 0.5 * (3.0 * x * x - 1.0))


def _accept_reject_bkg_angles(n, cl1, cl2, ck1, ck2, stream: _Stream, block: int = 1 << 20):
    # bound of each 1D factor on [-1,1]: 0.5 (1 + |c1| + |c2|)
    bound = 0.25 * (1.0 + abs(cl1) + abs(cl2)) * (1.0 + abs(ck1) + abs(ck2))
    got, parts = 0, []
    while got < n:
        u = stream.take(3 * block).reshape(block, 3)
        cl = 2.0 * u[:, 0] - 1.0
        ck = 2.0 * u[:, 1] - 1.0
        keep = u[:, 2] * bound < _legendre2(cl, cl1, cl2) * _legendre2(ck, ck1, ck2)
        parts.append(np.stack([cl[keep], ck[keep]]))
        got += int(keep.sum())
    return np.concatenate(parts, axis=1)[:, :n]


def gen_4d(n: int, seed: int, lam=FOURD_TRUTH, lo: float = MASS_LO, hi: float = MASS_HI) -> np.ndarray:
    """C3 events: array [4][n] = (m, cos theta_l, cos theta_K, phi)."""
    lam = tuple(float(x) for x in lam)
    f, mu, sigma, tau = lam[0:4]
    a = lam[4:12]
    cl1, cl2, ck1, ck2 = lam[12:16]
    n = int(n)
    m, is_sig = _mass_from_streams(n, f, mu, sigma, tau, lo, hi, _Stream(seed, 0), _Stream(seed, 1))
    out = np.empty((4, n), dtype=np.float64)
    out[0] = m
    n_sig = int(is_sig.sum())
    n_bkg = n - n_sig
    if n_sig:
        out[1:4, is_sig] = _accept_reject_angular(n_sig, a, _Stream(seed, 2))
    if n_bkg:
        bk = ~is_sig
        out[1:3, bk] = _accept_reject_bkg_angles(n_bkg, cl1, cl2, ck1, ck2, _Stream(seed, 3))
        out[3, bk] = math.pi * (2.0 * _Stream(seed, 4).take(n_bkg) - 1.0)
    return out


def gen_lambda_points(n_points: int, seed: int, centre, half_width) -> np.ndarray:
    """C1's parameter points: uniform in centre +- half_width, array [n_points][K]."""
    centre = np.asarray(centre, dtype=np.float64)
    half_width = np.asarray(half_width, dtype=np.float64)
    u = _Stream(seed, 7).take(n_points * centre.size).reshape(n_points, centre.size)
    return centre + (2.0 * u - 1.0) * half_width


def mass_sigma_stat(n_events: int) -> np.ndarray:
    return np.asarray(MASS_SQRTN_SIGMA) / math.sqrt(n_events)
