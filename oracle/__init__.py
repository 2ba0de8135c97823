"""CPU fp64 ORACLE for the MoreFit NLL + analytic gradient — TEST INFRASTRUCTURE ONLY.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It imports nothing from
``paper_2505_12414_b200`` (the CUDA path) and shares no code with it.

* ``mf_oracle.c``  — the plain per-event definitions (Eq. 1, 2, 4) and the
  long-double sums; compiled on first use with gcc into ``oracle/_build/``.
* ``fit()``        — the fit iteration of SURVEY.md §8(c) ("Fit"), step by step, in numpy.

Parity status: every function is pinned by ``tests/test_oracle_*.py`` (see the header of
``mf_oracle.c``); nothing here is "parity unpinned".
"""
from __future__ import annotations

import ctypes
import math
import os
import subprocess
from dataclasses import dataclass, field

import numpy as np

MASS, ANGULAR, FOURD = 0, 1, 2
NPARAMS = {MASS: 4, ANGULAR: 8, FOURD: 16}
NDIM = {MASS: 1, ANGULAR: 3, FOURD: 4}

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "mf_oracle.c")
_LIB_PATH = os.path.join(_HERE, "_build", "libmf_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile mf_oracle.c with gcc (no fast-math, no FMA contraction, OpenMP)."""
    os.makedirs(os.path.dirname(_LIB_PATH), exist_ok=True)
    if (not force and os.path.exists(_LIB_PATH)
            and os.path.getmtime(_LIB_PATH) >= os.path.getmtime(_SRC)):
        return _LIB_PATH
    tmp = _LIB_PATH + f".{os.getpid()}.tmp"
    subprocess.check_call(["gcc", "-O2", "-std=c11", "-fPIC", "-shared", "-fopenmp",
                           "-ffp-contract=off", "-fno-fast-math", "-o", tmp, _SRC, "-lm"])
    os.replace(tmp, _LIB_PATH)
    return _LIB_PATH


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        dp = ctypes.POINTER(ctypes.c_double)
        dpp = ctypes.POINTER(dp)
        lib.mfo_nll_grad.restype = ctypes.c_int64
        lib.mfo_nll_grad.argtypes = [ctypes.c_int, ctypes.c_int64, dpp, dp, ctypes.c_double,
                                     ctypes.c_double, ctypes.c_int, dp, dp]
        lib.mfo_nll_grad_w.restype = ctypes.c_int64
        lib.mfo_nll_grad_w.argtypes = [ctypes.c_int, ctypes.c_int64, dpp, dp, dp, ctypes.c_double,
                                       ctypes.c_double, ctypes.c_int, dp, dp]
        lib.mfo_nll_grad_hess_w.restype = ctypes.c_int64
        lib.mfo_nll_grad_hess_w.argtypes = [ctypes.c_int, ctypes.c_int64, dpp, dp, dp, ctypes.c_double, ctypes.c_double,
                                            dp, dp, dp, dp]
        lib.mfo_hess_points.restype = ctypes.c_int
        lib.mfo_hess_points.argtypes = [ctypes.c_int, ctypes.c_int64, dpp, dp, ctypes.c_double, ctypes.c_double, dp, dp, dp]
        lib.mfo_pdf.restype = ctypes.c_int
        lib.mfo_pdf.argtypes = [ctypes.c_int, ctypes.c_int64, dpp, dp, ctypes.c_double,
                                ctypes.c_double, dp, dp]
        lib.mfo_nll_grad_hess.restype = ctypes.c_int64
        lib.mfo_nll_grad_hess.argtypes = [ctypes.c_int, ctypes.c_int64, dpp, dp, ctypes.c_double, ctypes.c_double, dp, dp, dp]
        lib.mfo_mass_hess_points.restype = ctypes.c_int
        lib.mfo_mass_hess_points.argtypes = [ctypes.c_int64, dp, dp, ctypes.c_double, ctypes.c_double, dp, dp, dp]
        lib.mfo_mass_norms.restype = None
        lib.mfo_mass_norms.argtypes = [dp, ctypes.c_double, ctypes.c_double, dp]
        lib.mfo_angular_terms.restype = None
        lib.mfo_angular_terms.argtypes = [ctypes.c_double, ctypes.c_double, ctypes.c_double, dp]
        lib.mfo_max_threads.restype = ctypes.c_int
        _lib = lib
    return _lib


def _dptr(a: np.ndarray):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def _columns(kind: int, events) -> tuple[list[np.ndarray], int]:
    ev = np.asarray(events, dtype=np.float64)
    if ev.ndim == 1:
        ev = ev[None, :]
    if ev.shape[0] != NDIM[kind]:
        raise ValueError(f"kind {kind} needs {NDIM[kind]} columns, got {ev.shape[0]}")
    cols = [np.ascontiguousarray(ev[j]) for j in range(ev.shape[0])]
    return cols, int(ev.shape[1])


def _colptrs(cols):
    arr = (ctypes.POINTER(ctypes.c_double) * len(cols))()
    for j, c in enumerate(cols):
        arr[j] = _dptr(c)
    return arr


def check_domain(kind: int, lam) -> bool:
    """Parameter domain: finite, and for the mass part 0<=f<=1, sigma>0."""
    lam = np.asarray(lam, dtype=np.float64)
    if lam.shape != (NPARAMS[kind],) or not np.all(np.isfinite(lam)):
        return False
    if kind in (MASS, FOURD):
        if not (0.0 <= lam[0] <= 1.0) or not (lam[2] > 0.0):
            return False
    return True


def max_threads() -> int:
    return int(_load().mfo_max_threads())


def _weights(weights, n: int):
    if weights is None:
        return None
    w = np.ascontiguousarray(weights, dtype=np.float64)
    if w.shape != (n,):
        raise ValueError(f"weights must have shape ({n},)")
    return w


def nll_grad(kind: int, events, lam, lo: float = 0.0, hi: float = 0.0, nthreads: int = 1,
             want_grad: bool = True, weights=None):
    """(-ln L, d(-ln L)/d lambda, n_bad) over all events (Eq. 1); with ``weights`` the weighted sums
    -sum_i w_i ln P_i (reading R23)."""
    lib = _load()
    cols, n = _columns(kind, events)
    lam = np.ascontiguousarray(lam, dtype=np.float64)
    if not check_domain(kind, lam):
        raise ValueError("parameter outside its domain")
    w = _weights(weights, n)
    nll = ctypes.c_double(0.0)
    grad = np.zeros(NPARAMS[kind], dtype=np.float64)
    if w is None:
        nbad = lib.mfo_nll_grad(kind, n, _colptrs(cols), _dptr(lam), lo, hi, int(nthreads),
                                ctypes.byref(nll), _dptr(grad) if want_grad else None)
    else:
        nbad = lib.mfo_nll_grad_w(kind, n, _colptrs(cols), _dptr(w), _dptr(lam), lo, hi, int(nthreads),
                                  ctypes.byref(nll), _dptr(grad) if want_grad else None)
    if nbad < 0:
        raise ValueError("bad argument")
    return float(nll.value), (grad if want_grad else None), int(nbad)


def nll_grad_hess(kind: int, events, lam, lo: float = 0.0, hi: float = 0.0, weights=None, want_fisher: bool = False):
    """(-ln L, gradient [K], Hessian [K][K], n_bad) from the analytic second derivatives (
    SURVEY.md §8(f)-1), all three kinds, optionally weighted.  ``want_fisher``: also returns
    sum_i w_i^2 s_i s_i^T (s = d ln P/d lambda, reading R23) as a fifth element, before n_bad."""
    lib = _load()
    cols, n = _columns(kind, events)
    lam = np.ascontiguousarray(lam, dtype=np.float64)
    if not check_domain(kind, lam):
        raise ValueError("parameter outside its domain")
    w = _weights(weights, n)
    K = NPARAMS[kind]
    nll = ctypes.c_double(0.0)
    grad = np.zeros(K, dtype=np.float64)
    hess = np.zeros((K, K), dtype=np.float64)
    fisher = np.zeros((K, K), dtype=np.float64)
    nbad = lib.mfo_nll_grad_hess_w(kind, n, _colptrs(cols), _dptr(w) if w is not None else None, _dptr(lam), lo, hi,
                                   ctypes.byref(nll), _dptr(grad), _dptr(hess), _dptr(fisher))
    if nbad < 0:
        raise ValueError("bad argument")
    if want_fisher:
        return float(nll.value), grad, hess, fisher, int(nbad)
    return float(nll.value), grad, hess, int(nbad)


def nll_grad_hess_unweighted_c(kind: int, events, lam, lo: float = 0.0, hi: float = 0.0):
    """mfo_nll_grad_hess as first written (mass and angular kinds only); kept so that a test can show that the weighted
    routine with w = NULL reproduces it bit for bit."""
    lib = _load()
    cols, n = _columns(kind, events)
    lam = np.ascontiguousarray(lam, dtype=np.float64)
    K = NPARAMS[kind]
    nll = ctypes.c_double(0.0)
    grad = np.zeros(K, dtype=np.float64)
    hess = np.zeros((K, K), dtype=np.float64)
    nbad = lib.mfo_nll_grad_hess(kind, n, _colptrs(cols), _dptr(lam), lo, hi, ctypes.byref(nll), _dptr(grad), _dptr(hess))
    if nbad < 0:
        raise ValueError("bad argument (mass and angular kinds only)")
    return float(nll.value), grad, hess, int(nbad)


def hess_points(kind: int, events, lam, lo: float = 0.0, hi: float = 0.0):
    """Per event: P [n], d ln P/d lambda [n][K], d2 ln P/d lambda^2 [n][K][K]."""
    lib = _load()
    cols, n = _columns(kind, events)
    lam = np.ascontiguousarray(lam, dtype=np.float64)
    K = NPARAMS[kind]
    P = np.empty(n)
    g = np.empty((n, K))
    H = np.empty((n, K, K))
    if lib.mfo_hess_points(kind, n, _colptrs(cols), _dptr(lam), lo, hi, _dptr(P), _dptr(g), _dptr(H)) != 0:
        raise ValueError("bad argument")
    return P, g, H


def mass_hess_points(m, lam, lo: float, hi: float):
    """P [n], d ln P/d lambda [n][4] and the packed Hessian of ln P [n][10] (ff, fm, fs, ft, mm, ms, mt, ss, st, tt)."""
    lib = _load()
    m = np.ascontiguousarray(m, dtype=np.float64)
    lam = np.ascontiguousarray(lam, dtype=np.float64)
    P = np.empty(m.size)
    g = np.empty((m.size, 4))
    h = np.empty((m.size, 10))
    lib.mfo_mass_hess_points(m.size, _dptr(m), _dptr(lam), lo, hi, _dptr(P), _dptr(g), _dptr(h))
    return P, g, h


def pdf(kind: int, events, lam, lo: float = 0.0, hi: float = 0.0, want_grad: bool = True):
    """Per-event P(x_i|lambda) and d ln P/d lambda_k (array [K][n])."""
    lib = _load()
    cols, n = _columns(kind, events)
    lam = np.ascontiguousarray(lam, dtype=np.float64)
    p = np.empty(n, dtype=np.float64)
    d = np.empty((NPARAMS[kind], n), dtype=np.float64) if want_grad else None
    rc = lib.mfo_pdf(kind, n, _colptrs(cols), _dptr(lam), lo, hi, _dptr(p),
                     _dptr(d) if want_grad else None)
    if rc != 0:
        raise ValueError("bad argument")
    return p, d


def mass_norms(lam, lo: float, hi: float) -> dict:
    out = np.zeros(5)
    lam = np.ascontiguousarray(lam, dtype=np.float64)
    _load().mfo_mass_norms(_dptr(lam), lo, hi, _dptr(out))
    return dict(N1=out[0], dN1_dmu=out[1], dN1_dsigma=out[2], N2=out[3], dlnN2_dtau=out[4])


def angular_terms(cl: float, ck: float, phi: float) -> np.ndarray:
    """c * (the eleven terms of Eq. 4 in printed order, coefficient-free)."""
    out = np.zeros(11)
    _load().mfo_angular_terms(cl, ck, phi, _dptr(out))
    return out


# --------------------------------------------------------------------------- fit
@dataclass
class FitOptions:
    max_iter: int = 200          # BFGS iterations
    edm_tol: float = 1e-5        # switch from BFGS to the Newton polish when EDM < edm_tol
    armijo_c1: float = 1e-4
    backtrack: float = 0.5
    max_backtracks: int = 40
    polish_tol: float = 1e-9     # max_k |Newton step_k| / sigma_k at which the fit has converged
    max_polish: int = 8          # FD Hessians in the polish
    max_chord: int = 8           # Newton steps per FD Hessian
    fd_rel: float = 1e-5         # first FD step: fd_rel * max(|lambda_k|, 1)
    fd_sigma: float = 1e-4       # later FD steps: fd_sigma * sigma_k


@dataclass
class FitResult:
    lam: np.ndarray
    cov: np.ndarray
    nll: float
    n_calls: int
    converged: bool
    n_iter: int = 0
    history: list = field(default_factory=list)
    cov_hesse: np.ndarray | None = None   # H^-1 (equals cov for an unweighted fit)

    @property
    def sigma(self):
        return np.sqrt(np.diag(self.cov))


def fit(kind: int, events, start, fixed=None, lo: float = 0.0, hi: float = 0.0,
        opts: FitOptions | None = None, nthreads: int = 1, weights=None) -> FitResult:
    """Quasi-Newton fit of SURVEY.md §8(c) "Fit", in the order stated there:

    1. seed the inverse Hessian with a central-difference Hessian of the analytic gradient
       at the start point (diagonal only if that matrix is not positive definite);
    2. BFGS with inverse-Hessian update and a backtracking (Armijo) line search that rejects
       non-finite points, domain errors and P<=0 points, until EDM = g^T H^-1 g / 2 < edm_tol;
    3. polish: central-difference Hessian of the analytic gradient, then Newton steps with
       that Hessian until max_k |step_k|/sigma_k < polish_tol; cov = H^-1.

    With ``weights`` the minimised function is -sum_i w_i ln P_i and the returned covariance is the sandwich
    H^-1 F H^-1 with F = sum_i w_i^2 s_i s_i^T evaluated at the minimum (reading R23); the
    convergence test keeps using H^-1 (``cov_hesse``).
    """
    o = opts or FitOptions()
    K = NPARAMS[kind]
    x = np.array(start, dtype=np.float64)
    free = np.ones(K, bool) if fixed is None else ~np.asarray(fixed, bool)
    idx = np.flatnonzero(free)
    nf = idx.size
    calls = 0

    def F(xx):
        nonlocal calls
        calls += 1
        if not check_domain(kind, xx):
            return math.inf, None
        v, g, nbad = nll_grad(kind, events, xx, lo, hi, nthreads, weights=weights)
        if nbad or not math.isfinite(v) or not np.all(np.isfinite(g)):
            return math.inf, None
        return v, g[idx]

    def fd_hessian(xx, h):
        H = np.zeros((nf, nf))
        for a, k in enumerate(idx):
            xp = xx.copy(); xp[k] += h[a]
            xm = xx.copy(); xm[k] -= h[a]
            _, gp = F(xp)
            _, gm = F(xm)
            if gp is None or gm is None:
                return None
            H[a] = (gp - gm) / ((xp[k] - xm[k]))
        return 0.5 * (H + H.T)

    def inv_pd(H):
        try:
            np.linalg.cholesky(H)
        except np.linalg.LinAlgError:
            return None
        return np.linalg.inv(H)

    f, g = F(x)
    if g is None:
        raise ValueError("start point is not a valid parameter point")
    h0 = o.fd_rel * np.maximum(np.abs(x[idx]), 1.0)
    H0 = fd_hessian(x, h0)
    Hinv = inv_pd(H0) if H0 is not None else None
    if Hinv is None:
        d = np.abs(np.diag(H0)) if H0 is not None else np.ones(nf)
        Hinv = np.diag(1.0 / np.where(d > 0, d, 1.0))

    n_iter = 0
    for n_iter in range(1, o.max_iter + 1):
        edm = 0.5 * g @ Hinv @ g
        if edm < o.edm_tol:
            break
        p = -Hinv @ g
        slope = g @ p
        if slope >= 0:  # not a descent direction: reset the metric
            Hinv = np.diag(np.abs(np.diag(Hinv)))
            p = -Hinv @ g
            slope = g @ p
        alpha, ok = 1.0, False
        for _ in range(o.max_backtracks):
            xn = x.copy(); xn[idx] += alpha * p
            fn, gn = F(xn)
            if gn is not None and fn <= f + o.armijo_c1 * alpha * slope:
                ok = True
                break
            alpha *= o.backtrack
        if not ok:
            break
        s = xn[idx] - x[idx]
        y = gn - g
        sy = s @ y
        if sy > 1e-10 * np.linalg.norm(s) * np.linalg.norm(y):
            rho = 1.0 / sy
            V = np.eye(nf) - rho * np.outer(s, y)
            Hinv = V @ Hinv @ V.T + rho * np.outer(s, s)
        x, f, g = xn, fn, gn

    converged = False
    cov = Hinv
    h = o.fd_sigma * np.sqrt(np.abs(np.diag(Hinv)))
    for _ in range(o.max_polish):
        H = fd_hessian(x, h)
        c = inv_pd(H) if H is not None else None
        if c is None:
            break
        cov = c
        sig = np.sqrt(np.diag(cov))
        h = o.fd_sigma * sig
        moved = np.zeros(nf)
        done = False
        for _ in range(o.max_chord):
            step = -cov @ g
            if np.max(np.abs(step) / sig) < o.polish_tol:
                done = True
                break
            xn = x.copy(); xn[idx] += step
            fn, gn = F(xn)
            if gn is None:
                break
            moved += np.abs(step)
            x, f, g = xn, fn, gn
        if done and np.max(moved / sig) < 1e-3:
            converged = True
            break

    cov_full = np.zeros((K, K))
    cov_full[np.ix_(idx, idx)] = cov
    cov_hesse = cov_full
    if weights is not None:
        fisher = nll_grad_hess(kind, events, x, lo, hi, weights=weights, want_fisher=True)[3]
        cov_full = np.zeros((K, K))
        cov_full[np.ix_(idx, idx)] = cov @ fisher[np.ix_(idx, idx)] @ cov
    return FitResult(lam=x, cov=cov_full, nll=f, n_calls=calls, converged=converged, n_iter=n_iter, cov_hesse=cov_hesse)
