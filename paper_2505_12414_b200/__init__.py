"""paper_2505_12414_b200 — thin Python binding of the C-ABI library ``libmorefit_b200.so``.

Argument marshalling only: every step of the hot path (event-only precompute, fused
NLL + gradient, reductions, batched toys) runs in the library's sm_100a kernels, and the
fit driver is the library's host C++ (``include/morefit_b200.h`` documents each call).
There is no CPU fallback: if the library has not been built (``python -m
paper_2505_12414_b200.build``) importing the binding's objects raises, and without a CUDA
device ``Context()`` raises ``MoreFitError(MF_ERR_CUDA)``.

The names mirror the C entry points: ``Context`` (mf_ctx_*), ``Context.dataset_upload``
(mf_dataset_upload), ``Context.model_create`` (mf_model_create), ``Model.nll_grad``,
``Model.nll_grad_async``, ``Model.nll_grad_batch``, ``Model.fit``, ``Model.fit_batch``.
"""
from __future__ import annotations

import ctypes
import weakref
import os

import numpy as np

from . import build as _build

MF_OK, MF_ERR_ARG, MF_ERR_CUDA, MF_ERR_OOM, MF_ERR_DATA_RANGE, MF_ERR_PARAM_DOMAIN, MF_NONPOSITIVE_PDF = range(7)
MF_MASS_GAUSS_EXP, MF_ANGULAR_KSTMUMU, MF_MASS_X_ANGULAR = 0, 1, 2
MF_HOST, MF_DEVICE = 0, 1
MF_MAX_PARAMS = 16
NPARAMS = {MF_MASS_GAUSS_EXP: 4, MF_ANGULAR_KSTMUMU: 8, MF_MASS_X_ANGULAR: 16}
NDIM = {MF_MASS_GAUSS_EXP: 1, MF_ANGULAR_KSTMUMU: 3, MF_MASS_X_ANGULAR: 4}
_STATUS_NAMES = ["MF_OK", "MF_ERR_ARG", "MF_ERR_CUDA", "MF_ERR_OOM", "MF_ERR_DATA_RANGE",
                 "MF_ERR_PARAM_DOMAIN", "MF_NONPOSITIVE_PDF"]

EXPORTS = [
    "mf_ctx_create", "mf_ctx_destroy", "mf_last_error", "mf_ctx_kernel_launches",
    "mf_dataset_upload", "mf_generate_mass", "mf_generate_angular", "mf_generate_4d", "mf_dataset_download", "mf_dataset_set_weights", "mf_dataset_destroy", "mf_dataset_n_events", "mf_dataset_n_toys",
    "mf_model_create", "mf_model_destroy", "mf_model_nparams", "mf_model_n_events", "mf_model_n_toys",
    "mf_nll_grad", "mf_nll_grad_async", "mf_nll_grad_points", "mf_nll_grad_sweep", "mf_nll_grad_batch", "mf_nll_grad_batch_async",
    "mf_model_serve", "mf_model_is_served", "mf_model_has_hessian", "mf_model_is_weighted", "mf_nll_grad_hess", "mf_nll_grad_hess_fisher", "mf_nll_grad_hess_batch",
    "mf_fit_opts_default", "mf_fit", "mf_fit_batch", "mf_toy_study_mass", "mf_toy_study_angular",
    "mf_combine_partials", "mf_nll_grad_mass_noalloc",
]
MF_NOALLOC_MAX_EVENTS = 1 << 25


class MoreFitError(RuntimeError):
    def __init__(self, status: int, text: str = ""):
        self.status = int(status)
        name = _STATUS_NAMES[status] if 0 <= status < len(_STATUS_NAMES) else str(status)
        super().__init__(f"{name}: {text}" if text else name)


class FitOpts(ctypes.Structure):
    _fields_ = [("max_iter", ctypes.c_int), ("edm_tol", ctypes.c_double), ("armijo_c1", ctypes.c_double),
                ("backtrack", ctypes.c_double), ("max_backtracks", ctypes.c_int), ("polish_tol", ctypes.c_double),
                ("max_polish", ctypes.c_int), ("max_chord", ctypes.c_int), ("fd_rel", ctypes.c_double),
                ("fd_sigma", ctypes.c_double), ("analytic_hessian", ctypes.c_int)]


class _FitResultC(ctypes.Structure):
    _fields_ = [("lambda_hat", ctypes.c_double * MF_MAX_PARAMS),
                ("cov", ctypes.c_double * (MF_MAX_PARAMS * MF_MAX_PARAMS)),
                ("nll_min", ctypes.c_double), ("n_calls", ctypes.c_int), ("n_iter", ctypes.c_int),
                ("converged", ctypes.c_int)]


class FitResult:
    """Fitted parameters, HESSE covariance (K x K), -ln L at the minimum, call counts."""

    def __init__(self, c: _FitResultC, K: int):
        self.lam = np.array(c.lambda_hat[:K], dtype=np.float64)
        self.cov = np.array(c.cov[:K * K], dtype=np.float64).reshape(K, K)
        self.nll = float(c.nll_min)
        self.n_calls = int(c.n_calls)
        self.n_iter = int(c.n_iter)
        self.converged = bool(c.converged)

    @property
    def sigma(self) -> np.ndarray:
        return np.sqrt(np.diag(self.cov))


class BatchFitResult:
    """Results of mf_fit_batch as arrays: lam [T][K], cov [T][K][K], nll [T], n_calls [T], n_iter [T],
    converged [T] (bool), sigma [T][K].  Indexing or iterating yields per-toy FitResult-like views."""

    _DT = np.dtype([("lambda_hat", np.float64, (MF_MAX_PARAMS,)), ("cov", np.float64, (MF_MAX_PARAMS * MF_MAX_PARAMS,)),
                    ("nll_min", np.float64), ("n_calls", np.int32), ("n_iter", np.int32), ("converged", np.int32),
                    ("_pad", np.int32)])

    def __init__(self, raw, T: int, K: int):
        assert self._DT.itemsize == ctypes.sizeof(_FitResultC)
        a = raw if isinstance(raw, np.ndarray) else np.frombuffer(raw, dtype=self._DT, count=T)
        self.lam = a["lambda_hat"][:, :K].copy()
        self.cov = a["cov"][:, :K * K].reshape(T, K, K).copy()
        self.nll = a["nll_min"].copy()
        self.n_calls = a["n_calls"].copy()
        self.n_iter = a["n_iter"].copy()
        self.converged = a["converged"] != 0
        self.sigma = np.sqrt(np.abs(np.diagonal(self.cov, axis1=1, axis2=2)))

    def __len__(self):
        return self.lam.shape[0]

    def __getitem__(self, t):
        v = FitResult.__new__(FitResult)
        v.lam, v.cov, v.nll = self.lam[t], self.cov[t], float(self.nll[t])
        v.n_calls, v.n_iter, v.converged = int(self.n_calls[t]), int(self.n_iter[t]), bool(self.converged[t])
        return v

    def __iter__(self):
        return (self[t] for t in range(len(self)))


_lib = None


def lib_path() -> str:
    return _build.LIB_PATH


def load_library() -> ctypes.CDLL:
    """Loads lib/libmorefit_b200.so; raises if it has not been built (no fallback exists)."""
    global _lib
    if _lib is not None:
        return _lib
    path = lib_path()
    if not os.path.exists(path):
        raise ImportError(f"{path} is missing: build it with `python -m paper_2505_12414_b200.build` "
                          "(nvcc, sm_100a). There is no CPU fallback.")
    lib = ctypes.CDLL(path)
    vp, dp, i64 = ctypes.c_void_p, ctypes.POINTER(ctypes.c_double), ctypes.c_int64
    u8p = ctypes.POINTER(ctypes.c_uint8)
    lib.mf_ctx_create.restype = ctypes.c_int
    lib.mf_ctx_create.argtypes = [ctypes.c_int, vp, ctypes.POINTER(vp)]
    lib.mf_ctx_destroy.restype = None
    lib.mf_ctx_destroy.argtypes = [vp]
    lib.mf_last_error.restype = ctypes.c_char_p
    lib.mf_last_error.argtypes = [vp]
    lib.mf_ctx_kernel_launches.restype = i64
    lib.mf_ctx_kernel_launches.argtypes = [vp]
    lib.mf_dataset_upload.restype = ctypes.c_int
    lib.mf_dataset_upload.argtypes = [vp, ctypes.c_int, i64, i64, ctypes.POINTER(vp), ctypes.c_int, dp, dp,
                                      ctypes.POINTER(vp)]
    lib.mf_generate_mass.restype = ctypes.c_int
    lib.mf_generate_mass.argtypes = [vp, ctypes.c_uint64, i64, i64, dp, ctypes.c_double, ctypes.c_double, ctypes.POINTER(vp)]
    lib.mf_generate_angular.restype = ctypes.c_int
    lib.mf_generate_angular.argtypes = [vp, ctypes.c_uint64, i64, i64, dp, ctypes.POINTER(vp)]
    lib.mf_generate_4d.restype = ctypes.c_int
    lib.mf_generate_4d.argtypes = [vp, ctypes.c_uint64, i64, i64, dp, ctypes.c_double, ctypes.c_double, ctypes.POINTER(vp)]
    lib.mf_dataset_download.restype = ctypes.c_int
    lib.mf_dataset_download.argtypes = [vp, dp]
    lib.mf_dataset_set_weights.restype = ctypes.c_int
    lib.mf_dataset_set_weights.argtypes = [vp, vp, ctypes.c_int]
    lib.mf_dataset_destroy.restype = None
    lib.mf_dataset_destroy.argtypes = [vp]
    lib.mf_dataset_n_events.restype = i64
    lib.mf_dataset_n_events.argtypes = [vp]
    lib.mf_dataset_n_toys.restype = i64
    lib.mf_dataset_n_toys.argtypes = [vp]
    lib.mf_model_create.restype = ctypes.c_int
    lib.mf_model_create.argtypes = [vp, ctypes.c_int, vp, ctypes.POINTER(vp)]
    lib.mf_model_destroy.restype = None
    lib.mf_model_destroy.argtypes = [vp]
    lib.mf_model_nparams.restype = ctypes.c_int
    lib.mf_model_nparams.argtypes = [vp]
    lib.mf_model_n_events.restype = i64
    lib.mf_model_n_events.argtypes = [vp]
    lib.mf_model_n_toys.restype = i64
    lib.mf_model_n_toys.argtypes = [vp]
    lib.mf_nll_grad.restype = ctypes.c_int
    lib.mf_nll_grad.argtypes = [vp, dp, dp, dp]
    lib.mf_nll_grad_async.restype = ctypes.c_int
    lib.mf_nll_grad_async.argtypes = [vp, dp, vp]
    lib.mf_nll_grad_points.restype = ctypes.c_int
    lib.mf_nll_grad_points.argtypes = [vp, i64, dp, vp]
    lib.mf_nll_grad_batch.restype = ctypes.c_int
    lib.mf_nll_grad_batch.argtypes = [vp, i64, dp, u8p, dp, dp]
    lib.mf_nll_grad_batch_async.restype = ctypes.c_int
    lib.mf_nll_grad_batch_async.argtypes = [vp, i64, vp, vp]
    lib.mf_model_has_hessian.restype = ctypes.c_int
    lib.mf_model_has_hessian.argtypes = [vp]
    lib.mf_nll_grad_hess.restype = ctypes.c_int
    lib.mf_nll_grad_hess.argtypes = [vp, dp, dp, dp, dp]
    lib.mf_model_serve.restype = ctypes.c_int
    lib.mf_model_serve.argtypes = [vp, ctypes.c_int]
    lib.mf_model_is_served.restype = ctypes.c_int
    lib.mf_model_is_served.argtypes = [vp]
    lib.mf_model_is_weighted.restype = ctypes.c_int
    lib.mf_model_is_weighted.argtypes = [vp]
    lib.mf_nll_grad_hess_fisher.restype = ctypes.c_int
    lib.mf_nll_grad_hess_fisher.argtypes = [vp, dp, dp, dp, dp, dp]
    lib.mf_nll_grad_hess_batch.restype = ctypes.c_int
    lib.mf_nll_grad_hess_batch.argtypes = [vp, i64, dp, u8p, dp, dp, dp]
    lib.mf_fit_opts_default.restype = None
    lib.mf_fit_opts_default.argtypes = [ctypes.POINTER(FitOpts)]
    lib.mf_fit.restype = ctypes.c_int
    lib.mf_fit.argtypes = [vp, dp, u8p, ctypes.POINTER(FitOpts), ctypes.POINTER(_FitResultC)]
    lib.mf_fit_batch.restype = ctypes.c_int
    lib.mf_fit_batch.argtypes = [vp, i64, dp, u8p, ctypes.POINTER(FitOpts), ctypes.POINTER(_FitResultC)]
    lib.mf_toy_study_mass.restype = ctypes.c_int
    lib.mf_toy_study_mass.argtypes = [vp, ctypes.c_uint64, i64, i64, dp, ctypes.c_double, ctypes.c_double, ctypes.POINTER(FitOpts),
                                      ctypes.POINTER(_FitResultC)]
    lib.mf_toy_study_angular.restype = ctypes.c_int
    lib.mf_toy_study_angular.argtypes = [vp, ctypes.c_uint64, i64, i64, dp, ctypes.POINTER(FitOpts), ctypes.POINTER(_FitResultC)]
    lib.mf_nll_grad_mass_noalloc.restype = ctypes.c_int
    lib.mf_nll_grad_mass_noalloc.argtypes = [vp, vp, i64, ctypes.c_double, ctypes.c_double, dp, vp, vp]
    lib.mf_nll_grad_sweep.restype = ctypes.c_int
    lib.mf_nll_grad_sweep.argtypes = [vp, i64, dp, dp, dp, ctypes.POINTER(i64)]
    lib.mf_combine_partials.restype = ctypes.c_int
    lib.mf_combine_partials.argtypes = [ctypes.c_int, ctypes.c_int, dp, dp]
    _lib = lib
    return lib


def _dp(a: np.ndarray):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def _u8p(a):
    return None if a is None else a.ctypes.data_as(ctypes.POINTER(ctypes.c_uint8))


def combine_partials(rows) -> np.ndarray:
    """mf_combine_partials: rows [n_ranks][width] -> rank-ordered compensated column sums [width] (host only)."""
    rows = np.ascontiguousarray(rows, dtype=np.float64)
    if rows.ndim != 2:
        raise ValueError("rows must be [n_ranks][width]")
    out = np.empty(rows.shape[1], dtype=np.float64)
    st = load_library().mf_combine_partials(rows.shape[0], rows.shape[1], _dp(rows), _dp(out))
    if st != MF_OK:
        raise MoreFitError(st, "mf_combine_partials")
    return out


def default_fit_opts() -> FitOpts:
    o = FitOpts()
    load_library().mf_fit_opts_default(ctypes.byref(o))
    return o


class Context:
    """mf_ctx: a CUDA device and a borrowed stream (default: torch's current stream on it)."""

    def __init__(self, device: int = 0, stream: int | None = None):
        self._lib = load_library()
        self._h = ctypes.c_void_p()
        self._children = weakref.WeakSet()   # live datasets / models, closed before the context
        self._fit_buf = None                 # reused result buffer of the batched fits (fresh pages cost ~2 ms per 4096 toys)
        if stream is None:
            import torch  # device memory / streams come from PyTorch (plumbing only)
            if not torch.cuda.is_available():
                raise MoreFitError(MF_ERR_CUDA, "no CUDA device: the MoreFit hot path has no CPU fallback")
            stream = torch.cuda.current_stream(device).cuda_stream
        st = self._lib.mf_ctx_create(int(device), ctypes.c_void_p(stream), ctypes.byref(self._h))
        if st != MF_OK:
            raise MoreFitError(st, "mf_ctx_create failed (no usable CUDA device?)")
        self.device = int(device)

    def _fit_results(self, n_toys: int) -> np.ndarray:
        if self._fit_buf is None or self._fit_buf.size < n_toys:
            self._fit_buf = np.empty(n_toys, dtype=BatchFitResult._DT)
        return self._fit_buf[:n_toys]

    def _check(self, st: int):
        if st != MF_OK:
            raise MoreFitError(st, self._lib.mf_last_error(self._h).decode())

    @property
    def kernel_launches(self) -> int:
        return int(self._lib.mf_ctx_kernel_launches(self._h))

    def dataset_upload(self, columns, lo=None, hi=None, n_toys: int = 1) -> "Dataset":
        """columns: numpy array [ndim][n_toys*n_events] (or 1-D for ndim = 1; [n_toys][n_events] for
        ndim = 1 with n_toys > 1), or a list of CUDA torch tensors (device pointers, one per dimension)."""
        return Dataset(self, columns, lo, hi, n_toys)

    def generate_mass(self, seed0: int, n_toys: int, n_events: int, lam, lo: float, hi: float) -> "Dataset":
        """n_toys pseudo-experiments of the mass model generated on the device (no host copy)."""
        lam = np.ascontiguousarray(lam, dtype=np.float64)
        ds = Dataset.__new__(Dataset)
        ds._ctx, ds._lib, ds._h = self, self._lib, ctypes.c_void_p()
        self._check(self._lib.mf_generate_mass(self._h, int(seed0), int(n_toys), int(n_events), _dp(lam), float(lo), float(hi),
                                               ctypes.byref(ds._h)))
        self._children.add(ds)
        ds.ndim, ds.n_events, ds.n_toys = 1, int(n_events), int(n_toys)
        return ds

    def generate_4d(self, seed0: int, n_toys: int, n_events: int, lam, lo: float, hi: float) -> "Dataset":
        """n_toys pseudo-experiments of the 4D mass x angular model generated on the device."""
        lam = np.ascontiguousarray(lam, dtype=np.float64)
        if lam.shape != (16,):
            raise ValueError("lam must have 16 entries")
        ds = Dataset.__new__(Dataset)
        ds._ctx, ds._lib, ds._h = self, self._lib, ctypes.c_void_p()
        self._check(self._lib.mf_generate_4d(self._h, int(seed0), int(n_toys), int(n_events), _dp(lam), float(lo), float(hi),
                                             ctypes.byref(ds._h)))
        self._children.add(ds)
        ds.ndim, ds.n_events, ds.n_toys = 4, int(n_events), int(n_toys)
        return ds

    def generate_angular(self, seed0: int, n_toys: int, n_events: int, a) -> "Dataset":
        """n_toys pseudo-experiments of the angular model generated on the device by accept-reject."""
        a = np.ascontiguousarray(a, dtype=np.float64)
        ds = Dataset.__new__(Dataset)
        ds._ctx, ds._lib, ds._h = self, self._lib, ctypes.c_void_p()
        self._check(self._lib.mf_generate_angular(self._h, int(seed0), int(n_toys), int(n_events), _dp(a), ctypes.byref(ds._h)))
        self._children.add(ds)
        ds.ndim, ds.n_events, ds.n_toys = 3, int(n_events), int(n_toys)
        return ds

    def toy_study_mass(self, seed0: int, n_toys: int, n_events: int, lam_truth, lo: float, hi: float,
                       opts: "FitOpts | None" = None) -> "BatchFitResult":
        """Generate, fit and HESSE n_toys pseudo-experiments of the mass model on the device."""
        lam = np.ascontiguousarray(lam_truth, dtype=np.float64)
        res = self._fit_results(int(n_toys))
        self._check(self._lib.mf_toy_study_mass(self._h, int(seed0), int(n_toys), int(n_events), _dp(lam), float(lo), float(hi),
                                                None if opts is None else ctypes.byref(opts),
                                                res.ctypes.data_as(ctypes.POINTER(_FitResultC))))
        return BatchFitResult(res, int(n_toys), 4)

    def toy_study_angular(self, seed0: int, n_toys: int, n_events: int, a_truth, opts: "FitOpts | None" = None) -> "BatchFitResult":
        """Generate (accept-reject), fit and HESSE n_toys pseudo-experiments of the angular model on the device."""
        a = np.ascontiguousarray(a_truth, dtype=np.float64)
        if a.shape != (8,):
            raise ValueError("a_truth must have 8 entries")
        res = self._fit_results(int(n_toys))
        self._check(self._lib.mf_toy_study_angular(self._h, int(seed0), int(n_toys), int(n_events), _dp(a),
                                                   None if opts is None else ctypes.byref(opts),
                                                   res.ctypes.data_as(ctypes.POINTER(_FitResultC))))
        return BatchFitResult(res, int(n_toys), 8)

    def nll_grad_mass_noalloc(self, m_dev_ptr: int, n: int, lo: float, hi: float, lam, out_dev_ptr: int, stream: int = 0) -> None:
        """mf_nll_grad_mass_noalloc: one mass-model evaluation on n device-resident events (16-byte aligned pointer) that
        allocates nothing (fixed scratch in the library image, n <= MF_NOALLOC_MAX_EVENTS); 6 doubles (-ln L, gradient,
        n_bad) are written to out_dev_ptr in stream order.  Calls that overlap on the GPU race on the scratch."""
        lam = np.ascontiguousarray(lam, dtype=np.float64)
        if lam.shape != (4,):
            raise ValueError("lam must have 4 entries")
        self._check(self._lib.mf_nll_grad_mass_noalloc(self._h, ctypes.c_void_p(int(m_dev_ptr)), int(n), float(lo), float(hi),
                                                       _dp(lam), ctypes.c_void_p(int(out_dev_ptr)),
                                                       ctypes.c_void_p(int(stream)) if stream else None))

    def model_create(self, kind: int, dataset: "Dataset") -> "Model":
        return Model(self, kind, dataset)

    def close(self):
        """Destroys the context after every dataset and model made from it (the C-ABI's required order)."""
        if self._h:
            for child in list(self._children):
                child.close()
            self._lib.mf_ctx_destroy(self._h)
            self._h = ctypes.c_void_p()


class Dataset:
    def __init__(self, ctx: Context, columns, lo, hi, n_toys: int = 1):
        self._ctx, self._lib = ctx, ctx._lib
        self._h = ctypes.c_void_p()
        where = MF_HOST
        keep = []
        if isinstance(columns, (list, tuple)) and len(columns) and hasattr(columns[0], "data_ptr"):
            import torch
            for t in columns:
                if not (t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()):
                    raise ValueError("device columns must be contiguous float64 CUDA tensors")
            where = MF_DEVICE
            ndim = len(columns)
            total = int(columns[0].numel())
            ptrs = [int(t.data_ptr()) for t in columns]
            keep = list(columns)
            torch.cuda.current_stream(ctx.device).synchronize()
        else:
            arr = np.asarray(columns, dtype=np.float64)
            if arr.ndim == 1:
                arr = arr[None, :]
            elif arr.ndim == 2 and n_toys > 1 and arr.shape[0] == n_toys:
                arr = arr.reshape(1, -1)          # [n_toys][n_events] of a 1-D model
            elif arr.ndim == 3:
                arr = arr.reshape(arr.shape[0], -1)  # [ndim][n_toys][n_events]
            cols = [np.ascontiguousarray(arr[j]) for j in range(arr.shape[0])]
            ndim, total = len(cols), int(cols[0].size)
            ptrs = [c.ctypes.data for c in cols]
            keep = cols
        if total % n_toys:
            raise ValueError("column length is not a multiple of n_toys")
        cptr = (ctypes.c_void_p * ndim)(*ptrs)
        lo_a = None if lo is None else np.ascontiguousarray(np.atleast_1d(lo), dtype=np.float64)
        hi_a = None if hi is None else np.ascontiguousarray(np.atleast_1d(hi), dtype=np.float64)
        if lo_a is not None and lo_a.size == 1 and ndim == 4:   # mass range only: angular defaults
            lo_a = np.array([lo_a[0], -1.0, -1.0, -np.pi])
            hi_a = np.array([hi_a[0], 1.0, 1.0, np.pi])
        st = self._lib.mf_dataset_upload(ctx._h, ndim, total // n_toys, int(n_toys), cptr, where,
                                         None if lo_a is None else _dp(lo_a), None if hi_a is None else _dp(hi_a),
                                         ctypes.byref(self._h))
        del keep
        ctx._check(st)
        ctx._children.add(self)
        self.ndim, self.n_events, self.n_toys = ndim, total // n_toys, int(n_toys)

    def set_weights(self, weights) -> None:
        """Event weights (host array of n_events doubles, or None for unweighted); models created afterwards are weighted."""
        if weights is None:
            self._ctx._check(self._lib.mf_dataset_set_weights(self._h, None, MF_HOST))
            return
        w = np.ascontiguousarray(weights, dtype=np.float64)
        if w.shape != (self.n_events,):
            raise ValueError(f"weights must have shape ({self.n_events},)")
        self._ctx._check(self._lib.mf_dataset_set_weights(self._h, ctypes.c_void_p(w.ctypes.data), MF_HOST))

    def download(self) -> np.ndarray:
        """The events as a host array [ndim][n_toys][n_events]."""
        out = np.empty((self.ndim, self.n_toys, self.n_events), dtype=np.float64)
        self._ctx._check(self._lib.mf_dataset_download(self._h, _dp(out)))
        return out

    def close(self):
        if self._h:
            self._lib.mf_dataset_destroy(self._h)
            self._h = ctypes.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


class Model:
    def __init__(self, ctx: Context, kind: int, dataset: Dataset):
        self._ctx, self._lib = ctx, ctx._lib
        self._h = ctypes.c_void_p()
        ctx._check(self._lib.mf_model_create(ctx._h, int(kind), dataset._h, ctypes.byref(self._h)))
        ctx._children.add(self)
        self.kind = int(kind)
        self.K = int(self._lib.mf_model_nparams(self._h))
        self.n_events = int(self._lib.mf_model_n_events(self._h))
        self.n_toys = int(self._lib.mf_model_n_toys(self._h))

    def nll_grad(self, lam, want_grad: bool = True):
        """(-ln L, gradient) at lam; raises MoreFitError on a domain error or P <= 0.  (Marshalling buffers and their
        pointers are made once per model: this call is what a minimiser loops over.)"""
        io = self.__dict__.get("_io")
        if io is None:
            lam_b, grad_b, nll_b = np.empty(self.K), np.empty(self.K), ctypes.c_double()
            io = self._io = (lam_b, grad_b, nll_b, _dp(lam_b), _dp(grad_b), ctypes.byref(nll_b), self._lib.mf_nll_grad)
        lam_b, grad_b, nll_b, p_lam, p_grad, p_nll, fn = io
        lam_b[:] = lam                       # raises on a wrong length; converts to float64
        st = fn(self._h, p_lam, p_nll, p_grad if want_grad else None)
        if st != MF_OK:
            self._ctx._check(st)
        return nll_b.value, (grad_b.copy() if want_grad else None)

    def nll_grad_status(self, lam):
        """Like nll_grad but returns (status, nll, grad) instead of raising."""
        lam = np.ascontiguousarray(lam, dtype=np.float64)
        nll = ctypes.c_double(np.nan)
        grad = np.full(self.K, np.nan)
        st = self._lib.mf_nll_grad(self._h, _dp(lam), ctypes.byref(nll), _dp(grad))
        return int(st), float(nll.value), grad

    def nll_grad_async(self, lam, out_dev_ptr: int):
        """Enqueues one evaluation; K+2 doubles are written to the device pointer out_dev_ptr."""
        lam = np.ascontiguousarray(lam, dtype=np.float64)
        self._ctx._check(self._lib.mf_nll_grad_async(self._h, _dp(lam), ctypes.c_void_p(out_dev_ptr)))

    def nll_grad_points(self, lambdas, out_dev_ptr: int):
        """Enqueues len(lambdas) evaluations back to back; row p of the device array [n][K+2] at
        out_dev_ptr receives [-ln L, gradient, n_bad] at lambdas[p]."""
        lam = np.ascontiguousarray(lambdas, dtype=np.float64)
        if lam.ndim != 2 or lam.shape[1] != self.K:
            raise ValueError(f"lambdas must be [n][{self.K}]")
        self._ctx._check(self._lib.mf_nll_grad_points(self._h, lam.shape[0], _dp(lam), ctypes.c_void_p(out_dev_ptr)))

    def nll_grad_sweep(self, lambdas, want_grad: bool = True):
        """lambdas [n][K] (host) -> (nll [n], grad [n][K], number of points with P <= 0 events), results on the host."""
        lam = np.ascontiguousarray(lambdas, dtype=np.float64)
        if lam.ndim != 2 or lam.shape[1] != self.K:
            raise ValueError(f"lambdas must be [n][{self.K}]")
        n = lam.shape[0]
        nll = np.empty(n)
        grad = np.empty((n, self.K)) if want_grad else None
        nbad = ctypes.c_int64(0)
        self._ctx._check(self._lib.mf_nll_grad_sweep(self._h, n, _dp(lam), _dp(nll), None if grad is None else _dp(grad),
                                                     ctypes.byref(nbad)))
        return nll, grad, int(nbad.value)

    def nll_grad_batch(self, lambdas, active=None):
        """lambdas [T][K] -> (nll [T], grad [T][K]); inactive toys are NaN in the returned arrays."""
        lam = np.ascontiguousarray(lambdas, dtype=np.float64)
        T = self.n_toys
        if lam.shape != (T, self.K):
            raise ValueError(f"lambdas must be [{T}][{self.K}]")
        act = None if active is None else np.ascontiguousarray(active, dtype=np.uint8)
        nll = np.full(T, np.nan)
        grad = np.full((T, self.K), np.nan)
        self._ctx._check(self._lib.mf_nll_grad_batch(self._h, T, _dp(lam), _u8p(act), _dp(nll), _dp(grad)))
        return nll, grad

    @property
    def has_hessian(self) -> bool:
        return bool(self._lib.mf_model_has_hessian(self._h))

    def nll_grad_hess(self, lam):
        """(-ln L, gradient [K], Hessian [K][K]) from one launch (analytic second derivatives)."""
        lam = np.ascontiguousarray(lam, dtype=np.float64)
        nll = ctypes.c_double()
        grad = np.empty(self.K)
        hess = np.empty((self.K, self.K))
        self._ctx._check(self._lib.mf_nll_grad_hess(self._h, _dp(lam), ctypes.byref(nll), _dp(grad), _dp(hess)))
        return float(nll.value), grad, hess

    def serve(self, on: bool = True) -> None:
        """Keep a resident evaluation kernel for this model (mass model, single dataset): nll_grad / nll_grad_hess then
        cost no kernel launch.  serve(False) stops it."""
        self._ctx._check(self._lib.mf_model_serve(self._h, 1 if on else 0))

    @property
    def weighted(self) -> bool:
        return bool(self._lib.mf_model_is_weighted(self._h))

    def nll_grad_hess_fisher(self, lam):
        """(-ln L, gradient [K], Hessian [K][K], Fisher matrix sum w^2 s s^T [K][K]) from one pass (tensor-core contraction)."""
        lam = np.ascontiguousarray(lam, dtype=np.float64)
        nll = ctypes.c_double()
        grad = np.empty(self.K)
        hess = np.empty((self.K, self.K))
        fisher = np.empty((self.K, self.K))
        self._ctx._check(self._lib.mf_nll_grad_hess_fisher(self._h, _dp(lam), ctypes.byref(nll), _dp(grad), _dp(hess), _dp(fisher)))
        return float(nll.value), grad, hess, fisher

    def nll_grad_hess_batch(self, lambdas, active=None):
        """lambdas [T][K] -> (nll [T], grad [T][K], hess [T][K][K]); inactive toys are NaN."""
        lam = np.ascontiguousarray(lambdas, dtype=np.float64)
        T = self.n_toys
        act = None if active is None else np.ascontiguousarray(active, dtype=np.uint8)
        nll = np.full(T, np.nan)
        grad = np.full((T, self.K), np.nan)
        hess = np.full((T, self.K, self.K), np.nan)
        self._ctx._check(self._lib.mf_nll_grad_hess_batch(self._h, T, _dp(lam), _u8p(act), _dp(nll), _dp(grad), _dp(hess)))
        return nll, grad, hess

    def nll_grad_batch_async(self, lambdas_dev_ptr: int, out_dev_ptr: int):
        """All toys, device pointers in ([T][K]) and out ([T][K+2]), no host synchronisation."""
        self._ctx._check(self._lib.mf_nll_grad_batch_async(self._h, self.n_toys, ctypes.c_void_p(lambdas_dev_ptr),
                                                           ctypes.c_void_p(out_dev_ptr)))

    def fit(self, start, fixed=None, opts: FitOpts | None = None) -> FitResult:
        start = np.ascontiguousarray(start, dtype=np.float64)
        fx = None if fixed is None else np.ascontiguousarray(fixed, dtype=np.uint8)
        res = _FitResultC()
        st = self._lib.mf_fit(self._h, _dp(start), _u8p(fx), None if opts is None else ctypes.byref(opts),
                              ctypes.byref(res))
        self._ctx._check(st)
        return FitResult(res, self.K)

    def fit_batch(self, starts, fixed=None, opts: FitOpts | None = None) -> "BatchFitResult":
        T = self.n_toys
        starts = np.ascontiguousarray(starts, dtype=np.float64)
        if starts.shape == (self.K,):
            starts = np.ascontiguousarray(np.broadcast_to(starts, (T, self.K)))
        fx = None if fixed is None else np.ascontiguousarray(fixed, dtype=np.uint8)
        res = self._ctx._fit_results(T)   # filled by the library; BatchFitResult copies what it keeps
        st = self._lib.mf_fit_batch(self._h, T, _dp(starts), _u8p(fx), None if opts is None else ctypes.byref(opts),
                                    res.ctypes.data_as(ctypes.POINTER(_FitResultC)))
        self._ctx._check(st)
        return BatchFitResult(res, T, self.K)

    def close(self):
        if self._h:
            self._lib.mf_model_destroy(self._h)
            self._h = ctypes.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
