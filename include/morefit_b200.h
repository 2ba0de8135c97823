/*
 * morefit_b200.h — C-ABI boundary of the B200-native MoreFit hot path.
 *
 * The path: fused evaluation of the unbinned negative log-likelihood
 *     -ln L(lambda) = - sum_i ln P(x_i | lambda)            (Eq. 1)
 * and of its analytic gradient d(-ln L)/d lambda_k over N independent
 * events, for the model families named in BASELINE.json, plus the host quasi-Newton fit
 * driver that calls it.  SURVEY.md §8(a) lists the steps S0..S6, §8(b) this
 * boundary.  Every step of the path runs in the library's own sm_100a kernels; there is no
 * CPU fallback: without a CUDA device every compute entry point returns MF_ERR_CUDA.
 *
 * Conventions
 *   * All floating point is IEEE double (kernelT = evalT = double).
 *   * "host" / "device" beside a pointer says which memory it must point to.
 *   * The library copies what it needs: every caller array may be freed on return.
 *   * No call throws; every call returns an mf_status.  mf_last_error() gives a text for
 *     the last non-OK status of that context (valid until the next call on the context).
 *   * All device work of a context is enqueued on the CUDA stream given at creation
 *     (borrowed, e.g. torch.cuda.current_stream().cuda_stream; NULL = the legacy default
 *     stream).  Calls on one context must not be made concurrently from several threads.
 *   * Results are bit-identical for identical inputs through the same entry point on the same
 *     GPU: per-thread, per-warp, per-block and final sums are all taken in a fixed order
 *     (PAPER.md:65 uses Kahan reduction kernels; here one compensated fixed-order pass,
 *     SURVEY.md §8(a) S4/S5).  Different entry points tile the events differently (a lone call,
 *     a pipelined series, many points per launch, toys): their results agree to summation
 *     rounding (~1e-14 relative), not bit for bit.
 *   * Successive evaluations on the stream overlap (programmatic dependent launch); results
 *     still land in stream order.
 */
#ifndef MOREFIT_B200_H
#define MOREFIT_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    MF_OK = 0,
    MF_ERR_ARG = 1,          /* NULL pointer, wrong ndim / kind / size */
    MF_ERR_CUDA = 2,         /* CUDA runtime error or no device; text in mf_last_error */
    MF_ERR_OOM = 3,          /* host or device allocation failed */
    MF_ERR_DATA_RANGE = 4,   /* an event is non-finite or outside [lo, hi] */
    MF_ERR_PARAM_DOMAIN = 5, /* non-finite lambda, sigma <= 0 or f outside [0,1]: outputs untouched */
    MF_NONPOSITIVE_PDF = 6   /* P(x_i|lambda) <= 0, NaN, or underflowed (P N2 e^{-tau m} < 2^-1000) for >= 1 event:
                                nll = +inf, grad = NaN */
} mf_status;

/* Model families (BASELINE.json configs; parameter order = SURVEY.md §8(b)).
 *   MF_MASS_GAUSS_EXP   ndim 1 (m), K = 4: f, mu, sigma, tau.            PAPER.md:83-88 (Eq. 2)
 *   MF_ANGULAR_KSTMUMU  ndim 3 (cos theta_l, cos theta_K, phi), K = 8:
 *                       FL, S3, S4, S5, AFB, S7, S8, S9.                 PAPER.md:116-118 (Eq. 4)
 *   MF_MASS_X_ANGULAR   ndim 4 (m, cos theta_l, cos theta_K, phi), K = 16:
 *                       f, mu, sigma, tau, the 8 angular, cl1, cl2, ck1, ck2
 *                       P = f (G/N1) A + (1-f) (E/N2) L, L = l(cos theta_l) l(cos theta_K)/(2 pi),
 *                       l(x; c1, c2) = 1/2 [1 + c1 x + c2 (3x^2-1)/2]   (BASELINE.json configs[3]) */
typedef enum {
    MF_MASS_GAUSS_EXP = 0,
    MF_ANGULAR_KSTMUMU = 1,
    MF_MASS_X_ANGULAR = 2
} mf_model_kind;

typedef enum { MF_HOST = 0, MF_DEVICE = 1 } mf_mem;

#define MF_MAX_PARAMS 16
#define MF_MAX_DIMS 4

typedef struct mf_ctx mf_ctx;
typedef struct mf_dataset mf_dataset;
typedef struct mf_model mf_model;

/* ---- context ------------------------------------------------------------------------- */

/* Binds CUDA device `device` and the borrowed stream `cuda_stream` (a cudaStream_t, may be
 * NULL).  *out is set only on MF_OK.  MF_ERR_CUDA if the device cannot be used. */
mf_status mf_ctx_create(int device, void* cuda_stream, mf_ctx** out);
/* Frees the context.  Datasets and models made from it must be destroyed first. */
void mf_ctx_destroy(mf_ctx* ctx);
/* Text of the last error on this context ("" if none).  Never NULL.  ctx may be NULL. */
const char* mf_last_error(const mf_ctx* ctx);
/* Number of this library's kernels launched on the context since creation (bench.py's
 * gpu_launches claim is read from here). */
int64_t mf_ctx_kernel_launches(const mf_ctx* ctx);

/* ---- S0: data (PAPER.md:65 structure of arrays, padded) ------------ */

/* Copies `ndim` event columns to the device as a padded structure of arrays.
 *   columns[j]   host array of ndim pointers (always host); columns[j] points, in `where`
 *                memory, to n_toys*n_events doubles, toy-major (toy t at [t*n_events, (t+1)*n_events)).
 *   n_toys       1 for one dataset, T for T pseudo-experiments of n_events events each.
 *   lo, hi       host, ndim each: closed ranges.  For the mass dimension they are the
 *                normalisation range [m_a, m_b] of Eq. 2; the angular dimensions must be
 *                [-1,1], [-1,1], [-pi,pi] (checked to 1e-12).  NULL = those defaults (mass: error).
 * Each toy is padded to a multiple of 64 events with copies of its last event; padded
 * lanes are predicated to contribute exactly 0 (SURVEY.md §8(c) reading 10).
 * n_events == 0 is allowed (every sum is then 0).
 * MF_ERR_DATA_RANGE if any event is NaN/inf or outside its range (checked on the device). */
mf_status mf_dataset_upload(mf_ctx* ctx, int ndim, int64_t n_events, int64_t n_toys,
                            const double* const* columns, mf_mem where,
                            const double* lo, const double* hi, mf_dataset** out);
/* Event weights ("weighted fits"; reading R23): models created on the dataset
 * AFTER this call evaluate  -ln L_w = -sum_i w_i ln P(x_i | lambda)  (gradient and Hessian likewise) and mf_fit returns the
 * sandwich covariance H^-1 F H^-1 with F = sum_i w_i^2 s_i s_i^T (mf_nll_grad_hess_fisher).
 *   weights   n_events doubles in `where` memory (copied; any sign, e.g. sWeights), or NULL: back to unweighted.
 * Only datasets with n_toys == 1.  MF_ERR_DATA_RANGE if a weight is NaN/inf.  Weighted models are evaluated by the
 * second-order kernels (one launch pair per parameter point); the batched-toy entry points do not take weights. */
mf_status mf_dataset_set_weights(mf_dataset* ds, const double* weights, mf_mem where);
void mf_dataset_destroy(mf_dataset* ds);
int64_t mf_dataset_n_events(const mf_dataset* ds);
int64_t mf_dataset_n_toys(const mf_dataset* ds);

/* ---- on-device generation of pseudo-experiments ------------------------- */

/* Generates n_toys pseudo-experiments of n_events events each of the Gaussian + exponential mass model at lambda =
 * (f, mu, sigma, tau) on [lo, hi], directly into a device dataset (ndim = 1; use it with mf_model_create).  Toy t uses the
 * counter-based stream Philox4x32-10 keyed by seed0 + t; event i is a pure function of (seed0 + t, i), whatever the launch
 * geometry.  Recipe: mf_generate.cu.  lam: host, 4 doubles.  MF_ERR_PARAM_DOMAIN as for the mass model. */
mf_status mf_generate_mass(mf_ctx* ctx, uint64_t seed0, int64_t n_toys, int64_t n_events, const double* lam, double lo,
                           double hi, mf_dataset** out);

/* The same for the angular model (ndim = 3): accept-reject of uniform proposals in (cos theta_l, cos theta_K, phi) under
 * the paper's get_max() envelope 9/(32 pi) (4 + sum |S_i| + 4/3 |AFB|), flat acceptance; proposal k of an
 * event uses the draws 2k and 2k+1 of its Philox stream.  a: host, the 8 coefficients FL, S3, S4, S5, AFB, S7, S8, S9. */
mf_status mf_generate_angular(mf_ctx* ctx, uint64_t seed0, int64_t n_toys, int64_t n_events, const double* a, mf_dataset** out);

/* The same for the 4D model (ndim = 4: m, cos theta_l, cos theta_K, phi; BASELINE.json configs[3]).  lam: host, the 16
 * parameters f, mu, sigma, tau, the 8 angular coefficients, cl1, cl2, ck1, ck2.  Signal (probability f): Gaussian mass and
 * angular accept-reject as above; background: exponential mass by inverse CDF, flat phi, (cos theta_l, cos theta_K) by
 * accept-reject of the Legendre product under 1/2 (1 + |c1| + |c2|) per factor.
 * Draw layout of event i (Philox counter (i, draw), two uniforms per draw): draw 0 = (component choice, background mass);
 * signal: draws 1..64 Box-Muller mass candidates, draws 100+2k, 101+2k = angular proposal k (cos theta_l, cos theta_K |
 * phi, accept); background: draw 1 = (phi, unused), draws 100+2k, 101+2k = Legendre proposal k (cos theta_l,
 * cos theta_K | accept, unused). */
mf_status mf_generate_4d(mf_ctx* ctx, uint64_t seed0, int64_t n_toys, int64_t n_events, const double* lam, double lo, double hi,
                         mf_dataset** out);

/* Copies a dataset's events to the host: dst [ndim][n_toys][n_events] doubles. */
mf_status mf_dataset_download(const mf_dataset* ds, double* dst);

/* ---- S1: model (event-only precompute, Listing 4) --- */

/* Binds a model family to a dataset (ndim must match the kind) and runs the event-only
 * precompute once: for the angular kinds the nine merged basis columns
 * h_k = 9/(32 pi) g_k are cached in HBM.  The model keeps its own
 * reference to the dataset's device buffers: the dataset may be destroyed afterwards. */
mf_status mf_model_create(mf_ctx* ctx, mf_model_kind kind, const mf_dataset* ds, mf_model** out);
void mf_model_destroy(mf_model* model);
int mf_model_nparams(const mf_model* model);
int64_t mf_model_n_events(const mf_model* model);
int64_t mf_model_n_toys(const mf_model* model);

/* ---- S2..S6: value + gradient ------------------------------------------------------------ */

/* -ln L and d(-ln L)/d lambda_k at `lambda` over all events of a 1-toy dataset.
 *   lambda  host, K doubles.   nll  host, 1 double.   grad  host, K doubles or NULL.
 * One kernel launch (parameter-only constants of Eq. 3, are computed on
 * the host and passed as kernel arguments); the host then waits on a completion word in mapped memory.
 * MF_ERR_ARG if the dataset has n_toys != 1.  See mf_status for the domain / P<=0 cases. */
mf_status mf_nll_grad(mf_model* model, const double* lambda, double* nll, double* grad);

/* Same evaluation without a host synchronisation: enqueues the launch on the context's
 * stream and writes K+2 doubles to out_dev (DEVICE): [-ln L, grad[0..K-1], n_bad], where
 * n_bad is the number of events with P <= 0 (then -ln L = +inf, grad = NaN).  The
 * parameter-domain check is still made on the host before the launch. */
mf_status mf_nll_grad_async(mf_model* model, const double* lambda, double* out_dev);

/* n_points evaluations of the same dataset at n_points parameter points (BASELINE.json configs[1]:
 * "repeated NLL+gradient calls at 1,000 random parameter points"), enqueued without a host synchronisation.
 *   lambdas  host, [n_points][K].   out_dev  DEVICE, [n_points][K+2], row p = [-ln L, grad, n_bad] at point p.
 * Few points (mass model: fewer than 8, fewer than 4 up to 2e5 events; angular: fewer than 6; 4D: fewer than 10): mf_nll_grad_async n_points times (one launch each,
 * pipelined).  Otherwise, by family:
 *   mass     ONE launch whose CTA tile is (point, event chunk), the parameter-only constants of every point derived on
 *            the host and read by the kernel in place from a pinned, device-mapped staging ring (the dataset is read from
 *            HBM once and re-read from L2 by the other points; 8 B per event, ALU bound); consecutive calls overlap on the
 *            GPU (outputs still land in stream order);
 *   angular  one pass over the nine cached columns per 32 points: P = h0 + A.H and G = R.H^T as fp64 tensor-core
 *            contractions on 8 points x 8 events (mf_points.cuh), then a combine launch;
 *   4D       one pass over the twelve columns per 16 points: tensor-core contractions around the per-pair exponential
 *            (mf_points4d.cuh), then a combine launch; a call with a point at f = 0 or f = 1 uses the (point, chunk) tile.
 * Weighted models: one second-order evaluation (gradient mode) per point.
 * No allocation, clearing or synchronisation per call once the model's scratch has grown to its size.
 * Every point is validated first: MF_ERR_PARAM_DOMAIN (nothing enqueued) if one is outside the domain
 * (below the few-points threshold the earlier ones are enqueued). */
mf_status mf_nll_grad_points(mf_model* model, int64_t n_points, const double* lambdas, double* out_dev);

/* The same sweep with the results returned to the HOST: evaluates the n_points parameter points (as
 * mf_nll_grad_points does), copies the results back and synchronises.
 *   lambdas  host, [n_points][K].   nll  host, [n_points].   grad  host, [n_points][K] or NULL.
 *   n_bad    host, 1 integer or NULL: number of points at which some event had P <= 0 (those points have
 *            nll = +inf, grad = NaN; the call still returns MF_OK).
 * MF_ERR_PARAM_DOMAIN (nothing evaluated) if a point is outside the parameter domain. */
mf_status mf_nll_grad_sweep(mf_model* model, int64_t n_points, const double* lambdas, double* nll, double* grad,
                            int64_t* n_bad);

/* T pseudo-experiments at their own parameter points in ONE launch (BASELINE.json
 * configs[4]): a CTA tile is (toy, event chunk); the toys' parameter-only constants are
 * derived on the device by a small kernel launched just before it.
 *   n_toys   must equal the dataset's n_toys.
 *   lambdas  host, [n_toys][K].   active  host, n_toys bytes or NULL (= all active).
 *   nll      host, [n_toys].      grad    host, [n_toys][K] or NULL.
 * Inactive toys are skipped and their outputs left untouched.  A toy whose lambda is
 * outside the parameter domain, or that has an event with P <= 0, gets nll = +inf and
 * grad = NaN; the call still returns MF_OK. */
mf_status mf_nll_grad_batch(mf_model* model, int64_t n_toys, const double* lambdas,
                            const uint8_t* active, double* nll, double* grad);

/* The same evaluation for ALL toys without host copies or synchronisation: lambdas_dev is DEVICE [n_toys][K],
 * out_dev DEVICE [n_toys][K+2], row t = [-ln L, grad, n_bad] of toy t (n_bad = -1: lambda_t outside the domain).
 * Two launches are enqueued on the context's stream (parameter-only constants, then the fused kernel).
 * lambdas_dev may have been written by the caller's own kernel enqueued earlier on the same stream (a device-side
 * minimiser step): the constants kernel reads it only after the programmatic-launch wait, i.e. once that work has
 * completed and its writes are visible. */
mf_status mf_nll_grad_batch_async(mf_model* model, int64_t n_toys, const double* lambdas_dev, double* out_dev);

/* Resident evaluation kernel for the minimiser's one-point-at-a-time pattern (at small N an evaluation
 * costs its kernel submission).  on = 1: from the next mf_nll_grad / mf_nll_grad_hess on, the model's CTAs stay resident on
 * a stream of their own (one per SM, at most half an SM's registers) and are fed through mapped pinned memory: the call
 * writes the parameter-only constants and a request number, the last CTA writes the result and the number back; no kernel
 * launch and no completion latency per call.  The kernel leaves on mf_model_serve(model, 0), mf_model_destroy, or by
 * itself after 5 ms without a request (it is relaunched on the next call).  mf_fit serves its own evaluations this way
 * for the duration of the fit.  Only unweighted MF_MASS_GAUSS_EXP models with n_toys == 1 and n_events > 0 (MF_ERR_ARG
 * otherwise).  Other calls on the model or the context are unaffected and may run beside the resident kernel. */
mf_status mf_model_serve(mf_model* model, int on);
int mf_model_is_served(const mf_model* model);

/* ---- value + gradient + analytic Hessian ---------------------- */

/* 1 if the analytic Hessian is available for this model (every family, single datasets and batched toys). */
int mf_model_has_hessian(const mf_model* model);
/* 1 if the model was created on a dataset with event weights. */
int mf_model_is_weighted(const mf_model* model);

/* As mf_nll_grad, plus hess (host, K*K doubles, row-major, symmetric) = d2(-ln L)/d lambda_k d lambda_l from the same
 * pass over the data.  Unweighted mass and angular models: one launch that accumulates the second-derivative sums in
 * registers (mass: seven more moment sums; angular: the 36 products of the score components).  The 4D model (136
 * second-derivative sums) and every weighted model: the second-order kernel, which forms S^T diag(w) S and the
 * P_ab / P terms as fp64 tensor-core contractions over the event index (mf_second.cuh).
 * On MF_NONPOSITIVE_PDF hess is NaN. */
mf_status mf_nll_grad_hess(mf_model* model, const double* lambda, double* nll, double* grad, double* hess);

/* As mf_nll_grad_hess, plus fisher (host, K*K, row-major, symmetric) = sum_i w_i^2 s_i s_i^T with s_i = d ln P_i/d lambda
 * (w_i = 1 without weights): the matrix PAPER.md:53 calls the Fisher information matrix "required for weighted fits";
 * the covariance of a weighted fit is hess^-1 fisher hess^-1 at the minimum (reading R23).  Any model family,
 * n_toys == 1; hess may be NULL.  One launch pair (second-order kernel + combine). */
mf_status mf_nll_grad_hess_fisher(mf_model* model, const double* lambda, double* nll, double* grad, double* hess,
                                  double* fisher);

/* As mf_nll_grad_batch, plus hess (host, [n_toys][K*K]); inactive toys are left untouched.  Mass and angular families: one
 * launch for all toys; the 4D family: the second-order kernel toy by toy, in stream order, one synchronisation at the end. */
mf_status mf_nll_grad_hess_batch(mf_model* model, int64_t n_toys, const double* lambdas, const uint8_t* active,
                                 double* nll, double* grad, double* hess);

/* ---- fit driver (host quasi-Newton over the GPU value+gradient) ------- */

typedef struct {
    int max_iter;          /* BFGS iterations (default 200) */
    double edm_tol;        /* leave BFGS for the Newton polish when g^T H^-1 g / 2 < edm_tol (1e-5) */
    double armijo_c1;      /* sufficient-decrease constant (1e-4) */
    double backtrack;      /* step shrink factor (0.5) */
    int max_backtracks;    /* (40) */
    double polish_tol;     /* converged when max_k |Newton step_k| / sigma_k < polish_tol (1e-9) */
    int max_polish;        /* finite-difference Hessians in the polish (8) */
    int max_chord;         /* Newton steps per Hessian (8) */
    double fd_rel;         /* first FD step: fd_rel * max(|lambda_k|, 1) (1e-5) */
    double fd_sigma;       /* later FD steps: fd_sigma * sigma_k (1e-4) */
    int analytic_hessian;  /* 1 (default): use the analytic Hessian kernel where the model has one (mf_model_has_hessian):
                              every evaluation returns the Hessian, Newton steps, no finite-difference phases */
} mf_fit_opts;

/* Fills *opts with the defaults above. */
void mf_fit_opts_default(mf_fit_opts* opts);

typedef struct {
    double lambda_hat[MF_MAX_PARAMS];               /* fitted parameters (fixed ones = start) */
    double cov[MF_MAX_PARAMS * MF_MAX_PARAMS];      /* row-major K x K inverse Hessian (HESSE); 0 for fixed.
                                                       Weighted model: the sandwich H^-1 F H^-1 (reading R23) */
    double nll_min;
    int n_calls;                                    /* value+gradient evaluations used */
    int n_iter;                                     /* BFGS iterations */
    int converged;                                  /* 1 = polish criterion met */
} mf_fit_result;

/* Minimises -ln L from `start` (host, K).  fixed: host, K bytes (1 = keep at start; paper:
 * the parameter `constant` flag) or NULL.  opts NULL = defaults.
 * With the analytic Hessian (opts->analytic_hessian, every family with n_toys == 1): Newton steps with Armijo backtracking on the
 * Hessian returned by every evaluation, then Newton polish; cov = H^-1 at the minimum.
 * Otherwise (SURVEY.md §8(c) "Fit"): central-difference Hessian of the analytic gradient
 * at the start point seeds the inverse metric; BFGS with Armijo backtracking that rejects
 * domain errors and P<=0 points; then Newton steps on a fresh central-difference Hessian
 * until the step is below polish_tol sigma; cov = H^-1.
 * MF_ERR_PARAM_DOMAIN / MF_NONPOSITIVE_PDF if the start point itself is invalid. */
mf_status mf_fit(mf_model* model, const double* start, const uint8_t* fixed,
                 const mf_fit_opts* opts, mf_fit_result* result);

/* Fits all T toys of the model's dataset concurrently: T independent fit states advance
 * in lock step, one mf_nll_grad_batch launch per round with the finished toys masked out.
 *   starts   host, [n_toys][K].   results  host, n_toys entries.
 * A toy whose start point is invalid gets converged = 0 and n_calls = 1. */
mf_status mf_fit_batch(mf_model* model, int64_t n_toys, const double* starts,
                       const uint8_t* fixed, const mf_fit_opts* opts, mf_fit_result* results);

/* The paper's toy study for the mass model (Listing 6: `toystudy.toy(...)`): generates n_toys
 * pseudo-experiments of n_events events at lam_truth (mf_generate_mass, seeds seed0 + t), fits all of them concurrently from
 * lam_truth (mf_fit_batch) and returns the n_toys fit results (host) with their HESSE covariances.  No event leaves the device. */
mf_status mf_toy_study_mass(mf_ctx* ctx, uint64_t seed0, int64_t n_toys, int64_t n_events, const double* lam_truth, double lo,
                            double hi, const mf_fit_opts* opts, mf_fit_result* results);

/* The same for the angular model (the paper's second benchmark, Table 3): n_toys pseudo-experiments of
 * n_events events generated by accept-reject at a_truth (mf_generate_angular, seeds seed0 + t), fitted concurrently from
 * a_truth with Newton steps on the analytic Hessian, HESSE covariances returned.  a_truth: host, 8 doubles. */
mf_status mf_toy_study_angular(mf_ctx* ctx, uint64_t seed0, int64_t n_toys, int64_t n_events, const double* a_truth,
                               const mf_fit_opts* opts, mf_fit_result* results);

/* ---- an evaluation that allocates nothing ------------------------------------------------------------------ */

/* For callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid it):
 * ONE evaluation of -ln L(lambda) and its gradient for the mass model (Eq. 1; Eq. 2 / Eq. 3) on
 * events the caller already holds on the device, with no dataset or model object.  The kernel's cross-CTA scratch (one row of
 * partial sums per 8192 events, the completion ticket) is a fixed array of 246,016 bytes in the library's device image, held
 * by every GPU that loads the library until the process exits; nothing is allocated or freed by this call (no cudaMalloc,
 * cudaFree, cudaHostAlloc, no stream-ordered pool), it enqueues one 256-byte memset and one kernel and does not synchronise.
 *   m_dev    device, n doubles, 16-byte aligned, unpadded; NOT range-checked: every event must lie in [lo, hi].
 *   n        0 <= n <= MF_NOALLOC_MAX_EVENTS; more: MF_ERR_ARG, text in mf_last_error, nothing enqueued.
 *   lambda   host, 4 doubles (f, mu, sigma, tau), read before the call returns; MF_ERR_PARAM_DOMAIN as for mf_nll_grad.
 *   out_dev  device, 6 doubles, written in stream order: -ln L, the 4 gradient components, n_bad (events with P <= 0;
 *            when non-zero the value is +inf and the gradient NaN).
 *   stream   a cudaStream_t, or NULL for the context's stream.
 * Every call on a device shares the one scratch array: calls ordered on one stream are safe (the ticket word is cleared on
 * the stream before each kernel, rows are overwritten before they are read); calls that OVERLAP on the GPU — two streams,
 * two host threads, parallel graph branches — race on it and return garbage.  The first call on a device resolves the
 * array's device address (cudaGetSymbolAddress): make it once outside stream capture.  The result agrees with mf_nll_grad
 * to rounding (not bit for bit: fixed 8192-event chunks, general event body) and does not depend on the SM count. */
#define MF_NOALLOC_MAX_EVENTS 33554432 /* 2^25 */
mf_status mf_nll_grad_mass_noalloc(mf_ctx* ctx, const double* m_dev, int64_t n, double lo, double hi, const double* lambda,
                                   double* out_dev, void* stream);

/* ---- multi-GPU: S5 across ranks ------------------------------------------------------ */

/* Combines the partial sums of n_ranks event shards of ONE dataset (each rank's mf_nll_grad on its shard: -ln L and the
 * gradient are sums over events, Eq. 1) into the totals.  Host arithmetic, no device needed.
 *   rows  host, [n_ranks][width], rank r's `width` partial sums in row r (gathered by the caller, e.g. all_gather).
 *   out   host, [width].
 * Every column is added in RANK ORDER with two-sum compensation, so all ranks obtain bit-identical totals whatever the
 * collective's reduction tree; a column holding +inf or NaN (a shard with P <= 0) is added plainly and propagates. */
mf_status mf_combine_partials(int n_ranks, int width, const double* rows, double* out);

#ifdef __cplusplus
}
#endif
#endif /* MOREFIT_B200_H */
