// mf_fit.cpp — host quasi-Newton fit driver over the GPU value + gradient (north_star item 3;
// PAPER.md:41 "the minimiser calls this repeatedly at new parameter points", PAPER.md:154 HESSE).
//
// The algorithm is the one of SURVEY.md §8(c) "Fit":
//   1. central-difference Hessian of the analytic gradient at the start point -> inverse metric
//      (its diagonal if the matrix is not positive definite);
//   2. BFGS with inverse update and Armijo backtracking; a trial point that is outside the
//      parameter domain, has P <= 0 for an event, or is non-finite is a rejected step;
//      leave when EDM = g^T H^-1 g / 2 < edm_tol;
//   3. polish: central-difference Hessian, Newton steps with it until
//      max_k |step_k| / sigma_k < polish_tol; cov = H^-1 (the HESSE matrix).
//
// Where the model family has the analytic Hessian kernel (mf_model_has_hessian) and opts->analytic_hessian is set, every
// evaluation also returns d2(-ln L): steps 1 and 3 need no finite differences, step 2 uses the Newton metric of the
// accepted point (BFGS update only if that Hessian is not positive definite), and cov is the inverse of the Hessian at the
// final point.
//
// It is written as a resumable state machine (one FitState per fit: "give me the next point
// to evaluate" / "here is the value and gradient there") so that the same code drives one fit
// through mf_nll_grad and T concurrent toy fits through ONE mf_nll_grad_batch launch per round.
#include <algorithm>
#include <cmath>
#include <cstring>
#include <vector>

#include "mf_internal.h"

namespace {

// Dense symmetric helpers on nf x nf matrices stored row-major with leading dimension KM (the capacity of the fit
// state: 4, 8 or 16 parameters, so that 4096 concurrent 4-parameter toy fits carry 1 KB of state each, not 12 KB).
template <int KM>
struct MatT {
    double a[KM][KM];
};

// Cholesky factor (lower) of A; false if A is not positive definite.
template <class Mat>
bool cholesky(const Mat& A, int n, Mat& L)
{
    for (int i = 0; i < n; ++i) {
        for (int j = 0; j <= i; ++j) {
            double s = A.a[i][j];
            for (int k = 0; k < j; ++k) s -= L.a[i][k] * L.a[j][k];
            if (i == j) {
                if (!(s > 0.0) || !std::isfinite(s)) return false;
                L.a[i][i] = std::sqrt(s);
            } else {
                L.a[i][j] = s / L.a[j][j];
            }
        }
    }
    return true;
}

// inv = A^-1 for positive definite A; false otherwise.
template <class Mat>
bool inv_pd(const Mat& A, int n, Mat& inv)
{
    Mat L;
    if (!cholesky(A, n, L)) return false;
    // invert L (lower triangular) column by column, then A^-1 = L^-T L^-1
    Mat Li;
    for (int i = 0; i < n; ++i)
        for (int j = 0; j < n; ++j) Li.a[i][j] = 0.0;
    for (int j = 0; j < n; ++j) {
        Li.a[j][j] = 1.0 / L.a[j][j];
        for (int i = j + 1; i < n; ++i) {
            double s = 0.0;
            for (int k = j; k < i; ++k) s -= L.a[i][k] * Li.a[k][j];
            Li.a[i][j] = s / L.a[i][i];
        }
    }
    for (int i = 0; i < n; ++i)
        for (int j = 0; j <= i; ++j) {
            double s = 0.0;
            for (int k = i; k < n; ++k) s += Li.a[k][i] * Li.a[k][j];
            inv.a[i][j] = inv.a[j][i] = s;
        }
    return true;
}

template <int KMAX>
class FitStateT {
    using Mat = MatT<KMAX>;

public:
    void init(int K, const double* start, const uint8_t* fixed, const mf_fit_opts& o)
    {
        K_ = K;
        o_ = o;
        nf_ = 0;
        for (int k = 0; k < K; ++k) {
            x_[k] = start[k];
            if (!(fixed && fixed[k])) idx_[nf_++] = k;
        }
        phase_ = START;
        calls_ = 0;
        iter_ = 0;
        polish_ = 0;
        chord_ = 0;
        converged_ = false;
        failed_start_ = false;
        std::memcpy(req_, x_, sizeof(double) * K);
    }
    bool done() const { return phase_ == DONE; }
    const double* request() const { return req_; }
    // Analytic-Hessian mode (model families with the Hessian kernel; likelihood + gradient + Hessian
    // per iteration): every evaluation also returns d2(-ln L); no finite-difference phases, Newton metric.
    void use_analytic_hessian() { use_h_ = true; }

    // Result of evaluating request(): ok = finite value and gradient at a valid point.  hfull: K x K Hessian there
    // (analytic mode) or NULL.
    void feed(bool ok, double f, const double* gfull, const double* hfull = nullptr)
    {
        ++calls_;
        double g[KMAX];
        if (ok) {
            ok = std::isfinite(f);
            for (int a = 0; a < nf_; ++a) {
                g[a] = gfull[idx_[a]];
                ok = ok && std::isfinite(g[a]);
            }
        }
        Mat Hin{};
        bool h_ok = use_h_ && ok && hfull != nullptr;
        if (h_ok)
            for (int a = 0; a < nf_; ++a)
                for (int b = 0; b < nf_; ++b) {
                    Hin.a[a][b] = hfull[idx_[a] * K_ + idx_[b]];
                    h_ok = h_ok && std::isfinite(Hin.a[a][b]);
                }
        switch (phase_) {
        case START:
            if (!ok) {
                failed_start_ = true;
                f_ = f;
                phase_ = DONE;
                return;
            }
            f_ = f;
            std::memcpy(g_, g, sizeof(double) * nf_);
            if (nf_ == 0) {
                converged_ = true;
                phase_ = DONE;
                return;
            }
            if (use_h_) {  // the Hessian at the start point came with this evaluation
                H_ = Hin;
                Hx_ = Hin;
                hx_ok_ = h_ok;
                fd_ok_ = h_ok;
                after_seed();
                return;
            }
            for (int a = 0; a < nf_; ++a) h_[a] = o_.fd_rel * std::max(std::fabs(x_[idx_[a]]), 1.0);
            begin_fd(SEED_FD);
            return;
        case SEED_FD:
        case POLISH_FD:
            if (!fd_feed(ok, g)) return;  // more FD points to go
            if (phase_ == SEED_FD) after_seed();
            else after_polish_fd();
            return;
        case TRIAL:
            if (ok && f <= f_ + o_.armijo_c1 * alpha_ * slope_) {
                // accept; BFGS inverse update  H <- (I - rho s y^T) H (I - rho y s^T) + rho s s^T
                double s[KMAX], y[KMAX], sy = 0, ss = 0, yy = 0;
                for (int a = 0; a < nf_; ++a) {
                    s[a] = req_[idx_[a]] - x_[idx_[a]];
                    y[a] = g[a] - g_[a];
                    sy += s[a] * y[a];
                    ss += s[a] * s[a];
                    yy += y[a] * y[a];
                }
                Mat newton;
                if (use_h_ && h_ok && inv_pd(Hin, nf_, newton)) {
                    Hinv_ = newton;  // Newton metric at the accepted point
                } else if (sy > 1e-10 * std::sqrt(ss) * std::sqrt(yy)) {
                    const double rho = 1.0 / sy;
                    double Hy[KMAX];
                    double yHy = 0;
                    for (int a = 0; a < nf_; ++a) {
                        double t = 0;
                        for (int b = 0; b < nf_; ++b) t += Hinv_.a[a][b] * y[b];
                        Hy[a] = t;
                    }
                    for (int a = 0; a < nf_; ++a) yHy += y[a] * Hy[a];
                    for (int a = 0; a < nf_; ++a)
                        for (int b = 0; b < nf_; ++b)
                            Hinv_.a[a][b] += -rho * (s[a] * Hy[b] + Hy[a] * s[b]) + rho * (rho * yHy + 1.0) * s[a] * s[b];
                }
                std::memcpy(x_, req_, sizeof(double) * K_);
                f_ = f;
                std::memcpy(g_, g, sizeof(double) * nf_);
                Hx_ = Hin;
                hx_ok_ = h_ok;
                begin_bfgs_iter();
                return;
            }
            alpha_ *= o_.backtrack;
            if (++nbt_ >= o_.max_backtracks) {
                begin_polish();
                return;
            }
            set_trial();
            return;
        case CHORD:
            if (!ok) {  // Newton step left the valid region: take a new Hessian
                begin_polish();
                return;
            }
            for (int a = 0; a < nf_; ++a) moved_[a] += std::fabs(req_[idx_[a]] - x_[idx_[a]]);
            std::memcpy(x_, req_, sizeof(double) * K_);
            f_ = f;
            std::memcpy(g_, g, sizeof(double) * nf_);
            ++chord_;
            if (use_h_) {  // a fresh Hessian came with the point: true Newton steps, covariance always current
                Hx_ = Hin;
                hx_ok_ = h_ok;
                Mat c;
                if (h_ok && inv_pd(Hin, nf_, c)) {
                    cov_ = c;
                    for (int a = 0; a < nf_; ++a) {
                        sig_[a] = std::sqrt(cov_.a[a][a]);
                        moved_[a] = 0.0;  // the covariance was taken here
                    }
                }
            }
            begin_chord();
            return;
        default: return;
        }
    }

    void result(mf_fit_result* r) const
    {
        std::memset(r, 0, sizeof(*r));
        for (int k = 0; k < K_; ++k) r->lambda_hat[k] = x_[k];
        for (int a = 0; a < nf_; ++a)
            for (int b = 0; b < nf_; ++b) r->cov[idx_[a] * K_ + idx_[b]] = cov_.a[a][b];
        r->nll_min = f_;
        r->n_calls = calls_;
        r->n_iter = iter_;
        r->converged = converged_ ? 1 : 0;
    }
    bool failed_start() const { return failed_start_; }

private:
    enum Phase { START, SEED_FD, TRIAL, POLISH_FD, CHORD, DONE };

    void begin_fd(Phase ph)
    {
        phase_ = ph;
        fd_a_ = 0;
        fd_side_ = 0;
        fd_ok_ = true;
        set_fd_request();
    }
    void set_fd_request()
    {
        std::memcpy(req_, x_, sizeof(double) * K_);
        const int k = idx_[fd_a_];
        req_[k] = fd_side_ == 0 ? x_[k] + h_[fd_a_] : x_[k] - h_[fd_a_];
    }
    // returns true when all 2 nf points are in; H_ is then the symmetrised Hessian (if fd_ok_)
    bool fd_feed(bool ok, const double* g)
    {
        if (!ok) fd_ok_ = false;
        if (fd_side_ == 0) {
            if (ok) std::memcpy(gp_, g, sizeof(double) * nf_);
            xp_ = req_[idx_[fd_a_]];
            fd_side_ = 1;
            set_fd_request();
            return false;
        }
        if (ok && fd_ok_) {
            const double dx = xp_ - req_[idx_[fd_a_]];
            for (int b = 0; b < nf_; ++b) H_.a[fd_a_][b] = (gp_[b] - g[b]) / dx;
        }
        fd_side_ = 0;
        if (++fd_a_ < nf_) {
            set_fd_request();
            return false;
        }
        if (fd_ok_)
            for (int a = 0; a < nf_; ++a)
                for (int b = 0; b < a; ++b) H_.a[a][b] = H_.a[b][a] = 0.5 * (H_.a[a][b] + H_.a[b][a]);
        return true;
    }
    void after_seed()
    {
        bool have = fd_ok_ && inv_pd(H_, nf_, Hinv_);
        if (!have) {
            for (int a = 0; a < nf_; ++a)
                for (int b = 0; b < nf_; ++b) Hinv_.a[a][b] = 0.0;
            for (int a = 0; a < nf_; ++a) {
                const double d = fd_ok_ ? std::fabs(H_.a[a][a]) : 1.0;
                Hinv_.a[a][a] = 1.0 / (d > 0.0 ? d : 1.0);
            }
        }
        cov_ = Hinv_;
        begin_bfgs_iter();
    }
    void begin_bfgs_iter()
    {
        if (iter_ >= o_.max_iter) {
            begin_polish();
            return;
        }
        ++iter_;
        double edm = 0;
        for (int a = 0; a < nf_; ++a)
            for (int b = 0; b < nf_; ++b) edm += g_[a] * Hinv_.a[a][b] * g_[b];
        edm *= 0.5;
        if (edm < o_.edm_tol) {
            begin_polish();
            return;
        }
        slope_ = direction();
        if (slope_ >= 0.0) {  // not a descent direction: reset the metric to its diagonal
            for (int a = 0; a < nf_; ++a)
                for (int b = 0; b < nf_; ++b)
                    Hinv_.a[a][b] = (a == b) ? std::fabs(Hinv_.a[a][a]) : 0.0;
            slope_ = direction();
        }
        alpha_ = 1.0;
        nbt_ = 0;
        phase_ = TRIAL;
        set_trial();
    }
    double direction()
    {
        double slope = 0;
        for (int a = 0; a < nf_; ++a) {
            double t = 0;
            for (int b = 0; b < nf_; ++b) t -= Hinv_.a[a][b] * g_[b];
            p_[a] = t;
            slope += g_[a] * t;
        }
        return slope;
    }
    void set_trial()
    {
        std::memcpy(req_, x_, sizeof(double) * K_);
        for (int a = 0; a < nf_; ++a) req_[idx_[a]] = x_[idx_[a]] + alpha_ * p_[a];
    }
    void begin_polish()
    {
        if (polish_ == 0) {
            for (int a = 0; a < nf_; ++a) h_[a] = o_.fd_sigma * std::sqrt(std::fabs(Hinv_.a[a][a]));
            cov_ = Hinv_;
        }
        if (polish_ >= o_.max_polish) {
            phase_ = DONE;
            return;
        }
        ++polish_;
        if (use_h_) {  // the Hessian at x_ is already here
            H_ = Hx_;
            fd_ok_ = hx_ok_;
            after_polish_fd();
            return;
        }
        begin_fd(POLISH_FD);
    }
    void after_polish_fd()
    {
        Mat c;
        if (!fd_ok_ || !inv_pd(H_, nf_, c)) {
            phase_ = DONE;
            return;
        }
        cov_ = c;
        for (int a = 0; a < nf_; ++a) {
            sig_[a] = std::sqrt(cov_.a[a][a]);
            h_[a] = o_.fd_sigma * sig_[a];
            moved_[a] = 0.0;
        }
        chord_ = 0;
        begin_chord();
    }
    void begin_chord()
    {
        double step[KMAX], worst = 0;
        for (int a = 0; a < nf_; ++a) {
            double t = 0;
            for (int b = 0; b < nf_; ++b) t -= cov_.a[a][b] * g_[b];
            step[a] = t;
            worst = std::max(worst, std::fabs(t) / sig_[a]);
        }
        if (worst < o_.polish_tol) {
            double mv = 0;
            for (int a = 0; a < nf_; ++a) mv = std::max(mv, moved_[a] / sig_[a]);
            if (mv < 1e-3) {
                converged_ = true;
                phase_ = DONE;
                return;
            }
            begin_polish();  // moved far on this Hessian: refresh it (and the covariance)
            return;
        }
        if (chord_ >= o_.max_chord) {
            begin_polish();
            return;
        }
        phase_ = CHORD;
        std::memcpy(req_, x_, sizeof(double) * K_);
        for (int a = 0; a < nf_; ++a) req_[idx_[a]] = x_[idx_[a]] + step[a];
    }

    int K_ = 0, nf_ = 0, idx_[KMAX] = {};
    mf_fit_opts o_{};
    Phase phase_ = START;
    double x_[KMAX] = {}, req_[KMAX] = {}, f_ = 0, g_[KMAX] = {};
    Mat Hinv_{}, H_{}, cov_{};
    double h_[KMAX] = {}, gp_[KMAX] = {}, xp_ = 0;
    int fd_a_ = 0, fd_side_ = 0;
    bool fd_ok_ = true;
    double p_[KMAX] = {}, slope_ = 0, alpha_ = 1;
    int nbt_ = 0, iter_ = 0, calls_ = 0, polish_ = 0, chord_ = 0;
    double sig_[KMAX] = {}, moved_[KMAX] = {};
    bool converged_ = false, failed_start_ = false;
    bool use_h_ = false, hx_ok_ = false;
    Mat Hx_{};  // analytic mode: Hessian at x_
};

}  // namespace

extern "C" void mf_fit_opts_default(mf_fit_opts* o)
{
    if (!o) return;
    o->max_iter = 200;
    o->edm_tol = 1e-5;
    o->armijo_c1 = 1e-4;
    o->backtrack = 0.5;
    o->max_backtracks = 40;
    o->polish_tol = 1e-9;
    o->max_polish = 8;
    o->max_chord = 8;
    o->fd_rel = 1e-5;
    o->fd_sigma = 1e-4;
    o->analytic_hessian = 1;
}

template <int KM>
static mf_status fit_one(mf_model* m, const double* start, const uint8_t* fixed, const mf_fit_opts& o, mf_fit_result* result)
{
    FitStateT<KM> st;
    st.init(m->K, start, fixed, o);
    const bool analytic = o.analytic_hessian != 0 && mf_model_has_hessian(m);
    if (analytic) st.use_analytic_hessian();
    // the minimiser asks for one point at a time: serve the evaluations from a resident kernel for the duration of the fit
    // where the model family has one (kernel submission dominates at small N)
    struct Serve {
        mf_model* m;
        bool was_on;
        explicit Serve(mf_model* mm) : m(mm), was_on(mf_model_is_served(mm) != 0) { mf_server_begin(m); }
        ~Serve() { mf_server_end(m, was_on); }
    } serve(m);
    mf_status first = MF_OK;
    bool is_first = true;
    while (!st.done()) {
        double f = 0, g[KM], h[KM * KM];
        const mf_status rc = analytic ? mf_nll_grad_hess(m, st.request(), &f, g, h) : mf_nll_grad(m, st.request(), &f, g);
        if (rc != MF_OK && rc != MF_ERR_PARAM_DOMAIN && rc != MF_NONPOSITIVE_PDF) return rc;
        if (is_first) first = rc;
        is_first = false;
        st.feed(rc == MF_OK, f, g, analytic ? h : nullptr);
    }
    st.result(result);
    if (st.failed_start()) return mf_fail(m->ctx, first == MF_OK ? MF_NONPOSITIVE_PDF : first, "mf_fit: invalid start point");
    if (mf_model_is_weighted(m)) {
        // weighted fit: cov = H^-1 F H^-1 with F = sum_i w_i^2 s_i s_i^T at the minimum (reading R23);
        // result->cov holds H^-1 over the free parameters (zero rows / columns for the fixed ones)
        const int K = m->K;
        double f = 0, g[KM], F[KM * KM];
        const mf_status rc = mf_nll_grad_hess_fisher(m, result->lambda_hat, &f, g, nullptr, F);
        if (rc != MF_OK) return rc;
        double T[KM * KM], C[KM * KM];
        for (int i = 0; i < K; ++i)
            for (int j = 0; j < K; ++j) {
                double s = 0.0;
                for (int k = 0; k < K; ++k) s += result->cov[i * K + k] * F[k * K + j];
                T[i * K + j] = s;
            }
        for (int i = 0; i < K; ++i)
            for (int j = 0; j < K; ++j) {
                double s = 0.0;
                for (int k = 0; k < K; ++k) s += T[i * K + k] * result->cov[k * K + j];
                C[i * K + j] = s;
            }
        for (int i = 0; i < K; ++i)
            for (int j = 0; j <= i; ++j) result->cov[i * K + j] = result->cov[j * K + i] = 0.5 * (C[i * K + j] + C[j * K + i]);
    }
    return MF_OK;
}

extern "C" mf_status mf_fit(mf_model* m, const double* start, const uint8_t* fixed, const mf_fit_opts* opts,
                            mf_fit_result* result)
{
    if (!m || !start || !result) return mf_fail(m ? m->ctx : nullptr, MF_ERR_ARG, "mf_fit: NULL argument");
    if (m->n_toys != 1) return mf_fail(m->ctx, MF_ERR_ARG, "mf_fit: dataset has n_toys != 1; use mf_fit_batch");
    mf_fit_opts o;
    if (opts) o = *opts;
    else mf_fit_opts_default(&o);
    if (m->K <= 4) return fit_one<4>(m, start, fixed, o, result);
    if (m->K <= 8) return fit_one<8>(m, start, fixed, o, result);
    return fit_one<MF_MAX_PARAMS>(m, start, fixed, o, result);
}

template <int KM>
static mf_status fit_many(mf_model* m, int64_t n_toys, const double* starts, const uint8_t* fixed, const mf_fit_opts& o,
                          mf_fit_result* results)
{
    const int K = m->K;
    std::vector<FitStateT<KM>> st((size_t)n_toys);
    std::vector<double> lam((size_t)n_toys * K), nll((size_t)n_toys), grad((size_t)n_toys * K);
    std::vector<uint8_t> active((size_t)n_toys);
    const bool analytic = o.analytic_hessian != 0 && mf_model_has_hessian(m);  // n_toys > 1: mass and angular families
    std::vector<double> hess(analytic ? (size_t)n_toys * K * K : 0);
    // the T fit states are independent: their host-side updates run on all cores (static schedule; the results do not
    // depend on the thread count)
#pragma omp parallel for schedule(static) if (n_toys >= 256)
    for (int64_t t = 0; t < n_toys; ++t) {
        st[t].init(K, starts + t * K, fixed, o);
        if (analytic) st[t].use_analytic_hessian();
    }
    for (;;) {
        int64_t n_active = 0;
#pragma omp parallel for schedule(static) reduction(+ : n_active) if (n_toys >= 256)
        for (int64_t t = 0; t < n_toys; ++t) {
            active[t] = st[t].done() ? 0 : 1;
            if (active[t]) {
                std::memcpy(&lam[t * K], st[t].request(), sizeof(double) * K);
                ++n_active;
            }
        }
        if (n_active == 0) break;
        const mf_status rc = analytic ? mf_nll_grad_hess_batch(m, n_toys, lam.data(), active.data(), nll.data(), grad.data(), hess.data())
                                      : mf_nll_grad_batch(m, n_toys, lam.data(), active.data(), nll.data(), grad.data());
        if (rc != MF_OK) return rc;
#pragma omp parallel for schedule(static) if (n_toys >= 256)
        for (int64_t t = 0; t < n_toys; ++t)
            if (active[t]) st[t].feed(std::isfinite(nll[t]), nll[t], &grad[t * K], analytic ? &hess[t * K * K] : nullptr);
    }
#pragma omp parallel for schedule(static) if (n_toys >= 256)
    for (int64_t t = 0; t < n_toys; ++t) st[t].result(&results[t]);
    return MF_OK;
}

extern "C" mf_status mf_fit_batch(mf_model* m, int64_t n_toys, const double* starts, const uint8_t* fixed,
                                  const mf_fit_opts* opts, mf_fit_result* results)
{
    if (!m || !starts || !results) return mf_fail(m ? m->ctx : nullptr, MF_ERR_ARG, "mf_fit_batch: NULL argument");
    if (n_toys != m->n_toys) return mf_fail(m->ctx, MF_ERR_ARG, "mf_fit_batch: n_toys does not match the dataset");
    mf_fit_opts o;
    if (opts) o = *opts;
    else mf_fit_opts_default(&o);
    if (m->K <= 4) return fit_many<4>(m, n_toys, starts, fixed, o, results);
    if (m->K <= 8) return fit_many<8>(m, n_toys, starts, fixed, o, results);
    return fit_many<MF_MAX_PARAMS>(m, n_toys, starts, fixed, o, results);
}
