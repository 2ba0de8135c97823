/*
 * mf_oracle.c — plain, slow, fp64 CPU ORACLE for the MoreFit NLL + analytic gradient.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT PRODUCT CODE.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may build, link or call it.  It
 * shares no code, header, table or constant with paper_2505_12414_b200/ (the CUDA path)
 * and neither includes the other.
 *
 * What it computes (the plain definitions, PAPER.md line numbers):
 *   Eq. 1      -ln L(lambda) = - sum_i ln P(x_i | lambda)
 *   Eq. 2   mass model  P = f G/N1 + (1-f) e^{tau m}/N2
 *   Eq. 4 angular model d^3Gamma/dcos(theta_l) dcos(theta_K) dphi
 *   4D model (BASELINE.json configs[3]; not in the paper) P = f (G/N1) A + (1-f) (E/N2) L
 * and the hand-derived d ln P / d lambda_k of each.
 *
 * Deliberately NOT done here (those are the optimisations under test):
 * no parameter-only constants hoisted out of the event loop, no cached event-only
 * terms, no algebraic merging of the angular terms, no blocking or fusion.  Every event
 * re-evaluates the normalisations from the formulas.  Per-event arithmetic is IEEE
 * double (the paper's precision); sums over events are accumulated
 * in long double (x87 80-bit) so that the summation error of the oracle itself is
 * negligible against the 1e-11 / 1e-9 parity tolerances.  With OpenMP (nthreads > 1)
 * events are split into `nthreads` contiguous static chunks whose long-double sums
 * are combined in chunk order.
 *
 * Readings of the paper taken here:
 *   R6  N2 is evaluated as e^{tau a} expm1(tau (b-a)) / tau (tau != 0) and (b-a) at tau == 0;
 *       d ln N2 / d tau = a + w h(tau w), h(u) = 1/(1-e^{-u}) - 1/u evaluated in long
 *       double, by its Taylor series for |u| < 1e-2 (cancellation), h(0) = 1/2.
 *   R9  no extended (Poisson) term, unweighted events.
 *   R15 an event with P <= 0 (or NaN) makes -ln L = +inf and every gradient component NaN;
 *       the number of such events is returned.
 *
 * Pins (tests/test_oracle_*.py): unit integral by quadrature, positivity, score identity,
 * finite differences, scipy truncnorm/truncexpon, Gaussian closed-form MLE, the printed
 * constants of Listing 4, closed-form angular marginals, hand-evaluated points of Eq. 4.
 * The analytic Hessian at the end of the file (all three kinds) has its own pins
 * (tests/test_oracle_hessian.py): finite differences of the pinned gradient and the information identity.
 * Weighted sums and the Fisher matrix of weighted fits (reading R23: -ln L_w = -sum w_i ln P_i; covariance
 * H^-1 F H^-1 with F = sum w_i^2 s_i s_i^T) are pinned there too: unit weights reproduce the unweighted sums bit for
 * bit, integer weights equal event duplication, the sums rebuilt from the pinned per-event quantities, the closed
 * forms of a weighted Gaussian (MLE, H, F, sandwich), invariance under a rescaling of the weights, unit pull width.
 */
#include <math.h>
#include <stddef.h>
#include <stdint.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define MFO_MASS 0
#define MFO_ANGULAR 1
#define MFO_4D 2
#define MFO_MAXK 16

static const double MFO_PI = 3.14159265358979323846264338327950288;

/* ---------------------------------------------------------------- mass, Eq. 2 */

/* N1(mu, sigma) */
static double norm_gauss(double mu, double sigma, double a, double b)
{
    const double s2 = sqrt(2.0) * sigma;
    return 0.5 * (erf((mu - a) / s2) - erf((mu - b) / s2));
}

/* g(x) = Gaussian density */
static double gauss_density(double x, double mu, double sigma)
{
    const double d = x - mu;
    return exp(-(d * d) / (2.0 * sigma * sigma)) / (sqrt(2.0 * MFO_PI) * sigma);
}

/* dN1/dmu = g(a) - g(b);  dN1/dsigma = [(a-mu) g(a) - (b-mu) g(b)] / sigma */
static double dnorm_gauss_dmu(double mu, double sigma, double a, double b)
{
    return gauss_density(a, mu, sigma) - gauss_density(b, mu, sigma);
}
static double dnorm_gauss_dsigma(double mu, double sigma, double a, double b)
{
    return ((a - mu) * gauss_density(a, mu, sigma) - (b - mu) * gauss_density(b, mu, sigma)) / sigma;
}

/* N2(tau), reading R6 */
static double norm_exp(double tau, double a, double b)
{
    if (tau == 0.0) return b - a;
    return exp(tau * a) * expm1(tau * (b - a)) / tau;
}

/* d ln N2 / d tau = mean of m under the truncated exponential, reading R6 */
static double dlognorm_exp_dtau(double tau, double a, double b)
{
    const long double w = (long double)b - (long double)a;
    const long double u = (long double)tau * w;
    long double h;
    if (fabsl(u) < 1e-2L) {
        const long double u2 = u * u;
        /* 1/(1-e^-u) - 1/u = 1/2 + u/12 - u^3/720 + u^5/30240 - u^7/1209600 + ... */
        h = 0.5L + u * (1.0L / 12.0L + u2 * (-1.0L / 720.0L + u2 * (1.0L / 30240.0L + u2 * (-1.0L / 1209600.0L))));
    } else {
        h = -1.0L / expm1l(-u) - 1.0L / u;
    }
    return (double)((long double)a + w * h);
}

/* P and d ln P / d(f, mu, sigma, tau) for one event.  g may be NULL. */
static double mass_event(double m, const double *lam, double a, double b, double *g)
{
    const double f = lam[0], mu = lam[1], sigma = lam[2], tau = lam[3];
    const double G = gauss_density(m, mu, sigma);
    const double N1 = norm_gauss(mu, sigma, a, b);
    const double E = exp(tau * m);
    const double N2 = norm_exp(tau, a, b);
    const double S = f * G / N1;
    const double B = (1.0 - f) * E / N2;
    const double P = S + B;
    if (g) {
        g[0] = (G / N1 - E / N2) / P;
        g[1] = S * ((m - mu) / (sigma * sigma) - dnorm_gauss_dmu(mu, sigma, a, b) / N1) / P;
        g[2] = S * ((m - mu) * (m - mu) / (sigma * sigma * sigma) - 1.0 / sigma
                    - dnorm_gauss_dsigma(mu, sigma, a, b) / N1) / P;
        g[3] = B * (m - dlognorm_exp_dtau(tau, a, b)) / P;
    }
    return P;
}

/* ------------------------------------------------------------ angular, Eq. 4 */

/* The eleven angular terms of Eq. 4 in the order printed, WITHOUT the
 * coefficients: term[0..3] carry (1-FL), FL, (1-FL), -FL; term[4..10] carry
 * S3, S4, S5, AFB, S7, S8, S9.  The 4/3 of the AFB term is kept with the term. */
static void angular_terms(double cl, double ck, double phi, double t[11])
{
    const double cos2_l = cl * cl, cos2_k = ck * ck;
    const double sin2_l = 1.0 - cos2_l, sin2_k = 1.0 - cos2_k; /* sin^2 theta */
    const double sin_l = sqrt(sin2_l), sin_k = sqrt(sin2_k);   /* theta in [0,pi]: sin >= 0 */
    const double cos2theta_l = 2.0 * cos2_l - 1.0;             /* cos 2theta_l */
    const double sin2theta_l = 2.0 * sin_l * cl;               /* sin 2theta_l */
    const double sin2theta_k = 2.0 * sin_k * ck;               /* sin 2theta_K */
    t[0] = 0.75 * sin2_k;
    t[1] = cos2_k;
    t[2] = 0.25 * sin2_k * cos2theta_l;
    t[3] = cos2_k * cos2theta_l;
    t[4] = sin2_k * sin2_l * cos(2.0 * phi);
    t[5] = sin2theta_k * sin2theta_l * cos(phi);
    t[6] = sin2theta_k * sin_l * cos(phi);
    t[7] = (4.0 / 3.0) * sin2_k * cl;
    t[8] = sin2theta_k * sin_l * sin(phi);
    t[9] = sin2theta_k * sin2theta_l * sin(phi);
    t[10] = sin2_k * sin2_l * sin(2.0 * phi);
}

/* A(Omega) and dA/d(FL,S3,S4,S5,AFB,S7,S8,S9) (NOT divided by A).  dA may be NULL. */
static double angular_value(double cl, double ck, double phi, const double *a, double *dA)
{
    const double c = 9.0 / (32.0 * MFO_PI);
    double t[11];
    angular_terms(cl, ck, phi, t);
    const double FL = a[0];
    double A = (1.0 - FL) * t[0] + FL * t[1] + (1.0 - FL) * t[2] - FL * t[3];
    for (int k = 1; k < 8; ++k) A += a[k] * t[3 + k];
    A *= c;
    if (dA) {
        dA[0] = c * (-t[0] + t[1] - t[2] - t[3]);
        for (int k = 1; k < 8; ++k) dA[k] = c * t[3 + k];
    }
    return A;
}

static double angular_event(double cl, double ck, double phi, const double *lam, double *g)
{
    double dA[8];
    const double A = angular_value(cl, ck, phi, lam, dA);
    if (g)
        for (int k = 0; k < 8; ++k) g[k] = dA[k] / A;
    return A;
}

/* ------------------------------------------- 4D, BASELINE.json configs[3] */

/* l(x; c1, c2) = 1/2 [1 + c1 P1(x) + c2 P2(x)], normalised on [-1,1] */
static double legendre2(double x, double c1, double c2)
{
    return 0.5 * (1.0 + c1 * x + c2 * 0.5 * (3.0 * x * x - 1.0));
}

/* lambda = (f, mu, sigma, tau, FL..S9, cl1, cl2, ck1, ck2) */
static double fourd_event(double m, double cl, double ck, double phi, const double *lam,
                          double a, double b, double *g)
{
    const double f = lam[0], mu = lam[1], sigma = lam[2], tau = lam[3];
    const double *ang = lam + 4;
    const double cl1 = lam[12], cl2 = lam[13], ck1 = lam[14], ck2 = lam[15];
    const double G = gauss_density(m, mu, sigma);
    const double N1 = norm_gauss(mu, sigma, a, b);
    const double E = exp(tau * m);
    const double N2 = norm_exp(tau, a, b);
    double dA[8];
    const double A = angular_value(cl, ck, phi, ang, dA);
    const double Ll = legendre2(cl, cl1, cl2), Lk = legendre2(ck, ck1, ck2);
    const double L = Ll * Lk / (2.0 * MFO_PI);
    const double S = f * (G / N1) * A;
    const double B = (1.0 - f) * (E / N2) * L;
    const double P = S + B;
    if (g) {
        g[0] = ((G / N1) * A - (E / N2) * L) / P;
        g[1] = S * ((m - mu) / (sigma * sigma) - dnorm_gauss_dmu(mu, sigma, a, b) / N1) / P;
        g[2] = S * ((m - mu) * (m - mu) / (sigma * sigma * sigma) - 1.0 / sigma
                    - dnorm_gauss_dsigma(mu, sigma, a, b) / N1) / P;
        g[3] = B * (m - dlognorm_exp_dtau(tau, a, b)) / P;
        for (int k = 0; k < 8; ++k) g[4 + k] = f * (G / N1) * dA[k] / P;
        const double Bm = (1.0 - f) * (E / N2) / (2.0 * MFO_PI);
        g[12] = Bm * (0.5 * cl) * Lk / P;
        g[13] = Bm * (0.5 * 0.5 * (3.0 * cl * cl - 1.0)) * Lk / P;
        g[14] = Bm * Ll * (0.5 * ck) / P;
        g[15] = Bm * Ll * (0.5 * 0.5 * (3.0 * ck * ck - 1.0)) / P;
    }
    return P;
}

/* ------------------------------------------------------------------- API */

int mfo_nparams(int kind)
{
    return kind == MFO_MASS ? 4 : kind == MFO_ANGULAR ? 8 : kind == MFO_4D ? 16 : -1;
}
int mfo_ndim(int kind)
{
    return kind == MFO_MASS ? 1 : kind == MFO_ANGULAR ? 3 : kind == MFO_4D ? 4 : -1;
}

static double eval_event(int kind, const double *const *cols, int64_t i, const double *lam,
                         double lo, double hi, double *g)
{
    switch (kind) {
    case MFO_MASS: return mass_event(cols[0][i], lam, lo, hi, g);
    case MFO_ANGULAR: return angular_event(cols[0][i], cols[1][i], cols[2][i], lam, g);
    default: return fourd_event(cols[0][i], cols[1][i], cols[2][i], cols[3][i], lam, lo, hi, g);
    }
}

/* Per-event P(x_i | lambda) and d ln P / d lambda_k (dlnp laid out [K][n], may be NULL). */
int mfo_pdf(int kind, int64_t n, const double *const *cols, const double *lam, double lo,
            double hi, double *p, double *dlnp)
{
    const int K = mfo_nparams(kind);
    if (K < 0) return -1;
    for (int64_t i = 0; i < n; ++i) {
        double g[MFO_MAXK];
        p[i] = eval_event(kind, cols, i, lam, lo, hi, dlnp ? g : NULL);
        if (dlnp)
            for (int k = 0; k < K; ++k) dlnp[(int64_t)k * n + i] = g[k];
    }
    return 0;
}

/* The two normalisations and their derivatives, exposed so that tests can pin them. */
void mfo_mass_norms(const double *lam, double lo, double hi, double *out /*[5]*/)
{
    out[0] = norm_gauss(lam[1], lam[2], lo, hi);
    out[1] = dnorm_gauss_dmu(lam[1], lam[2], lo, hi);
    out[2] = dnorm_gauss_dsigma(lam[1], lam[2], lo, hi);
    out[3] = norm_exp(lam[3], lo, hi);
    out[4] = dlognorm_exp_dtau(lam[3], lo, hi);
}

/* The eleven terms of Eq. 4 times c = 9/(32 pi), exposed so that tests can pin them. */
void mfo_angular_terms(double cl, double ck, double phi, double *out /*[11]*/)
{
    angular_terms(cl, ck, phi, out);
    for (int j = 0; j < 11; ++j) out[j] *= 9.0 / (32.0 * MFO_PI);
}

static void chunk_sums(int kind, const double *const *cols, const double *w /* event weights or NULL (= 1) */, int64_t i0,
                       int64_t i1, const double *lam, double lo, double hi, int K, int want_grad,
                       long double *acc /*[K+1]*/, int64_t *nbad)
{
    for (int k = 0; k <= K; ++k) acc[k] = 0.0L;
    int64_t bad = 0;
    for (int64_t i = i0; i < i1; ++i) {
        double g[MFO_MAXK];
        const double P = eval_event(kind, cols, i, lam, lo, hi, want_grad ? g : NULL);
        if (!(P > 0.0)) { ++bad; continue; }
        const long double wi = w ? (long double)w[i] : 1.0L; /* times 1.0L is exact: the unweighted sums are unchanged */
        acc[0] += wi * (long double)log(P);
        if (want_grad)
            for (int k = 0; k < K; ++k) acc[1 + k] += wi * (long double)g[k];
    }
    *nbad = bad;
}

/*
 * -ln L and its gradient over n events (Eq. 1).  cols: ndim pointers to n doubles each.
 * grad may be NULL.  Returns the number of events with P <= 0 or NaN (then *nll = +inf,
 * grad = NaN), or -1 on a bad argument.
 */
int64_t mfo_nll_grad_w(int kind, int64_t n, const double *const *cols, const double *w, const double *lam, double lo,
                       double hi, int nthreads, double *nll, double *grad);

int64_t mfo_nll_grad(int kind, int64_t n, const double *const *cols, const double *lam, double lo,
                     double hi, int nthreads, double *nll, double *grad)
{
    return mfo_nll_grad_w(kind, n, cols, NULL, lam, lo, hi, nthreads, nll, grad);
}

/*
 * The same with event weights w_i ("weighted fits"; reading R23):
 *     -ln L_w(lambda) = - sum_i w_i ln P(x_i | lambda),   gradient likewise.
 * w == NULL means w_i = 1 (bit-identical to the unweighted sums).  Weights may be negative (sWeights); an event
 * with P <= 0 is counted as bad whatever its weight.
 */
int64_t mfo_nll_grad_w(int kind, int64_t n, const double *const *cols, const double *w, const double *lam, double lo,
                       double hi, int nthreads, double *nll, double *grad)
{
    const int K = mfo_nparams(kind);
    if (K < 0 || n < 0) return -1;
    if (nthreads < 1) nthreads = 1;
    if (nthreads > 1024) nthreads = 1024;
    long double part[1024][MFO_MAXK + 1];
    int64_t bad[1024];
    const int want_grad = grad != NULL;
#ifdef _OPENMP
#pragma omp parallel for num_threads(nthreads) schedule(static, 1)
#endif
    for (int c = 0; c < nthreads; ++c) {
        const int64_t i0 = n * c / nthreads, i1 = n * (c + 1) / nthreads;
        chunk_sums(kind, cols, w, i0, i1, lam, lo, hi, K, want_grad, part[c], &bad[c]);
    }
    long double tot[MFO_MAXK + 1];
    int64_t nbad = 0;
    for (int k = 0; k <= K; ++k) tot[k] = 0.0L;
    for (int c = 0; c < nthreads; ++c) { /* chunk order: deterministic */
        nbad += bad[c];
        for (int k = 0; k <= K; ++k) tot[k] += part[c][k];
    }
    if (nbad) {
        *nll = INFINITY;
        if (grad) for (int k = 0; k < K; ++k) grad[k] = NAN;
        return nbad;
    }
    *nll = (double)(-tot[0]);
    if (grad) for (int k = 0; k < K; ++k) grad[k] = (double)(-tot[1 + k]);
    return 0;
}

int mfo_max_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ================================================================================================
 * Second derivatives (analytic Hessian by symbolic second
 * differentiation of ln P).  Written through the derivatives of P itself,
 *     d2 ln P / da db = P_ab / P - P_a P_b / P^2,
 * with P = f s(m; mu, sigma) + (1 - f) b(m; tau), s = G/N1, b = e^{tau m}/N2.
 * Pins (tests/test_oracle_hessian.py): Richardson central differences of mfo_nll_grad's gradient, and the
 * information identity  int P (l_ab + l_a l_b) dm = 0  by quadrature for all ten (a, b).
 * ================================================================================================ */

/* d^2 ln N2 / d tau^2 = w^2 h'(tau w), h(u) = 1/(1 - e^-u) - 1/u, h'(u) = 1/u^2 - 1/(4 sinh^2(u/2)) */
static double d2lognorm_exp_dtau2(double tau, double a, double b)
{
    const long double w = (long double)b - (long double)a;
    const long double u = (long double)tau * w;
    long double hp;
    if (fabsl(u) < 1e-2L) {
        const long double u2 = u * u;
        hp = 1.0L / 12.0L + u2 * (-1.0L / 240.0L + u2 * (1.0L / 6048.0L + u2 * (-1.0L / 172800.0L)));
    } else {
        const long double sh = sinhl(0.5L * u);
        hp = 1.0L / (u * u) - 1.0L / (4.0L * sh * sh);
    }
    return (double)(w * w * hp);
}

/* Hessian of ln P for one mass event, h[10] in the order ff, fm, fs, ft, mm, ms, mt, ss, st, tt
 * (m = mu, s = sigma, t = tau); g[4] = gradient of ln P.  Returns P. */
static double mass_event_hess(double m, const double *lam, double a, double b, double *g, double *h)
{
    const double f = lam[0], mu = lam[1], sigma = lam[2], tau = lam[3];
    const double s2 = sigma * sigma, s3 = s2 * sigma, s4 = s2 * s2;
    const double d = m - mu;
    const double N1 = norm_gauss(mu, sigma, a, b);
    const double ga = gauss_density(a, mu, sigma), gb = gauss_density(b, mu, sigma);
    /* derivatives of N1: dg(x)/dmu = g (x-mu)/sigma^2, dg(x)/dsigma = g ((x-mu)^2/sigma^3 - 1/sigma) */
    const double da = a - mu, db = b - mu;
    const double N1_m = ga - gb;
    const double N1_s = (da * ga - db * gb) / sigma;
    const double ga_s = ga * (da * da / s3 - 1.0 / sigma), gb_s = gb * (db * db / s3 - 1.0 / sigma);
    const double N1_mm = ga * da / s2 - gb * db / s2;
    const double N1_ms = ga_s - gb_s;
    const double N1_ss = (da * ga_s - db * gb_s) / sigma - (da * ga - db * gb) / s2;
    /* s = G/N1 and its logarithmic derivatives */
    const double s = gauss_density(m, mu, sigma) / N1;
    const double al_m = d / s2 - N1_m / N1;
    const double al_s = d * d / s3 - 1.0 / sigma - N1_s / N1;
    const double al_mm = -1.0 / s2 - (N1_mm / N1 - (N1_m / N1) * (N1_m / N1));
    const double al_ms = -2.0 * d / s3 - (N1_ms / N1 - (N1_m / N1) * (N1_s / N1));
    const double al_ss = -3.0 * d * d / s4 + 1.0 / s2 - (N1_ss / N1 - (N1_s / N1) * (N1_s / N1));
    const double s_m = s * al_m, s_s = s * al_s;
    const double s_mm = s * (al_m * al_m + al_mm), s_ms = s * (al_m * al_s + al_ms), s_ss = s * (al_s * al_s + al_ss);
    /* b = E/N2 */
    const double bb = exp(tau * m) / norm_exp(tau, a, b);
    const double be = m - dlognorm_exp_dtau(tau, a, b);
    const double b_t = bb * be;
    const double b_tt = bb * (be * be - d2lognorm_exp_dtau2(tau, a, b));
    const double P = f * s + (1.0 - f) * bb;
    const double Pf = s - bb, Pm = f * s_m, Ps = f * s_s, Pt = (1.0 - f) * b_t;
    const double P1[4] = {Pf, Pm, Ps, Pt};
    /*                  ff   fm   fs    ft     mm        ms        mt   ss        st   tt */
    const double P2[10] = {0.0, s_m, s_s, -b_t, f * s_mm, f * s_ms, 0.0, f * s_ss, 0.0, (1.0 - f) * b_tt};
    if (g) for (int k = 0; k < 4; ++k) g[k] = P1[k] / P;
    int q = 0;
    for (int i = 0; i < 4; ++i)
        for (int j = i; j < 4; ++j, ++q) h[q] = P2[q] / P - (P1[i] / P) * (P1[j] / P);
    return P;
}

/* exposed for the quadrature pins: P, gradient and packed Hessian of ln P at mass values m[0..n-1] */
int mfo_mass_hess_points(int64_t n, const double *m, const double *lam, double lo, double hi, double *P, double *g /*[n][4]*/,
                         double *h /*[n][10]*/)
{
    for (int64_t i = 0; i < n; ++i) P[i] = mass_event_hess(m[i], lam, lo, hi, g + 4 * i, h + 10 * i);
    return 0;
}

/*
 * -ln L, its gradient and its Hessian (row-major K x K, symmetric) over n events, for the mass (K = 4) and
 * angular (K = 8) kinds.  Angular: P = A is linear in its coefficients, so d2 ln P / da db = -A_a A_b / A^2.
 * Sums in long double, single pass in event order.  Returns the number of events with P <= 0 (then nll = +inf,
 * everything else NaN), -1 on a bad argument (including the 4D kind: its Hessian is reached through
 * mfo_nll_grad_hess_w below, which with w = NULL returns for the mass and angular kinds exactly what this routine does).
 */
int64_t mfo_nll_grad_hess(int kind, int64_t n, const double *const *cols, const double *lam, double lo, double hi,
                          double *nll, double *grad, double *hess)
{
    if (!(kind == MFO_MASS || kind == MFO_ANGULAR) || n < 0) return -1;
    const int K = mfo_nparams(kind);
    long double s0 = 0.0L, sg[8], sh[64];
    for (int i = 0; i < 8; ++i) sg[i] = 0.0L;
    for (int i = 0; i < 64; ++i) sh[i] = 0.0L;
    int64_t bad = 0;
    for (int64_t e = 0; e < n; ++e) {
        double g[8], P;
        if (kind == MFO_MASS) {
            double h[10];
            P = mass_event_hess(cols[0][e], lam, lo, hi, g, h);
            if (!(P > 0.0)) { ++bad; continue; }
            int q = 0;
            for (int i = 0; i < 4; ++i)
                for (int j = i; j < 4; ++j, ++q) {
                    sh[i * K + j] += (long double)h[q];
                    if (j != i) sh[j * K + i] += (long double)h[q];
                }
        } else {
            double dA[8];
            P = angular_value(cols[0][e], cols[1][e], cols[2][e], lam, dA);
            if (!(P > 0.0)) { ++bad; continue; }
            for (int i = 0; i < 8; ++i) g[i] = dA[i] / P;
            for (int i = 0; i < 8; ++i)
                for (int j = 0; j < 8; ++j) sh[i * K + j] += (long double)(-(dA[i] / P) * (dA[j] / P));
        }
        s0 += (long double)log(P);
        for (int i = 0; i < K; ++i) sg[i] += (long double)g[i];
    }
    if (bad) {
        *nll = INFINITY;
        for (int i = 0; i < K; ++i) grad[i] = NAN;
        for (int i = 0; i < K * K; ++i) hess[i] = NAN;
        return bad;
    }
    *nll = (double)(-s0);
    for (int i = 0; i < K; ++i) grad[i] = (double)(-sg[i]);
    for (int i = 0; i < K * K; ++i) hess[i] = (double)(-sh[i]);
    return 0;
}

/* ================================================================================================
 * 4D model: second derivatives, again through the derivatives of P:
 *     P = f s(m; mu, sigma) A(Omega; a) + (1 - f) b(m; tau) L(Omega; c),   d2 ln P / dx dy = P_xy / P - P_x P_y / P^2.
 * A is linear in its eight coefficients and L = l(cos theta_l; cl1, cl2) l(cos theta_K; ck1, ck2) / (2 pi) is linear in
 * each Legendre coefficient, so the only non-zero second derivatives of P are
 *     (f, x) for every other x;  (mu|sigma, mu|sigma);  (mu|sigma, a_k);  (tau, tau);  (tau, c);  (cl_i, ck_j).
 * Pins (tests/test_oracle_hessian.py): Richardson central differences of the pinned gradient, and the information
 * identity  int P (l_xy + l_x l_y) dm dOmega = 0  for all 136 pairs on the quadrature grid of test_oracle_4d.py.
 * ================================================================================================ */

/* s = G/N1, b = e^{tau m}/N2 and their first and second parameter derivatives for one mass value
 * (the same formulas as in mass_event_hess, collected for the 4D model). */
typedef struct {
    double s, s_m, s_s, s_mm, s_ms, s_ss; /* signal shape and its (mu, sigma) derivatives */
    double b, b_t, b_tt;                  /* background shape and its tau derivatives */
} mass_parts;

static void mass_shape_derivs(double m, double mu, double sigma, double tau, double a, double b, mass_parts *o)
{
    const double s2 = sigma * sigma, s3 = s2 * sigma, s4 = s2 * s2;
    const double d = m - mu;
    const double N1 = norm_gauss(mu, sigma, a, b);
    const double ga = gauss_density(a, mu, sigma), gb = gauss_density(b, mu, sigma);
    const double da = a - mu, db = b - mu;
    const double N1_m = ga - gb;
    const double N1_s = (da * ga - db * gb) / sigma;
    const double ga_s = ga * (da * da / s3 - 1.0 / sigma), gb_s = gb * (db * db / s3 - 1.0 / sigma);
    const double N1_mm = ga * da / s2 - gb * db / s2;
    const double N1_ms = ga_s - gb_s;
    const double N1_ss = (da * ga_s - db * gb_s) / sigma - (da * ga - db * gb) / s2;
    const double s = gauss_density(m, mu, sigma) / N1;
    const double al_m = d / s2 - N1_m / N1;
    const double al_s = d * d / s3 - 1.0 / sigma - N1_s / N1;
    const double al_mm = -1.0 / s2 - (N1_mm / N1 - (N1_m / N1) * (N1_m / N1));
    const double al_ms = -2.0 * d / s3 - (N1_ms / N1 - (N1_m / N1) * (N1_s / N1));
    const double al_ss = -3.0 * d * d / s4 + 1.0 / s2 - (N1_ss / N1 - (N1_s / N1) * (N1_s / N1));
    o->s = s;
    o->s_m = s * al_m;
    o->s_s = s * al_s;
    o->s_mm = s * (al_m * al_m + al_mm);
    o->s_ms = s * (al_m * al_s + al_ms);
    o->s_ss = s * (al_s * al_s + al_ss);
    const double bb = exp(tau * m) / norm_exp(tau, a, b);
    const double be = m - dlognorm_exp_dtau(tau, a, b);
    o->b = bb;
    o->b_t = bb * be;
    o->b_tt = bb * (be * be - d2lognorm_exp_dtau2(tau, a, b));
}

/* P, g[16] = d ln P / d lambda, H[16][16] = d2 ln P / d lambda^2 (full, symmetric) for one 4D event.
 * lambda = (f, mu, sigma, tau, FL..S9, cl1, cl2, ck1, ck2). */
static double fourd_event_hess(double m, double cl, double ck, double phi, const double *lam, double a, double b,
                               double *g, double *H)
{
    const double f = lam[0], mu = lam[1], sigma = lam[2], tau = lam[3];
    const double cl1 = lam[12], cl2 = lam[13], ck1 = lam[14], ck2 = lam[15];
    mass_parts q;
    mass_shape_derivs(m, mu, sigma, tau, a, b, &q);
    double dA[8];
    const double A = angular_value(cl, ck, phi, lam + 4, dA);
    const double Ll = legendre2(cl, cl1, cl2), Lk = legendre2(ck, ck1, ck2);
    const double twopi = 2.0 * MFO_PI;
    const double L = Ll * Lk / twopi;
    /* dl/dc1 = x/2, dl/dc2 = (3x^2 - 1)/4 */
    const double dLl[2] = {0.5 * cl, 0.5 * 0.5 * (3.0 * cl * cl - 1.0)};
    const double dLk[2] = {0.5 * ck, 0.5 * 0.5 * (3.0 * ck * ck - 1.0)};
    const double dL[4] = {dLl[0] * Lk / twopi, dLl[1] * Lk / twopi, Ll * dLk[0] / twopi, Ll * dLk[1] / twopi};
    const double P = f * q.s * A + (1.0 - f) * q.b * L;
    double P1[16], P2[16][16];
    for (int i = 0; i < 16; ++i)
        for (int j = 0; j < 16; ++j) P2[i][j] = 0.0;
    P1[0] = q.s * A - q.b * L;
    P1[1] = f * q.s_m * A;
    P1[2] = f * q.s_s * A;
    P1[3] = (1.0 - f) * q.b_t * L;
    for (int k = 0; k < 8; ++k) P1[4 + k] = f * q.s * dA[k];
    for (int k = 0; k < 4; ++k) P1[12 + k] = (1.0 - f) * q.b * dL[k];
    /* row f */
    P2[0][1] = q.s_m * A;
    P2[0][2] = q.s_s * A;
    P2[0][3] = -q.b_t * L;
    for (int k = 0; k < 8; ++k) P2[0][4 + k] = q.s * dA[k];
    for (int k = 0; k < 4; ++k) P2[0][12 + k] = -q.b * dL[k];
    /* (mu, sigma) block and its couplings to the angular coefficients */
    P2[1][1] = f * q.s_mm * A;
    P2[1][2] = f * q.s_ms * A;
    P2[2][2] = f * q.s_ss * A;
    for (int k = 0; k < 8; ++k) {
        P2[1][4 + k] = f * q.s_m * dA[k];
        P2[2][4 + k] = f * q.s_s * dA[k];
    }
    /* tau and the Legendre coefficients */
    P2[3][3] = (1.0 - f) * q.b_tt * L;
    for (int k = 0; k < 4; ++k) P2[3][12 + k] = (1.0 - f) * q.b_t * dL[k];
    for (int i = 0; i < 2; ++i)
        for (int j = 0; j < 2; ++j) P2[12 + i][14 + j] = (1.0 - f) * q.b * dLl[i] * dLk[j] / twopi;
    for (int i = 0; i < 16; ++i)
        for (int j = 0; j < i; ++j) P2[i][j] = P2[j][i];
    for (int i = 0; i < 16; ++i) g[i] = P1[i] / P;
    for (int i = 0; i < 16; ++i)
        for (int j = 0; j < 16; ++j) H[i * 16 + j] = P2[i][j] / P - (P1[i] / P) * (P1[j] / P);
    return P;
}

/* P, gradient and full Hessian of ln P for one event of any kind (g[K], H[K*K]). */
static double event_hess(int kind, const double *const *cols, int64_t e, const double *lam, double lo, double hi, double *g,
                         double *H)
{
    if (kind == MFO_MASS) {
        double h[10];
        const double P = mass_event_hess(cols[0][e], lam, lo, hi, g, h);
        int q = 0;
        for (int i = 0; i < 4; ++i)
            for (int j = i; j < 4; ++j, ++q) H[i * 4 + j] = H[j * 4 + i] = h[q];
        return P;
    }
    if (kind == MFO_ANGULAR) {
        double dA[8];
        const double P = angular_value(cols[0][e], cols[1][e], cols[2][e], lam, dA);
        for (int i = 0; i < 8; ++i) g[i] = dA[i] / P;
        for (int i = 0; i < 8; ++i)
            for (int j = 0; j < 8; ++j) H[i * 8 + j] = -(dA[i] / P) * (dA[j] / P);
        return P;
    }
    return fourd_event_hess(cols[0][e], cols[1][e], cols[2][e], cols[3][e], lam, lo, hi, g, H);
}

/* exposed for the quadrature pins: per-event P [n], d ln P [n][K], d2 ln P [n][K][K] */
int mfo_hess_points(int kind, int64_t n, const double *const *cols, const double *lam, double lo, double hi, double *P,
                    double *g, double *H)
{
    const int K = mfo_nparams(kind);
    if (K < 0) return -1;
    for (int64_t e = 0; e < n; ++e) P[e] = event_hess(kind, cols, e, lam, lo, hi, g + e * K, H + e * K * K);
    return 0;
}

/*
 * Weighted second-order sums for every kind ("the Fisher information matrix can be
 * calculated analytically, which is required for weighted fits [22]"; reading R23):
 *     -ln L_w = - sum_i w_i ln P_i
 *     grad    = - sum_i w_i  d ln P_i / d lambda
 *     hess    = - sum_i w_i  d2 ln P_i / d lambda^2                 (K x K, may be NULL)
 *     fisher  =   sum_i w_i^2 (d ln P_i/d lambda)(d ln P_i/d lambda)^T   (K x K, may be NULL)
 * The covariance of a weighted fit is  hess^-1 fisher hess^-1  at the minimum (the sandwich of [22]); for w_i = 1 its
 * expectation equals hess^-1.  w == NULL means w_i = 1: hess is then what mfo_nll_grad_hess returns, bit for bit, and
 * this is also the only route to the 4D Hessian.  Sums in long double, one pass in event order.
 * Returns the number of events with P <= 0 (then nll = +inf, everything else NaN), -1 on a bad argument.
 */
int64_t mfo_nll_grad_hess_w(int kind, int64_t n, const double *const *cols, const double *w, const double *lam, double lo,
                            double hi, double *nll, double *grad, double *hess, double *fisher)
{
    const int K = mfo_nparams(kind);
    if (K < 0 || n < 0) return -1;
    long double s0 = 0.0L, sg[MFO_MAXK], sh[MFO_MAXK * MFO_MAXK], sf[MFO_MAXK * MFO_MAXK];
    for (int i = 0; i < K; ++i) sg[i] = 0.0L;
    for (int i = 0; i < K * K; ++i) sh[i] = sf[i] = 0.0L;
    int64_t bad = 0;
    for (int64_t e = 0; e < n; ++e) {
        double g[MFO_MAXK], H[MFO_MAXK * MFO_MAXK];
        const double P = event_hess(kind, cols, e, lam, lo, hi, g, H);
        if (!(P > 0.0)) { ++bad; continue; }
        const long double wi = w ? (long double)w[e] : 1.0L;
        s0 += wi * (long double)log(P);
        for (int i = 0; i < K; ++i) sg[i] += wi * (long double)g[i];
        for (int i = 0; i < K * K; ++i) sh[i] += wi * (long double)H[i];
        for (int i = 0; i < K; ++i)
            for (int j = 0; j < K; ++j) sf[i * K + j] += wi * wi * (long double)(g[i] * g[j]);
    }
    if (bad) {
        *nll = INFINITY;
        for (int i = 0; i < K; ++i) grad[i] = NAN;
        for (int i = 0; i < K * K; ++i) {
            if (hess) hess[i] = NAN;
            if (fisher) fisher[i] = NAN;
        }
        return bad;
    }
    *nll = (double)(-s0);
    for (int i = 0; i < K; ++i) grad[i] = (double)(-sg[i]);
    for (int i = 0; i < K * K; ++i) {
        if (hess) hess[i] = (double)(-sh[i]);
        if (fisher) fisher[i] = (double)sf[i];
    }
    return 0;
}
