// mf_models.cuh — the three PDF families of the hot path: parameter-only constants (S2) and
// the per-event value + gradient body (S3).  SURVEY.md §8(a); Eq. 2 (83-88),
// Eq. 3 (90-100), Eq. 4 (116-118), Listing 5 (351-385).
//
// Notation follows the paper: f = f_sig, mu, sigma = sigma_m, tau = alpha (BASELINE.json
// calls the slope tau), N1 / N2 the two normalisations of Eq. 2, [m_a, m_b] the mass range.
//
// What is NOT the paper's kernel:
//  * value and all K derivatives are produced in one pass in registers (the paper emits
//    one kernel per quantity from its differentiated graph);
//  * the mass mixture is evaluated in ratio form with ONE exponential per event:
//        R   = (G/N1)/(E/N2) = exp(-b0 (m-mu)^2 - tau m + ln(c1/c2))
//        P   = (E/N2) [(1-f) + f R],   ln P = tau m + ln c2 + ln[(1-f) + f R]
//    instead of Eq. 3's b1 exp(..) + b2 exp(..) (two exponentials); b0, c1, c2 and the
//    derivatives of ln N1, ln N2 are the buffered parameter-only terms;
//  * the kernels accumulate model-specific SUMS (mass: the product of the D_i and five moments
//    of u = R/D, r = 1/D) and one thread per evaluation turns them into -ln L and the gradient
//    (M::finish); sum_i tau m_i is an event-only constant times tau;
//  * the eleven angular terms of Listing 4 are merged into nine columns h_0..h_8 with
//    P = h0 + FL h1 + S3 h2 + S4 h3 + S5 h4 + AFB h5 + S7 h6 + S8 h7 + S9 h8.
#pragma once
#include <cmath>
#include <cstdint>

#ifdef __CUDACC__
#include "mf_math.cuh"
#define MF_HD __host__ __device__
#define MF_D __device__ __forceinline__
#else
#define MF_HD
#endif

namespace mf {

constexpr double kPi = 3.141592653589793238462643383279502884;
constexpr double kLnSqrt2Pi = 0.918938533204672741780329736405617639;  // ln sqrt(2 pi)
constexpr double kSqrt2Pi = 2.506628274631000502415765284811045253;
constexpr double kSqrtHalf = 0.707106781186547524400844362104849039;
constexpr double kAngNorm = 9.0 / (32.0 * kPi);                        // 9/(32 pi), Eq. 4
constexpr double kInv8Pi = 1.0 / (8.0 * kPi);

// ------------------------------------------------------------------------------------------
// Parameter-only constants (S2).  One MF_HD implementation: the host runs it once per
// mf_nll_grad call ("calculating these terms only once on the host for each
// parameter update"), the batched-toy kernel runs it once per CTA for its toy's lambda_t.
// ------------------------------------------------------------------------------------------

// Langevin function coth(x) - 1/x without cancellation: continued fraction
// x/(3 + x^2/(5 + x^2/(7 + ...))) for |x| <= 2, closed form beyond.
MF_HD inline double langevin(double x)
{
    const double ax = fabs(x);
    if (ax > 2.0) {
        // coth(x) = 1 + 2/expm1(2x); no cancellation against 1/x here (coth >= 1, 1/x <= 0.5)
        const double cth = 1.0 + 2.0 / expm1(2.0 * ax);
        const double v = cth - 1.0 / ax;
        return x < 0.0 ? -v : v;
    }
    const double x2 = x * x;
    double t = 43.0;  // depth 20: truncation error < 1e-30 for |x| <= 2
    for (int n = 41; n >= 3; n -= 2) t = (double)n + x2 / t;
    return x / t;
}

struct MassConsts {
    double f, omf;   // f_sig, 1 - f_sig
    double mu, tau;
    double nb0;      // -b0 = -1/(2 sigma^2)                       (Eq. 3 b0)
    double lnk;      // ln(c1/c2), c1 = 1/(sqrt(2pi) sigma N1), c2 = 1/N2   (Eq. 3 b1/f, b2/(1-f))
    double lnc2;     // -ln N2
    double is2;      // 1/sigma^2
    double is3;      // 1/sigma^3
    double kmu;      // d ln N1 / d mu
    double ksig;     // 1/sigma + d ln N1 / d sigma
    double ma;       // m_a (reference point for the tau derivative)
    double ktau;     // d ln N2 / d tau - m_a = w [1/2 + Langevin(tau w / 2)/2],  w = m_b - m_a
    // second derivatives of the normalisations (analytic Hessian; MassHessModel)
    double is4;      // 1/sigma^4
    double ct;       // mu - m_a - ktau:  m - d ln N2/d tau = d + ct
    double n1mm, n1ms, n1ss;  // d2 ln N1 / d(mu, sigma)^2
    double n2tt;     // d2 ln N2 / d tau^2 = w^2 L'(tau w / 2) / 4
    // 1.0 if this parameter point allows the event loop's fast path (MassModel::events<E, true>), else 0.0:
    //   * 1 - f >= 1/4, so that D = (1-f) + f R >= 1/4 and the sums over r = 1/D can be derived from those over u = R/D
    //     (f u + (1-f) r = 1 for every event) without amplifying their rounding by more than 4;
    //   * every exponent argument lies in (-700, 69): no clamp in the exponential, D < 2^100, so the product of 8 factors D
    //     cannot leave the normal range and no event can have "P <= 0".
    double fast;
};

// derivative of the Langevin function, 1/x^2 - 1/sinh^2(x) (series below |x| = 0.1: cancellation)
MF_HD inline double langevin_prime(double x)
{
    const double x2 = x * x;
    if (fabs(x) < 0.1)
        return 1.0 / 3.0 + x2 * (-1.0 / 15.0 + x2 * (2.0 / 189.0 + x2 * (-1.0 / 675.0 + x2 * (2.0 / 10395.0))));
    if (fabs(x) > 350.0) return 1.0 / x2;
    const double sh = sinh(x);
    return 1.0 / x2 - 1.0 / (sh * sh);
}

// Returns false if lambda = (f, mu, sigma, tau) is outside the parameter domain
// (non-finite, sigma <= 0, f outside [0,1]).
MF_HD inline bool mass_consts(const double* lam, double ma, double mb, MassConsts& c)
{
    const double f = lam[0], mu = lam[1], sigma = lam[2], tau = lam[3];
    if (!(isfinite(f) && isfinite(mu) && isfinite(sigma) && isfinite(tau))) return false;
    if (!(f >= 0.0 && f <= 1.0) || !(sigma > 0.0)) return false;
    const double is = 1.0 / sigma;
    // N1
    const double za = (mu - ma) * is * kSqrtHalf, zb = (mu - mb) * is * kSqrtHalf;
    const double N1 = 0.5 * (erf(za) - erf(zb));
    // Gaussian density at the range ends: dN1/dmu = g(a) - g(b); dN1/dsigma = [(a-mu)g(a) - (b-mu)g(b)]/sigma
    const double ga = exp(-za * za) * is / kSqrt2Pi, gb = exp(-zb * zb) * is / kSqrt2Pi;
    const double iN1 = 1.0 / N1;
    // N2, cancellation-free (SURVEY §8(c) reading 6)
    const double w = mb - ma;
    const double lnN2 = (tau == 0.0) ? log(w) : tau * ma + log(expm1(tau * w) / tau);
    c.f = f;
    c.omf = 1.0 - f;
    c.mu = mu;
    c.tau = tau;
    c.nb0 = -0.5 * is * is;
    c.lnc2 = -lnN2;
    c.lnk = (-kLnSqrt2Pi - log(sigma) - log(N1)) + lnN2;
    c.is2 = is * is;
    c.is3 = is * is * is;
    c.kmu = (ga - gb) * iN1;
    c.ksig = is + ((ma - mu) * ga - (mb - mu) * gb) * is * iN1;
    c.ma = ma;
    c.ktau = w * (0.5 + 0.5 * langevin(0.5 * tau * w));
    {
        const double da = ma - mu, db = mb - mu, is2 = is * is, is3 = is2 * is;
        const double N1m = ga - gb, N1s = (da * ga - db * gb) * is;
        const double ga_s = ga * (da * da * is3 - is), gb_s = gb * (db * db * is3 - is);
        const double N1mm = (ga * da - gb * db) * is2, N1ms = ga_s - gb_s;
        const double N1ss = (da * ga_s - db * gb_s) * is - (da * ga - db * gb) * is2;
        c.n1mm = N1mm * iN1 - (N1m * iN1) * (N1m * iN1);
        c.n1ms = N1ms * iN1 - (N1m * iN1) * (N1s * iN1);
        c.n1ss = N1ss * iN1 - (N1s * iN1) * (N1s * iN1);
        c.n2tt = 0.25 * w * w * langevin_prime(0.5 * tau * w);
        c.is4 = is2 * is2;
        c.ct = (mu - ma) - c.ktau;
    }
    // The kernels evaluate R = exp(-b0 (m-mu)^2 - tau m + lnk) with a range-restricted exp: refuse
    // parameter points whose normalisations are not representable (N1 or N2 under/overflow) or
    // whose largest possible exponent argument leaves the finite range.
    if (!(isfinite(c.lnk) && isfinite(c.lnc2) && isfinite(c.kmu) && isfinite(c.ksig) && isfinite(c.nb0) &&
          isfinite(c.is3)))
        return false;
    const double mmax = fmax(fabs(ma), fabs(mb));
    if (!(c.lnk + fabs(tau) * mmax < 700.0)) return false;
    // ... and whose most negative one is beyond the range in which mf_exp32 reduces its argument
    const double dmax = fmax(fabs(ma - mu), fabs(mb - mu));
    if (!(-c.nb0 * dmax * dmax + fabs(tau) * mmax + fabs(c.lnk) < 1e12)) return false;
    // bounds of ln R = -b0 d^2 - tau m + lnk over the range: -b0 d^2 <= 0
    const double arg_hi = c.lnk + fabs(tau) * mmax, arg_lo = c.nb0 * dmax * dmax - fabs(tau) * mmax + c.lnk;
#ifdef MF_MASS_NO_FAST
    c.fast = 0.0;  // ablation: always the general path
#else
    c.fast = (c.omf >= 0.25 && arg_hi < 69.0 && arg_lo > -700.0) ? 1.0 : 0.0;
#endif
    return true;
}

struct AngularConsts {
    double a[8];  // FL, S3, S4, S5, AFB, S7, S8, S9 (PAPER.md:369-376 order)
};

MF_HD inline bool angular_consts(const double* lam, AngularConsts& c)
{
    bool ok = true;
    for (int k = 0; k < 8; ++k) {
        c.a[k] = lam[k];
        ok = ok && isfinite(lam[k]);
    }
    return ok;
}

struct FourDConsts {
    MassConsts m;
    double a[8];                // angular coefficients
    double cl1, cl2, ck1, ck2;  // Legendre coefficients of the background
    double kappa;               // (1-f)/(8 pi): (1-f) L = kappa * ll * lk with ll = 2 l(cos theta_l) etc.
};

MF_HD inline bool fourd_consts(const double* lam, double ma, double mb, FourDConsts& c)
{
    bool ok = mass_consts(lam, ma, mb, c.m);
    for (int k = 0; k < 8; ++k) {
        c.a[k] = lam[4 + k];
        ok = ok && isfinite(lam[4 + k]);
    }
    c.cl1 = lam[12];
    c.cl2 = lam[13];
    c.ck1 = lam[14];
    c.ck2 = lam[15];
    ok = ok && isfinite(c.cl1) && isfinite(c.cl2) && isfinite(c.ck1) && isfinite(c.ck2);
    c.kappa = ok ? c.m.omf * kInv8Pi : 0.0;
    return ok;
}

#ifdef __CUDACC__
// ------------------------------------------------------------------------------------------
// Per-event bodies (S3) and the per-call finish.
//
// The kernels keep NACC running sums per thread.  Sum 0 is always ln of the product of the factor
// of P_i that needs a logarithm (LogProd, mf_math.cuh: sum of logs = log of the product, one
// logarithm per thread).  Sums 1..NACC-1 are model specific.  After the fixed-order reduction ONE
// thread per evaluation calls M::finish(), which turns the NACC sums into -ln L and the K gradient
// components using the parameter-only constants and the event-only constant sum_m = sum_i m_i
// (precomputed once per dataset: ln P_i contains tau m_i, so its sum needs no
// per-event work).  `bad` counts events whose P is not a positive normal number (SURVEY.md §8(c)
// reading 15); when it ends up non-zero the sums are discarded, so they are accumulated
// unconditionally.  PRED = true is the ragged-tail variant: lanes with valid == false contribute
// exactly 0 (reading 10).  t_lane is this lane's entry of the exp table (mf_exp32).
// ------------------------------------------------------------------------------------------

// a b - c d with the rounding errors of both products recovered (the two terms nearly cancel at a
// likelihood maximum)
MF_D double diff_of_products(double a, double b, double c, double d)
{
    const double p = a * b, q = c * d;
    const double ep = fma(a, b, -p), eq = fma(c, d, -q);
    return (p - q) + (ep - eq);
}

struct MassModel {
    static constexpr int K = 4;
    static constexpr int NCOL = 1;  // m
    static constexpr int NOUT = K + 1;  // -ln L, gradient
    static constexpr int NACC = 6;  // ln prod D, and with u = (G/N1)/P', r = (E/N2)/P' (P' = P N2 e^{-tau m}, d = m - mu):
                                    // sum u, sum r, sum u d, sum u d^2, sum r d
    // tuning knobs (defaults = the measured best on B200)
#ifndef MF_MASS_EVENTS
#define MF_MASS_EVENTS 8
#endif
#ifndef MF_MASS_GRID
#define MF_MASS_GRID 2
#endif
#ifndef MF_MASS_RESIDENT
#define MF_MASS_RESIDENT 2
#endif
    static constexpr int EVENTS_PER_CALL = MF_MASS_EVENTS;  // independent events interleaved per thread (a 256-event group is 8 per thread)
    static constexpr int CTAS_PER_SM = MF_MASS_GRID;    // grid of a lone (synchronous) evaluation: CTAs per SM
#ifndef MF_MASS_BATCH_RESIDENT
#define MF_MASS_BATCH_RESIDENT 4
#endif
#ifndef MF_MASS_BATCH_BLOCK
#define MF_MASS_BATCH_BLOCK 128
#endif
    static constexpr int BATCH_BLOCK = MF_MASS_BATCH_BLOCK;  // threads per CTA of the batched kernel
    static constexpr int BATCH_RESIDENT_CTAS = MF_MASS_BATCH_RESIDENT;  // the batched kernel: more, smaller-budget CTAs
    static constexpr int RESIDENT_CTAS = MF_MASS_RESIDENT;  // register budget: CTAs of the next evaluation co-reside under PDL
    using Consts = MassConsts;

    template <bool PRED>
    static MF_D void event(const double* x, const Consts& c, double* acc, LogProd& lp, unsigned& bad, bool valid,
                           double t_lane)
    {
        const double m = x[0];
        const double d = m - c.mu;
        const double t = d * d;
        // ln R = -b0 d^2 - tau m + ln(c1/c2)
        const double arg = fma(c.nb0, t, fma(-c.tau, m, c.lnk));  // < 700 by the check in mass_consts
        const double R = mf_exp32(arg, t_lane);  // (G/N1)/(E/N2)
        const double D = fma(c.f, R, c.omf);     // P N2 e^{-tau m} = (1-f) + f R
        const double r = mf_rcp(D);
        const double u = R * r;
        if (!PRED || valid) {
            lp.mul(D, bad);
            acc[1] += u;
            acc[2] += r;
            acc[3] = fma(u, d, acc[3]);
            acc[4] = fma(u, t, acc[4]);
            acc[5] = fma(r, d, acc[5]);
        }
    }

    static constexpr bool HAS_FAST = true;
    static MF_D bool is_fast(const Consts& c) { return c.fast != 0.0; }

    // E full events at once (the body of the event loop), written operation by operation across the E
    // events so that the instruction stream is interleaved as issued and constants are shared operands.
    // FAST (Consts::fast, decided per parameter point where the constants are made): D is known to lie in [1/4, 2^100], so
    //   * the E factors are multiplied by a tree and enter the running product as ONE bounded factor: one exponent
    //     extraction per E events (the caller's renorm()) instead of one per event, and no "P <= 0" test;
    //   * the exponential needs no clamp;
    //   * sum r and sum r d are not accumulated: f u + (1-f) r = 1 gives them from sum u, sum u d and the event-only
    //     constant sum_i m_i (finish).  24 fp64 instructions per event instead of 26.
    template <int E, bool FAST>
    static MF_D void events(const double (&m)[E], const Consts& c, double* acc, LogProd& lp, unsigned& bad, double t_lane)
    {
        double d[E], t[E], arg[E], R[E], D[E], r[E], u[E];
#pragma unroll
        for (int e = 0; e < E; ++e) d[e] = m[e] - c.mu;
#pragma unroll
        for (int e = 0; e < E; ++e) arg[e] = fma(-c.tau, m[e], c.lnk);
#pragma unroll
        for (int e = 0; e < E; ++e) t[e] = d[e] * d[e];
#pragma unroll
        for (int e = 0; e < E; ++e) arg[e] = fma(c.nb0, t[e], arg[e]);
        mf_exp32_v<E, FAST>(arg, t_lane, R);
#pragma unroll
        for (int e = 0; e < E; ++e) D[e] = fma(c.f, R[e], c.omf);
        if constexpr (FAST) {
            static_assert(E <= 8 && (E & (E - 1)) == 0, "the product of E factors below 2^100 must stay below 2^900");
            // product tree of the E factors: P[l][i] = product of factors i 2^l .. (i+1) 2^l - 1
            constexpr int L = (E == 8) ? 3 : (E == 4) ? 2 : (E == 2) ? 1 : 0;  // levels of the tree
            double P[4][E];
#pragma unroll
            for (int e = 0; e < E; ++e) P[0][e] = D[e];
#pragma unroll
            for (int l = 0; l < L; ++l)
#pragma unroll
                for (int i = 0; i < (E >> (l + 1)); ++i) P[l + 1][i] = P[l][2 * i] * P[l][2 * i + 1];
            lp.mul_bounded(P[L][0]);
            // ONE Newton reciprocal for the E events, of the root of the tree, pushed back down: the reciprocal of a node is
            // its sibling's product times the parent's reciprocal (2 - 2/E multiplications per event instead of a 3-DFMA
            // Newton step, a MUFU and a register move each)
            double I[4][E];
            I[L][0] = mf_rcp(P[L][0]);
#pragma unroll
            for (int l = L; l > 0; --l)
#pragma unroll
                for (int i = 0; i < (E >> l); ++i) {
                    I[l - 1][2 * i] = P[l - 1][2 * i + 1] * I[l][i];
                    I[l - 1][2 * i + 1] = P[l - 1][2 * i] * I[l][i];
                }
#pragma unroll
            for (int e = 0; e < E; ++e) u[e] = R[e] * I[0][e];
#pragma unroll
            for (int e = 0; e < E; ++e) {
                acc[1] += u[e];
                acc[3] = fma(u[e], d[e], acc[3]);
                acc[4] = fma(u[e], t[e], acc[4]);
            }
        } else {
#pragma unroll
            for (int e = 0; e < E; ++e) r[e] = mf_rcp(D[e]);
#pragma unroll
            for (int e = 0; e < E; ++e) u[e] = R[e] * r[e];
#pragma unroll
            for (int e = 0; e < E; ++e) {
                lp.mul(D[e], bad);
                acc[1] += u[e];
                acc[2] += r[e];
                acc[3] = fma(u[e], d[e], acc[3]);
                acc[4] = fma(u[e], t[e], acc[4]);
                acc[5] = fma(r[e], d[e], acc[5]);
            }
        }
    }

    // ln P = tau m - ln N2 + ln D
    // d ln P/df = u - r;  d/dmu = f u (d/sigma^2 - kmu);  d/dsigma = f u (d^2/sigma^3 - ksig);
    // d/dtau = (1-f) r (m - m_a - ktau) = (1-f) r (d + mu - m_a - ktau)
    // sum_m = (hi, lo) of the event-only constant sum_i m_i.
    static MF_D void finish_general(const Consts& c, const double* s, double n, double2 sum_m, double* out)
    {
        out[0] = -(s[0] + fma(c.tau, sum_m.x, fma(c.tau, sum_m.y, n * c.lnc2)));
        out[1] = -(s[1] - s[2]);
        out[2] = -c.f * diff_of_products(c.is2, s[3], c.kmu, s[1]);
        out[3] = -c.f * diff_of_products(c.is3, s[4], c.ksig, s[1]);
        out[4] = -c.omf * fma((c.mu - c.ma) - c.ktau, s[2], s[5]);
    }

    // Fast path: s[2] (sum r) and s[5] (sum r d) were not accumulated.  With f u + (1-f) r = 1 for every event:
    //   (1-f) sum r   = N - f sum u            ->  sum u - sum r = (sum u - N) / (1-f)
    //   (1-f) sum r d = sum d - f sum u d,   sum d = sum_i m_i - N mu  (double-double: the two terms nearly cancel)
    static MF_D void finish(const Consts& c, const double* s, double n, double2 sum_m, double* out)
    {
        if (c.fast == 0.0) {
            finish_general(c, s, n, sum_m, out);
            return;
        }
        const double Su = s[1], Sud = s[3], Sut = s[4];
        const double p = n * c.mu, pe = fma(n, c.mu, -p);       // N mu = p + pe exactly
        const double Sd = (sum_m.x - p) + (sum_m.y - pe);
        out[0] = -(s[0] + fma(c.tau, sum_m.x, fma(c.tau, sum_m.y, n * c.lnc2)));
        out[1] = -(Su - n) / c.omf;
        out[2] = -c.f * diff_of_products(c.is2, Sud, c.kmu, Su);
        out[3] = -c.f * diff_of_products(c.is3, Sut, c.ksig, Su);
        out[4] = -fma(c.ct, fma(-c.f, Su, n), fma(-c.f, Sud, Sd));
    }
};

// ------------------------------------------------------------------------------------------
// Mass model with the analytic Hessian (value, gradient and
// Hessian in one evaluation give Newton convergence in 2-3 iterations).  With w = f u the signal
// weight, 1 - w = (1-f) r, A = ln R and q = m - d ln N2/d tau = d + ct:
//   l_ff = -(u - r)^2                       l_f,theta = u r A_theta            (A_tau = -q)
//   l_theta,theta' = w (1-w) A_theta A_theta' + w A_theta,theta'   (- (1-w) d2 ln N2/dtau^2 for tau,tau)
// A_mu = d/s^2 - kmu, A_sigma = d^2/s^3 - ksig are polynomials in d, so the Hessian needs seven more
// moment sums: sum u^2, r^2, z, z d, z d^2, z d^3, z d^4 with z = u r.  36 fp64 instructions per event.
// Output: -ln L, gradient[4], then the upper triangle ff, fm, fs, ft, mm, ms, mt, ss, st, tt of d2(-ln L).
// ------------------------------------------------------------------------------------------
struct MassHessModel {
    static constexpr int K = 4;
    static constexpr int NCOL = 1;
    static constexpr int NOUT = 1 + 4 + 10;
    static constexpr int NACC = 13;
    static constexpr int EVENTS_PER_CALL = 4;  // 4 events at once (13 sums leave fewer registers)
    static constexpr int CTAS_PER_SM = 2;
    static constexpr int RESIDENT_CTAS = 2;
    static constexpr int BATCH_RESIDENT_CTAS = 4;
    static constexpr int BATCH_BLOCK = 128;
    using Consts = MassConsts;
    static constexpr bool HAS_FAST = true;
    static MF_D bool is_fast(const Consts& c) { return c.fast != 0.0; }

    // FAST: as MassModel's, but only the integer side (no clamp, one exponent extraction per E events, no "P <= 0" test);
    // all 13 sums are accumulated.
    template <int E, bool FAST>
    static MF_D void events(const double (&m)[E], const Consts& c, double* acc, LogProd& lp, unsigned& bad, double t_lane)
    {
        double d[E], t[E], arg[E], R[E], D[E], r[E], u[E], z[E];
#pragma unroll
        for (int e = 0; e < E; ++e) d[e] = m[e] - c.mu;
#pragma unroll
        for (int e = 0; e < E; ++e) arg[e] = fma(-c.tau, m[e], c.lnk);
#pragma unroll
        for (int e = 0; e < E; ++e) t[e] = d[e] * d[e];
#pragma unroll
        for (int e = 0; e < E; ++e) arg[e] = fma(c.nb0, t[e], arg[e]);
        mf_exp32_v<E, FAST>(arg, t_lane, R);
#pragma unroll
        for (int e = 0; e < E; ++e) D[e] = fma(c.f, R[e], c.omf);
#pragma unroll
        for (int e = 0; e < E; ++e) r[e] = mf_rcp(D[e]);
#pragma unroll
        for (int e = 0; e < E; ++e) u[e] = R[e] * r[e];
#pragma unroll
        for (int e = 0; e < E; ++e) z[e] = u[e] * r[e];
        if constexpr (FAST) {
            static_assert(E <= 8, "the product of E factors below 2^100 must stay below 2^900");
            double P[E];
#pragma unroll
            for (int e = 0; e < E; ++e) P[e] = D[e];
#pragma unroll
            for (int s = 1; s < E; s <<= 1)
#pragma unroll
                for (int e = 0; e + s < E; e += 2 * s) P[e] *= P[e + s];
            lp.mul_bounded(P[0]);
        }
#pragma unroll
        for (int e = 0; e < E; ++e) {
            if constexpr (!FAST) lp.mul(D[e], bad);
            acc[1] += u[e];
            acc[2] += r[e];
            acc[3] = fma(u[e], d[e], acc[3]);
            acc[4] = fma(u[e], t[e], acc[4]);
            acc[5] = fma(r[e], d[e], acc[5]);
            acc[6] = fma(u[e], u[e], acc[6]);
            acc[7] = fma(r[e], r[e], acc[7]);
            acc[8] += z[e];
            const double zd = z[e] * d[e];
            acc[9] += zd;
            acc[10] = fma(zd, d[e], acc[10]);
            acc[11] = fma(zd, t[e], acc[11]);
            acc[12] = fma(z[e] * t[e], t[e], acc[12]);
        }
    }

    template <bool PRED>
    static MF_D void event(const double* x, const Consts& c, double* acc, LogProd& lp, unsigned& bad, bool valid,
                           double t_lane)
    {
        // every lane evaluates (the exponential shuffles across the whole warp); invalid lanes discard the result
        double tmp[NACC];
#pragma unroll
        for (int k = 0; k < NACC; ++k) tmp[k] = 0.0;
        LogProd lp2;
        unsigned bad2 = 0;
        const double m1[1] = {x[0]};
        events<1, false>(m1, c, tmp, lp2, bad2, t_lane);
        if (!PRED || valid) {
#pragma unroll
            for (int k = 1; k < NACC; ++k) acc[k] += tmp[k];
            lp.prod *= lp2.prod;
            lp.esum += lp2.esum;
            bad += bad2;
        }
    }

    static MF_D void finish(const Consts& c, const double* s, double n, double2 sum_m, double* out)
    {
        MassModel::finish_general(c, s, n, sum_m, out);
        const double Su = s[1], Sr = s[2], Sud = s[3], Sud2 = s[4];
        const double Suu = s[6], Srr = s[7], Sz = s[8], Szd = s[9], Szd2 = s[10], Szd3 = s[11], Szd4 = s[12];
        const double fo = c.f * c.omf, ct = c.ct, kmu = c.kmu, ksig = c.ksig, is2 = c.is2, is3 = c.is3;
        const double Szq = fma(ct, Sz, Szd);          // sum z q
        const double Szdq = fma(ct, Szd, Szd2);       // sum z d q
        const double Szd2q = fma(ct, Szd2, Szd3);     // sum z d^2 q
        const double l_ff = -((Suu - 2.0 * Sz) + Srr);
        const double l_fm = diff_of_products(is2, Szd, kmu, Sz);
        const double l_fs = diff_of_products(is3, Szd2, ksig, Sz);
        const double l_ft = -Szq;
        const double l_mm = fo * (is2 * is2 * Szd2 - 2.0 * is2 * kmu * Szd + kmu * kmu * Sz) - c.f * (is2 + c.n1mm) * Su;
        const double l_ms = fo * (is2 * is3 * Szd3 - is2 * ksig * Szd - kmu * is3 * Szd2 + kmu * ksig * Sz) -
                            c.f * (2.0 * is3 * Sud + c.n1ms * Su);
        const double l_mt = -fo * diff_of_products(is2, Szdq, kmu, Szq);
        const double l_ss = fo * (is3 * is3 * Szd4 - 2.0 * is3 * ksig * Szd2 + ksig * ksig * Sz) +
                            c.f * ((is2 - c.n1ss) * Su - 3.0 * c.is4 * Sud2);
        const double l_st = -fo * diff_of_products(is3, Szd2q, ksig, Szq);
        const double l_tt = fo * (Szd2 + 2.0 * ct * Szd + ct * ct * Sz) - c.omf * c.n2tt * Sr;
        out[5] = -l_ff;
        out[6] = -l_fm;
        out[7] = -l_fs;
        out[8] = -l_ft;
        out[9] = -l_mm;
        out[10] = -l_ms;
        out[11] = -l_mt;
        out[12] = -l_ss;
        out[13] = -l_st;
        out[14] = -l_tt;
    }
};

struct AngularModel {
    static constexpr bool HAS_FAST = false;
    static constexpr int K = 8;
    static constexpr int NCOL = 9;  // h_0..h_8 (cached, already times 9/(32 pi))
    static constexpr int NOUT = K + 1;
    static constexpr int NACC = 9;  // ln prod P, sum h_k / P
    static constexpr int ITEMS_PER_ITER = 1;  // memory bound: depth comes from the prefetched next item
    static constexpr int PREFETCH = 0;
    static constexpr int CTAS_PER_SM = 2;
    static constexpr int RESIDENT_CTAS = 2;
    static constexpr int BATCH_RESIDENT_CTAS = 2;
    static constexpr int BATCH_BLOCK = 256;
    using Consts = AngularConsts;

    template <bool PRED>
    static MF_D void event(const double* x, const Consts& c, double* acc, LogProd& lp, unsigned& bad, bool valid,
                           double)
    {
        double P = fma(c.a[0], x[1], x[0]);
#pragma unroll
        for (int k = 1; k < 8; ++k) P = fma(c.a[k], x[1 + k], P);
        const double r = mf_rcp(P);
        if (!PRED || valid) {
            lp.mul(P, bad);
#pragma unroll
            for (int k = 0; k < 8; ++k) acc[1 + k] = fma(x[1 + k], r, acc[1 + k]);
        }
    }

    static MF_D void finish(const Consts&, const double* s, double, double2, double* out)
    {
#pragma unroll
        for (int k = 0; k < NACC; ++k) out[k] = -s[k];
    }
};

// Angular model with the analytic Hessian.  P is linear in its coefficients, so with the score components
// s_k = h_k / P:  d2 ln P / da_k da_l = -s_k s_l, i.e. d2(-ln L) = sum_i s_k s_l (positive semi-definite: -ln L is convex).
// 36 more sums than AngularModel; still one pass over the nine cached columns.
// Output: -ln L, gradient[8], then the upper triangle (k <= l, row by row) of d2(-ln L).
struct AngularHessModel {
    static constexpr bool HAS_FAST = false;
    static constexpr int K = 8;
    static constexpr int NCOL = 9;
    static constexpr int NOUT = 1 + 8 + 36;
    static constexpr int NACC = 1 + 8 + 36;
    static constexpr int ITEMS_PER_ITER = 1;
    static constexpr int PREFETCH = 0;
    static constexpr int CTAS_PER_SM = 1;
    static constexpr int RESIDENT_CTAS = 1;  // 45 sums + two 9-column register buffers
    static constexpr int BATCH_RESIDENT_CTAS = 1;
    static constexpr int BATCH_BLOCK = 256;
    using Consts = AngularConsts;

    template <bool PRED>
    static MF_D void event(const double* x, const Consts& c, double* acc, LogProd& lp, unsigned& bad, bool valid,
                           double)
    {
        double P = fma(c.a[0], x[1], x[0]);
#pragma unroll
        for (int k = 1; k < 8; ++k) P = fma(c.a[k], x[1 + k], P);
        const double r = mf_rcp(P);
        if (!PRED || valid) {
            lp.mul(P, bad);
            double s[8];
#pragma unroll
            for (int k = 0; k < 8; ++k) {
                s[k] = x[1 + k] * r;
                acc[1 + k] += s[k];
            }
            int q = 9;
#pragma unroll
            for (int k = 0; k < 8; ++k)
#pragma unroll
                for (int l = k; l < 8; ++l, ++q) acc[q] = fma(s[k], s[l], acc[q]);
        }
    }

    static MF_D void finish(const Consts&, const double* s, double, double2, double* out)
    {
#pragma unroll
        for (int k = 0; k < 9; ++k) out[k] = -s[k];
#pragma unroll
        for (int k = 9; k < NOUT; ++k) out[k] = s[k];
    }
};

struct FourDModel {
    static constexpr bool HAS_FAST = false;
    static constexpr int K = 16;
    static constexpr int NCOL = 12;  // m, cos theta_l, cos theta_K, h_0..h_8
    static constexpr int NOUT = K + 1;
    static constexpr int NACC = 17;  // ln prod D, then sum d ln P / d lambda_k
    static constexpr int ITEMS_PER_ITER = 1;
    static constexpr int PREFETCH = 0;
    static constexpr int RESIDENT_CTAS = 1;
    static constexpr int BATCH_RESIDENT_CTAS = 1;
    static constexpr int BATCH_BLOCK = 256;
    static constexpr int CTAS_PER_SM = 2;  // grid of the shared-memory-staged kernel (the register-buffer kernel, 255 registers, 1 resident CTA/SM, serves only n < 1024)
    using Consts = FourDConsts;

    template <bool PRED>
    static MF_D void event(const double* x, const Consts& c, double* acc, LogProd& lp, unsigned& bad, bool valid,
                           double t_lane)
    {
        const MassConsts& q = c.m;
        const double m = x[0], cl = x[1], ck = x[2];
        const double* h = x + 3;
        // angular signal A(Omega)
        double A = fma(c.a[0], h[1], h[0]);
#pragma unroll
        for (int k = 1; k < 8; ++k) A = fma(c.a[k], h[1 + k], A);
        // background angles: ll = 2 l(cos theta_l), lk = 2 l(cos theta_K); L = ll lk / (8 pi)
        const double p2l = fma(1.5 * cl, cl, -0.5), p2k = fma(1.5 * ck, ck, -0.5);
        const double ll = fma(c.cl2, p2l, fma(c.cl1, cl, 1.0));
        const double lk = fma(c.ck2, p2k, fma(c.ck1, ck, 1.0));
        const double d = m - q.mu;
        const double t = d * d;
        const double arg = fma(q.nb0, t, fma(-q.tau, m, q.lnk));  // < 700 by the check in mass_consts
        const double R = mf_exp32(arg, t_lane);   // (G/N1)/(E/N2)
        const double omfL = c.kappa * (ll * lk);  // (1-f) L
        const double fR = q.f * R;
        const double D = fma(fR, A, omfL);        // P N2 e^{-tau m}
        const double r = mf_rcp(D);
        const double ws = fR * A * r;             // f (G/N1) A / P
        const double wb = omfL * r;               // (1-f)(E/N2) L / P
        const double gf = fma(R * A, r, -(ll * lk) * kInv8Pi * r);
        const double hmu = fma(d, q.is2, -q.kmu);
        const double hsig = fma(t, q.is3, -q.ksig);
        const double htau = (m - q.ma) - q.ktau;
        const double qa = fR * r;                 // f (G/N1) / P
        const double qb = c.kappa * r;            // (1-f)(E/N2)/(8 pi P)
        const double qbl = qb * lk, qbk = qb * ll;
        if (!PRED || valid) {
            lp.mul(D, bad);
            acc[1] += gf;
            acc[2] = fma(ws, hmu, acc[2]);
            acc[3] = fma(ws, hsig, acc[3]);
            acc[4] = fma(wb, htau, acc[4]);
#pragma unroll
            for (int k = 0; k < 8; ++k) acc[5 + k] = fma(qa, h[1 + k], acc[5 + k]);
            acc[13] = fma(qbl, cl, acc[13]);
            acc[14] = fma(qbl, p2l, acc[14]);
            acc[15] = fma(qbk, ck, acc[15]);
            acc[16] = fma(qbk, p2k, acc[16]);
        }
    }

    // ln P = tau m - ln N2 + ln D
    static MF_D void finish(const Consts& c, const double* s, double n, double2 sum_m, double* out)
    {
        out[0] = -(s[0] + fma(c.m.tau, sum_m.x, fma(c.m.tau, sum_m.y, n * c.m.lnc2)));
#pragma unroll
        for (int k = 1; k < NACC; ++k) out[k] = -s[k];
    }
};
#endif  // __CUDACC__

}  // namespace mf
