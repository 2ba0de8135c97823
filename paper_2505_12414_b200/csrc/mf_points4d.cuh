// mf_points4d.cuh — many parameter points on ONE 4D dataset in a single pass over the data, the
// counterpart of mf_points.cuh for the mass x angular model (BASELINE.json configs[3]).
//
// Per (point p, event e) pair the mass part needs an exponential (mu, sigma, tau differ per point), so unlike the angular
// model the pair is not a pure contraction; but everything around the exponential is:
//     A[p][e]   = h0(e) + sum_k a_pk h_k(e)                       [M x 8] . [8 x N]     (as mf_points.cuh)
//     LL[p][e]  = 1 + cl1_p cos(theta_l) + cl2_p P2(cos theta_l)   [M x 3] . [3 x N]
//     LK[p][e]  = kappa_p (1 + ck1_p cos(theta_K) + ck2_p P2(..))   [M x 3] . [3 x N]     kappa = (1-f)/(8 pi)
//     R'        = exp(nb0 d^2 - tau m' + q0),  d = m' - mu'        per pair, 15 fp64 instructions (q0 carries ln f: R' = f R)
//     D         = R' A + LL LK  ( = P N2 e^{-tau m}),  r = 1/D
//     G_a[p][k] = sum_e (R' r) h_k(e),  G_cl[p][.] = sum_e (r LK) [cos, P2](theta_l),  G_ck[p][.] = sum_e (r LL) [cos, P2](theta_K)
// run as DMMA m8n8k4 on 8 points x 8 events (4 + 6 per tile), in the accumulator layout of mf_points.cuh: lane (g, t) holds
// point g and events 2t, 2t+1, and the weights R' r, r LK, r LL it has just computed are the A operands of the second
// contractions.  The four mass-parameter sums (sum ws, sum ws h_mu, sum ws h_sigma, sum wb h_tau) stay per-thread FMA
// accumulators of SIGNED per-event terms: written as moments (sum ws m'^k) they would each carry the rounding of a sum of
// 1e2..1e7 where the gradient is the 1e-9-accurate difference of two of them.
// m' = m - mref with mref the middle of the mass range (an event-only shift that keeps nb0 d^2 small enough to add to).
#pragma once
#include "mf_points.cuh"

namespace mf {

constexpr int kP4PointConsts = 4;   // per point, in shared memory: mu', nb0, tau, q0
constexpr int kP4StageDoubles = 12;  // per lane and stage: f1[2], f2, f0, cl(fg), ck(fg), c2, m2 = 96 bytes
constexpr int kP4FinishConsts = 12;  // per point, for the combine kernel: 1/f, 1/(1-f), tau, lnc2, kappa, is2, kmu, is3, ksig,
                                     // mu - m_a - ktau, m_a + ktau, spare

struct FourDPointsArgs {
    const double* col[12];       // m, cos theta_l, cos theta_K, h_0..h_8
    int64_t n, n_pad;
    double mref;
    const double* coef;          // device [n_points][16] lambda (angular coefficients at [4..12), Legendre at [12..16))
    const double* pconst;        // device [n_points][kP4PointConsts]
    int n_points;
    double* partials;            // [n_points][17][G]
    unsigned* bad_partials;      // [n_points][G]
};

// Calls of up to kP4InlinePoints points carry their per-point data in the kernels' parameter blocks (as the angular kernel's,
// mf_points.cuh): no copy between such a call and the previous kernel on the stream, both kernels launched programmatically.
constexpr int kP4InlinePoints = 96;
struct FourDPointsInlineArgs {
    FourDPointsArgs a;
    double coef[kP4InlinePoints * 16];
    double pconst[kP4InlinePoints * kP4PointConsts];
};

template <int NPB>
__device__ __forceinline__ void fourd_points_mma_body(const FourDPointsArgs& a, const double* __restrict__ coef,
                                                      const double* __restrict__ pconst);

template <int NPB>
__global__ void __launch_bounds__(kBlock, 2) fourd_points_mma_kernel(const __grid_constant__ FourDPointsArgs a)
{
    fourd_points_mma_body<NPB>(a, a.coef, a.pconst);
}

template <int NPB>
__global__ void __launch_bounds__(kBlock, 2) fourd_points_mma_inline_kernel(const __grid_constant__ FourDPointsInlineArgs ia)
{
    fourd_points_mma_body<NPB>(ia.a, ia.coef, ia.pconst);
}

template <int NPB>
__device__ __forceinline__ void fourd_points_mma_body(const FourDPointsArgs& a, const double* __restrict__ coef,
                                                      const double* __restrict__ pconst)
{
    pdl_launch_dependents();
    // dynamic shared memory: the per-lane staging of the event fragments (two stages, filled by cp.async: loads in flight cost
    // no registers), reused after the event loop for the cross-warp reduction
    extern __shared__ __align__(16) unsigned char p4_raw[];
    double (*stg)[kBlock][kP4StageDoubles] = reinterpret_cast<double (*)[kBlock][kP4StageDoubles]>(p4_raw);
    double (*red)[NPB][8][17] = reinterpret_cast<double (*)[NPB][8][17]>(p4_raw);
    static_assert(sizeof(double) * kWarps * NPB * 8 * 17 <= sizeof(double) * 2 * kBlock * kP4StageDoubles, "reduction fits the staging area");
    __shared__ unsigned red_bad[kWarps][NPB][8];
    __shared__ double s_pc[NPB * 8][kP4PointConsts];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int fg = lane >> 2, ft = lane & 3;
    const int64_t G = gridDim.x;
    const int p0 = blockIdx.y * (8 * NPB);
    for (int i = threadIdx.x; i < NPB * 8 * kP4PointConsts; i += kBlock) {
        const int p = p0 + i / kP4PointConsts;
        (&s_pc[0][0])[i] = (p < a.n_points) ? pconst[(int64_t)p0 * kP4PointConsts + i] : 0.0;
    }
    // A fragments of the first contractions: lane (fg, ft) holds, for point p = p0 + 8 pb + fg,
    //   ca[pb][kk] coefficient of h_{1 + 4 kk + ft};  cl_[pb] = (1, cl1, cl2, 0)[ft];  ck_[pb] = kappa (1, ck1, ck2, 0)[ft]
    double ca[NPB][2], cll[NPB], clk[NPB];
#pragma unroll
    for (int pb = 0; pb < NPB; ++pb) {
        const int p = p0 + 8 * pb + fg;
        const bool live = p < a.n_points;
        const double* lam = coef + (int64_t)(live ? p : 0) * 16;
#pragma unroll
        for (int kk = 0; kk < 2; ++kk) ca[pb][kk] = live ? lam[4 + 4 * kk + ft] : 0.0;
        const double kappa = live ? (1.0 - lam[0]) * kInv8Pi : 0.0;
        cll[pb] = (ft == 0) ? 1.0 : (ft == 3 || !live) ? 0.0 : lam[11 + ft];
        clk[pb] = (ft == 0) ? kappa : (ft == 3 || !live) ? 0.0 : kappa * lam[13 + ft];
    }
    __syncthreads();
    double gA[NPB][2], gL[NPB][2], gK[NPB][2];  // tiles: angular gradient; r LK x (cl, P2l, ...); r LL x (.., .., ck, P2k)
    double ams[NPB][3];                         // per-thread: sum ws, ws d, ws d^2 (d = m - mu)
    LogProd lp[NPB];
    unsigned bad[NPB];
#pragma unroll
    for (int pb = 0; pb < NPB; ++pb) {
        gA[pb][0] = gA[pb][1] = gL[pb][0] = gL[pb][1] = gK[pb][0] = gK[pb][1] = 0.0;
        ams[pb][0] = ams[pb][1] = ams[pb][2] = 0.0;
        bad[pb] = 0;
    }
    const double t_lane = mf_exp32_lane_entry();
    const int64_t n_groups = a.n_pad / 8, step = G * kWarps;
    struct Frag {
        double f1[2];     // h_{1 + 4 kk + ft}(event fg)
        double2 f2, f0;   // h_{1 + fg}(events 2 ft, 2 ft + 1); h_0(events 2 ft, 2 ft + 1)
        double bl, bk;    // (1, cos theta_l, P2, 0)[ft] and (1, cos theta_K, P2, 0)[ft] at event fg
        double2 x2;       // second-contraction B for the Legendre gradients: column fg of (cl, P2l, ck, P2k, 0..) at events 2 ft, 2 ft + 1
        double2 m2;       // m' at events 2 ft, 2 ft + 1
    };
    // issue: this lane's raw values of group grp -> stage st (asynchronous copies); fetch: stage st -> fragments
    auto issue = [&](int64_t grp, int st) {
        const int64_t e0 = grp * 8;
        const unsigned dst = (unsigned)__cvta_generic_to_shared(&stg[st][threadIdx.x][0]);
        auto cp8 = [&](int slot, const double* src) {
            asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(dst + 8u * slot), "l"(src) : "memory");
        };
        auto cp16 = [&](int slot, const double* src) {
            asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"(dst + 8u * slot), "l"(src) : "memory");
        };
        cp8(0, a.col[4 + ft] + e0 + fg);
        cp8(1, a.col[8 + ft] + e0 + fg);
        cp16(2, a.col[4 + fg] + e0 + 2 * ft);
        cp16(4, a.col[3] + e0 + 2 * ft);
        cp8(6, a.col[1] + e0 + fg);
        cp8(7, a.col[2] + e0 + fg);
        cp16(8, a.col[(fg & 2) ? 2 : 1] + e0 + 2 * ft);   // cl (fg 0, 1) or ck (fg 2, 3)
        cp16(10, a.col[0] + e0 + 2 * ft);
        asm volatile("cp.async.commit_group;" ::: "memory");
    };
    auto fetch = [&](int st, Frag& f) {
        const double* q = &stg[st][threadIdx.x][0];
        f.f1[0] = q[0];
        f.f1[1] = q[1];
        f.f2 = *reinterpret_cast<const double2*>(q + 2);
        f.f0 = *reinterpret_cast<const double2*>(q + 4);
        const double cl = q[6], ck = q[7];
        f.bl = (ft == 0) ? 1.0 : (ft == 1) ? cl : (ft == 2) ? fma(1.5 * cl, cl, -0.5) : 0.0;
        f.bk = (ft == 0) ? 1.0 : (ft == 1) ? ck : (ft == 2) ? fma(1.5 * ck, ck, -0.5) : 0.0;
        const double2 c2 = *reinterpret_cast<const double2*>(q + 8);
        const double2 q2 = make_double2(fma(1.5 * c2.x, c2.x, -0.5), fma(1.5 * c2.y, c2.y, -0.5));
        f.x2 = (fg >= 4) ? make_double2(0.0, 0.0) : (fg & 1) ? q2 : c2;
        const double2 mm = *reinterpret_cast<const double2*>(q + 10);
        f.m2 = make_double2(mm.x - a.mref, mm.y - a.mref);
    };
    auto process = [&](int64_t grp, const Frag& f) {
        const bool masked = grp * 8 + 8 > a.n;  // warp-uniform: only the dataset's last groups hold padded events
        const int64_t e = grp * 8 + 2 * ft;
        const bool v0 = e < a.n, v1 = e + 1 < a.n;
        double A[NPB][2], LL[NPB][2], LK[NPB][2];
#pragma unroll
        for (int pb = 0; pb < NPB; ++pb) {
            A[pb][0] = f.f0.x;
            A[pb][1] = f.f0.y;
            LL[pb][0] = LL[pb][1] = LK[pb][0] = LK[pb][1] = 0.0;
        }
#pragma unroll
        for (int kk = 0; kk < 2; ++kk)
#pragma unroll
            for (int pb = 0; pb < NPB; ++pb) dmma_m8n8k4(A[pb][0], A[pb][1], ca[pb][kk], f.f1[kk]);
#pragma unroll
        for (int pb = 0; pb < NPB; ++pb) dmma_m8n8k4(LL[pb][0], LL[pb][1], cll[pb], f.bl);
#pragma unroll
        for (int pb = 0; pb < NPB; ++pb) dmma_m8n8k4(LK[pb][0], LK[pb][1], clk[pb], f.bk);
        double qa[NPB][2], wl[NPB][2], wk[NPB][2];
#pragma unroll
        for (int pb = 0; pb < NPB; ++pb) {
            const double* pc = s_pc[8 * pb + fg];
            const double mu = pc[0], nb0 = pc[1], tau = pc[2], q0 = pc[3];
            const double m[2] = {f.m2.x, f.m2.y};
            double arg[2], d[2], t[2], R[2];
#pragma unroll
            for (int j = 0; j < 2; ++j) {
                d[j] = m[j] - mu;
                t[j] = d[j] * d[j];
                arg[j] = fma(nb0, t[j], fma(-tau, m[j], q0));
            }
            mf_exp32_v<2, false>(arg, t_lane, R);  // f (G/N1)/(E/N2)
#pragma unroll
            for (int j = 0; j < 2; ++j) {
                const double Lp = LL[pb][j] * LK[pb][j];       // (1-f) L
                double D = fma(R[j], A[pb][j], Lp);             // P N2 e^{-tau m}
                const bool v = j ? v1 : v0;
                if (masked && !v) D = 1.0;
                double r = mf_rcp(D);
                if (masked && !v) r = 0.0;
                lp[pb].mul(D, bad[pb]);
                const double q = R[j] * r;                      // f (G/N1) / P
                const double ws = q * A[pb][j];                 // signal weight of the event; the background's is 1 - ws
                qa[pb][j] = q;
                wl[pb][j] = r * LK[pb][j];
                wk[pb][j] = r * LL[pb][j];
                // raw moments of ws; the parameter-only factors and the background sums (from sum_i 1, sum_i m_i) are applied
                // once per point by the combine kernel
                ams[pb][0] += ws;
                ams[pb][1] = fma(ws, d[j], ams[pb][1]);
                ams[pb][2] = fma(ws, t[j], ams[pb][2]);
            }
        }
#pragma unroll
        for (int pb = 0; pb < NPB; ++pb) dmma_m8n8k4(gA[pb][0], gA[pb][1], qa[pb][0], f.f2.x);
#pragma unroll
        for (int pb = 0; pb < NPB; ++pb) dmma_m8n8k4(gA[pb][0], gA[pb][1], qa[pb][1], f.f2.y);
#pragma unroll
        for (int pb = 0; pb < NPB; ++pb) dmma_m8n8k4(gL[pb][0], gL[pb][1], wl[pb][0], f.x2.x);
#pragma unroll
        for (int pb = 0; pb < NPB; ++pb) dmma_m8n8k4(gL[pb][0], gL[pb][1], wl[pb][1], f.x2.y);
#pragma unroll
        for (int pb = 0; pb < NPB; ++pb) dmma_m8n8k4(gK[pb][0], gK[pb][1], wk[pb][0], f.x2.x);
#pragma unroll
        for (int pb = 0; pb < NPB; ++pb) dmma_m8n8k4(gK[pb][0], gK[pb][1], wk[pb][1], f.x2.y);
    };
    int64_t gi = blockIdx.x + G * warp;
    unsigned since_renorm = 0;
    int st = 0;
    if (gi < n_groups) issue(gi, 0);
    while (gi < n_groups) {
        if (gi + step < n_groups) {
            issue(gi + step, st ^ 1);
            asm volatile("cp.async.wait_group 1;" ::: "memory");  // everything but the group just requested has landed
        } else {
            asm volatile("cp.async.wait_group 0;" ::: "memory");
        }
        Frag f;
        fetch(st, f);
        process(gi, f);
        gi += step;
        st ^= 1;
        if (++since_renorm == 256) {
            since_renorm = 0;
#pragma unroll
            for (int pb = 0; pb < NPB; ++pb) lp[pb].renorm();
        }
    }
    __syncthreads();  // the staging area becomes the reduction buffer
    // lane (fg, ft) holds per-thread sums for point fg over its events: add the four ft lanes; tiles are complete per lane
#pragma unroll
    for (int pb = 0; pb < NPB; ++pb) {
        double v[5] = {lp[pb].log(), ams[pb][0], ams[pb][1], ams[pb][2], 0.0};
#pragma unroll
        for (int i = 0; i < 5; ++i) {
            v[i] += __shfl_xor_sync(0xffffffffu, v[i], 1);
            v[i] += __shfl_xor_sync(0xffffffffu, v[i], 2);
        }
        unsigned b = bad[pb];
        b += __shfl_xor_sync(0xffffffffu, b, 1);
        b += __shfl_xor_sync(0xffffffffu, b, 2);
        double* rr = red[warp][pb][fg];
        if (ft == 0) {
#pragma unroll
            for (int i = 0; i < 5; ++i) rr[i] = v[i];
            red_bad[warp][pb][fg] = b;
        }
        rr[5 + 2 * ft] = gA[pb][0];      // angular coefficients 2 ft, 2 ft + 1
        rr[6 + 2 * ft] = gA[pb][1];
        if (ft == 0) {                   // tile columns 0, 1: cos theta_l, P2
            rr[13] = gL[pb][0];
            rr[14] = gL[pb][1];
        }
        if (ft == 1) {                   // tile columns 2, 3: cos theta_K, P2
            rr[15] = gK[pb][0];
            rr[16] = gK[pb][1];
        }
    }
    __syncthreads();
    pdl_wait();  // the partial sums are shared with the previous call, whose combine kernel must have read them
    for (int q = threadIdx.x; q < NPB * 8 * 18; q += kBlock) {
        const int pl = q / 18, k = q % 18;  // local point, quantity (17: bad count)
        const int p = p0 + pl;
        if (p >= a.n_points) continue;
        if (k < 17) {
            double s = 0.0;
#pragma unroll
            for (int w = 0; w < kWarps; ++w) s += red[w][pl >> 3][pl & 7][k];
            a.partials[((int64_t)p * 17 + k) * G + blockIdx.x] = s;
        } else {
            unsigned b = 0;
#pragma unroll
            for (int w = 0; w < kWarps; ++w) b += red_bad[w][pl >> 3][pl & 7];
            a.bad_partials[(int64_t)p * G + blockIdx.x] = b;
        }
    }
}

// One CTA per point, one warp per quantity (17 sums + the bad-event count; warp_combine_partials, mf_points.cuh), then the
// K + 2 = 18 outputs.
// Sums: 0 ln prod D; 1 sum ws; 2 sum ws d; 3 sum ws d^2; 4 unused; 5..12 angular; 13, 14 cl1, cl2; 15, 16 ck1, ck2 (/ kappa).
constexpr int kP4CombineThreads = 32 * 18;
struct FourDCombineInlineArgs {
    const double* partials;
    const unsigned* bad_partials;
    int G, n_points;
    const double2* sum_m;
    double n;
    double* out;
    double fconst[kP4InlinePoints * kP4FinishConsts];
};

__device__ __forceinline__ void fourd_points_combine_body(const double* __restrict__ partials, const unsigned* __restrict__ bad_partials,
                                                          int G, int n_points, const double* __restrict__ fconst,
                                                          const double2* __restrict__ sum_m, double n, double* __restrict__ out);

__global__ void __launch_bounds__(kP4CombineThreads) fourd_points_combine_kernel(const double* __restrict__ partials,
                                                                                const unsigned* __restrict__ bad_partials, int G,
                                                                                int n_points, const double* __restrict__ fconst,
                                                                                const double2* __restrict__ sum_m, double n,
                                                                                double* __restrict__ out)
{
    fourd_points_combine_body(partials, bad_partials, G, n_points, fconst, sum_m, n, out);
}

__global__ void __launch_bounds__(kP4CombineThreads) fourd_points_combine_inline_kernel(const __grid_constant__ FourDCombineInlineArgs c)
{
    fourd_points_combine_body(c.partials, c.bad_partials, c.G, c.n_points, c.fconst, c.sum_m, c.n, c.out);
}

__device__ __forceinline__ void fourd_points_combine_body(const double* __restrict__ partials, const unsigned* __restrict__ bad_partials,
                                                          int G, int n_points, const double* __restrict__ fconst,
                                                          const double2* __restrict__ sum_m, double n, double* __restrict__ out)
{
    pdl_launch_dependents();
    pdl_wait();  // the main kernel of this call has completed
    __shared__ double s[17];
    __shared__ unsigned s_nb;
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, p = blockIdx.x;
    if (p >= n_points) return;
    if (w < 17) {
        const double v = warp_combine_partials(partials + ((int64_t)p * 17 + w) * G, G, lane);
        if (lane == 0) s[w] = v;
    } else {
        const unsigned b = warp_combine_bad(bad_partials + (int64_t)p * G, G, lane);
        if (lane == 0) s_nb = b;
    }
    __syncthreads();
    const int k = threadIdx.x;
    if (k > 17) return;
    const unsigned nb = s_nb;
    double* op = out + (int64_t)p * 18;
    if (k == 17) {
        op[17] = (double)nb;
        return;
    }
    const double* fc = fconst + (int64_t)p * kP4FinishConsts;
    const double inv_f = fc[0], inv_omf = fc[1], tau = fc[2], lnc2 = fc[3], kappa = fc[4];
    double o;
    if (k == 0) {
        const double2 sm = __ldg(sum_m);
        o = -(s[0] + fma(tau, sm.x, fma(tau, sm.y, n * lnc2)));
    } else if (k == 1) {
        o = -(inv_f * s[1] - inv_omf * (n - s[1]));  // sum (R A - L') / D from sum ws: ws / f - (1 - ws) / (1 - f)
    } else if (k == 2) {  // d/dmu = -sum ws (d is2 - kmu): the two terms nearly cancel at a minimum
        o = -diff_of_products(fc[5], s[2], fc[6], s[1]);
    } else if (k == 3) {  // d/dsigma = -sum ws (d^2 is3 - ksig)
        o = -diff_of_products(fc[7], s[3], fc[8], s[1]);
    } else if (k == 4) {
        // d/dtau = -sum wb (m - m_a - ktau) with wb = 1 - ws for every valid event:
        //   sum_i (m_i - c) - sum ws (m - c),  c = m_a + ktau,  m - c = d + (mu - c);  sum_i m_i as its (hi, lo) pair
        const double2 sm = __ldg(sum_m);
        const double c = fc[10], pr = n * c, pe = fma(n, c, -pr);
        const double all = (sm.x - pr) + (sm.y - pe);
        o = -(all - fma(fc[9], s[1], s[2]));
    } else if (k >= 15) {
        o = -kappa * s[k];
    } else {
        o = -s[k];
    }
    op[k] = !nb ? o : (k == 0) ? __longlong_as_double(0x7ff0000000000000LL) : __longlong_as_double(0x7ff8000000000000LL);
}

}  // namespace mf
