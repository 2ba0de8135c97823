// mf_points.cuh — many parameter points on ONE dataset in a single pass over the data, angular model
// ("multi-lambda evaluation in one pass ... the only case where F C becomes a real contraction worth
// testing on tensor cores"; north_star: "tensor cores only if the batched angular basis product F(N x K) C(K x M) is shown
// by ncu to be a real contraction").
//
// With M parameter points the cached-basis model is two contractions around one reciprocal:
//     P[p][e]   = sum_k a_pk h_k(e)            (k = 0..8, a_p0 = 1)        [M x 9] . [9 x N]
//     r[p][e]   = 1 / P[p][e],   ln L_p = sum_e ln P[p][e]                 (log of the running product, LogProd)
//     G[p][k]   = sum_e r[p][e] h_k(e)         (k = 1..8)                  [M x N] . [N x 8]
// Both run as DMMA m8n8k4 (mma.sync f64) on 8 points x 8 events at a time:
//   step 1: A = coefficients (8 points x 4 k, registers, loaded once), B = basis values (4 k x 8 events), two k-steps for
//           h_1..h_8, the accumulator tile initialised with the coefficient-free h_0 -> lane (g, t) holds
//           P(point g; events 2t, 2t+1);
//   step 2: A = r (8 points x 4 events) — exactly the two values each lane already holds if k-step j takes events
//           {2t + j}: no transposition, no shuffle; B = h_{1+g}(event 2t + j), one 16-byte load -> G tile (8 points x 8 k).
// Every 8-event group is fetched once per pass (two layouts, 576 B each, 64-byte segments from L2 / HBM, staged per lane in
// shared memory by cp.async so that the loads in flight cost no registers) and serves all the points of the pass, so the arithmetic intensity grows with M and the kernel is bound by the fp64 pipe: per
// (point, event) pair 4/64 DMMA (each holds the pipe of its SM sub-partition for 16 clocks) + one reciprocal (3 DFMA) + one
// DMUL, i.e. 0.31 pipe-clocks per pair per SM, the same as the hand-written DFMA form — which however issues 2.4
// instructions per pair instead of 0.6 and whose three-register DFMAs run at 2/3 rate.
#pragma once
#include "mf_kernels.cuh"
#include "mf_second.cuh"  // dmma_m8n8k4

namespace mf {

struct AngPointsArgs {
    const double* col[9];   // h_0..h_8
    int64_t n, n_pad;
    const double* coef;     // device [n_points][8]: FL, S3, S4, S5, AFB, S7, S8, S9 per point; NULL: in the parameter block
    int n_points;
    double* partials;       // [n_points][9][G]
    unsigned* bad_partials; // [n_points][G]
};

// Calls of up to kAngInlinePoints points carry the coefficients in the kernel's parameter block (16 KB): no copy sits between
// such a call and the previous kernel on the stream, so under the programmatic launch its CTAs start in the tail of the previous
// call (both kernels release their successor at entry; the main kernel waits for its predecessor — the previous call's combine
// kernel, which itself waited for that call's main kernel — only before it writes the partial sums the calls share, the
// combine kernel before it reads them).
constexpr int kAngInlinePoints = 256;
template <int MAXP>  // 32 or kAngInlinePoints: small calls carry a small block (2 KB instead of 16 KB per launch)
struct AngPointsInlineArgs {
    AngPointsArgs a;
    double coef[MAXP * 8];
};

// NPB point blocks of 8 points per CTA pass; grid = (G, ceil(n_points / (8 NPB))); dynamic shared memory: ang_points_smem<NPB>().
template <int NPB>
constexpr size_t ang_points_smem()
{
    return sizeof(double) * ((2 * kBlock * 6 > kWarps * NPB * 8 * 9) ? 2 * kBlock * 6 : kWarps * NPB * 8 * 9);
}

template <int NPB>
__device__ __forceinline__ void angular_points_mma_body(const AngPointsArgs& a, const double* __restrict__ coef);

template <int NPB>
__global__ void __launch_bounds__(kBlock, (NPB <= 2) ? 3 : (NPB <= 4) ? 2 : 1) angular_points_mma_kernel(const __grid_constant__ AngPointsArgs a)
{
    angular_points_mma_body<NPB>(a, a.coef);
}

template <int NPB, int MAXP>
__global__ void __launch_bounds__(kBlock, (NPB <= 2) ? 3 : (NPB <= 4) ? 2 : 1)
    angular_points_mma_inline_kernel(const __grid_constant__ AngPointsInlineArgs<MAXP> ia)
{
    angular_points_mma_body<NPB>(ia.a, ia.coef);
}

template <int NPB>
__device__ __forceinline__ void angular_points_mma_body(const AngPointsArgs& a, const double* __restrict__ coef)
{
    pdl_launch_dependents();
    // dynamic shared memory: per-lane staging of the event fragments (two stages filled by cp.async: loads in flight cost no
    // registers), reused after the event loop for the cross-warp reduction
    extern __shared__ __align__(16) unsigned char ap_raw[];
    double (*stg)[kBlock][6] = reinterpret_cast<double (*)[kBlock][6]>(ap_raw);
    double (*red)[NPB][8][9] = reinterpret_cast<double (*)[NPB][8][9]>(ap_raw);
    __shared__ unsigned red_bad[kWarps][NPB][8];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int fg = lane >> 2, ft = lane & 3;
    const int64_t G = gridDim.x;
    const int p0 = blockIdx.y * (8 * NPB);  // first point of this pass
    // step-1 A fragments: lane (fg, ft) holds the coefficient of h_{1 + 4 kk + ft} of point p = p0 + 8 pb + fg
    double ca[NPB][2];
#pragma unroll
    for (int pb = 0; pb < NPB; ++pb) {
        const int p = p0 + 8 * pb + fg;
        const bool live = p < a.n_points;
#pragma unroll
        for (int kk = 0; kk < 2; ++kk) ca[pb][kk] = live ? coef[(int64_t)p * 8 + 4 * kk + ft] : 0.0;
    }
    double g[NPB][2];
    LogProd lp[NPB];
    unsigned bad[NPB];
#pragma unroll
    for (int pb = 0; pb < NPB; ++pb) {
        g[pb][0] = g[pb][1] = 0.0;
        bad[pb] = 0;
    }
    const int64_t n_groups = a.n_pad / 8, step = G * kWarps;
    // fragments of a group: f1[kk] = h_{1 + 4 kk + ft}(event fg), f2 = h_{1 + fg}(events 2 ft, 2 ft + 1),
    // f0 = h_0(events 2 ft, 2 ft + 1): the coefficient-free term, the initial value of every P tile
    struct Frag {
        double f1[2];
        double2 f2, f0;
    };
    // issue: this lane's values of group grp -> stage st (asynchronous copies); fetch: stage st -> fragments
    // this lane's four source pointers at group 0 (set once: no indexed loads of the column table in the loop)
    const double* const src_a = a.col[1 + ft] + fg;
    const double* const src_b = a.col[5 + ft] + fg;
    const double* const src_c = a.col[1 + fg] + 2 * ft;
    const double* const src_d = a.col[0] + 2 * ft;
    const unsigned dst0 = (unsigned)__cvta_generic_to_shared(&stg[0][threadIdx.x][0]);
    auto issue = [&](int64_t grp, int st) {
        const int64_t e0 = grp * 8;
        const unsigned dst = dst0 + (unsigned)(st * (int)sizeof(stg[0]));
        asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(dst), "l"(src_a + e0) : "memory");
        asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(dst + 8u), "l"(src_b + e0) : "memory");
        asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"(dst + 16u), "l"(src_c + e0) : "memory");
        asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"(dst + 32u), "l"(src_d + e0) : "memory");
        asm volatile("cp.async.commit_group;" ::: "memory");
    };
    auto fetch = [&](int st, Frag& f) {
        const double* q = &stg[st][threadIdx.x][0];
        f.f1[0] = q[0];
        f.f1[1] = q[1];
        f.f2 = *reinterpret_cast<const double2*>(q + 2);
        f.f0 = *reinterpret_cast<const double2*>(q + 4);
    };
    // One group for all the point blocks of the pass, written stage by stage across the NPB independent blocks so that
    // dependent instructions are NPB apart.  Only the dataset's last groups can hold padded events (copies of the last
    // event): there `masked` makes them contribute exactly nothing.
    auto process = [&](int64_t grp, const Frag& f) {
        const double2 f2 = f.f2;
        double c[NPB][2], r[NPB][2];
#pragma unroll
        for (int pb = 0; pb < NPB; ++pb) {
            c[pb][0] = f.f0.x;
            c[pb][1] = f.f0.y;
        }
#pragma unroll
        for (int kk = 0; kk < 2; ++kk)
#pragma unroll
            for (int pb = 0; pb < NPB; ++pb) dmma_m8n8k4(c[pb][0], c[pb][1], ca[pb][kk], f.f1[kk]);
        const bool masked = grp * 8 + 8 > a.n;  // warp-uniform
        const int64_t e = grp * 8 + 2 * ft;
        const bool v0 = e < a.n, v1 = e + 1 < a.n;
        if (masked) {
#pragma unroll
            for (int pb = 0; pb < NPB; ++pb) {
                c[pb][0] = v0 ? c[pb][0] : 1.0;
                c[pb][1] = v1 ? c[pb][1] : 1.0;
            }
        }
#pragma unroll
        for (int pb = 0; pb < NPB; ++pb) {
            r[pb][0] = mf_rcp(c[pb][0]);
            r[pb][1] = mf_rcp(c[pb][1]);
        }
        if (masked) {
#pragma unroll
            for (int pb = 0; pb < NPB; ++pb) {
                r[pb][0] = v0 ? r[pb][0] : 0.0;
                r[pb][1] = v1 ? r[pb][1] : 0.0;
            }
        }
#pragma unroll
        for (int pb = 0; pb < NPB; ++pb) dmma_m8n8k4(g[pb][0], g[pb][1], r[pb][0], f2.x);
#pragma unroll
        for (int pb = 0; pb < NPB; ++pb) dmma_m8n8k4(g[pb][0], g[pb][1], r[pb][1], f2.y);
        // ln L: the PDF values of a group are multiplied into the running products as they are when all of them lie in
        // [2^-60, 2^16) (one integer max per value decides; the exponent is then extracted every fourth group: at most
        // 8 x 60 bits of drift); otherwise (a bad or an extreme value somewhere in the lane's 2 NPB values) the general
        // multiplication, which extracts every exponent and counts the bad events
        constexpr int kLo = (1023 - 60) << 20;
        constexpr unsigned kRange = 76u << 20;
        unsigned u = 0;
#pragma unroll
        for (int pb = 0; pb < NPB; ++pb) {
            u = max(u, (unsigned)(__double2hiint(c[pb][0]) - kLo));
            u = max(u, (unsigned)(__double2hiint(c[pb][1]) - kLo));
        }
        if (u < kRange) {
#pragma unroll
            for (int pb = 0; pb < NPB; ++pb) {
                lp[pb].mul_bounded(c[pb][0]);
                lp[pb].mul_bounded(c[pb][1]);
            }
        } else {
#pragma unroll
            for (int pb = 0; pb < NPB; ++pb) {
                lp[pb].mul(c[pb][0], bad[pb]);
                lp[pb].mul(c[pb][1], bad[pb]);
            }
        }
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
        if (++since_renorm == 4) {  // 8 factors in [2^-60, 2^16) (or mantissas in [1, 2)) per running product since the last one
            since_renorm = 0;
#pragma unroll
            for (int pb = 0; pb < NPB; ++pb) lp[pb].renorm();
        }
    }
    __syncthreads();  // the staging area becomes the reduction buffer
    // lane (fg, ft): ln of the product over its events for point fg of every block; sum over the four ft lanes
#pragma unroll
    for (int pb = 0; pb < NPB; ++pb) {
        double l = lp[pb].log();
        l += __shfl_xor_sync(0xffffffffu, l, 1);
        l += __shfl_xor_sync(0xffffffffu, l, 2);
        unsigned b = bad[pb];
        b += __shfl_xor_sync(0xffffffffu, b, 1);
        b += __shfl_xor_sync(0xffffffffu, b, 2);
        if (ft == 0) {
            red[warp][pb][fg][0] = l;
            red_bad[warp][pb][fg] = b;
        }
        red[warp][pb][fg][1 + 2 * ft] = g[pb][0];
        red[warp][pb][fg][2 + 2 * ft] = g[pb][1];
    }
    __syncthreads();
    pdl_wait();  // the partial sums are shared with the previous call, whose combine kernel must have read them
    for (int q = threadIdx.x; q < NPB * 8 * 10; q += kBlock) {
        const int pl = q / 10, k = q % 10;  // local point, quantity (9: bad count)
        const int p = p0 + pl;
        if (p >= a.n_points) continue;
        if (k < 9) {
            double s = 0.0;
#pragma unroll
            for (int w = 0; w < kWarps; ++w) s += red[w][pl >> 3][pl & 7][k];
            a.partials[((int64_t)p * 9 + k) * G + blockIdx.x] = s;
        } else {
            unsigned b = 0;
#pragma unroll
            for (int w = 0; w < kWarps; ++w) b += red_bad[w][pl >> 3][pl & 7];
            a.bad_partials[(int64_t)p * G + blockIdx.x] = b;
        }
    }
}

// One CTA per point, one warp per quantity (9 sums + the bad-event count): out[p] = (-ln L, gradient[8], n_bad).  (One warp per
// POINT walking its 9 rows one after the other took 16 us whatever the number of points: a chain of dependent L2 round trips.)
constexpr int kAngCombineThreads = 32 * 10;
__global__ void __launch_bounds__(kAngCombineThreads) angular_points_combine_kernel(const double* __restrict__ partials,
                                                                                   const unsigned* __restrict__ bad_partials, int G,
                                                                                   int n_points, double* __restrict__ out)
{
    __shared__ double s_sum[9];
    __shared__ unsigned s_nb;
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, p = blockIdx.x;
    pdl_launch_dependents();
    pdl_wait();  // the main kernel of this call has completed
    if (p >= n_points) return;
    if (w < 9) {
        const double s = warp_combine_partials(partials + ((int64_t)p * 9 + w) * G, G, lane);
        if (lane == 0) s_sum[w] = s;
    } else {
        const unsigned nb = warp_combine_bad(bad_partials + (int64_t)p * G, G, lane);
        if (lane == 0) s_nb = nb;
    }
    __syncthreads();
    const unsigned nb = s_nb;
    double* o = out + (int64_t)p * 10;
    if (threadIdx.x < 9)
        o[threadIdx.x] = !nb                ? -s_sum[threadIdx.x]
                         : (threadIdx.x == 0) ? __longlong_as_double(0x7ff0000000000000LL)
                                              : __longlong_as_double(0x7ff8000000000000LL);
    else if (threadIdx.x == 9)
        o[9] = (double)nb;
}

}  // namespace mf
