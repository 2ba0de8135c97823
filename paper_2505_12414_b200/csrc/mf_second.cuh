// mf_second.cuh — second-order sums of the likelihood by fp64 tensor-core contraction:
// in ONE pass over the data
//     -ln L_w = -sum_i w_i ln P_i,   its gradient,   its Hessian  -sum_i w_i d2 ln P_i,   F = sum_i w_i^2 s_i s_i^T
// for all three model families, weighted or not (analytic Hessian by second differentiation of
// ln P; "the Fisher information matrix ... required for weighted fits", reading R23).
//
// Why tensor cores here and nowhere else on the path: with s = d ln P / d lambda the Hessian of ln P is
// P_ab / P - s_a s_b, so the sums over events are dominated by  S^T diag(w) S  with S the [N x K] matrix of scores — a real
// contraction over the event index (K = 16: 136 products per event for the 4D model, too many accumulators for one thread).
// The non-zero P_ab / P terms are products of a few event-only quantities X (1, d, d^2, ...) with score-like
// quantities, i.e. a second contraction  X^T diag(w) Y.  Both run as DMMA m8n8k4 (mma.sync f64): four events per
// instruction, the 8 x 8 accumulator tiles live distributed over the warp (two doubles per lane per tile).
// Measured on B200 (mfp_dmma_rate): DMMA reaches the nominal fp64 rate (1.86e13 FMA/s) but shares the pipe with DFMA, so
// the gain is not in flops (the padded tiles cost about twice the FMAs of the sparse hand-written sums) but in issue slots
// (1 instruction per 256 FMAs) and registers (no per-thread accumulator array).
//
// Per-event "vectors" of a model S (all finite for any finite event):
//   Y[S::NY]  y_a for a < K with score s_a = phi_a y_a (phi_a a parameter-only factor 1, f or 1-f, applied in finish, so
//             that nothing is divided by f or 1-f), then model-specific helper entries;
//   X[8]      X_0 = 1, then event-only quantities.
// Tile sums (each an 8 x 8 tile of doubles):
//   XY[tj]      = sum_i w_i X_r(i) Y_{8 tj + c}(i)                      (row 0: the weighted gradient sums)
//   YY[ti<=tj]  = sum_i w_i Y_{8 ti + r}(i) Y_{8 tj + c}(i)             (MODE >= 1; score tiles only: 8 ti, 8 tj < K)
//   FF[ti<=tj]  = the same with w_i^2                                  (MODE == 2)
// plus the plain per-thread sum of w_i ln D_i.  S::finish turns the combined sums into the outputs.
#pragma once
#include "mf_kernels.cuh"

namespace mf {

__device__ __forceinline__ void dmma_m8n8k4(double& c0, double& c1, double a, double b)
{
    asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(c0), "+d"(c1)
                 : "d"(a), "d"(b));
}

constexpr int kSecondRow = 36;  // doubles per row of the per-warp vector buffer: 32 events + 4 (conflict-free fragment reads)
constexpr int kSecondItem = 32;  // events per warp item: one per lane

template <class S>
struct SecondArgs {
    const double* col[S::NCOL];
    const double* w;   // event weights [n_pad] (padding 0) or NULL (= 1)
    int64_t n, n_pad;
    typename S::Consts c;
    double* partials;        // [NQ][gridDim.x]
    unsigned* bad_partials;  // [gridDim.x]
};

template <class S, int MODE>
struct SecondLayout {
    static constexpr int NT = S::NY / 8;          // Y tiles (scores, then helpers)
    static constexpr int NTK = (S::K + 7) / 8;    // Y tiles that hold scores: only their products enter YY and FF
    static constexpr int NYY = NTK * (NTK + 1) / 2;
    static constexpr int NTILES = NT + (MODE >= 1 ? NYY : 0) + (MODE >= 2 ? NYY : 0);
    static constexpr int NQ = 1 + 64 * NTILES;  // quantity 0: sum w ln D
    static constexpr int NV = 8 + S::NY + 1;    // X, Y, w
    static constexpr int K = S::K;
    static constexpr int NH = K * (K + 1) / 2;
    static constexpr int NOUT = 1 + K + (MODE >= 1 ? NH : 0) + (MODE >= 2 ? NH : 0);  // n_bad follows at [NOUT]
    // CTA size: 16 warps where the register budget allows (128 per thread), else 12; one CTA per SM
    static constexpr int THREADS = (S::NY > 8 && MODE >= 2) ? 384 : 512;
    static constexpr int WARPS = THREADS / 32;
    __host__ __device__ static constexpr int yy_tile(int ti, int tj)  // ti <= tj, row-major upper triangle
    {
        return ti * NTK - ti * (ti - 1) / 2 + (tj - ti);
    }
    static constexpr size_t smem_bytes() { return sizeof(double) * (size_t)WARPS * NV * kSecondRow + sizeof(double2) * kLogTableSize; }
};

// Warps are independent: a warp item is 32 consecutive events, one per lane, read with one coalesced 256-byte load per
// column; items are dealt block-cyclically over all warps of the grid; the next item's lines are requested from L2 while
// the current one is evaluated.  No CTA-wide barrier inside the event loop.
template <class S, int MODE>
__global__ void __launch_bounds__(SecondLayout<S, MODE>::THREADS, 1) nll_second_kernel(const __grid_constant__ SecondArgs<S> a)
{
    using L = SecondLayout<S, MODE>;
    constexpr int NT = L::NT, NTK = L::NTK, NYY = L::NYY, NV = L::NV, RS = kSecondRow, WARPS = L::WARPS, THREADS = L::THREADS;
    extern __shared__ __align__(128) unsigned char sec_raw[];
    double (*sv)[NV][RS] = reinterpret_cast<double (*)[NV][RS]>(sec_raw);
    double2* s_tab = reinterpret_cast<double2*>(sec_raw + sizeof(double) * WARPS * NV * RS);
    __shared__ double s_w0[WARPS];
    __shared__ unsigned s_wbad[WARPS];

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int fg = lane >> 2, ft = lane & 3;  // fragment coordinates: row / column group and event within the group of four
    const bool weighted = a.w != nullptr;
    const int64_t n_items = a.n_pad / kSecondItem, G = gridDim.x;
    load_log_table(s_tab);
    __syncthreads();
    double cxy[NT][2], cyy[MODE >= 1 ? NYY : 1][2], cff[MODE >= 2 ? NYY : 1][2];
#pragma unroll
    for (int i = 0; i < NT; ++i) cxy[i][0] = cxy[i][1] = 0.0;
#pragma unroll
    for (int i = 0; i < (MODE >= 1 ? NYY : 1); ++i) cyy[i][0] = cyy[i][1] = 0.0;
#pragma unroll
    for (int i = 0; i < (MODE >= 2 ? NYY : 1); ++i) cff[i][0] = cff[i][1] = 0.0;
    double acc0 = 0.0;
    unsigned bad = 0;
    const double t_lane = mf_exp32_lane_entry();
    const int64_t step = G * WARPS;
    for (int64_t item = blockIdx.x + G * warp; item < n_items; item += step) {
        const int64_t e = item * kSecondItem + lane;
        double x[S::NCOL], wgt = 1.0;
#pragma unroll
        for (int c = 0; c < S::NCOL; ++c) x[c] = __ldg(a.col[c] + e);
        if (weighted) wgt = __ldg(a.w + e);
        if (item + step < n_items) {  // next item of this warp: 256 bytes per column = two lines
            const int64_t en = (item + step) * kSecondItem;
            if (lane < 2 * S::NCOL) asm volatile("prefetch.global.L2 [%0];" ::"l"(a.col[lane >> 1] + en + 16 * (lane & 1)));
            if (weighted && lane >= 30) asm volatile("prefetch.global.L2 [%0];" ::"l"(a.w + en + 16 * (lane & 1)));
        }
        const bool valid = e < a.n;
        if (!valid) wgt = 0.0;
        {
            double X[8], Y[S::NY];
            const double D = S::vectors(x, a.c, X, Y, t_lane);
            const int hx = __double2hiint(D);
            const bool isbad = (unsigned)(hx - 0x01700000) >= 0x7E800000u;  // not in [2^-1000, inf): "P <= 0" (as LogProd::mul)
            bad += (valid && isbad) ? 1u : 0u;
            acc0 = fma(wgt, mf_log(isbad ? 1.0 : D, s_tab), acc0);
#pragma unroll
            for (int j = 0; j < 8; ++j) sv[warp][j][lane] = X[j];
#pragma unroll
            for (int j = 0; j < S::NY; ++j) sv[warp][8 + j][lane] = isbad ? 0.0 : Y[j];
            sv[warp][NV - 1][lane] = wgt;
        }
        __syncwarp();
        // the warp's 32 events, four per DMMA: lane (fg, ft) supplies row / column fg of event ft of the group
#pragma unroll
        for (int q = 0; q < 8; ++q) {
            const int ev = 4 * q + ft;
            const double wv = sv[warp][NV - 1][ev];
            const double xa = sv[warp][fg][ev] * wv;
            double y[NT];
#pragma unroll
            for (int ti = 0; ti < NT; ++ti) y[ti] = sv[warp][8 + 8 * ti + fg][ev];
#pragma unroll
            for (int tj = 0; tj < NT; ++tj) dmma_m8n8k4(cxy[tj][0], cxy[tj][1], xa, y[tj]);
            if constexpr (MODE >= 1) {
#pragma unroll
                for (int ti = 0; ti < NTK; ++ti) {
                    const double ya = y[ti] * wv;
#pragma unroll
                    for (int tj = ti; tj < NTK; ++tj) dmma_m8n8k4(cyy[L::yy_tile(ti, tj)][0], cyy[L::yy_tile(ti, tj)][1], ya, y[tj]);
                    if constexpr (MODE >= 2) {
                        const double yaa = ya * wv;
#pragma unroll
                        for (int tj = ti; tj < NTK; ++tj) dmma_m8n8k4(cff[L::yy_tile(ti, tj)][0], cff[L::yy_tile(ti, tj)][1], yaa, y[tj]);
                    }
                }
            }
        }
        __syncwarp();  // every lane has read the vectors before the next item overwrites them
    }
    // ---- warp -> block: tile accumulators through the (now free) vector buffers, summed in warp order
    static_assert(64 * L::NTILES <= NV * RS, "a warp's tiles fit its vector buffer");
    double* red = &sv[warp][0][0];  // [NTILES][64], element (row, col) of a tile at 8 row + col = 2 lane + {0, 1}
#pragma unroll
    for (int i = 0; i < NT; ++i) {
        red[64 * i + 2 * lane] = cxy[i][0];
        red[64 * i + 2 * lane + 1] = cxy[i][1];
    }
    if constexpr (MODE >= 1) {
#pragma unroll
        for (int i = 0; i < NYY; ++i) {
            red[64 * (NT + i) + 2 * lane] = cyy[i][0];
            red[64 * (NT + i) + 2 * lane + 1] = cyy[i][1];
        }
    }
    if constexpr (MODE >= 2) {
#pragma unroll
        for (int i = 0; i < NYY; ++i) {
            red[64 * (NT + NYY + i) + 2 * lane] = cff[i][0];
            red[64 * (NT + NYY + i) + 2 * lane + 1] = cff[i][1];
        }
    }
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) acc0 += __shfl_xor_sync(0xffffffffu, acc0, off);
    bad = __reduce_add_sync(0xffffffffu, bad);
    if (lane == 0) {
        s_w0[warp] = acc0;
        s_wbad[warp] = bad;
    }
    __syncthreads();
    for (int q = tid; q < 64 * L::NTILES; q += THREADS) {
        double s = 0.0;
#pragma unroll
        for (int w = 0; w < WARPS; ++w) s += (&sv[w][0][0])[q];
        a.partials[(int64_t)(1 + q) * G + blockIdx.x] = s;
    }
    if (tid == 0) {
        double s = 0.0;
        unsigned b = 0;
#pragma unroll
        for (int w = 0; w < WARPS; ++w) {
            s += s_w0[w];
            b += s_wbad[w];
        }
        a.partials[blockIdx.x] = s;
        a.bad_partials[blockIdx.x] = b;
    }
}

// Fixed-order compensated combine of the CTA partials (one warp per quantity), then S::finish by the CTA that draws the
// last ticket.  grid = ceil(NQ / 8) CTAs of 256 threads.
template <class S>
struct SecondCombineArgs {
    const double* partials;        // [NQ][G]
    const unsigned* bad_partials;  // [G]
    int G;
    double* sums;                  // [NQ]
    unsigned* ticket;              // zero on entry, reset by the last CTA
    typename S::Consts c;
    double* out;                   // [NOUT + 1]
    unsigned long long* done_flag; // mapped host word that receives done_value after `out` is written, or NULL
    unsigned long long done_value;
};

template <class S, int MODE>
__global__ void __launch_bounds__(kBlock) second_combine_kernel(const __grid_constant__ SecondCombineArgs<S> a)
{
    using L = SecondLayout<S, MODE>;
    __shared__ bool s_last;
    __shared__ double s_sum[L::NQ];
    __shared__ unsigned s_nb;
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const int q = blockIdx.x * kWarps + w;
    if (q < L::NQ) {
        const double s = warp_combine_partials(a.partials + (int64_t)q * a.G, a.G, lane);
        if (lane == 0) a.sums[q] = s;
    }
    __syncthreads();
    if (threadIdx.x == 0) s_last = (ticket_take(a.ticket) == gridDim.x - 1);
    __syncthreads();
    if (!s_last) return;
    for (int i = threadIdx.x; i < L::NQ; i += kBlock) s_sum[i] = __ldcg(a.sums + i);
    if (w == 0) {
        unsigned nb = 0;
        for (int i = lane; i < a.G; i += 32) nb += __ldcg(a.bad_partials + i);
        nb = __reduce_add_sync(0xffffffffu, nb);
        if (lane == 0) s_nb = nb;
    }
    __syncthreads();
    const unsigned nb = s_nb;
    for (int o = threadIdx.x; o < L::NOUT; o += kBlock) {
        const double v = S::template finish<MODE>(a.c, s_sum, o);
        a.out[o] = !nb ? v : (o == 0) ? __longlong_as_double(0x7ff0000000000000LL) : __longlong_as_double(0x7ff8000000000000LL);
    }
    if (threadIdx.x == 0) {
        a.out[L::NOUT] = (double)nb;
        *a.ticket = 0u;
    }
    if (a.done_flag) {  // synchronous call: `out` is mapped host memory and the host spins on this word
        __threadfence_system();
        __syncthreads();
        if (threadIdx.x == 0) {
            __threadfence_system();
            *reinterpret_cast<volatile unsigned long long*>(a.done_flag) = a.done_value;
        }
    }
}

// ---- access to the combined tile sums inside S::finish ---------------------------------------------------------------
template <class S, int MODE>
struct SecondSums {
    using L = SecondLayout<S, MODE>;
    const double* s;
    __device__ __forceinline__ double w_ln_d() const { return s[0]; }
    // sum_i w_i X_r Y_j
    __device__ __forceinline__ double xy(int r, int j) const { return s[1 + 64 * (j >> 3) + 8 * r + (j & 7)]; }
    // sum_i w_i Y_i Y_j (any order)
    __device__ __forceinline__ double yy(int i, int j) const
    {
        if (i > j) {
            const int t = i;
            i = j;
            j = t;
        }
        return s[1 + 64 * (L::NT + L::yy_tile(i >> 3, j >> 3)) + 8 * (i & 7) + (j & 7)];
    }
    // sum_i w_i^2 Y_i Y_j
    __device__ __forceinline__ double ff(int i, int j) const
    {
        if (i > j) {
            const int t = i;
            i = j;
            j = t;
        }
        return s[1 + 64 * (L::NT + L::NYY + L::yy_tile(i >> 3, j >> 3)) + 8 * (i & 7) + (j & 7)];
    }
};

// output index o -> (kind, a, b): kind 0 = -ln L, 1 = gradient a, 2 = Hessian (a <= b), 3 = Fisher (a <= b)
template <int K>
__device__ __forceinline__ void second_out_index(int o, int& kind, int& a, int& b)
{
    constexpr int NH = K * (K + 1) / 2;
    a = b = 0;
    if (o == 0) {
        kind = 0;
        return;
    }
    if (o <= K) {
        kind = 1;
        a = o - 1;
        return;
    }
    int q = o - 1 - K;
    kind = 2;
    if (q >= NH) {
        q -= NH;
        kind = 3;
    }
    int i = 0;
    while (q >= K - i) {
        q -= K - i;
        ++i;
    }
    a = i;
    b = i + q;
}

// ---- the three families ---------------------------------------------------------------------------------------------

// Mass model.  u = R/D, r = 1/D (D = (1-f) + f R = P N2 e^{-tau m}); al_m = d/sigma^2 - kmu, al_s = d^2/sigma^3 - ksig,
// be = m - d ln N2/d tau = d + ct.  y = (u - r, u al_m, u al_s, r be), phi = (1, f, f, 1-f).
// Helpers: Y4 = u, Y5 = r, Y6 = 1.  X = (1, d, d^2, d^3, d^4).
struct MassSecond {
    static constexpr int K = 4, NCOL = 1, NY = 8;
    using Consts = MassConsts;
    static MF_D double vectors(const double* x, const Consts& c, double* X, double* Y, double t_lane)
    {
        const double m = x[0];
        const double d = m - c.mu, t = d * d;
        const double arg = fma(c.nb0, t, fma(-c.tau, m, c.lnk));
        const double R = mf_exp32(arg, t_lane);
        const double D = fma(c.f, R, c.omf);
        const double r = mf_rcp(D);
        const double u = R * r;
        Y[0] = u - r;
        Y[1] = u * fma(d, c.is2, -c.kmu);
        Y[2] = u * fma(t, c.is3, -c.ksig);
        Y[3] = r * (d + c.ct);
        Y[4] = u;
        Y[5] = r;
        Y[6] = 1.0;
        Y[7] = 0.0;
        X[0] = 1.0;
        X[1] = d;
        X[2] = t;
        X[3] = t * d;
        X[4] = t * t;
        X[5] = X[6] = X[7] = 0.0;
        return D;
    }
    static MF_D double phi(const Consts& c, int a) { return a == 0 ? 1.0 : a == 3 ? c.omf : c.f; }
    // sum_i w_i P_ab / P for a <= b
    template <class T>
    static MF_D double pp(const Consts& c, const T& S, int a, int b)
    {
        const double M0 = S.xy(0, 4), M1 = S.xy(1, 4), M2 = S.xy(2, 4), M3 = S.xy(3, 4), M4 = S.xy(4, 4);
        const double B0 = S.xy(0, 5), B1 = S.xy(1, 5), B2 = S.xy(2, 5);
        const double is2 = c.is2, is3 = c.is3, kmu = c.kmu, ksig = c.ksig;
        if (a == 0) return b == 0 ? 0.0 : b == 3 ? -S.xy(0, 3) : S.xy(0, b);
        if (a == 1 && b == 1) return c.f * (is2 * is2 * M2 - 2.0 * is2 * kmu * M1 + (kmu * kmu - is2 - c.n1mm) * M0);
        if (a == 1 && b == 2)
            return c.f * (is2 * is3 * M3 - kmu * is3 * M2 - (is2 * ksig + 2.0 * is3) * M1 + (kmu * ksig - c.n1ms) * M0);
        if (a == 2 && b == 2)
            return c.f * (is3 * is3 * M4 - (2.0 * is3 * ksig + 3.0 * c.is4) * M2 + (ksig * ksig + is2 - c.n1ss) * M0);
        if (a == 3 && b == 3) return c.omf * (B2 + 2.0 * c.ct * B1 + (c.ct * c.ct - c.n2tt) * B0);
        return 0.0;
    }
    template <int MODE>
    static MF_D double finish(const Consts& c, const double* s, int o)
    {
        const SecondSums<MassSecond, MODE> S{s};
        int kind, a, b;
        second_out_index<K>(o, kind, a, b);
        if (kind == 0) {
            const double Sw = S.xy(0, 6), Swm = fma(c.mu, Sw, S.xy(1, 6));
            return -(S.w_ln_d() + fma(c.tau, Swm, Sw * c.lnc2));
        }
        if (kind == 1) return -phi(c, a) * S.xy(0, a);
        if (kind == 2) return phi(c, a) * phi(c, b) * S.yy(a, b) - pp(c, S, a, b);
        return phi(c, a) * phi(c, b) * S.ff(a, b);
    }
};

// Angular model: P linear in its coefficients, y_k = h_{k+1} / P = s_k, no second derivatives of P.
struct AngularSecond {
    static constexpr int K = 8, NCOL = 9, NY = 8;
    using Consts = AngularConsts;
    static MF_D double vectors(const double* x, const Consts& c, double* X, double* Y, double)
    {
        double P = fma(c.a[0], x[1], x[0]);
#pragma unroll
        for (int k = 1; k < 8; ++k) P = fma(c.a[k], x[1 + k], P);
        const double r = mf_rcp(P);
#pragma unroll
        for (int k = 0; k < 8; ++k) Y[k] = x[1 + k] * r;
        X[0] = 1.0;
#pragma unroll
        for (int k = 1; k < 8; ++k) X[k] = 0.0;
        return P;
    }
    template <int MODE>
    static MF_D double finish(const Consts&, const double* s, int o)
    {
        const SecondSums<AngularSecond, MODE> S{s};
        int kind, a, b;
        second_out_index<K>(o, kind, a, b);
        if (kind == 0) return -S.w_ln_d();
        if (kind == 1) return -S.xy(0, a);
        if (kind == 2) return S.yy(a, b);
        return S.ff(a, b);
    }
};

// 4D model.  D = f R A + (1-f) L' (L' = ll lk / (8 pi)), r = 1/D, us = R A r (signal weight / f), ub = L' r (background
// weight / (1-f)), qq = r / (8 pi).
//   y = (us - ub, us al_m, us al_s, ub be, R r h_1..h_8, qq lk cl, qq lk p2l, qq ll ck, qq ll p2k),
//   phi = (1, f, f, 1-f, f x 8, (1-f) x 4).
// Helpers: Y16 = us, Y17 = ub, Y18 = qq cl, Y19 = qq p2l, Y20 = 1.  X = (1, d, d^2, d^3, d^4, ck, p2k).
struct FourDSecond {
    static constexpr int K = 16, NCOL = 12, NY = 24;
    using Consts = FourDConsts;
    static MF_D double vectors(const double* x, const Consts& c, double* X, double* Y, double t_lane)
    {
        const MassConsts& q = c.m;
        const double m = x[0], cl = x[1], ck = x[2];
        const double* h = x + 3;
        double A = fma(c.a[0], h[1], h[0]);
#pragma unroll
        for (int k = 1; k < 8; ++k) A = fma(c.a[k], h[1 + k], A);
        const double p2l = fma(1.5 * cl, cl, -0.5), p2k = fma(1.5 * ck, ck, -0.5);
        const double ll = fma(c.cl2, p2l, fma(c.cl1, cl, 1.0));
        const double lk = fma(c.ck2, p2k, fma(c.ck1, ck, 1.0));
        const double d = m - q.mu, t = d * d;
        const double arg = fma(q.nb0, t, fma(-q.tau, m, q.lnk));
        const double R = mf_exp32(arg, t_lane);
        const double Lp = (ll * lk) * kInv8Pi;
        const double D = fma(q.f * R, A, q.omf * Lp);
        const double r = mf_rcp(D);
        const double Rr = R * r;
        const double us = Rr * A, ub = Lp * r, qq = kInv8Pi * r;
        Y[0] = us - ub;
        Y[1] = us * fma(d, q.is2, -q.kmu);
        Y[2] = us * fma(t, q.is3, -q.ksig);
        Y[3] = ub * (d + q.ct);
#pragma unroll
        for (int k = 0; k < 8; ++k) Y[4 + k] = Rr * h[1 + k];
        const double ql = qq * lk, qk = qq * ll;
        Y[12] = ql * cl;
        Y[13] = ql * p2l;
        Y[14] = qk * ck;
        Y[15] = qk * p2k;
        Y[16] = us;
        Y[17] = ub;
        Y[18] = qq * cl;
        Y[19] = qq * p2l;
        Y[20] = 1.0;
        Y[21] = Y[22] = Y[23] = 0.0;
        X[0] = 1.0;
        X[1] = d;
        X[2] = t;
        X[3] = t * d;
        X[4] = t * t;
        X[5] = ck;
        X[6] = p2k;
        X[7] = 0.0;
        return D;
    }
    static MF_D double phi(const Consts& c, int a) { return a == 0 ? 1.0 : (a == 3 || a >= 12) ? c.m.omf : c.m.f; }
    template <class T>
    static MF_D double pp(const Consts& cc, const T& S, int a, int b)
    {
        const MassConsts& c = cc.m;
        const double is2 = c.is2, is3 = c.is3, kmu = c.kmu, ksig = c.ksig;
        if (a == 0) return b == 0 ? 0.0 : (b == 3 || b >= 12) ? -S.xy(0, b) : S.xy(0, b);
        if (a <= 2 && b <= 2) {
            const double M0 = S.xy(0, 16), M1 = S.xy(1, 16), M2 = S.xy(2, 16), M3 = S.xy(3, 16), M4 = S.xy(4, 16);
            if (a == 1 && b == 1) return c.f * (is2 * is2 * M2 - 2.0 * is2 * kmu * M1 + (kmu * kmu - is2 - c.n1mm) * M0);
            if (a == 1 && b == 2)
                return c.f * (is2 * is3 * M3 - kmu * is3 * M2 - (is2 * ksig + 2.0 * is3) * M1 + (kmu * ksig - c.n1ms) * M0);
            return c.f * (is3 * is3 * M4 - (2.0 * is3 * ksig + 3.0 * c.is4) * M2 + (ksig * ksig + is2 - c.n1ss) * M0);
        }
        if (a == 1 && b >= 4 && b < 12) return c.f * (is2 * S.xy(1, b) - kmu * S.xy(0, b));
        if (a == 2 && b >= 4 && b < 12) return c.f * (is3 * S.xy(2, b) - ksig * S.xy(0, b));
        if (a == 3 && b == 3) {
            const double B0 = S.xy(0, 17), B1 = S.xy(1, 17), B2 = S.xy(2, 17);
            return c.omf * (B2 + 2.0 * c.ct * B1 + (c.ct * c.ct - c.n2tt) * B0);
        }
        if (a == 3 && b >= 12) return c.omf * fma(c.ct, S.xy(0, b), S.xy(1, b));
        if ((a == 12 || a == 13) && (b == 14 || b == 15)) return c.omf * S.xy(5 + (b - 14), 18 + (a - 12));
        return 0.0;
    }
    template <int MODE>
    static MF_D double finish(const Consts& c, const double* s, int o)
    {
        const SecondSums<FourDSecond, MODE> S{s};
        int kind, a, b;
        second_out_index<K>(o, kind, a, b);
        if (kind == 0) {
            const double Sw = S.xy(0, 20), Swm = fma(c.m.mu, Sw, S.xy(1, 20));
            return -(S.w_ln_d() + fma(c.m.tau, Swm, Sw * c.m.lnc2));
        }
        if (kind == 1) return -phi(c, a) * S.xy(0, a);
        if (kind == 2) return phi(c, a) * phi(c, b) * S.yy(a, b) - pp(c, S, a, b);
        return phi(c, a) * phi(c, b) * S.ff(a, b);
    }
};

}  // namespace mf
