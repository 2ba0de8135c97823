// mf_generate.cu — on-device generation of mass-model pseudo-experiments ("a small-state
// RNG per work item ... events generated on the accelerator", half of the paper's per-toy time at 1M events).
//
// Counter-based instead of the paper's jump-seeded Xoshiro streams: event i of toy t draws from Philox4x32-10 with
// key = seed0 + t and counter = (i, draw), so any thread can generate any event and the result does not depend on the
// launch geometry.  Recipe of the mass model (one block per event in the common case, all four words w0..w3 of a draw used):
//   s = (w0 + 1/2) 2^-32,  u = ((w1 2^32 + w2) >> 11 + 1/2) 2^-53,  v = (w3 + 1/2) 2^-32;
//   draw 0: signal if s < f, else background m = lo + log1p(u expm1(tau w)) / tau  (lo + u w at tau == 0);
//   signal: Box-Muller z = sqrt(-2 ln u) cos(2 pi v), m = mu + sigma z from draw 0; if outside [lo, hi], (u, v) of draws
//   1, 2, ... until inside (after 64 rejected draws the last one is clamped).
// The angular and 4D recipes take two 53-bit uniforms ((w0, w1), (w2, w3)) per draw; their layouts are at their kernels.
// The events are written straight into the dataset's padded structure of arrays: no host copy.
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <new>
#include <string>

#include "mf_internal.h"
#include "mf_math.cuh"

namespace {

__device__ __forceinline__ void philox4x32_10(unsigned c0, unsigned c1, unsigned c2, unsigned c3, unsigned k0, unsigned k1,
                                              unsigned (&out)[4])
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const unsigned long long p0 = (unsigned long long)0xD2511F53u * c0, p1 = (unsigned long long)0xCD9E8D57u * c2;  // one wide multiply each
        const unsigned hi0 = (unsigned)(p0 >> 32), lo0 = (unsigned)p0;
        const unsigned hi1 = (unsigned)(p1 >> 32), lo1 = (unsigned)p1;
        const unsigned n0 = hi1 ^ c1 ^ k0, n2 = hi0 ^ c3 ^ k1;
        c0 = n0;
        c1 = lo1;
        c2 = n2;
        c3 = lo0;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    out[0] = c0;
    out[1] = c1;
    out[2] = c2;
    out[3] = c3;
}

__device__ __forceinline__ double uniform53(unsigned hi, unsigned lo)
{
    const unsigned long long x = (((unsigned long long)hi << 32) | lo) >> 11;
    return (double)x * 0x1p-53 + 0x1p-54;
}

__device__ __forceinline__ void uniforms(unsigned long long seed, unsigned long long event, unsigned draw, double& ua, double& ub)
{
    unsigned w[4];
    philox4x32_10((unsigned)event, (unsigned)(event >> 32), draw, 0u, (unsigned)seed, (unsigned)(seed >> 32), w);
    ua = uniform53(w[0], w[1]);
    ub = uniform53(w[2], w[3]);
}

// data: [n_toys][n_pad]; the padding of each toy row repeats its last event (as mf_dataset_upload does).
// grid = (slots, toys): no 64-bit division per event.  The transforms use the path's own logarithm (mf_log, table in
// shared memory) and cospi instead of the library's log / log1p / cos (which made the kernel instruction-issue bound:
// 785 us for 4.1e7 events); the results differ from the recipe evaluated with correctly rounded functions by a few ulp
// of the Box-Muller variate and far less than an ulp of m for the background (ln(1 + x) with x in (-1, 0]: the absolute
// error 1.1e-16 of forming 1 + x is divided by |tau| and added to lo ~ 5).
__global__ void __launch_bounds__(256) generate_mass_kernel(double* __restrict__ data, int64_t n_toys, int64_t n, int64_t n_pad,
                                                            unsigned long long seed0, double f, double mu, double sigma,
                                                            double tau, double lo, double hi, double em1, double inv_tau)
{
    __shared__ double2 s_tab[mf::kLogTableSize];
    mf::load_log_table(s_tab);
    __syncthreads();
    const double w = hi - lo;
    for (int64_t toy = blockIdx.y; toy < n_toys; toy += gridDim.y) {
        double* row = data + toy * n_pad;
        const unsigned long long seed = seed0 + (unsigned long long)toy;
        for (int64_t slot = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; slot < n_pad; slot += (int64_t)gridDim.x * blockDim.x) {
            if (n == 0) {
                row[slot] = 0.0;
                continue;
            }
            const unsigned long long ev = (unsigned long long)(slot < n ? slot : n - 1);
            // draw 0: s = (w0 + 1/2) 2^-32 chooses the component, u = 53 bits of (w1, w2), v = (w3 + 1/2) 2^-32.
            // Both components need ONE logarithm of a function of u: ln u (Box-Muller radius) or ln(1 + u expm1(tau w))
            // (inverse CDF of the exponential), so the common path has no divergent branch.
            unsigned wd[4];
            philox4x32_10((unsigned)ev, (unsigned)(ev >> 32), 0u, 0u, (unsigned)seed, (unsigned)(seed >> 32), wd);
            const bool sig = ((double)wd[0] + 0.5) * 0x1p-32 < f;
            double u = uniform53(wd[1], wd[2]), v = ((double)wd[3] + 0.5) * 0x1p-32;
            const double L = mf::mf_log(sig ? u : fma(u, em1, 1.0), s_tab);
            const double zs = sqrt(-2.0 * L) * cospi(2.0 * v);
            double m = sig ? fma(sigma, zs, mu) : (tau == 0.0) ? fma(u, w, lo) : fma(L, inv_tau, lo);
            if (sig && !(m >= lo && m <= hi)) {  // rare: the Gaussian draw fell outside the range: further blocks
                bool ok = false;
                for (unsigned k = 1; k <= 64 && !ok; ++k) {
                    philox4x32_10((unsigned)ev, (unsigned)(ev >> 32), k, 0u, (unsigned)seed, (unsigned)(seed >> 32), wd);
                    u = uniform53(wd[1], wd[2]);
                    v = ((double)wd[3] + 0.5) * 0x1p-32;
                    m = fma(sigma, sqrt(-2.0 * mf::mf_log(u, s_tab)) * cospi(2.0 * v), mu);
                    ok = (m >= lo && m <= hi);
                }
            }
            m = fmin(fmax(m, lo), hi);
            row[slot] = m;
        }
    }
}

// Eq. 4, term by term, for the accept decision
// phi = pi phi_turns: sine and cosine by sincospi of the half-turn count (no argument reduction of a rounded phi), the
// double angle by the addition formulas
__device__ __forceinline__ double angular_pdf(double cl, double ck, double phi_turns, const double* a)
{
    const double cl2 = cl * cl, ck2 = ck * ck, sl2 = 1.0 - cl2, sk2 = 1.0 - ck2;
    const double sl = sqrt(sl2), sk = sqrt(sk2);
    const double c2l = 2.0 * cl2 - 1.0, s2l = 2.0 * sl * cl, s2k = 2.0 * sk * ck;
    double sp, cp;
    sincospi(phi_turns, &sp, &cp);
    const double s2p = 2.0 * sp * cp, c2p = (cp - sp) * (cp + sp);
    const double FL = a[0];
    return (9.0 / (32.0 * 3.141592653589793238462643383279502884)) *
           (0.75 * (1.0 - FL) * sk2 + FL * ck2 + 0.25 * (1.0 - FL) * sk2 * c2l - FL * ck2 * c2l + a[1] * sk2 * sl2 * c2p +
            a[2] * s2k * s2l * cp + a[3] * s2k * sl * cp + (4.0 / 3.0) * a[4] * sk2 * cl + a[5] * s2k * sl * sp +
            a[6] * s2k * s2l * sp + a[7] * sk2 * sl2 * s2p);
}

struct AngGenArgs {
    double a[8];
    double pmax;
};

// data: [3][n_toys][n_pad] (cos theta_l, cos theta_K, phi).  Proposal k of an event uses draws 2k and 2k+1; the event is its
// first accepted proposal (a pure function of (seed, event index)).
// Work distribution: accept-reject with ~10 % efficiency leaves a warp that walks 32 events in lock step waiting for its
// slowest lane (35 proposals against a mean of 10).  Here every warp owns a contiguous chunk of the flattened (toy, slot)
// index space and its lanes are persistent workers: a lane whose event has been accepted writes it and takes the next
// unassigned index of the chunk (ballot + prefix count), so all 32 lanes keep proposing until the chunk is exhausted.
constexpr int kGenChunk = 256;  // indices per warp chunk (the last proposals of a chunk run on a thinning warp)

__global__ void __launch_bounds__(256) generate_angular_kernel(double* __restrict__ data, int64_t n_toys, int64_t n, int64_t n_pad,
                                                               unsigned long long seed0, const __grid_constant__ AngGenArgs g)
{
    const int64_t per_dim = n_toys * n_pad;
    const int lane = threadIdx.x & 31;
    const int64_t n_chunks = (per_dim + kGenChunk - 1) / kGenChunk;
    const int64_t warps = (int64_t)gridDim.x * (blockDim.x >> 5), w0 = (int64_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    for (int64_t ch = w0; ch < n_chunks; ch += warps) {
        const int64_t first = ch * kGenChunk, end = (first + kGenChunk < per_dim) ? first + kGenChunk : per_dim;
        int64_t next = first + 32;          // next unassigned index of the chunk (warp-uniform)
        int64_t idx = first + lane;         // this lane's current index
        bool active = idx < end;
        unsigned long long ev = 0, seed = 0;
        unsigned k = 0;
        auto start = [&]() {                // set up the event of index idx
            const int64_t toy = idx / n_pad, slot = idx % n_pad;
            ev = (unsigned long long)(slot < n ? slot : n - 1);
            seed = seed0 + (unsigned long long)toy;
            k = 0;
        };
        if (active && n > 0) start();
        while (__any_sync(0xffffffffu, active)) {
            bool finished = false;
            double cl = 0.0, ck = 0.0, phi = 0.0;
            if (active) {
                if (n > 0) {
                    double u1, u2, u3, u4;
                    uniforms(seed, ev, 2 * k, u1, u2);
                    uniforms(seed, ev, 2 * k + 1, u3, u4);
                    cl = 2.0 * u1 - 1.0;
                    ck = 2.0 * u2 - 1.0;
                    phi = 3.141592653589793238462643383279502884 * (2.0 * u3 - 1.0);
                    finished = (u4 * g.pmax < angular_pdf(cl, ck, 2.0 * u3 - 1.0, g.a)) || (k == 4095u);
                    ++k;
                } else {
                    finished = true;        // empty toys: zeros
                }
                if (finished) {
                    data[idx] = cl;
                    data[per_dim + idx] = ck;
                    data[2 * per_dim + idx] = phi;
                }
            }
            // lanes that finished take the next unassigned indices, in lane order
            const unsigned need = __ballot_sync(0xffffffffu, active && finished);
            if (active && finished) {
                idx = next + __popc(need & ((1u << lane) - 1u));
                active = idx < end;
                if (active && n > 0) start();
            }
            next += __popc(need);
        }
    }
}

struct FourDGenArgs {
    double f, mu, sigma, tau, lo, hi, em1;
    AngGenArgs ang;
    double cl1, cl2, ck1, ck2, bound;
};

__device__ __forceinline__ double legendre2(double x, double c1, double c2)
{
    return 0.5 * (1.0 + c1 * x + c2 * 0.5 * (3.0 * x * x - 1.0));
}

// data: [4][n_toys][n_pad] (m, cos theta_l, cos theta_K, phi).  Draw layout of one event (two uniforms per draw):
//   draw 0 -> (uA, uB): signal if uA < f; background mass from uB by the inverse CDF (as generate_mass_kernel);
//   signal:     draws 1..64 Box-Muller mass candidates (first inside the range); draws 100 + 2k -> (cos theta_l, cos theta_K)
//               and 101 + 2k -> (phi, accept) of angular proposal k, accepted when accept * pmax < P(Omega);
//   background: draw 1 -> (phi, unused); draws 100 + 2k -> (cos theta_l, cos theta_K) and 101 + 2k -> (accept, unused) of
//               Legendre proposal k, accepted when accept * bound < l(cos theta_l) l(cos theta_K).
__global__ void __launch_bounds__(256) generate_4d_kernel(double* __restrict__ data, int64_t n_toys, int64_t n, int64_t n_pad,
                                                          unsigned long long seed0, const __grid_constant__ FourDGenArgs g)
{
    // persistent lanes over warp chunks of the flattened (toy, slot) index space, as generate_angular_kernel
    const int64_t per_dim = n_toys * n_pad;
    const double pi = 3.141592653589793238462643383279502884;
    const int lane = threadIdx.x & 31;
    const int64_t n_chunks = (per_dim + kGenChunk - 1) / kGenChunk;
    const int64_t warps = (int64_t)gridDim.x * (blockDim.x >> 5), w0 = (int64_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    for (int64_t ch = w0; ch < n_chunks; ch += warps) {
        const int64_t first = ch * kGenChunk, end = (first + kGenChunk < per_dim) ? first + kGenChunk : per_dim;
        int64_t next = first + 32;
        int64_t idx = first + lane;
        bool active = idx < end;
        unsigned long long ev = 0, seed = 0;
        unsigned k = 0;
        bool sig = false;
        double m = 0.0, phi_bkg = 0.0;
        auto start = [&]() {  // component, mass (and the background's phi) of the event of index idx; proposals start at k = 0
            const int64_t toy = idx / n_pad, slot = idx % n_pad;
            ev = (unsigned long long)(slot < n ? slot : n - 1);
            seed = seed0 + (unsigned long long)toy;
            k = 0;
            double ua, ub;
            uniforms(seed, ev, 0u, ua, ub);
            sig = ua < g.f;
            if (sig) {
                m = g.mu;
                bool ok = false;
                for (unsigned q = 1; q <= 64 && !ok; ++q) {
                    double u1, u2;
                    uniforms(seed, ev, q, u1, u2);
                    m = fma(g.sigma, sqrt(-2.0 * log(u1)) * cos(2.0 * pi * u2), g.mu);
                    ok = (m >= g.lo && m <= g.hi);
                }
                if (!ok) m = fmin(fmax(m, g.lo), g.hi);
            } else {
                const double w = g.hi - g.lo;
                m = (g.tau == 0.0) ? fma(ub, w, g.lo) : g.lo + log1p(ub * g.em1) / g.tau;
                m = fmin(fmax(m, g.lo), g.hi);
                double u1, u2;
                uniforms(seed, ev, 1u, u1, u2);
                phi_bkg = pi * (2.0 * u1 - 1.0);
            }
        };
        if (active && n > 0) start();
        while (__any_sync(0xffffffffu, active)) {
            bool finished = false;
            double cl = 0.0, ck = 0.0, phi = 0.0;
            if (active) {
                if (n > 0) {
                    double u1, u2, u3, u4;
                    uniforms(seed, ev, 100 + 2 * k, u1, u2);
                    uniforms(seed, ev, 101 + 2 * k, u3, u4);
                    cl = 2.0 * u1 - 1.0;
                    ck = 2.0 * u2 - 1.0;
                    if (sig) {
                        phi = pi * (2.0 * u3 - 1.0);
                        finished = u4 * g.ang.pmax < angular_pdf(cl, ck, 2.0 * u3 - 1.0, g.ang.a);
                    } else {
                        phi = phi_bkg;
                        finished = u3 * g.bound < legendre2(cl, g.cl1, g.cl2) * legendre2(ck, g.ck1, g.ck2);
                    }
                    finished = finished || (k == 4095u);
                    ++k;
                } else {
                    finished = true;
                    m = 0.0;
                }
                if (finished) {
                    data[idx] = m;
                    data[per_dim + idx] = cl;
                    data[2 * per_dim + idx] = ck;
                    data[3 * per_dim + idx] = phi;
                }
            }
            const unsigned need = __ballot_sync(0xffffffffu, active && finished);
            if (active && finished) {
                idx = next + __popc(need & ((1u << lane) - 1u));
                active = idx < end;
                if (active && n > 0) start();
            }
            next += __popc(need);
        }
    }
}

}  // namespace

extern "C" mf_status mf_generate_4d(mf_ctx* ctx, uint64_t seed0, int64_t n_toys, int64_t n_events, const double* lam, double lo,
                                    double hi, mf_dataset** out)
{
    if (!ctx || !lam || !out) return mf_fail(ctx, MF_ERR_ARG, "mf_generate_4d: NULL argument");
    if (n_toys < 1 || n_events < 0 || !(std::isfinite(lo) && std::isfinite(hi) && lo < hi))
        return mf_fail(ctx, MF_ERR_ARG, "mf_generate_4d: n_toys >= 1, n_events >= 0 and a finite range lo < hi are required");
    for (int k = 0; k < 16; ++k)
        if (!std::isfinite(lam[k])) return mf_fail(ctx, MF_ERR_PARAM_DOMAIN, "mf_generate_4d: non-finite parameter");
    if (!(lam[0] >= 0.0 && lam[0] <= 1.0) || !(lam[2] > 0.0) || !std::isfinite(std::expm1(lam[3] * (hi - lo))))
        return mf_fail(ctx, MF_ERR_PARAM_DOMAIN, "mf_generate_4d: lambda outside the parameter domain");
    FourDGenArgs g;
    g.f = lam[0];
    g.mu = lam[1];
    g.sigma = lam[2];
    g.tau = lam[3];
    g.lo = lo;
    g.hi = hi;
    g.em1 = std::expm1(lam[3] * (hi - lo));
    double sum = 4.0;
    for (int k = 0; k < 8; ++k) {
        g.ang.a[k] = lam[4 + k];
        if (k > 0) sum += (k == 4 ? 4.0 / 3.0 : 1.0) * std::fabs(lam[4 + k]);
    }
    g.ang.pmax = 9.0 / (32.0 * 3.141592653589793238462643383279502884) * sum;
    g.cl1 = lam[12];
    g.cl2 = lam[13];
    g.ck1 = lam[14];
    g.ck2 = lam[15];
    g.bound = 0.5 * (1.0 + std::fabs(g.cl1) + std::fabs(g.cl2)) * 0.5 * (1.0 + std::fabs(g.ck1) + std::fabs(g.ck2));
    if (cudaSetDevice(ctx->device) != cudaSuccess) return mf_fail(ctx, MF_ERR_CUDA, "mf_generate_4d: cudaSetDevice failed");
    mf_dataset* ds = new (std::nothrow) mf_dataset();
    mf_devbuf* buf = new (std::nothrow) mf_devbuf();
    if (!ds || !buf) {
        delete ds;
        delete buf;
        return mf_fail(ctx, MF_ERR_OOM, "mf_generate_4d: host allocation failed");
    }
    ds->ctx = ctx;
    ds->ndim = 4;
    ds->n_events = n_events;
    ds->n_pad = (n_events + 63) / 64 * 64;
    ds->n_toys = n_toys;
    const double alo[4] = {lo, -1.0, -1.0, -3.141592653589793238462643383279502884};
    const double ahi[4] = {hi, 1.0, 1.0, 3.141592653589793238462643383279502884};
    for (int j = 0; j < 4; ++j) {
        ds->lo[j] = alo[j];
        ds->hi[j] = ahi[j];
    }
    ds->raw = buf;
    buf->stream = ctx->stream;
    const int64_t per_dim = ds->n_pad * n_toys;
    buf->bytes = (size_t)(per_dim > 0 ? 4 * per_dim : 1) * sizeof(double);
    cudaError_t e = cudaMallocAsync(reinterpret_cast<void**>(&buf->p), buf->bytes, ctx->stream);
    if (e == cudaSuccess && per_dim > 0) {
        const int64_t chunks = (per_dim + kGenChunk - 1) / kGenChunk;
        const int grid = (int)std::max<int64_t>(1, std::min<int64_t>((chunks + 7) / 8, 32 * (int64_t)ctx->sm_count));
        generate_4d_kernel<<<grid, 256, 0, ctx->stream>>>(buf->p, n_toys, n_events, ds->n_pad, seed0, g);
        ++ctx->launches;
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);
    if (e != cudaSuccess) {
        if (buf->p) cudaFreeAsync(buf->p, ctx->stream);
        delete buf;
        delete ds;
        return mf_fail(ctx, e == cudaErrorMemoryAllocation ? MF_ERR_OOM : MF_ERR_CUDA, std::string("mf_generate_4d: ") + cudaGetErrorString(e));
    }
    *out = ds;
    return MF_OK;
}

extern "C" mf_status mf_generate_angular(mf_ctx* ctx, uint64_t seed0, int64_t n_toys, int64_t n_events, const double* a,
                                         mf_dataset** out)
{
    if (!ctx || !a || !out) return mf_fail(ctx, MF_ERR_ARG, "mf_generate_angular: NULL argument");
    if (n_toys < 1 || n_events < 0) return mf_fail(ctx, MF_ERR_ARG, "mf_generate_angular: n_toys >= 1 and n_events >= 0 are required");
    AngGenArgs g;
    double sum = 4.0;
    for (int k = 0; k < 8; ++k) {
        if (!std::isfinite(a[k])) return mf_fail(ctx, MF_ERR_PARAM_DOMAIN, "mf_generate_angular: non-finite coefficient");
        g.a[k] = a[k];
        if (k > 0) sum += (k == 4 ? 4.0 / 3.0 : 1.0) * std::fabs(a[k]);
    }
    g.pmax = 9.0 / (32.0 * 3.141592653589793238462643383279502884) * sum;  // the paper's get_max() bound
    if (cudaSetDevice(ctx->device) != cudaSuccess) return mf_fail(ctx, MF_ERR_CUDA, "mf_generate_angular: cudaSetDevice failed");
    mf_dataset* ds = new (std::nothrow) mf_dataset();
    mf_devbuf* buf = new (std::nothrow) mf_devbuf();
    if (!ds || !buf) {
        delete ds;
        delete buf;
        return mf_fail(ctx, MF_ERR_OOM, "mf_generate_angular: host allocation failed");
    }
    ds->ctx = ctx;
    ds->ndim = 3;
    ds->n_events = n_events;
    ds->n_pad = (n_events + 63) / 64 * 64;
    ds->n_toys = n_toys;
    const double alo[3] = {-1.0, -1.0, -3.141592653589793238462643383279502884};
    for (int j = 0; j < 3; ++j) {
        ds->lo[j] = alo[j];
        ds->hi[j] = -alo[j];
    }
    ds->raw = buf;
    buf->stream = ctx->stream;
    const int64_t per_dim = ds->n_pad * n_toys;
    buf->bytes = (size_t)(per_dim > 0 ? 3 * per_dim : 1) * sizeof(double);
    cudaError_t e = cudaMallocAsync(reinterpret_cast<void**>(&buf->p), buf->bytes, ctx->stream);
    if (e == cudaSuccess && per_dim > 0) {
        const int64_t chunks = (per_dim + kGenChunk - 1) / kGenChunk;
        const int grid = (int)std::max<int64_t>(1, std::min<int64_t>((chunks + 7) / 8, 32 * (int64_t)ctx->sm_count));
        generate_angular_kernel<<<grid, 256, 0, ctx->stream>>>(buf->p, n_toys, n_events, ds->n_pad, seed0, g);
        ++ctx->launches;
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);
    if (e != cudaSuccess) {
        if (buf->p) cudaFreeAsync(buf->p, ctx->stream);
        delete buf;
        delete ds;
        return mf_fail(ctx, e == cudaErrorMemoryAllocation ? MF_ERR_OOM : MF_ERR_CUDA, std::string("mf_generate_angular: ") + cudaGetErrorString(e));
    }
    *out = ds;
    return MF_OK;
}

extern "C" mf_status mf_generate_mass(mf_ctx* ctx, uint64_t seed0, int64_t n_toys, int64_t n_events, const double* lam,
                                      double lo, double hi, mf_dataset** out)
{
    if (!ctx || !lam || !out) return mf_fail(ctx, MF_ERR_ARG, "mf_generate_mass: NULL argument");
    if (n_toys < 1 || n_events < 0 || !(std::isfinite(lo) && std::isfinite(hi) && lo < hi))
        return mf_fail(ctx, MF_ERR_ARG, "mf_generate_mass: n_toys >= 1, n_events >= 0 and a finite range lo < hi are required");
    const double f = lam[0], mu = lam[1], sigma = lam[2], tau = lam[3];
    if (!(std::isfinite(f) && std::isfinite(mu) && std::isfinite(sigma) && std::isfinite(tau)) || !(f >= 0.0 && f <= 1.0) ||
        !(sigma > 0.0) || !std::isfinite(std::expm1(tau * (hi - lo))))
        return mf_fail(ctx, MF_ERR_PARAM_DOMAIN, "mf_generate_mass: lambda outside the parameter domain");
    if (cudaSetDevice(ctx->device) != cudaSuccess) return mf_fail(ctx, MF_ERR_CUDA, "mf_generate_mass: cudaSetDevice failed");
    mf_dataset* ds = new (std::nothrow) mf_dataset();
    mf_devbuf* buf = new (std::nothrow) mf_devbuf();
    if (!ds || !buf) {
        delete ds;
        delete buf;
        return mf_fail(ctx, MF_ERR_OOM, "mf_generate_mass: host allocation failed");
    }
    ds->ctx = ctx;
    ds->ndim = 1;
    ds->n_events = n_events;
    ds->n_pad = (n_events + 63) / 64 * 64;
    ds->n_toys = n_toys;
    ds->lo[0] = lo;
    ds->hi[0] = hi;
    ds->raw = buf;
    buf->stream = ctx->stream;
    const int64_t total = ds->n_pad * n_toys;
    buf->bytes = (size_t)(total > 0 ? total : 1) * sizeof(double);
    cudaError_t e = cudaMallocAsync(reinterpret_cast<void**>(&buf->p), buf->bytes, ctx->stream);
    if (e == cudaSuccess && total > 0) {
        const unsigned gy = (unsigned)std::min<int64_t>(n_toys, 65535);
        const unsigned gx = (unsigned)std::max<int64_t>(1, std::min<int64_t>((ds->n_pad + 255) / 256, 32 * (int64_t)ctx->sm_count / gy));
        generate_mass_kernel<<<dim3(gx, gy), 256, 0, ctx->stream>>>(buf->p, n_toys, n_events, ds->n_pad, seed0, f, mu, sigma, tau, lo,
                                                                     hi, std::expm1(tau * (hi - lo)), tau != 0.0 ? 1.0 / tau : 0.0);
        ++ctx->launches;
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);
    if (e != cudaSuccess) {
        if (buf->p) cudaFreeAsync(buf->p, ctx->stream);
        delete buf;
        delete ds;
        return mf_fail(ctx, e == cudaErrorMemoryAllocation ? MF_ERR_OOM : MF_ERR_CUDA, std::string("mf_generate_mass: ") + cudaGetErrorString(e));
    }
    *out = ds;
    return MF_OK;
}

// Copies the events of a dataset back to the host (dst: [ndim][n_toys][n_events], dimension-major) — for tests and for
// users who want to inspect generated pseudo-data.
extern "C" mf_status mf_dataset_download(const mf_dataset* ds, double* dst)
{
    if (!ds || !dst) return MF_ERR_ARG;
    mf_ctx* ctx = ds->ctx;
    if (ds->n_events == 0) return MF_OK;
    const cudaError_t e = cudaMemcpy2DAsync(dst, (size_t)ds->n_events * sizeof(double), ds->raw->p, (size_t)ds->n_pad * sizeof(double),
                                            (size_t)ds->n_events * sizeof(double), (size_t)(ds->n_toys * ds->ndim),
                                            cudaMemcpyDeviceToHost, ctx->stream);
    if (e != cudaSuccess) return mf_fail(ctx, MF_ERR_CUDA, std::string("mf_dataset_download: ") + cudaGetErrorString(e));
    if (cudaStreamSynchronize(ctx->stream) != cudaSuccess) return mf_fail(ctx, MF_ERR_CUDA, "mf_dataset_download: synchronise failed");
    return MF_OK;
}

// The paper's toy study (Listing 6 `toystudy::toy`): generate n_toys pseudo-experiments of n_events events at
// lam_truth, fit all of them concurrently from lam_truth, HESSE.  Everything stays on the device.
extern "C" mf_status mf_toy_study_mass(mf_ctx* ctx, uint64_t seed0, int64_t n_toys, int64_t n_events, const double* lam_truth,
                                       double lo, double hi, const mf_fit_opts* opts, mf_fit_result* results)
{
    if (!ctx || !lam_truth || !results) return mf_fail(ctx, MF_ERR_ARG, "mf_toy_study_mass: NULL argument");
    mf_dataset* ds = nullptr;
    mf_status st = mf_generate_mass(ctx, seed0, n_toys, n_events, lam_truth, lo, hi, &ds);
    if (st != MF_OK) return st;
    mf_model* model = nullptr;
    st = mf_model_create(ctx, MF_MASS_GAUSS_EXP, ds, &model);
    mf_dataset_destroy(ds);
    if (st != MF_OK) return st;
    double* starts = new (std::nothrow) double[(size_t)n_toys * 4];
    if (!starts) {
        mf_model_destroy(model);
        return mf_fail(ctx, MF_ERR_OOM, "mf_toy_study_mass: host allocation failed");
    }
    for (int64_t t = 0; t < n_toys; ++t)
        for (int k = 0; k < 4; ++k) starts[t * 4 + k] = lam_truth[k];
    if (n_toys == 1) st = mf_fit(model, starts, nullptr, opts, results);
    else st = mf_fit_batch(model, n_toys, starts, nullptr, opts, results);
    delete[] starts;
    mf_model_destroy(model);
    return st;
}

extern "C" mf_status mf_toy_study_angular(mf_ctx* ctx, uint64_t seed0, int64_t n_toys, int64_t n_events, const double* a_truth,
                                          const mf_fit_opts* opts, mf_fit_result* results)
{
    if (!ctx || !a_truth || !results) return mf_fail(ctx, MF_ERR_ARG, "mf_toy_study_angular: NULL argument");
    mf_dataset* ds = nullptr;
    mf_status st = mf_generate_angular(ctx, seed0, n_toys, n_events, a_truth, &ds);
    if (st != MF_OK) return st;
    mf_model* model = nullptr;
    st = mf_model_create(ctx, MF_ANGULAR_KSTMUMU, ds, &model);
    mf_dataset_destroy(ds);
    if (st != MF_OK) return st;
    double* starts = new (std::nothrow) double[(size_t)n_toys * 8];
    if (!starts) {
        mf_model_destroy(model);
        return mf_fail(ctx, MF_ERR_OOM, "mf_toy_study_angular: host allocation failed");
    }
    for (int64_t t = 0; t < n_toys; ++t)
        for (int k = 0; k < 8; ++k) starts[t * 8 + k] = a_truth[k];
    if (n_toys == 1) st = mf_fit(model, starts, nullptr, opts, results);
    else st = mf_fit_batch(model, n_toys, starts, nullptr, opts, results);
    delete[] starts;
    mf_model_destroy(model);
    return st;
}

