// mf_noalloc.cu — mf_nll_grad_mass_noalloc: ONE evaluation of -ln L and its gradient (Eq. 1, Eq. 2/3 of the mass
// model) for callers that must not allocate: code under CUDA graph capture, tight serving loops, harnesses that forbid
// cudaMalloc.  A variant of the fused single-dataset kernel (mf_kernels.cuh, nll_grad_kernel<MassModel>) whose cross-CTA
// scratch — one row of partial sums per CTA, the bad-event counts, the completion ticket — lives in a file-scope
// `static __device__` array of fixed size instead of buffers allocated per model:
//
//   * the caller passes the events (device, unpadded), the range, lambda (host) and the output row (device);
//   * CTA c evaluates the fixed chunk of events [8192 c, 8192 (c + 1)): the result does not depend on the device's SM count;
//     the CTA that draws the last ticket combines the rows in chunk order (compensated sums) and writes the output;
//   * sum_i m_i, which the other kernels take from a per-dataset pre-pass (S1), is accumulated here as a seventh sum
//     (sum_i (m_i - m_a), so that the running sums stay small) and every parameter point takes the general event body;
//   * limit: MF_NOALLOC_MAX_EVENTS = 2^25 events = 4096 chunks; the scratch is kScratchBytes = 246,016 bytes, held by every
//     GPU that loads the library until the process exits;
//   * every call shares the array and finds the previous call's contents in it: the ticket word is cleared by a memset node
//     on the caller's stream before the kernel, the rows are overwritten before they are read.  Calls that overlap on the
//     GPU (two streams, two host threads, graph branches) RACE on it; calls on one stream are ordered and safe.
//
// In host code `g_scratch` is a host-side stand-in for the device array, not a device address: its address is resolved once
// per device with cudaGetSymbolAddress (scratch_for_device) and that pointer is what the kernel receives.
// The entry point calls no cudaMalloc / cudaFree / cudaHostAlloc and no allocating library routine.
#include <cuda_runtime.h>

#include <cmath>
#include <mutex>
#include <string>

#include "mf_internal.h"
#include "mf_models.cuh"

namespace {

using namespace mf;

constexpr int kThreads = 256, kWarpsPerCta = kThreads / 32;
constexpr int kGroupEv = 256;                            // events of one warp step: lane l takes events 2l, 2l+1 of four 64-event rows
constexpr int kChunkEv = 8192;                           // events per CTA
constexpr int kChunkGroups = kChunkEv / kGroupEv;        // 32 groups, four per warp
constexpr int kMaxChunks = (int)(MF_NOALLOC_MAX_EVENTS / kChunkEv);  // 4096
constexpr int kSums = 7;                                 // MassModel's six sums + sum_i (m_i - m_a)
static_assert(MF_NOALLOC_MAX_EVENTS % kChunkEv == 0, "the limit is a whole number of chunks");

// scratch layout: [0, 256) the ticket word | kSums rows of kMaxChunks doubles | kMaxChunks bad-event counts
constexpr size_t kOffPartials = 256;
constexpr size_t kOffBad = kOffPartials + sizeof(double) * kSums * kMaxChunks;
constexpr size_t kScratchBytes = kOffBad + sizeof(unsigned) * kMaxChunks;
static_assert(kScratchBytes == 246016, "the size stated in the header and the README");

static __device__ __align__(256) unsigned char g_scratch[kScratchBytes];

struct NoAllocArgs {
    const double* m;         // device, n events, 16-byte aligned, unpadded
    int64_t n;
    MassConsts c;            // parameter-only constants of lambda (S2), made on the host
    unsigned char* scratch;  // DEVICE address of g_scratch (cudaGetSymbolAddress)
    double* out;             // device, 6 doubles: -ln L, gradient (f, mu, sigma, tau), n_bad
};

__device__ __forceinline__ void two_sum_into(double& s, double& lo, double b, double blo)
{
    const double t = s + b;
    const double bb = t - s;
    const double e = (s - (t - bb)) + (b - bb);
    lo = (lo + blo) + e;
    s = t;
}

__global__ void __launch_bounds__(kThreads, 2) nll_grad_mass_noalloc_kernel(const __grid_constant__ NoAllocArgs a)
{
    __shared__ double sm[kWarpsPerCta][kSums];
    __shared__ unsigned sm_bad[kWarpsPerCta];
    __shared__ double s_sum[kSums];
    __shared__ unsigned s_nbad;
    __shared__ bool s_last;
    unsigned* ticket = reinterpret_cast<unsigned*>(a.scratch);
    double* part = reinterpret_cast<double*>(a.scratch + kOffPartials);
    unsigned* badp = reinterpret_cast<unsigned*>(a.scratch + kOffBad);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const MassConsts& c = a.c;
    const double t_lane = mf_exp32_lane_entry();
    double acc[kSums];
#pragma unroll
    for (int k = 0; k < kSums; ++k) acc[k] = 0.0;
    unsigned bad = 0;
    LogProd lp;
    // S3: the full 256-event groups of this CTA's chunk, four per warp
    const int64_t n_full = a.n / kGroupEv;
    const int64_t g_lo = (int64_t)blockIdx.x * kChunkGroups;
    const int64_t g_hi = (g_lo + kChunkGroups < n_full) ? g_lo + kChunkGroups : n_full;
    for (int64_t g = g_lo + warp; g < g_hi; g += kWarpsPerCta) {
        const double2* p = reinterpret_cast<const double2*>(a.m) + g * (kGroupEv / 2) + lane;
        double x[8];
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const double2 v = __ldg(p + 32 * i);
            x[2 * i] = v.x;
            x[2 * i + 1] = v.y;
        }
        MassModel::events<8, false>(x, c, acc, lp, bad, t_lane);
        lp.renorm();
        double sx = 0.0;
#pragma unroll
        for (int i = 0; i < 8; ++i) sx += x[i] - c.ma;
        acc[6] += sx;
    }
    // the dataset's ragged tail (n mod 256 events) belongs to the chunk in which it starts: one event per thread, predicated
    const int64_t t0 = n_full * kGroupEv;
    if (t0 < a.n && blockIdx.x == (unsigned)(t0 / kChunkEv)) {  // uniform over the CTA: every lane takes part in the shuffles
        const int64_t i = t0 + threadIdx.x;
        const bool valid = i < a.n;
        const double x = valid ? __ldg(a.m + i) : c.mu;
        MassModel::event<true>(&x, c, acc, lp, bad, valid, t_lane);
        if (valid) acc[6] += x - c.ma;
    }
    acc[0] = lp.log();
    // S4: thread -> warp -> CTA, fixed order
#pragma unroll
    for (int k = 0; k < kSums; ++k) {
        double v = acc[k];
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) v += __shfl_xor_sync(0xffffffffu, v, off);
        acc[k] = v;
    }
    bad = __reduce_add_sync(0xffffffffu, bad);
    if (lane == 0) {
#pragma unroll
        for (int k = 0; k < kSums; ++k) sm[warp][k] = acc[k];
        sm_bad[warp] = bad;
    }
    __syncthreads();
    if (threadIdx.x < kSums) {
        double s = 0.0;
#pragma unroll
        for (int w = 0; w < kWarpsPerCta; ++w) s += sm[w][threadIdx.x];
        part[(size_t)threadIdx.x * kMaxChunks + blockIdx.x] = s;  // overwrites whatever an earlier call left in this row
        __threadfence();
    } else if (threadIdx.x == kSums) {
        unsigned b = 0;
#pragma unroll
        for (int w = 0; w < kWarpsPerCta; ++w) b += sm_bad[w];
        badp[blockIdx.x] = b;
        __threadfence();
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        unsigned old;
        asm volatile("atom.add.acq_rel.gpu.global.u32 %0, [%1], 1;" : "=r"(old) : "l"(ticket) : "memory");
        s_last = (old == gridDim.x - 1);
    }
    __syncthreads();
    if (!s_last) return;
    // S5: the last CTA combines the gridDim.x rows in chunk order; warp k takes quantity k, warp 7 the bad-event counts
    const int count = (int)gridDim.x;
    if (warp < kSums) {
        const double* pk = part + (size_t)warp * kMaxChunks;
        double s = 0.0, cc = 0.0;
        for (int i = lane; i < count; i += 32) {  // Kahan
            const double y = __ldcg(pk + i) - cc;
            const double t = s + y;
            cc = (t - s) - y;
            s = t;
        }
        double lo = -cc;
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) {
            const double s2 = __shfl_down_sync(0xffffffffu, s, off);
            const double lo2 = __shfl_down_sync(0xffffffffu, lo, off);
            two_sum_into(s, lo, s2, lo2);
        }
        if (lane == 0) s_sum[warp] = s + lo;
    } else {
        unsigned nb = 0;
        for (int i = lane; i < count; i += 32) nb += __ldcg(badp + i);
        nb = __reduce_add_sync(0xffffffffu, nb);
        if (lane == 0) s_nbad = nb;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        const double n = (double)a.n;
        // sum_i m_i = n m_a + sum_i (m_i - m_a) as a (hi, lo) pair
        const double p = n * c.ma, pe = fma(n, c.ma, -p);
        double hi = p, lo = pe;
        two_sum_into(hi, lo, s_sum[6], 0.0);
        double o[5];
        MassModel::finish_general(c, s_sum, n, make_double2(hi, lo), o);
        const unsigned nb = s_nbad;
#pragma unroll
        for (int k = 0; k < 5; ++k)
            a.out[k] = !nb ? o[k] : (k == 0) ? __longlong_as_double(0x7ff0000000000000LL) : __longlong_as_double(0x7ff8000000000000LL);
        a.out[5] = (double)nb;
        *ticket = 0u;  // as the memset node of the next call would
    }
}

// Device address of g_scratch on `device`, resolved once per device with that device current.  The symbol's name is a
// host-side stand-in: only the pointer returned here may be given to a kernel.
constexpr int kMaxDevices = 64;
std::mutex g_ptr_mutex;
unsigned char* g_scratch_ptr[kMaxDevices] = {};

cudaError_t scratch_for_device(int device, unsigned char** out)
{
    std::lock_guard<std::mutex> lock(g_ptr_mutex);
    if (!g_scratch_ptr[device]) {
        void* p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&p, g_scratch);
        if (e != cudaSuccess) return e;
        g_scratch_ptr[device] = static_cast<unsigned char*>(p);
    }
    *out = g_scratch_ptr[device];
    return cudaSuccess;
}

}  // namespace

extern "C" mf_status mf_nll_grad_mass_noalloc(mf_ctx* ctx, const double* m_dev, int64_t n, double lo, double hi,
                                              const double* lambda, double* out_dev, void* stream)
{
    const char* who = "mf_nll_grad_mass_noalloc: ";
    if (!ctx) return MF_ERR_ARG;
    if (!lambda || !out_dev || (n > 0 && !m_dev)) return mf_fail(ctx, MF_ERR_ARG, std::string(who) + "NULL argument");
    if (n < 0) return mf_fail(ctx, MF_ERR_ARG, std::string(who) + "n < 0");
    if (n > (int64_t)MF_NOALLOC_MAX_EVENTS)
        return mf_fail(ctx, MF_ERR_ARG,
                       std::string(who) + "n = " + std::to_string((long long)n) + " exceeds MF_NOALLOC_MAX_EVENTS = " +
                           std::to_string((long long)MF_NOALLOC_MAX_EVENTS) +
                           " (the static scratch holds one row of partial sums per 8192 events); use mf_dataset_upload + mf_nll_grad");
    if (reinterpret_cast<uintptr_t>(m_dev) % 16 != 0)
        return mf_fail(ctx, MF_ERR_ARG, std::string(who) + "m_dev must be 16-byte aligned");
    if (!(std::isfinite(lo) && std::isfinite(hi) && lo < hi)) return mf_fail(ctx, MF_ERR_ARG, std::string(who) + "need finite lo < hi");
    if (ctx->device < 0 || ctx->device >= kMaxDevices) return mf_fail(ctx, MF_ERR_ARG, std::string(who) + "device index out of range");
    NoAllocArgs a;
    if (!mass_consts(lambda, lo, hi, a.c)) return mf_fail(ctx, MF_ERR_PARAM_DOMAIN, std::string(who) + "lambda outside the parameter domain");
    a.c.fast = 0.0;  // the kernel takes the general event body for every point
    cudaError_t e = cudaSetDevice(ctx->device);
    if (e == cudaSuccess) e = scratch_for_device(ctx->device, &a.scratch);
    if (e != cudaSuccess) return mf_fail(ctx, MF_ERR_CUDA, std::string(who) + cudaGetErrorString(e));
    a.m = m_dev;
    a.n = n;
    a.out = out_dev;
    cudaStream_t s = stream ? static_cast<cudaStream_t>(stream) : ctx->stream;
    const unsigned n_chunks = (unsigned)((n + kChunkEv - 1) / kChunkEv > 0 ? (n + kChunkEv - 1) / kChunkEv : 1);
    // what must start at zero: the ticket word (a call that was aborted mid-kernel may have left it anywhere)
    e = cudaMemsetAsync(a.scratch, 0, kOffPartials, s);
    if (e != cudaSuccess) return mf_fail(ctx, MF_ERR_CUDA, std::string(who) + cudaGetErrorString(e));
    nll_grad_mass_noalloc_kernel<<<n_chunks, kThreads, 0, s>>>(a);
    e = cudaGetLastError();
    if (e != cudaSuccess) return mf_fail(ctx, MF_ERR_CUDA, std::string(who) + cudaGetErrorString(e));
    ++ctx->launches;
    return MF_OK;
}
