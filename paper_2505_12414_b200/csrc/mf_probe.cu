// mf_probe.cu — measurement and test probes, built into their OWN library (lib/libmorefit_b200_probe.so, declared in
// mf_probe.h); they are not part of the product library nor of its public header.
//   * the two roofline denominators that MEASURED_PEAKS.json does not hold: the fp64-pipe issue
//     rate (register-only DFMA chains) and the read bandwidth of a working set that is re-read in a loop (L2-resident
//     when it fits the 126 MB L2, HBM otherwise) — used by bench.py;
//   * element-wise evaluation of the kernels' own device math (mf_math.cuh) — used by the accuracy tests.
// Every entry takes the CUDA device and stream directly and returns 0 or the cudaError_t that stopped it.
#include <cuda_runtime.h>

#include <cstdint>

#include "mf_math.cuh"
#include "mf_probe.h"

namespace {

// 8 independent DFMA chains per thread: enough ILP to cover the pipe latency at any occupancy.
__global__ void __launch_bounds__(256) dfma_chain_kernel(double* out, int iters, double a, double b)
{
    double x0 = threadIdx.x, x1 = x0 + 1, x2 = x0 + 2, x3 = x0 + 3, x4 = x0 + 4, x5 = x0 + 5, x6 = x0 + 6, x7 = x0 + 7;
#pragma unroll 1
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            x0 = fma(x0, a, b); x1 = fma(x1, a, b); x2 = fma(x2, a, b); x3 = fma(x3, a, b);
            x4 = fma(x4, a, b); x5 = fma(x5, a, b); x6 = fma(x6, a, b); x7 = fma(x7, a, b);
        }
    }
    const double s = ((x0 + x1) + (x2 + x3)) + ((x4 + x5) + (x6 + x7));
    if (s == 123.456) out[0] = s;  // never true for these inputs; keeps the chains alive
}

// fp64 tensor-core rate (DMMA m8n8k4) and whether it shares the issue rate of the vector fp64 pipe: N_MMA independent
// accumulator tiles and N_FMA independent DFMA chains per warp and iteration (either may be 0).
__device__ __forceinline__ void dmma(double& c0, double& c1, double a, double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};" : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

template <int N_MMA, int N_FMA>
__global__ void __launch_bounds__(256) dmma_mix_kernel(double* out, int iters, double a, double b)
{
    double c[8][2], x[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        c[i][0] = threadIdx.x + i;
        c[i][1] = threadIdx.x - i;
        x[i] = threadIdx.x + 0.5 * i;
    }
#pragma unroll 1
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < 4; ++u) {
#pragma unroll
            for (int i = 0; i < N_MMA; ++i) dmma(c[i][0], c[i][1], a, b);
#pragma unroll
            for (int i = 0; i < N_FMA; ++i) x[i] = fma(x[i], a, b);
        }
    }
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < 8; ++i) s += c[i][0] + c[i][1] + x[i];
    if (s == 123.456) out[0] = s;
}

__global__ void __launch_bounds__(256) read_kernel(const double2* __restrict__ p, size_t n_vec, int repeats, double* out)
{
    double s = 0.0;
    for (int r = 0; r < repeats; ++r)
        for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n_vec; i += (size_t)gridDim.x * blockDim.x) {
            const double2 v = __ldg(p + i);
            s += v.x + v.y;
        }
    if (s == 123.456) out[0] = s;
}


// Element-wise evaluation of the device math of mf_math.cuh (op 0: mf_exp, 1: mf_log, 2: mf_rcp, 3: mf_exp32).
__global__ void __launch_bounds__(256) math_kernel(int op, int64_t n, const double* __restrict__ x, double* __restrict__ y)
{
    __shared__ double2 s_tab[mf::kLogTableSize];
    mf::load_log_table(s_tab);
    __syncthreads();
    const double t_lane = mf::mf_exp32_lane_entry();
    // whole warps iterate together (mf_exp32 shuffles across the warp); lanes past n compute on 0
    const int64_t n_round = (n + 31) / 32 * 32;
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n_round; i += (int64_t)gridDim.x * blockDim.x) {
        const double v = i < n ? x[i] : 0.0;
        const double r = op == 3 ? mf::mf_exp32(v, t_lane) : op == 0 ? mf::mf_exp(v) : op == 1 ? mf::mf_log(v, s_tab) : mf::mf_rcp(v);
        if (i < n) y[i] = r;
    }
}

}  // namespace

#define MF_CUDA(ctx, call)                  \
    do {                                    \
        cudaError_t e__ = (call);           \
        if (e__ != cudaSuccess) return (int)e__; \
    } while (0)

struct ProbeCtx {
    int device;
    cudaStream_t stream;
    int sm_count;
};

static int probe_ctx(int device, void* stream, ProbeCtx* c)
{
    c->device = device;
    c->stream = static_cast<cudaStream_t>(stream);
    c->sm_count = 0;
    MF_CUDA(c, cudaSetDevice(device));
    MF_CUDA(c, cudaDeviceGetAttribute(&c->sm_count, cudaDevAttrMultiProcessorCount, device));
    return 0;
}

extern "C" int mfp_fp64_rate(int device, void* stream, double* dfma_per_second)
{
    if (!dfma_per_second) return (int)cudaErrorInvalidValue;
    ProbeCtx pc, *ctx = &pc;
    if (const int e = probe_ctx(device, stream, ctx)) return e;
    double* d_out = nullptr;
    MF_CUDA(ctx, cudaMalloc(&d_out, sizeof(double)));
    cudaEvent_t e0, e1;
    MF_CUDA(ctx, cudaEventCreate(&e0));
    MF_CUDA(ctx, cudaEventCreate(&e1));
    const int grid = ctx->sm_count * 4, iters = 4096;
    double best = 0.0;
    for (int rep = 0; rep < 6; ++rep) {
        MF_CUDA(ctx, cudaEventRecord(e0, ctx->stream));
        dfma_chain_kernel<<<grid, 256, 0, ctx->stream>>>(d_out, iters, 0.999999, 1e-9);
        MF_CUDA(ctx, cudaEventRecord(e1, ctx->stream));
        MF_CUDA(ctx, cudaEventSynchronize(e1));
        float ms = 0;
        MF_CUDA(ctx, cudaEventElapsedTime(&ms, e0, e1));
        const double rate = (double)grid * 256.0 * 64.0 * iters / (ms * 1e-3);
        if (rep > 0 && rate > best) best = rate;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(d_out);
    *dfma_per_second = best;
    return 0;
}

template <int N_MMA, int N_FMA>
static int time_mix(ProbeCtx* ctx, double* d_out, double* seconds)
{
    cudaEvent_t e0, e1;
    MF_CUDA(ctx, cudaEventCreate(&e0));
    MF_CUDA(ctx, cudaEventCreate(&e1));
    const int grid = ctx->sm_count * 4, iters = 2048;
    double best = 1e30;
    for (int rep = 0; rep < 5; ++rep) {
        MF_CUDA(ctx, cudaEventRecord(e0, ctx->stream));
        dmma_mix_kernel<N_MMA, N_FMA><<<grid, 256, 0, ctx->stream>>>(d_out, iters, 0.999999, 1e-9);
        MF_CUDA(ctx, cudaEventRecord(e1, ctx->stream));
        MF_CUDA(ctx, cudaEventSynchronize(e1));
        float ms = 0;
        MF_CUDA(ctx, cudaEventElapsedTime(&ms, e0, e1));
        if (rep > 0 && ms * 1e-3 < best) best = ms * 1e-3;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    *seconds = best;
    return 0;
}

extern "C" int mfp_dmma_rate(int device, void* stream, double* out4)
{
    if (!out4) return (int)cudaErrorInvalidValue;
    ProbeCtx pc, *ctx = &pc;
    if (const int e = probe_ctx(device, stream, ctx)) return e;
    double* d_out = nullptr;
    MF_CUDA(ctx, cudaMalloc(&d_out, sizeof(double)));
    const double warps = (double)ctx->sm_count * 4 * 8, steps = 2048.0 * 4;
    double t_mma = 0, t_fma = 0, t_both = 0, t_both2 = 0;
    if (const int e = time_mix<4, 0>(ctx, d_out, &t_mma)) return e;
    if (const int e = time_mix<0, 8>(ctx, d_out, &t_fma)) return e;
    if (const int e = time_mix<4, 8>(ctx, d_out, &t_both)) return e;
    if (const int e = time_mix<1, 8>(ctx, d_out, &t_both2)) return e;
    cudaFree(d_out);
    out4[0] = warps * steps * 4 * 256.0 / t_mma;        // DMMA alone: fp64 FMAs per second (m8n8k4 = 256 FMAs)
    out4[1] = warps * steps * 8 * 32.0 / t_fma;         // DFMA alone: FMAs per second
    out4[2] = t_both / (t_mma + t_fma);                 // 4 DMMA + 8 DFMA: 1.0 = the two serialise, max/sum = they overlap fully
    out4[3] = t_both2 / (t_fma + 0.25 * t_mma);         // 1 DMMA + 8 DFMA
    return 0;
}

extern "C" int mfp_read_bandwidth(int device, void* stream, size_t bytes, int repeats, double* bytes_per_second)
{
    if (!bytes_per_second || bytes < 4096 || repeats < 1) return (int)cudaErrorInvalidValue;
    ProbeCtx pc, *ctx = &pc;
    if (const int e = probe_ctx(device, stream, ctx)) return e;
    const size_t n_vec = bytes / sizeof(double2);
    double2* buf = nullptr;
    double* d_out = nullptr;
    MF_CUDA(ctx, cudaMalloc(&buf, n_vec * sizeof(double2)));
    MF_CUDA(ctx, cudaMalloc(&d_out, sizeof(double)));
    MF_CUDA(ctx, cudaMemsetAsync(buf, 0, n_vec * sizeof(double2), ctx->stream));
    cudaEvent_t e0, e1;
    MF_CUDA(ctx, cudaEventCreate(&e0));
    MF_CUDA(ctx, cudaEventCreate(&e1));
    const int grid = ctx->sm_count * 8;
    double best = 0.0;
    for (int rep = 0; rep < 4; ++rep) {
        MF_CUDA(ctx, cudaEventRecord(e0, ctx->stream));
        read_kernel<<<grid, 256, 0, ctx->stream>>>(buf, n_vec, repeats, d_out);
        MF_CUDA(ctx, cudaEventRecord(e1, ctx->stream));
        MF_CUDA(ctx, cudaEventSynchronize(e1));
        float ms = 0;
        MF_CUDA(ctx, cudaEventElapsedTime(&ms, e0, e1));
        const double rate = (double)n_vec * sizeof(double2) * repeats / (ms * 1e-3);
        if (rep > 0 && rate > best) best = rate;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(buf);
    cudaFree(d_out);
    *bytes_per_second = best;
    return 0;
}

extern "C" int mfp_math(int device, void* stream, int op, int64_t n, const double* x_host, double* y_host)
{
    if (!x_host || !y_host || n < 1 || op < 0 || op > 3) return (int)cudaErrorInvalidValue;
    ProbeCtx pc, *ctx = &pc;
    if (const int e = probe_ctx(device, stream, ctx)) return e;
    double *dx = nullptr, *dy = nullptr;
    MF_CUDA(ctx, cudaMalloc(&dx, sizeof(double) * n));
    MF_CUDA(ctx, cudaMalloc(&dy, sizeof(double) * n));
    MF_CUDA(ctx, cudaMemcpyAsync(dx, x_host, sizeof(double) * n, cudaMemcpyHostToDevice, ctx->stream));
    math_kernel<<<(int)((n + 255) / 256 > 1184 ? 1184 : (n + 255) / 256), 256, 0, ctx->stream>>>(op, n, dx, dy);
    MF_CUDA(ctx, cudaGetLastError());
    MF_CUDA(ctx, cudaMemcpyAsync(y_host, dy, sizeof(double) * n, cudaMemcpyDeviceToHost, ctx->stream));
    MF_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    cudaFree(dx);
    cudaFree(dy);
    return 0;
}
