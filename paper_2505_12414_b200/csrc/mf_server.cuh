// mf_server.cuh — a resident evaluation kernel for the minimiser's one-point-at-a-time access pattern (mass model).
//
// at small N the cost of an evaluation is kernel submission, not arithmetic.  A launch-per-evaluation call
// costs ~12 us from C at N = 1e4 (launch latency + completion latency around a 3 us kernel).  Here the CTAs stay resident
// (one per SM, 256 threads, at most 128 registers so that other kernels still fit beside them) and are fed through memory:
//   host     writes the parameter-only constants (S2) and then a request number into MAPPED PINNED host memory;
//   CTA 0    polls the request slot over PCIe (one 256-byte warp-wide read detects and fetches a request), copies it into
//            device memory and releases a device-side copy of the number;
//   all CTAs poll the device-side number (L2), run the same event loop / block reduction as nll_grad_kernel on their share
//            of the events, write block partials and take a ticket; the last CTA combines in fixed order (final_combine),
//            writes the K + 2 (or 1 + K + K(K+1)/2 + 1) doubles and then the request number into mapped host memory;
//   host     spins on that number.
// The kernel leaves when asked to (request number kServerExit) or after `idle_ns` without a request (a safety net: a
// forgotten server must not occupy the GPU, and tools that serialise kernels must not hang); the host relaunches on demand.
// Results are bit-identical to the launch-per-evaluation path with the same grid (same partition, same order).
#pragma once
#include "mf_kernels.cuh"

namespace mf {

constexpr unsigned long long kServerExit = ~0ull;
// Request slot: four 64-byte lines, each [request number, 7 payload words]; payload word 0 = kind, 1.. = MassConsts.  A
// 64-byte line is read atomically over PCIe, and the host stores a line's payload before its number, so a line whose number
// is new carries the new payload: ONE 256-byte warp-wide read detects and fetches a request.
constexpr int kServerReqLines = 4, kServerReqPayload = 7 * kServerReqLines;
constexpr int kServerRepDone = 62, kServerRepExited = 61;                   // words of the reply slot (out[] from word 0)

struct ServerRelay {  // device memory
    unsigned long long seq;
    double payload[kServerReqPayload];  // [0] = kind (as a 64-bit integer), [1..] = MassConsts
};

struct ServerArgs {
    const double* col0;
    int64_t n, n_items;
    const double2* sum_m;
    const unsigned long long* req;  // device alias of the mapped request slot (four 64-byte lines, see above)
    double* rep;                    // device alias of the mapped reply slot (64 words)
    ServerRelay* relay;
    double* partials;               // [13][gridDim.x]
    unsigned* bad_partials;         // [gridDim.x]
    unsigned* ticket;
    unsigned long long first_seq;   // requests up to this number have been served
    unsigned long long idle_ns;
};

__device__ __forceinline__ unsigned long long ld_acquire_sys_u64(const unsigned long long* p)
{
    unsigned long long v;
    asm volatile("ld.acquire.sys.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ unsigned long long globaltimer_ns()
{
    unsigned long long t;
    asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t));
    return t;
}

template <class M>
__device__ __forceinline__ void server_eval(const ServerArgs& a, const MassConsts& c, unsigned long long seq)
{
    constexpr int NACC = M::NACC;
    __shared__ double sm[kWarps][NACC];
    __shared__ double s_sum[NACC];
    __shared__ unsigned sm_bad[kWarps];
    __shared__ unsigned s_bad_block;
    __shared__ bool s_last;
    double acc[NACC];
#pragma unroll
    for (int k = 0; k < NACC; ++k) acc[k] = 0.0;
    unsigned bad = 0;
    const int64_t G = gridDim.x;
    const double* col[1] = {a.col0};
    accumulate<M>(col, a.n, a.n_items, blockIdx.x + G * (threadIdx.x >> 5), G * kWarps,
                  [&]() -> const MassConsts& { return c; }, acc, bad);
    const double s = block_reduce<NACC>(acc, bad, sm, sm_bad, &s_bad_block);  // contains a __syncthreads()
    if (threadIdx.x < NACC)
        a.partials[threadIdx.x * G + blockIdx.x] = s;
    else if (threadIdx.x == NACC)
        a.bad_partials[blockIdx.x] = s_bad_block;
    __syncthreads();
    if (threadIdx.x == 0) s_last = (ticket_take(a.ticket) == gridDim.x - 1);
    __syncthreads();
    if (s_last) {
        final_combine<M>(a.partials, G, (int)G, a.bad_partials, c, (double)a.n, a.sum_m ? __ldg(a.sum_m) : make_double2(0.0, 0.0),
                         s_sum, a.rep, reinterpret_cast<unsigned long long*>(a.rep + kServerRepDone), seq);
        if (threadIdx.x == 0) *a.ticket = 0u;
    }
    __syncthreads();
}

__global__ void __launch_bounds__(kBlock, 2) nll_server_kernel(const __grid_constant__ ServerArgs a)
{
    __shared__ MassConsts s_c;
    __shared__ unsigned long long s_seq;
    __shared__ long long s_kind;
    constexpr int CW = (int)(sizeof(MassConsts) / sizeof(double));
    unsigned long long last = a.first_seq;
    for (;;) {
        if (blockIdx.x == 0) {
            if (threadIdx.x < 32) {  // warp 0 polls the mapped request slot: one coalesced 256-byte PCIe read per poll
                const int lane = threadIdx.x;
                const unsigned long long t0 = globaltimer_ns();
                unsigned long long v, s;
                for (unsigned spins = 1;; ++spins) {
                    asm volatile("ld.relaxed.sys.global.u64 %0, [%1];" : "=l"(v) : "l"(a.req + lane) : "memory");
                    s = __shfl_sync(0xffffffffu, v, 0);
                    const bool same = s == __shfl_sync(0xffffffffu, v, 8) && s == __shfl_sync(0xffffffffu, v, 16) &&
                                      s == __shfl_sync(0xffffffffu, v, 24);
                    if (same && s != last) break;
                    if ((spins & 15) == 0 && globaltimer_ns() - t0 > a.idle_ns) {
                        s = kServerExit;
                        break;
                    }
                }
                if (s != kServerExit && (lane & 7) != 0)
                    reinterpret_cast<unsigned long long*>(a.relay->payload)[7 * (lane >> 3) + (lane & 7) - 1] = v;
                __syncwarp();
                if (lane == 0) {
                    gen_store(&a.relay->seq, s);  // release: the request is in device memory
                    s_seq = s;
                }
            }
        } else if (threadIdx.x == 0) {
            unsigned long long s;
            for (unsigned spins = 1; (s = gen_load(&a.relay->seq)) == last; ++spins)
                if (spins > 4096) __nanosleep(256);
            s_seq = s;
        }
        __syncthreads();
        const unsigned long long s = s_seq;
        if (s == kServerExit) {
            if (blockIdx.x == 0 && threadIdx.x == 0) {
                *reinterpret_cast<volatile unsigned long long*>(a.rep + kServerRepExited) = 1ull;
                __threadfence_system();
            }
            return;
        }
        static_assert(CW + 1 <= kServerReqPayload, "request payload too small");
        if (threadIdx.x < CW) reinterpret_cast<double*>(&s_c)[threadIdx.x] = __ldcg(a.relay->payload + 1 + threadIdx.x);
        if (threadIdx.x == 0) s_kind = __ldcg(reinterpret_cast<const long long*>(a.relay->payload));
        __syncthreads();
        if (s_kind == 0) server_eval<MassModel>(a, s_c, s);
        else server_eval<MassHessModel>(a, s_c, s);
        last = s;
    }
}

}  // namespace mf
