// mf_kernels.cuh — the fused NLL + gradient kernels (S3..S6 of SURVEY.md §8(a)).
//
// Work decomposition (both kernels).  The unit of work is a WARP ITEM: 64 consecutive
// events, lane l owning events 2l and 2l+1, read from every column as ONE coalesced
// 16-byte load per lane (512 contiguous bytes per warp per column; PAPER.md:65 structure
// of arrays).  Items are dealt block-cyclically — item j goes to CTA j % G, warp
// (j / G) % 8 — so that the leftover of the last round spreads over all SMs instead of
// queueing behind a few CTAs.  Each thread keeps K+1 plain fp64 sums over its few dozen
// events (SURVEY.md §7 "register budget"); compensation is applied where the long sums
// are: across block partials (Kahan, fixed order).
//
// Reduction (S4, S5; PAPER.md:65 does this with repeated Kahan reduction kernels, each a
// submission — here it is part of the same launch):
//   thread sums -> xor-shuffle tree per warp -> 8 warp sums added in warp order ->
//   block partial in global memory -> the CTA that takes the last ticket combines all
//   block partials: lane l Kahan-sums partials l, l+32, ... in index order, the 32
//   (sum, compensation) pairs are merged by a fixed two-sum tree.
// The order never depends on which CTA finishes last, so results are bit-reproducible.
#pragma once
#include <cuda_runtime.h>

#include <cstdint>

#include "mf_models.cuh"

namespace mf {

constexpr int kBlock = 256;
constexpr int kWarps = kBlock / 32;
constexpr int kItem = 64;  // events per warp item
constexpr int kRing = 4;    // scratch slots of the single-dataset kernel: evaluation e uses slot e % kRing
constexpr int kFinalBatch = 10;  // partials per lane loaded together in the final pass (covers 2 CTAs/SM x 148 SMs)

template <class M>
struct EvalArgs {
    const double* col[M::NCOL];  // column bases (this toy's row for the single kernel)
    int64_t n;                   // valid events
    int64_t n_items;             // n_pad / 64
    typename M::Consts c;        // parameter-only constants (S2), computed on the host
    const double2* sum_m;        // device: event-only constant sum_i m_i as (hi, lo) (S1), or NULL for models without a mass dimension
    // scratch slot of this evaluation (ring of kRing slots, so that successive evaluations do not
    // serialise on one scratch area; see "pipelining" below)
    double* partials;            // [NACC][gridDim.x]
    unsigned* bad_partials;      // [gridDim.x]
    unsigned* ticket;            // zero on entry, reset to zero by the last CTA
    unsigned long long* gen;     // evaluations completed on this slot
    unsigned long long need;     // value of *gen at which the slot is free for this evaluation
    double* out;                 // [NOUT+1]: -lnL, grad (, Hessian), n_bad
    unsigned long long* done_flag;   // mapped host word that receives done_value after `out` is written, or NULL
    unsigned long long done_value;
};

template <class M>
struct BatchArgs {
    const double* col[M::NCOL];  // column bases of toy 0; toy t is at + t * toy_stride
    int64_t toy_stride;          // n_pad
    int shared_data;             // 1: every slot evaluates toy 0 (several parameter points on ONE dataset)
    int64_t n;                   // valid events per toy
    int64_t n_items;             // n_pad / 64 per toy
    int chunks;                  // CTAs per toy
    double ma, mb;               // mass range for the constants prologue
    const double2* sum_m;        // [n_toys] event-only constants sum_i m_i per toy as (hi, lo), or NULL
    const double* lam;           // [n_active][K]
    int lam_external;            // 1: lam was written by the caller's own work on the stream (mf_nll_grad_batch_async), so it
                                 // may only be read after griddepcontrol.wait; 0: written by a stream-ordered copy of ours
    typename M::Consts* consts;  // [n_active] parameter-only constants (S2), written by batch_consts_kernel
    int* consts_ok;              // [n_active] 0 = lambda outside the parameter domain
    const int* ids;              // [n_active] toy index of each active slot; NULL = identity (all toys active)
    double* partials;            // [n_active][NACC][chunks]   (chunks > 1)
    unsigned* bad_partials;      // [n_active][chunks]
    unsigned* ticket;            // [n_active]
    double* out;                 // [n_active][K+2]
    int ahead;                   // > 0 (chunks == 1, one-column models): the CTA of slot s requests, group by group while it
                                 // evaluates its own toy, the events of slot s + ahead from HBM into L2 (ahead = the number of
                                 // co-resident CTAs: the CTA that will follow it on its SM); 0: off
    int n_active;
};

template <class M>
__device__ __forceinline__ bool make_consts(const double* lam, double ma, double mb, typename M::Consts& c);
template <>
__device__ __forceinline__ bool make_consts<MassModel>(const double* lam, double ma, double mb, MassConsts& c)
{
    return mass_consts(lam, ma, mb, c);
}
template <>
__device__ __forceinline__ bool make_consts<MassHessModel>(const double* lam, double ma, double mb, MassConsts& c)
{
    return mass_consts(lam, ma, mb, c);
}
template <>
__device__ __forceinline__ bool make_consts<AngularModel>(const double* lam, double, double, AngularConsts& c)
{
    return angular_consts(lam, c);
}
template <>
__device__ __forceinline__ bool make_consts<AngularHessModel>(const double* lam, double, double, AngularConsts& c)
{
    return angular_consts(lam, c);
}
template <>
__device__ __forceinline__ bool make_consts<FourDModel>(const double* lam, double ma, double mb, FourDConsts& c)
{
    return fourd_consts(lam, ma, mb, c);
}

// ---- pipelining of back-to-back evaluations on one stream (programmatic dependent launch) -------
// Every kernel lets its successor start at once (launch_dependents at entry) and waits for its
// predecessor to COMPLETE (griddepcontrol.wait) only where stream order matters:
//   * single-dataset kernel: the event loop reads only the immutable columns, partial sums go to
//     this evaluation's own scratch slot (ring of kRing), so only the CTA that does the final
//     combine waits, immediately before it writes the output.  Kernels therefore complete in
//     stream order, outputs land in stream order, and everything else overlaps.  A slot is reused
//     by evaluation e + kRing; its CTAs check the slot's completion counter first (it is always
//     already there unless > kRing evaluations are in flight; the kernel they would wait for has
//     all its CTAs running, because a dependent grid is only launched after every CTA of its
//     predecessor has started, so the check cannot deadlock);
//   * batched kernel: waits before its first global write.
// Without the launch attribute both instructions are no-ops.
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;"); }
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

// Ticket with release/acquire semantics at GPU scope.  Called by ONE thread after a __syncthreads():
// the barrier orders the CTA's partial-sum stores before the release, and the CTA that draws the last
// ticket acquires every other CTA's stores (then a second __syncthreads() hands them to its threads,
// which read the partials with L1-bypassing loads).  One fence per CTA instead of one
// sequentially-consistent fence per storing thread.
__device__ __forceinline__ unsigned long long gen_load(const unsigned long long* g)
{
    unsigned long long v;
    asm volatile("ld.acquire.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(g) : "memory");
    return v;
}
__device__ __forceinline__ void gen_store(unsigned long long* g, unsigned long long v)
{
    asm volatile("st.release.gpu.global.u64 [%0], %1;" ::"l"(g), "l"(v) : "memory");
}
__device__ __forceinline__ unsigned ticket_take(unsigned* ticket)
{
    unsigned old;
    asm volatile("atom.add.acq_rel.gpu.global.u32 %0, [%1], 1;" : "=r"(old) : "l"(ticket) : "memory");
    return old;
}

// ---- S3: the event loop of one warp ---------------------------------------------------------

template <class M>
__device__ __forceinline__ void load_item(const double* const* col, int64_t j, int lane, double* xa, double* xb)
{
#pragma unroll
    for (int c = 0; c < M::NCOL; ++c) {
        const double2 v = __ldg(reinterpret_cast<const double2*>(col[c] + kItem * j) + lane);
        xa[c] = v.x;
        xb[c] = v.y;
    }
}

// One group = U items (j, j + step, ...) of this warp; only item n_items - 1 can be ragged.
template <class M, int U>
__device__ __forceinline__ void load_group(const double* const* col, int64_t n_items, int64_t j, int64_t step, int lane,
                                           double (&buf)[U][2][M::NCOL])
{
#pragma unroll
    for (int u = 0; u < U; ++u)
        if (j + u * step < n_items) load_item<M>(col, j + u * step, lane, buf[u][0], buf[u][1]);
}

template <class M, int U>
__device__ __forceinline__ void compute_group(int64_t n, int64_t n_items, int64_t j, int64_t step, int lane,
                                              const double (&buf)[U][2][M::NCOL], const typename M::Consts& c,
                                              double* acc, LogProd& lp, unsigned& bad, double t_lane)
{
    const int64_t jl = j + (U - 1) * step;  // last item of the group
    if (jl < n_items && kItem * (jl + 1) <= n) {
        // fast path: 2U independent events, no predicates, free for the compiler to interleave
#pragma unroll
        for (int u = 0; u < U; ++u) {
            M::template event<false>(buf[u][0], c, acc, lp, bad, true, t_lane);
            M::template event<false>(buf[u][1], c, acc, lp, bad, true, t_lane);
        }
    } else {
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const int64_t ju = j + u * step;
            if (ju < n_items) {
                const int64_t e = kItem * ju + 2 * lane;
                M::template event<true>(buf[u][0], c, acc, lp, bad, e < n, t_lane);
                M::template event<true>(buf[u][1], c, acc, lp, bad, e + 1 < n, t_lane);
            }
        }
    }
    lp.renorm();  // at most 2U mantissas in [1,2) since the last one
}

// The event loop of one warp for the one-column (ALU-bound) models.  The unit is a GROUP of kGroupItems = 4 consecutive
// items = 256 consecutive events = 2 KB: lane l owns events 2l, 2l+1 of each of the four 64-event rows, read as four
// 16-byte loads at immediate offsets from ONE pointer (one 64-bit pointer add and one 32-bit counter per group).
// Groups g0, g0 + gstep, ... .  Latency: direct form (data from L2: one dataset, many points or launches): the other three
// warps of the SM sub-partition cover the L2 latency of the four loads; an L1 prefetch of the next group (round 1) was
// measured to do nothing (ncu: 5 % L1 hit rate on those loads; without it the C1 sweep is 0.7 % faster) and keeping the next
// group in registers made ptxas copy the buffer twice per iteration.  Staged form (data from HBM: batched toys): below.
// FAST selects the model's fast event body (M::events<E, true>; decided per parameter point, M::is_fast).  The last,
// partial group of the dataset (fewer than four items, or a ragged last item) is evaluated item by item by the warp it
// falls to; only a ragged item is predicated.
constexpr int kGroupItems = 4;
constexpr int kGroupEvents = 2 * kGroupItems;  // per thread

__device__ __forceinline__ void load_group4(const double2* __restrict__ p, double (&m)[kGroupEvents])
{
#pragma unroll
    for (int i = 0; i < kGroupItems; ++i) {
        const double2 v = __ldg(p + 32 * i);
        m[2 * i] = v.x;
        m[2 * i + 1] = v.y;
    }
}

// pf_bytes != 0 (staged form only): while group g is evaluated, the same group of ANOTHER dataset (pf_bytes further on: the
// toy that a later CTA will evaluate) is requested from HBM into L2 — one 64-byte-strided prefetch per lane covers the 2 KB.
// STG > 0: the warp's groups are staged through shared memory by per-lane asynchronous copies (cp.async, 16 bytes each, every
// lane copies and later reads only its own four double2), STG groups deep: the copies of the next STG - 1 groups are in
// flight while a group is evaluated, at no cost in registers.  For data that come from HBM (batched toys), where the
// direct form leaves the latency exposed (ncu: 22 % of the warp samples on the first use of a loaded value).
// stg: this warp's staging area, STG x 4 x 32 double2.
// state of the staging pipeline of one warp (STG > 0): started by stage_begin() BEFORE the parameter-only constants are
// waited for, so that the first copies are in flight during that wait
struct StagePipe {
    const double2* pi;  // next group to request
    unsigned s0;        // shared-memory address of this lane's slot in stage 0, item 0
    int ahead;          // groups requested and not yet evaluated
};

__device__ __forceinline__ void stage_issue(unsigned s0, const double2* src, int st)
{
#pragma unroll
    for (int i = 0; i < kGroupItems; ++i)
        asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(s0 + (unsigned)((st * kGroupItems + i) * 32 * 16)),
                     "l"(src + 32 * i)
                     : "memory");
}

// this warp's full groups g0, g0 + gstep, ... < n_full: pointer of lane `lane` into the first, pointer step, count
__device__ __forceinline__ int group_range(const double* col0, int64_t n, int g0, int gstep, int lane, const double2*& p,
                                           int64_t& pstep)
{
    const int n_full = (int)((n / kItem) / kGroupItems);
    p = reinterpret_cast<const double2*>(col0) + (int64_t)g0 * (32 * kGroupItems) + lane;
    pstep = (int64_t)gstep * (32 * kGroupItems);
    return (g0 < n_full) ? (n_full - g0 + gstep - 1) / gstep : 0;
}

template <int STG>
__device__ __forceinline__ void stage_begin(StagePipe& sp, const double* col0, int64_t n, int g0, int gstep, int lane, double2* stg,
                                            int64_t pf_bytes)
{
    const double2* p;
    int64_t pstep;
    const int left = group_range(col0, n, g0, gstep, lane, p, pstep);
    sp.pi = p;
    sp.s0 = (unsigned)__cvta_generic_to_shared(stg + lane);
    sp.ahead = 0;
#pragma unroll
    for (int k = 0; k < STG - 1; ++k) {  // groups 0 .. STG-2 of this warp (one commit per slot, empty if the warp has fewer)
        if (k < left) {
            stage_issue(sp.s0, sp.pi, k);
            if (pf_bytes) asm volatile("prefetch.global.L2 [%0];" ::"l"(reinterpret_cast<const char*>(sp.pi) + pf_bytes));
            sp.pi += pstep;
            ++sp.ahead;
        }
        asm volatile("cp.async.commit_group;" ::: "memory");
    }
}

template <class M, bool FAST, int STG = 0>
__device__ __forceinline__ void group_loop(const double* col0, int64_t n, int64_t n_items, int g0, int gstep, int lane,
                                           const typename M::Consts& c, double* acc, LogProd& lp, unsigned& bad, double t_lane,
                                           int64_t pf_bytes = 0, double2* stg = nullptr, StagePipe* spp = nullptr)
{
    constexpr int E = M::EVENTS_PER_CALL;  // events the model evaluates together (interleaved instruction streams)
    static_assert(kGroupEvents % E == 0, "a group is a whole number of calls");
    const int n_full = (int)((n / kItem) / kGroupItems);  // groups 0 .. n_full-1 hold 256 valid events
    const double2* p = reinterpret_cast<const double2*>(col0) + (int64_t)g0 * (32 * kGroupItems) + lane;
    const int64_t pstep = (int64_t)gstep * (32 * kGroupItems);
    // this warp's full groups: g0, g0 + gstep, ... < n_full
    int left = (g0 < n_full) ? (n_full - g0 + gstep - 1) / gstep : 0;
    const int g = g0 + left * gstep;  // this warp's first group index >= n_full
    if constexpr (STG > 0) {
        const unsigned s0 = spp->s0;
        const double2* pi = spp->pi;
        int ahead = spp->ahead;
        int st = 0, st_in = STG - 1;
        while (left > 0) {
            if (ahead < left) {  // one more group of this warp to request
                stage_issue(s0, pi, st_in);
                if (pf_bytes) asm volatile("prefetch.global.L2 [%0];" ::"l"(reinterpret_cast<const char*>(pi) + pf_bytes));
                pi += pstep;
                ++ahead;
            }
            asm volatile("cp.async.commit_group;" ::: "memory");
            asm volatile("cp.async.wait_group %0;" ::"n"(STG - 1) : "memory");  // the oldest group has landed
            double m[kGroupEvents];
#pragma unroll
            for (int i = 0; i < kGroupItems; ++i) {
                const double2 v = stg[(st * kGroupItems + i) * 32 + lane];
                m[2 * i] = v.x;
                m[2 * i + 1] = v.y;
            }
            --left;
            --ahead;
            st = (st + 1 == STG) ? 0 : st + 1;
            st_in = (st_in + 1 == STG) ? 0 : st_in + 1;
#pragma unroll
            for (int q = 0; q < kGroupEvents / E; ++q) {
                const double(&mq)[E] = *reinterpret_cast<const double(*)[E]>(&m[q * E]);
                M::template events<E, FAST>(mq, c, acc, lp, bad, t_lane);
                lp.renorm();
            }
        }
    } else {
        while (left > 0) {
            double m[kGroupEvents];
            load_group4(p, m);
            --left;
            p += pstep;
#pragma unroll
            for (int q = 0; q < kGroupEvents / E; ++q) {
                const double(&mq)[E] = *reinterpret_cast<const double(*)[E]>(&m[q * E]);
                M::template events<E, FAST>(mq, c, acc, lp, bad, t_lane);
                lp.renorm();
            }
        }
    }
    // the dataset's last, partial group: index n_full, if it exists and is one of this warp's
    if (g == n_full && (int64_t)n_full * kGroupItems < n_items) {
        const int64_t n_full_items = n / kItem;
#pragma unroll 1
        for (int64_t j = (int64_t)n_full * kGroupItems; j < n_items; ++j) {
            const double2 v = __ldg(reinterpret_cast<const double2*>(col0) + j * 32 + lane);
            const double x2[2] = {v.x, v.y};
            if (j < n_full_items) {
                M::template events<2, FAST>(x2, c, acc, lp, bad, t_lane);
            } else {
                const int64_t e = kItem * j + 2 * lane;
                M::template event<true>(&x2[0], c, acc, lp, bad, e < n, t_lane);
                M::template event<true>(&x2[1], c, acc, lp, bad, e + 1 < n, t_lane);
            }
            lp.renorm();
        }
    }
}

// The events of one warp.  Two schedules:
//  * one column, ALU bound (M::NCOL == 1): 256-event groups j0, j0 + step, ... (group_loop above);
//  * many columns, HBM bound: items (64 events) j0, j0 + step, ..., U items per iteration, software-pipelined with two
//    register buffers (the loads of the next group are in flight while the current group is evaluated).
// get_c() yields the parameter-only constants; it is called AFTER the first loads have been issued, so that a kernel
// which must first fetch them (batched toys) overlaps that with the data latency.
template <class M, int STG = 0, class GetC>
__device__ __forceinline__ void accumulate(const double* const* col, int64_t n, int64_t n_items, int64_t j0,
                                           int64_t step, GetC get_c, double* acc, unsigned& bad, int64_t pf_delta = 0,
                                           double2* stg = nullptr)
{
    const int lane = threadIdx.x & 31;
    const double t_lane = mf_exp32_lane_entry();
    LogProd lp;
    if constexpr (M::NCOL == 1) {
        const int g0 = (int)j0, gstep = (int)step;  // group indices fit 32 bits (n_pad / 256; the host checks)
        // lane l's pointer is 16 l bytes into the group; its prefetch goes to byte 64 l of the other dataset's group
        const int64_t pf_bytes = pf_delta ? pf_delta * (int64_t)sizeof(double) + 48 * lane : 0;
        StagePipe sp;
        if constexpr (STG > 0) stage_begin<STG>(sp, col[0], n, g0, gstep, lane, stg, pf_bytes);
        decltype(auto) c = get_c();
        if constexpr (M::HAS_FAST) {
            if (M::is_fast(c))  // uniform over the CTA: one parameter point per CTA
                group_loop<M, true, STG>(col[0], n, n_items, g0, gstep, lane, c, acc, lp, bad, t_lane, pf_bytes, stg, &sp);
            else
                group_loop<M, false, STG>(col[0], n, n_items, g0, gstep, lane, c, acc, lp, bad, t_lane, pf_bytes, stg, &sp);
        } else {
            group_loop<M, false, STG>(col[0], n, n_items, g0, gstep, lane, c, acc, lp, bad, t_lane, pf_bytes, stg, &sp);
        }
    } else {
        decltype(auto) c = get_c();
        constexpr int U = M::ITEMS_PER_ITER;
        double A[U][2][M::NCOL], B[U][2][M::NCOL];
        int64_t j = j0;
        load_group<M, U>(col, n_items, j, step, lane, A);
        while (j < n_items) {
            load_group<M, U>(col, n_items, j + U * step, step, lane, B);
            compute_group<M, U>(n, n_items, j, step, lane, A, c, acc, lp, bad, t_lane);
            j += U * step;
            if (j >= n_items) break;
            load_group<M, U>(col, n_items, j + U * step, step, lane, A);
            compute_group<M, U>(n, n_items, j, step, lane, B, c, acc, lp, bad, t_lane);
            j += U * step;
        }
    }
    acc[0] = lp.log();  // the one logarithm of this thread
}

// ---- S4: thread -> warp -> block ---------------------------------------------------------------

// After the call threads 0..NACC-1 hold the block sum of quantity threadIdx.x, thread NACC the
// block's bad-event count (in *bad_out).
template <int NACC, int WARPS = kWarps>
__device__ __forceinline__ double block_reduce(double* acc, unsigned bad, double (*sm)[NACC], unsigned* sm_bad,
                                               unsigned* bad_out)
{
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
#pragma unroll
    for (int k = 0; k < NACC; ++k) {
        double v = acc[k];
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) v += __shfl_xor_sync(0xffffffffu, v, off);
        acc[k] = v;
    }
    bad = __reduce_add_sync(0xffffffffu, bad);
    if (lane == 0) {
#pragma unroll
        for (int k = 0; k < NACC; ++k) sm[w][k] = acc[k];
        sm_bad[w] = bad;
    }
    __syncthreads();
    double s = 0.0;
    if (threadIdx.x < NACC) {
#pragma unroll
        for (int i = 0; i < WARPS; ++i) s += sm[i][threadIdx.x];
    } else if (threadIdx.x == NACC) {
        unsigned b = 0;
#pragma unroll
        for (int i = 0; i < WARPS; ++i) b += sm_bad[i];
        *bad_out = b;
    }
    return s;
}

// Fixed-order compensated sum of G partials by one warp: lane l adds partials l, l + 32, ... (Kahan), the 32 (sum, compensation)
// pairs are merged by a two-sum tree.  The loads of a lane are issued eight at a time, independently of the running sum.
__device__ __forceinline__ double warp_combine_partials(const double* __restrict__ pk, int G, int lane)
{
    double s = 0.0, cc = 0.0;
    for (int base = lane; base < G; base += 256) {
        double v[8];
#pragma unroll
        for (int j = 0; j < 8; ++j) v[j] = (base + 32 * j < G) ? __ldcg(pk + base + 32 * j) : 0.0;
#pragma unroll
        for (int j = 0; j < 8; ++j)
            if (base + 32 * j < G) {
                const double y = v[j] - cc;
                const double t = s + y;
                cc = (t - s) - y;
                s = t;
            }
    }
    double lo = -cc;
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
        const double s2 = __shfl_down_sync(0xffffffffu, s, off);
        const double lo2 = __shfl_down_sync(0xffffffffu, lo, off);
        const double t = s + s2;
        const double bb = t - s;
        const double e = (s - (t - bb)) + (s2 - bb);
        lo = (lo + lo2) + e;
        s = t;
    }
    return s + lo;  // lane 0
}

__device__ __forceinline__ unsigned warp_combine_bad(const unsigned* __restrict__ bp, int G, int lane)
{
    unsigned nb = 0;
    for (int i = lane; i < G; i += 32) nb += __ldcg(bp + i);
    return __reduce_add_sync(0xffffffffu, nb);
}

// ---- S5: fixed-order compensated combine of `count` partials per quantity, then M::finish ---------

// Called by every thread of the CTA that drew the last ticket.  Warp w combines quantities w, w + 8,
// ...; partial i of quantity k is at p[k * stride_k + i].  Thread 0 then turns the NACC sums into
// out[0] = -ln L, out[1..K] = gradient, out[K+1] = n_bad (+inf / NaN if n_bad), after waiting for the
// previous kernel on the stream (outputs land in stream order).
template <class M, int WARPS = kWarps>
__device__ __forceinline__ void final_combine(const double* p, int64_t stride_k, int count, const unsigned* badp,
                                              const typename M::Consts& c, double n, double2 sum_m, double* s_sum,
                                              double* out, unsigned long long* done_flag = nullptr,
                                              unsigned long long done_value = 0)
{
    constexpr int NACC = M::NACC, NOUT = M::NOUT;
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    unsigned nb = 0;
    if (w == 0) {
        for (int i = lane; i < count; i += 32) nb += __ldcg(badp + i);
        nb = __reduce_add_sync(0xffffffffu, nb);
    }
    for (int k = w; k < NACC; k += WARPS) {
        const double* pk = p + k * stride_k;
        double s = 0.0, cc = 0.0;  // Kahan: true sum ~ s - cc
        for (int i0 = lane; i0 < count; i0 += 32 * kFinalBatch) {
            double v[kFinalBatch];  // issue the loads of a batch together, then add them in index order
#pragma unroll
            for (int u = 0; u < kFinalBatch; ++u) {
                const int i = i0 + 32 * u;
                v[u] = (i < count) ? __ldcg(pk + i) : 0.0;
            }
#pragma unroll
            for (int u = 0; u < kFinalBatch; ++u) {
                const double y = v[u] - cc;
                const double t = s + y;
                cc = (t - s) - y;
                s = t;
            }
        }
        double lo = -cc;
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) {
            const double s2 = __shfl_down_sync(0xffffffffu, s, off);
            const double lo2 = __shfl_down_sync(0xffffffffu, lo, off);
            const double t = s + s2;  // two-sum
            const double bb = t - s;
            const double e = (s - (t - bb)) + (s2 - bb);
            lo = (lo + lo2) + e;
            s = t;
        }
        if (lane == 0) s_sum[k] = s + lo;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        double o[NOUT];
        M::finish(c, s_sum, n, sum_m, o);
        pdl_wait();
#pragma unroll
        for (int k = 0; k < NOUT; ++k)
            out[k] = !nb ? o[k] : (k == 0) ? __longlong_as_double(0x7ff0000000000000LL) : __longlong_as_double(0x7ff8000000000000LL);
        out[NOUT] = (double)nb;
        if (done_flag) {  // synchronous call: the host spins on this word instead of a stream synchronise
            __threadfence_system();
            *reinterpret_cast<volatile unsigned long long*>(done_flag) = done_value;
        }
    }
}

// ---- the fused single-dataset kernels (mf_nll_grad) ---------------------------------------------

// S4 + S5 of a single-dataset evaluation: thread sums -> block partial in this evaluation's scratch slot -> the CTA
// that draws the last ticket combines and finishes.  Called by every thread of every CTA.
template <class M>
__device__ __forceinline__ void reduce_and_finish(const EvalArgs<M>& a, double* acc, unsigned bad)
{
    constexpr int NACC = M::NACC;
    __shared__ double sm[kWarps][NACC];
    __shared__ double s_sum[NACC];
    __shared__ unsigned sm_bad[kWarps];
    __shared__ unsigned s_bad_block;
    __shared__ bool s_last;
    const int64_t G = gridDim.x;
    if (threadIdx.x == 0)
        while (gen_load(a.gen) < a.need) __nanosleep(64);  // slot still in use by evaluation e - kRing (rare)
    const double s = block_reduce<NACC>(acc, bad, sm, sm_bad, &s_bad_block);  // contains a __syncthreads()
    if (threadIdx.x < NACC)
        a.partials[threadIdx.x * G + blockIdx.x] = s;
    else if (threadIdx.x == NACC)
        a.bad_partials[blockIdx.x] = s_bad_block;
    __syncthreads();
    if (threadIdx.x == 0) s_last = (ticket_take(a.ticket) == gridDim.x - 1);
    __syncthreads();
    if (s_last) {
        final_combine<M>(a.partials, G, (int)G, a.bad_partials, a.c, (double)a.n, a.sum_m ? __ldg(a.sum_m) : make_double2(0.0, 0.0),
                         s_sum, a.out, a.done_flag, a.done_value);
        if (threadIdx.x == 0) {  // every partial has been read: final_combine synchronises the CTA before its thread 0 returns
            *a.ticket = 0u;
            gen_store(a.gen, a.need + 1);  // releases the slot (and the ticket reset) to evaluation e + kRing
        }
    }
}


template <class M>
__global__ void __launch_bounds__(kBlock, M::RESIDENT_CTAS) nll_grad_kernel(const __grid_constant__ EvalArgs<M> a)
{
    constexpr int NACC = M::NACC;
    pdl_launch_dependents();
    double acc[NACC];
#pragma unroll
    for (int k = 0; k < NACC; ++k) acc[k] = 0.0;
    unsigned bad = 0;
    const int64_t G = gridDim.x;
    accumulate<M>(a.col, a.n, a.n_items, blockIdx.x + G * (threadIdx.x >> 5), G * kWarps,
                  [&]() -> const typename M::Consts& { return a.c; }, acc, bad);

    reduce_and_finish<M>(a, acc, bad);
}

// The same evaluation for the many-column, HBM-bound models, with the event columns staged through shared memory by
// the bulk asynchronous copy engine (cp.async.bulk + mbarrier: "TMA" in its 1-D form): a tile is 256 consecutive events
// of every column (NCOL x 2 KB), STAGES tiles are in flight per CTA whatever the register budget, thread t evaluates
// event t of the tile.  Thread 0 re-arms a stage as soon as the CTA has consumed it.  Tiles are dealt block-cyclically.
constexpr int kTmaStages = 4;

template <class M>
constexpr size_t tma_smem_bytes()
{
    return sizeof(double) * kTmaStages * M::NCOL * kBlock + sizeof(unsigned long long) * kTmaStages;
}

template <class M>
__global__ void __launch_bounds__(kBlock, 2) nll_grad_tma_kernel(const __grid_constant__ EvalArgs<M> a)
{
    constexpr int NACC = M::NACC, NC = M::NCOL, TILE = kBlock, STAGES = kTmaStages;
    extern __shared__ __align__(128) unsigned char tma_raw[];
    double (*buf)[NC][TILE] = reinterpret_cast<double (*)[NC][TILE]>(tma_raw);
    unsigned long long* bar = reinterpret_cast<unsigned long long*>(tma_raw + sizeof(double) * STAGES * NC * TILE);
    const int tid = threadIdx.x;
    const int64_t n_pad = a.n_items * kItem, n_tiles = (n_pad + TILE - 1) / TILE, G = gridDim.x;
    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < STAGES; ++s)
            asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"((unsigned)__cvta_generic_to_shared(&bar[s])));
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    pdl_launch_dependents();
    auto issue = [&](int s, int64_t tile) {  // thread 0: arm stage s with tile `tile`
        const int64_t first = tile * TILE;
        const unsigned len = (unsigned)((n_pad - first < TILE) ? (n_pad - first) : TILE);  // multiple of 64 events
        const unsigned bytes = len * (unsigned)sizeof(double);
        const unsigned mb = (unsigned)__cvta_generic_to_shared(&bar[s]);
        asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(mb), "r"(bytes * NC) : "memory");
#pragma unroll
        for (int c = 0; c < NC; ++c)
            asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                             (unsigned)__cvta_generic_to_shared(&buf[s][c][0])),
                         "l"(a.col[c] + first), "r"(bytes), "r"(mb)
                         : "memory");
    };
    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < STAGES; ++s)
            if (blockIdx.x + s * G < n_tiles) issue(s, blockIdx.x + s * G);
    }
    double acc[NACC];
#pragma unroll
    for (int k = 0; k < NACC; ++k) acc[k] = 0.0;
    unsigned bad = 0;
    LogProd lp;
    const double t_lane = mf_exp32_lane_entry();
    int i = 0;
    for (int64_t tile = blockIdx.x; tile < n_tiles; tile += G, ++i) {
        const int s = i % STAGES;
        const unsigned phase = (unsigned)(i / STAGES) & 1u, mb = (unsigned)__cvta_generic_to_shared(&bar[s]);
        unsigned done = 0;
        while (!done)
            asm volatile("{ .reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2; selp.u32 %0, 1, 0, p; }"
                         : "=r"(done)
                         : "r"(mb), "r"(phase)
                         : "memory");
        const int64_t e = tile * TILE + tid;
        double x[NC];
        if (e < n_pad) {
#pragma unroll
            for (int c = 0; c < NC; ++c) x[c] = buf[s][c][tid];
        } else {
#pragma unroll
            for (int c = 0; c < NC; ++c) x[c] = 1.0;  // beyond the padded columns: any finite value, the lane is invalid
        }
        if ((tile + 1) * TILE <= a.n) M::template event<false>(x, a.c, acc, lp, bad, true, t_lane);
        else M::template event<true>(x, a.c, acc, lp, bad, e < a.n, t_lane);
        lp.renorm();
        __syncthreads();  // the whole CTA has consumed stage s
        if (tid == 0 && tile + STAGES * G < n_tiles) issue(s, tile + STAGES * G);
    }
    acc[0] = lp.log();
    reduce_and_finish<M>(a, acc, bad);
}

// ---- the batched-toy kernels (mf_nll_grad_batch) -------------------------------------------------

// S2 for every active toy in parallel: one thread per toy derives the parameter-only constants
// (erf, exp, expm1, log: ~2 us of serial work) from lambda_t, instead of one thread of every CTA doing
// it while the other 255 wait.
template <class M>
__global__ void __launch_bounds__(128) batch_consts_kernel(const __grid_constant__ BatchArgs<M> a, int n_active)
{
    pdl_launch_dependents();
    const int slot = blockIdx.x * blockDim.x + threadIdx.x;
    if (slot >= n_active) return;
    typename M::Consts c;
    // lambda written by the caller's preceding work on the stream is complete and visible only after the wait (a
    // programmatic launch may start this kernel before its predecessor has flushed); our own stream-ordered copy is
    // complete before this kernel can start, and the constants are then derived while the previous evaluation drains
    if (a.lam_external) pdl_wait();
    const int ok = make_consts<M>(a.lam + (int64_t)slot * M::K, a.ma, a.mb, c) ? 1 : 0;
    pdl_wait();
    a.consts[slot] = c;
    a.consts_ok[slot] = ok;
}

// CTA <-> (toy, event chunk)

// STG > 0 (one-column models, one CTA per toy): the events are staged through shared memory, STG groups deep (group_loop)
// BLOCK > 0: threads per CTA instead of M::BATCH_BLOCK, at the same number of resident threads per SM.  With many toys per
// call smaller CTAs are faster — the per-warp prologue and reduction (~450 instructions) are then paid by fewer warps per
// toy and CTAs retire more evenly (measured, 10^4-event toys: 16384 toys 307 us with 4-warp CTAs, 295 with 2, 281 with 1);
// with few toys larger CTAs finish a toy sooner (592 toys: 20 / 32 / 47 us).  The host picks by the number of active toys.
template <class M, int BLOCK>
struct BatchShape {
    static constexpr int kThreads = BLOCK > 0 ? BLOCK : M::BATCH_BLOCK;
    static constexpr int kResident = M::BATCH_BLOCK * M::BATCH_RESIDENT_CTAS / kThreads;
};

template <class M, int STG = 0, int BLOCK = 0>
__global__ void __launch_bounds__(BatchShape<M, BLOCK>::kThreads, BatchShape<M, BLOCK>::kResident)
    nll_grad_batch_kernel(const __grid_constant__ BatchArgs<M> a)
{
    constexpr int NACC = M::NACC;
    constexpr int kBlock = BatchShape<M, BLOCK>::kThreads, kWarps = kBlock / 32;  // this kernel's own CTA size
    __shared__ __align__(16) double2 s_stage[(STG > 0 ? STG : 1) * kGroupItems * 32 * (STG > 0 ? kWarps : 0) + 1];
    static_assert(kBlock >= 32 && kBlock % 32 == 0 && NACC + 1 <= kBlock, "CTA too small for the reduction");
    __shared__ double sm[kWarps][NACC];
    __shared__ double s_sum[NACC];
    __shared__ unsigned sm_bad[kWarps];
    __shared__ unsigned s_bad_block;
    __shared__ bool s_last;
    __shared__ typename M::Consts s_c;
    __shared__ int s_ok;
    __shared__ double2 s_summ;

    pdl_launch_dependents();
    const int slot = blockIdx.x / a.chunks, chunk = blockIdx.x % a.chunks;
    // ids == NULL: every toy is active.  ids is only ever the library's own array, filled by a stream-ordered copy that is
    // complete before the constants kernel (this kernel's predecessor) can start, so it may be read ahead of the wait.
    const int64_t toy = a.shared_data ? 0 : a.ids ? a.ids[slot] : slot;
    int64_t pf_delta = 0;  // doubles from this toy's events to those of the toy `ahead` slots further on
    if (STG > 0 && M::NCOL == 1 && a.ahead > 0 && slot + a.ahead < a.n_active) {
        const int64_t next = a.ids ? a.ids[slot + a.ahead] : slot + a.ahead;
        pf_delta = (next - toy) * a.toy_stride;
    }
    if (a.chunks == 1 && !a.shared_data && (STG == 0 || a.ahead <= 0 || slot < a.ahead)) {
        // this CTA streams its toy's columns once from HBM: ask for them now (L2 prefetch, 128-byte lines), so
        // that they arrive while the constants are fetched and the first loads of the event loop hit L2
        // (with `ahead` only the first wave: later toys were requested by their predecessors)
        const int64_t lines = (a.n_items * kItem * (int64_t)sizeof(double) + 127) / 128;
#pragma unroll
        for (int q = 0; q < M::NCOL; ++q) {
            const char* base = reinterpret_cast<const char*>(a.col[q] + toy * a.toy_stride);
            for (int64_t l = threadIdx.x; l < lines; l += kBlock) asm volatile("prefetch.global.L2 [%0];" ::"l"(base + 128 * l));
        }
    }
    // S2 for this toy: parameter-only constants of lambda_t (batch_consts_kernel, the previous launch).  Many points on one
    // dataset (shared_data): the host wrote the constants before the launch (pinned, device-mapped memory, or a stream-ordered
    // copy), so the event loop does NOT wait for the previous kernel on the stream: under a programmatic launch the CTAs of this
    // call fill the tail of the previous one; the wait comes before the first write to the scratch the calls share (below).
    if (!a.shared_data) pdl_wait();
    {
        constexpr int W = (int)(sizeof(typename M::Consts) / sizeof(double));
        static_assert(sizeof(typename M::Consts) % sizeof(double) == 0 && W <= kBlock, "Consts is an array of doubles");
        if (threadIdx.x < W)
            reinterpret_cast<double*>(&s_c)[threadIdx.x] = reinterpret_cast<const double*>(a.consts + slot)[threadIdx.x];
        if (threadIdx.x == 0) s_ok = a.consts_ok[slot];
        // the event-only constant of the toy (S1, complete long ago): fetched now, not when thread 0 finishes the toy
        if (STG > 0 && threadIdx.x == kBlock - 1) s_summ = a.sum_m ? a.sum_m[toy] : make_double2(0.0, 0.0);
    }
    constexpr int NOUT = M::NOUT;  // -ln L, gradient (and Hessian for the *Hess models); n_bad follows at [NOUT]
    double* out = a.out + (int64_t)slot * (NOUT + 1);
    double2 sum_m = make_double2(0.0, 0.0);
    if (STG == 0 && a.sum_m) sum_m = a.sum_m[toy];
    const double* col[M::NCOL];
#pragma unroll
    for (int i = 0; i < M::NCOL; ++i) col[i] = a.col[i] + toy * a.toy_stride;

    double acc[NACC];
#pragma unroll
    for (int k = 0; k < NACC; ++k) acc[k] = 0.0;
    unsigned bad = 0;
    const int64_t C = a.chunks;
    // the constants become visible (barrier) only after the first event loads are in flight
    accumulate<M, STG>(col, a.n, a.n_items, chunk + C * (threadIdx.x >> 5), C * kWarps,
                       [&]() -> const typename M::Consts& {
                           __syncthreads();
                           return s_c;
                       },
                       acc, bad, pf_delta, s_stage + (threadIdx.x >> 5) * (STG * kGroupItems * 32));
    if (!s_ok) {  // outside the parameter domain (the sums above are garbage and unused): +inf / NaN, n_bad = -1
        if (chunk == 0 && threadIdx.x <= NOUT)
            out[threadIdx.x] = threadIdx.x == 0       ? __longlong_as_double(0x7ff0000000000000LL)
                               : threadIdx.x == NOUT  ? -1.0
                                                      : __longlong_as_double(0x7ff8000000000000LL);
        return;
    }
    const typename M::Consts& c = s_c;
    if (STG > 0) sum_m = s_summ;

    const double s = block_reduce<NACC, kWarps>(acc, bad, sm, sm_bad, &s_bad_block);
    if (a.chunks == 1) {  // the CTA holds the toy's complete sums: no cross-CTA pass
        if constexpr (NACC + 1 <= 32) {  // the block sums and the bad count are held by threads of warp 0
            if (threadIdx.x >= 32) return;
            if (threadIdx.x < NACC) s_sum[threadIdx.x] = s;
            __syncwarp();
        } else {
            if (threadIdx.x < NACC) s_sum[threadIdx.x] = s;
            __syncthreads();
        }
        if (threadIdx.x == 0) {
            const unsigned nb = s_bad_block;
            double o[NOUT];
            M::finish(c, s_sum, (double)a.n, sum_m, o);
            pdl_wait();
#pragma unroll
            for (int k = 0; k < NOUT; ++k)
                out[k] = !nb ? o[k] : (k == 0) ? __longlong_as_double(0x7ff0000000000000LL) : __longlong_as_double(0x7ff8000000000000LL);
            out[NOUT] = (double)nb;
        }
        return;
    }
    pdl_wait();
    double* part = a.partials + (int64_t)slot * NACC * C;
    unsigned* badp = a.bad_partials + (int64_t)slot * C;
    if (threadIdx.x < NACC)
        part[threadIdx.x * C + chunk] = s;
    else if (threadIdx.x == NACC)
        badp[chunk] = s_bad_block;
    __syncthreads();
    if (threadIdx.x == 0) s_last = (ticket_take(a.ticket + slot) == (unsigned)a.chunks - 1);
    __syncthreads();
    if (s_last) {
        final_combine<M, kWarps>(part, C, (int)C, badp, c, (double)a.n, sum_m, s_sum, out);
        if (threadIdx.x == 0) a.ticket[slot] = 0u;
    }
}

// ---- S1: event-only constants: sum_i m_i per toy ------------------------------

// Deterministic two-level sum, returned as a (hi, lo) pair: the fast path of the mass model forms
// sum_i (m_i - mu) = sum_i m_i - N mu from it, two terms that nearly cancel.  Level 1: CTA (toy, chunk) sums events [chunk * len, (chunk+1) * len) of its
// toy — thread t Kahan-sums events t, t + 256, ..., the 256 (sum, compensation) pairs are merged by a
// fixed two-sum tree in shared memory — and writes the pair to part[toy][chunk].  Level 2 (chunks > 1):
// one thread per toy adds the chunk pairs in chunk order.
__device__ __forceinline__ void two_sum_acc(double& s, double& lo, double b, double blo)
{
    const double t = s + b;
    const double bb = t - s;
    const double e = (s - (t - bb)) + (b - bb);
    lo = (lo + blo) + e;
    s = t;
}

__device__ __forceinline__ double2 fast_two_sum(double hi, double lo)  // |hi| >= |lo|: renormalised (hi, lo) pair
{
    const double s = hi + lo;
    return make_double2(s, lo - (s - hi));
}

__global__ void __launch_bounds__(256) column_sum_kernel(const double* __restrict__ col, int64_t n, int64_t n_pad,
                                                         int chunks, double2* __restrict__ part, double2* __restrict__ out)
{
    __shared__ double sh[256], sl[256];
    const int toy = blockIdx.x / chunks, chunk = blockIdx.x % chunks;
    const int64_t len = (n + chunks - 1) / chunks;
    const int64_t lo_i = chunk * len, hi_i = (lo_i + len < n) ? lo_i + len : n;
    const double* x = col + (int64_t)toy * n_pad;
    double s = 0.0, cc = 0.0;
    for (int64_t i = lo_i + threadIdx.x; i < hi_i; i += 256) {
        const double y = x[i] - cc;
        const double t = s + y;
        cc = (t - s) - y;
        s = t;
    }
    sh[threadIdx.x] = s;
    sl[threadIdx.x] = -cc;
    __syncthreads();
    for (int off = 128; off > 0; off >>= 1) {
        if (threadIdx.x < off) {
            double a = sh[threadIdx.x], alo = sl[threadIdx.x];
            two_sum_acc(a, alo, sh[threadIdx.x + off], sl[threadIdx.x + off]);
            sh[threadIdx.x] = a;
            sl[threadIdx.x] = alo;
        }
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        if (chunks == 1)
            out[toy] = fast_two_sum(sh[0], sl[0]);
        else
            part[blockIdx.x] = make_double2(sh[0], sl[0]);
    }
}

__global__ void column_sum_finish_kernel(const double2* __restrict__ part, int chunks, int64_t n_toys, double2* __restrict__ out)
{
    const int64_t toy = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (toy >= n_toys) return;
    double s = 0.0, lo = 0.0;
    for (int c = 0; c < chunks; ++c) {
        const double2 p = part[toy * chunks + c];
        two_sum_acc(s, lo, p.x, p.y);
    }
    out[toy] = fast_two_sum(s, lo);
}

// ---- S1: event-only precompute (Listing 4) ------------------

// Writes the nine merged angular basis columns h_k = 9/(32 pi) g_k for every (padded) event.
// cl, ck, phi and h are [rows][n_pad] flattened; h column k is at h + k * total.
__global__ void __launch_bounds__(256) angular_precompute_kernel(const double* __restrict__ cl_,
                                                                 const double* __restrict__ ck_,
                                                                 const double* __restrict__ phi_, double* __restrict__ h,
                                                                 int64_t total)
{
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < total; i += (int64_t)gridDim.x * blockDim.x) {
        const double cl = cl_[i], ck = ck_[i], phi = phi_[i];
        const double cl2 = cl * cl, ck2 = ck * ck;
        const double sl2 = 1.0 - cl2, sk2 = 1.0 - ck2;
        const double sl = sqrt(sl2), sk = sqrt(sk2);  // theta in [0, pi]: sin theta >= 0
        double sp, cp;
        sincos(phi, &sp, &cp);
        const double c2p = (cp - sp) * (cp + sp), s2p = 2.0 * sp * cp;  // cos 2phi, sin 2phi
        const double g0 = 0.5 * sk2 * (1.0 + cl2);
        const double sksl = sk * ck * sl;  // sin(2 theta_K) sin(theta_l) / 2
        h[0 * total + i] = kAngNorm * g0;
        h[1 * total + i] = kAngNorm * (2.0 * ck2 * sl2 - g0);
        h[2 * total + i] = kAngNorm * (sk2 * sl2 * c2p);
        h[3 * total + i] = kAngNorm * (4.0 * sksl * cl * cp);
        h[4 * total + i] = kAngNorm * (2.0 * sksl * cp);
        h[5 * total + i] = kAngNorm * ((4.0 / 3.0) * sk2 * cl);
        h[6 * total + i] = kAngNorm * (2.0 * sksl * sp);
        h[7 * total + i] = kAngNorm * (4.0 * sksl * cl * sp);
        h[8 * total + i] = kAngNorm * (sk2 * sl2 * s2p);
    }
}

// ---- S0 helpers -----------------------------------------------------------------------------------

// Fills the padding of every toy row with that row's last valid event (rows = ndim * n_toys).
__global__ void pad_rows_kernel(double* data, int64_t rows, int64_t n, int64_t n_pad)
{
    const int64_t npadding = n_pad - n;
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < rows * npadding;
         i += (int64_t)gridDim.x * blockDim.x) {
        const int64_t r = i / npadding, o = i % npadding;
        data[r * n_pad + n + o] = (n > 0) ? data[r * n_pad + n - 1] : 0.0;
    }
}

// Counts entries of one dimension ([n_toys][n_pad], valid part only) that are not inside [lo, hi].
__global__ void range_check_kernel(const double* data, int64_t n_toys, int64_t n, int64_t n_pad, double lo, double hi,
                                   unsigned long long* count)
{
    unsigned long long local = 0;
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n_toys * n;
         i += (int64_t)gridDim.x * blockDim.x) {
        const double v = data[(i / n) * n_pad + (i % n)];
        if (!(v >= lo && v <= hi)) ++local;
    }
    if (local) atomicAdd(count, local);
}

}  // namespace mf
