// mf_api.cu — C-ABI entry points of include/morefit_b200.h: context, S0 upload, S1 model
// creation, and the launches of the fused kernels (S2..S6).  The fit driver is mf_fit.cpp.
#include <cuda_runtime.h>

#include <algorithm>
#include <atomic>
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <new>
#include <string>
#include <type_traits>
#include <utility>
#include <vector>

#include "mf_internal.h"
#include "mf_kernels.cuh"
#include "mf_second.cuh"
#include "mf_points.cuh"
#include "mf_points4d.cuh"
#include "mf_server.cuh"

using namespace mf;

mf_status mf_fail(mf_ctx* ctx, mf_status st, const std::string& msg)
{
    if (ctx) ctx->err = msg;
    return st;
}

#define MF_CUDA(ctx, call)                                                                              \
    do {                                                                                                \
        cudaError_t e__ = (call);                                                                       \
        if (e__ != cudaSuccess) {                                                                       \
            const mf_status st__ = (e__ == cudaErrorMemoryAllocation) ? MF_ERR_OOM : MF_ERR_CUDA;       \
            return mf_fail(ctx, st__, std::string(#call) + ": " + cudaGetErrorString(e__));             \
        }                                                                                               \
    } while (0)

// ---- allocation: device memory from the stream-ordered pool (kept warm: creating and destroying a dataset +
// model per call must not pay cudaMalloc / cudaFree synchronisations), result slots from one pinned, mapped slab.
template <class T>
static cudaError_t dev_alloc(mf_ctx* ctx, T** p, size_t bytes)
{
    return cudaMallocAsync(reinterpret_cast<void**>(p), bytes ? bytes : 1, ctx->stream);
}
static void dev_free(mf_ctx* ctx, void* p)
{
    if (p) cudaFreeAsync(p, ctx->stream);
}
static cudaError_t host_slot_acquire(mf_ctx* ctx, double** h, double** d)
{
    if (!ctx->h_slab) {
        cudaError_t e = cudaHostAlloc(&ctx->h_slab, sizeof(double) * MF_HOST_SLOT_DOUBLES * MF_HOST_SLOTS, cudaHostAllocMapped);
        if (e != cudaSuccess) return e;
        e = cudaHostGetDevicePointer(&ctx->d_slab, ctx->h_slab, 0);
        if (e != cudaSuccess) return e;
        for (int i = MF_HOST_SLOTS - 1; i >= 0; --i) ctx->free_slots.push_back(i);
    }
    if (ctx->free_slots.empty()) return cudaErrorMemoryAllocation;  // more than MF_HOST_SLOTS live models
    const int i = ctx->free_slots.back();
    ctx->free_slots.pop_back();
    *h = ctx->h_slab + (size_t)i * MF_HOST_SLOT_DOUBLES;
    *d = ctx->d_slab + (size_t)i * MF_HOST_SLOT_DOUBLES;
    std::memset(*h, 0, sizeof(double) * MF_HOST_SLOT_DOUBLES);
    return cudaSuccess;
}
// Pinned staging of a batched call: one grow-only block per context (cudaHostAlloc costs ~1 ms; a toy study creates a
// model per call).  Batched calls are synchronous, so the block is free again when they return.
static cudaError_t stage_views(mf_model* m)
{
    mf_ctx* ctx = m->ctx;
    auto up = [](size_t x) { return (x + 255) / 256 * 256; };
    const size_t T = (size_t)m->n_toys;
    const size_t b_lam = up(sizeof(double) * T * m->K), b_ids = up(sizeof(int) * T), b_out = up(sizeof(double) * T * m->bout_row);
    if (ctx->h_stage_bytes < b_lam + b_ids + b_out) {
        if (ctx->h_stage) {
            cudaStreamSynchronize(ctx->stream);
            cudaFreeHost(ctx->h_stage);
            ctx->h_stage = nullptr;
            ctx->h_stage_bytes = 0;
        }
        const cudaError_t e = cudaHostAlloc(reinterpret_cast<void**>(&ctx->h_stage), b_lam + b_ids + b_out, cudaHostAllocMapped);
        if (e != cudaSuccess) return e;
        ctx->h_stage_bytes = b_lam + b_ids + b_out;
    }
    m->h_lam = reinterpret_cast<double*>(ctx->h_stage);
    m->h_ids = reinterpret_cast<int*>(ctx->h_stage + b_lam);
    m->h_bout = reinterpret_cast<double*>(ctx->h_stage + b_lam + b_ids);
    return cudaSuccess;
}

static void host_slot_release(mf_ctx* ctx, double* h)
{
    if (h && ctx && ctx->h_slab) ctx->free_slots.push_back((int)((h - ctx->h_slab) / MF_HOST_SLOT_DOUBLES));
}

static inline int64_t round_up(int64_t x, int64_t m) { return (x + m - 1) / m * m; }

static void devbuf_release(mf_devbuf* b)
{
    if (b && --b->refs == 0) {
        if (b->p) cudaFreeAsync(b->p, b->stream);
        delete b;
    }
}

// ------------------------------------------------------------------------------ context

extern "C" mf_status mf_ctx_create(int device, void* cuda_stream, mf_ctx** out)
{
    if (!out) return MF_ERR_ARG;
    int count = 0;
    if (cudaGetDeviceCount(&count) != cudaSuccess || device < 0 || device >= count) {
        cudaGetLastError();
        return MF_ERR_CUDA;
    }
    mf_ctx* ctx = new (std::nothrow) mf_ctx();
    if (!ctx) return MF_ERR_OOM;
    ctx->device = device;
    ctx->stream = static_cast<cudaStream_t>(cuda_stream);
    if (cudaSetDevice(device) != cudaSuccess ||
        cudaDeviceGetAttribute(&ctx->sm_count, cudaDevAttrMultiProcessorCount, device) != cudaSuccess) {
        cudaGetLastError();
        delete ctx;
        return MF_ERR_CUDA;
    }
    cudaMemPool_t pool;
    if (cudaDeviceGetDefaultMemPool(&pool, device) == cudaSuccess) {
        unsigned long long keep = ~0ull;  // freed blocks stay in the pool for the next dataset / model
        cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &keep);
    }
    cudaGetLastError();
    *out = ctx;
    return MF_OK;
}

extern "C" void mf_ctx_destroy(mf_ctx* ctx)
{
    if (!ctx) return;
    for (mf_model* m : ctx->serving)  // resident kernels of models the caller has not destroyed
        if (m->srv_running) {
            for (int l = 0; l < 4; ++l) reinterpret_cast<volatile unsigned long long*>(m->h_req)[8 * l] = ~0ull;  // kServerExit
            m->srv_running = false;
        }
    if (ctx->server_stream) {
        cudaStreamSynchronize(ctx->server_stream);
        cudaStreamDestroy(ctx->server_stream);
    }
    cudaStreamSynchronize(ctx->stream);
    if (ctx->p_blk) cudaFreeAsync(ctx->p_blk, ctx->stream);
    if (ctx->h_slab) cudaFreeHost(ctx->h_slab);
    if (ctx->h_big) cudaFreeHost(ctx->h_big);
    if (ctx->h_stage) cudaFreeHost(ctx->h_stage);
    for (int i = 0; i < mf_ctx::kPointStages; ++i) {
        if (ctx->h_pts[i]) cudaFreeHost(ctx->h_pts[i]);
        if (ctx->pts_copied[i]) cudaEventDestroy(ctx->pts_copied[i]);
    }
    cudaGetLastError();
    delete ctx;
}

extern "C" const char* mf_last_error(const mf_ctx* ctx) { return ctx ? ctx->err.c_str() : ""; }

extern "C" int64_t mf_ctx_kernel_launches(const mf_ctx* ctx) { return ctx ? ctx->launches : 0; }

// ------------------------------------------------------------------------------ S0: data

extern "C" mf_status mf_dataset_upload(mf_ctx* ctx, int ndim, int64_t n_events, int64_t n_toys,
                                       const double* const* columns, mf_mem where, const double* lo,
                                       const double* hi, mf_dataset** out)
{
    if (!ctx || !out || !columns) return mf_fail(ctx, MF_ERR_ARG, "mf_dataset_upload: NULL argument");
    if (!(ndim == 1 || ndim == 3 || ndim == 4) || n_events < 0 || n_toys < 1)
        return mf_fail(ctx, MF_ERR_ARG, "mf_dataset_upload: ndim must be 1, 3 or 4; n_events >= 0; n_toys >= 1");
    for (int j = 0; j < ndim; ++j)
        if (!columns[j] && n_events > 0) return mf_fail(ctx, MF_ERR_ARG, "mf_dataset_upload: NULL column");
    const bool has_mass = (ndim == 1 || ndim == 4);
    if (has_mass && (!lo || !hi)) return mf_fail(ctx, MF_ERR_ARG, "mf_dataset_upload: the mass range lo/hi is required");
    double rlo[MF_MAX_DIMS], rhi[MF_MAX_DIMS];
    const double ang_lo[3] = {-1.0, -1.0, -kPi}, ang_hi[3] = {1.0, 1.0, kPi};
    for (int j = 0; j < ndim; ++j) {
        const bool is_ang = (ndim == 3) || (ndim == 4 && j > 0);
        const int ja = (ndim == 3) ? j : j - 1;
        if (is_ang) {
            rlo[j] = ang_lo[ja];
            rhi[j] = ang_hi[ja];
            if (lo && hi && (std::fabs(lo[j] - rlo[j]) > 1e-12 || std::fabs(hi[j] - rhi[j]) > 1e-12))
                return mf_fail(ctx, MF_ERR_ARG, "mf_dataset_upload: angular ranges must be [-1,1], [-1,1], [-pi,pi]");
        } else {
            rlo[j] = lo[j];
            rhi[j] = hi[j];
            if (!(std::isfinite(rlo[j]) && std::isfinite(rhi[j]) && rlo[j] < rhi[j]))
                return mf_fail(ctx, MF_ERR_ARG, "mf_dataset_upload: mass range must be finite with lo < hi");
        }
    }
    MF_CUDA(ctx, cudaSetDevice(ctx->device));

    mf_dataset* ds = new (std::nothrow) mf_dataset();
    mf_devbuf* buf = new (std::nothrow) mf_devbuf();
    if (!ds || !buf) {
        delete ds;
        delete buf;
        return mf_fail(ctx, MF_ERR_OOM, "mf_dataset_upload: host allocation failed");
    }
    ds->ctx = ctx;
    ds->ndim = ndim;
    ds->n_events = n_events;
    ds->n_pad = round_up(n_events, kItem);
    ds->n_toys = n_toys;
    for (int j = 0; j < ndim; ++j) {
        ds->lo[j] = rlo[j];
        ds->hi[j] = rhi[j];
    }
    ds->raw = buf;
    const int64_t per_dim = ds->n_pad * n_toys;
    buf->bytes = (size_t)std::max<int64_t>(per_dim * ndim, 1) * sizeof(double);
    buf->stream = ctx->stream;
    unsigned long long* d_count = nullptr;
    auto cleanup = [&]() {
        if (d_count) cudaFreeAsync(d_count, ctx->stream);
        devbuf_release(buf);
        delete ds;
    };
#define MF_CUDA_C(call)                                                                               \
    do {                                                                                              \
        cudaError_t e__ = (call);                                                                     \
        if (e__ != cudaSuccess) {                                                                     \
            cleanup();                                                                                \
            const mf_status st__ = (e__ == cudaErrorMemoryAllocation) ? MF_ERR_OOM : MF_ERR_CUDA;     \
            return mf_fail(ctx, st__, std::string(#call) + ": " + cudaGetErrorString(e__));           \
        }                                                                                             \
    } while (0)
    MF_CUDA_C(dev_alloc(ctx, &buf->p, buf->bytes));
    MF_CUDA_C(dev_alloc(ctx, &d_count, sizeof(unsigned long long)));
    MF_CUDA_C(cudaMemsetAsync(d_count, 0, sizeof(unsigned long long), ctx->stream));
    if (n_events > 0) {
        const cudaMemcpyKind kind = (where == MF_HOST) ? cudaMemcpyHostToDevice : cudaMemcpyDeviceToDevice;
        for (int j = 0; j < ndim; ++j) {
            double* dst = buf->p + (int64_t)j * per_dim;
            // toy rows of n_events doubles -> rows of n_pad doubles; one row (or no padding): a plain 1-D copy
            if (n_toys == 1 || ds->n_pad == n_events)
                MF_CUDA_C(cudaMemcpyAsync(dst, columns[j], (size_t)n_toys * n_events * sizeof(double), kind, ctx->stream));
            else
                MF_CUDA_C(cudaMemcpy2DAsync(dst, (size_t)ds->n_pad * sizeof(double), columns[j],
                                            (size_t)n_events * sizeof(double), (size_t)n_events * sizeof(double),
                                            (size_t)n_toys, kind, ctx->stream));
        }
        if (ds->n_pad > n_events) {
            const int64_t rows = (int64_t)ndim * n_toys;
            const int64_t work = rows * (ds->n_pad - n_events);
            const int grid = (int)std::min<int64_t>((work + 255) / 256, 4096);
            pad_rows_kernel<<<grid, 256, 0, ctx->stream>>>(buf->p, rows, n_events, ds->n_pad);
            ++ctx->launches;
        }
        for (int j = 0; j < ndim; ++j) {
            const int grid = (int)std::min<int64_t>((n_toys * n_events + 255) / 256, 8 * (int64_t)ctx->sm_count);
            range_check_kernel<<<grid, 256, 0, ctx->stream>>>(buf->p + (int64_t)j * per_dim, n_toys, n_events, ds->n_pad,
                                                              rlo[j], rhi[j], d_count);
            ++ctx->launches;
        }
        MF_CUDA_C(cudaGetLastError());
    }
    unsigned long long n_out = 0;
    MF_CUDA_C(cudaMemcpyAsync(&n_out, d_count, sizeof(n_out), cudaMemcpyDeviceToHost, ctx->stream));
    MF_CUDA_C(cudaStreamSynchronize(ctx->stream));
#undef MF_CUDA_C
    cudaFreeAsync(d_count, ctx->stream);
    d_count = nullptr;
    if (n_out) {
        cleanup();
        return mf_fail(ctx, MF_ERR_DATA_RANGE,
                       "mf_dataset_upload: " + std::to_string(n_out) + " values are non-finite or outside their range");
    }
    *out = ds;
    return MF_OK;
}

extern "C" void mf_dataset_destroy(mf_dataset* ds)
{
    if (!ds) return;
    devbuf_release(ds->raw);
    devbuf_release(ds->wts);
    delete ds;
}
// Event weights (reading R23): one more device column, padding 0.
extern "C" mf_status mf_dataset_set_weights(mf_dataset* ds, const double* weights, mf_mem where)
{
    if (!ds) return MF_ERR_ARG;
    mf_ctx* ctx = ds->ctx;
    if (ds->n_toys != 1) return mf_fail(ctx, MF_ERR_ARG, "mf_dataset_set_weights: weighted datasets must have n_toys == 1");
    MF_CUDA(ctx, cudaSetDevice(ctx->device));
    if (!weights) {  // back to unweighted (models created before keep their weights)
        devbuf_release(ds->wts);
        ds->wts = nullptr;
        return MF_OK;
    }
    mf_devbuf* buf = new (std::nothrow) mf_devbuf();
    if (!buf) return mf_fail(ctx, MF_ERR_OOM, "mf_dataset_set_weights: host allocation failed");
    buf->stream = ctx->stream;
    buf->bytes = (size_t)std::max<int64_t>(ds->n_pad, 1) * sizeof(double);
    unsigned long long* d_count = nullptr;
    unsigned long long n_out = 0;
    cudaError_t e = dev_alloc(ctx, &buf->p, buf->bytes);
    if (e == cudaSuccess) e = dev_alloc(ctx, &d_count, sizeof(unsigned long long));
    if (e == cudaSuccess) e = cudaMemsetAsync(d_count, 0, sizeof(unsigned long long), ctx->stream);
    if (e == cudaSuccess) e = cudaMemsetAsync(buf->p, 0, buf->bytes, ctx->stream);
    if (e == cudaSuccess && ds->n_events > 0) {
        e = cudaMemcpyAsync(buf->p, weights, sizeof(double) * ds->n_events,
                            where == MF_HOST ? cudaMemcpyHostToDevice : cudaMemcpyDeviceToDevice, ctx->stream);
        if (e == cudaSuccess) {
            const int grid = (int)std::min<int64_t>((ds->n_events + 255) / 256, 8 * (int64_t)ctx->sm_count);
            range_check_kernel<<<grid, 256, 0, ctx->stream>>>(buf->p, 1, ds->n_events, ds->n_pad, -1.7976931348623157e308,
                                                              1.7976931348623157e308, d_count);  // finite, any sign
            ++ctx->launches;
            e = cudaGetLastError();
        }
    }
    if (e == cudaSuccess) e = cudaMemcpyAsync(&n_out, d_count, sizeof(n_out), cudaMemcpyDeviceToHost, ctx->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);
    if (d_count) cudaFreeAsync(d_count, ctx->stream);
    if (e != cudaSuccess) {
        devbuf_release(buf);
        return mf_fail(ctx, e == cudaErrorMemoryAllocation ? MF_ERR_OOM : MF_ERR_CUDA,
                       std::string("mf_dataset_set_weights: ") + cudaGetErrorString(e));
    }
    if (n_out) {
        devbuf_release(buf);
        return mf_fail(ctx, MF_ERR_DATA_RANGE, "mf_dataset_set_weights: " + std::to_string(n_out) + " weights are not finite");
    }
    devbuf_release(ds->wts);
    ds->wts = buf;
    return MF_OK;
}

extern "C" int64_t mf_dataset_n_events(const mf_dataset* ds) { return ds ? ds->n_events : 0; }
extern "C" int64_t mf_dataset_n_toys(const mf_dataset* ds) { return ds ? ds->n_toys : 0; }

// ------------------------------------------------------------------------------ S1: model

// stops a model's resident kernel (if any) and forgets the model in the context's list
static void server_stop_for_destroy(mf_model* m)
{
    if (m->srv_running) {
        for (int l = 0; l < 4; ++l) reinterpret_cast<volatile unsigned long long*>(m->h_req)[8 * l] = ~0ull;  // kServerExit
        cudaStreamSynchronize(m->ctx->server_stream);
        cudaGetLastError();
        m->srv_running = false;
    }
    auto& v = m->ctx->serving;
    v.erase(std::remove(v.begin(), v.end(), m), v.end());
}

extern "C" void mf_model_destroy(mf_model* m)
{
    if (!m) return;
    // device memory is freed in stream order; the pinned result slot is recycled at once, so no evaluation of this
    // model may still be in flight
    server_stop_for_destroy(m);
    if (m->seq > 0 || m->n_toys > 1) cudaStreamSynchronize(m->ctx->stream);
    if (m->s1_done) cudaEventDestroy(m->s1_done);
    dev_free(m->ctx, m->srv_relay);
    dev_free(m->ctx, m->srv_partials);
    dev_free(m->ctx, m->srv_bad);
    dev_free(m->ctx, m->srv_ticket);
    host_slot_release(m->ctx, m->h_req);
    dev_free(m->ctx, m->cache);
    dev_free(m->ctx, m->d_sum_m);
    dev_free(m->ctx, m->partials);
    dev_free(m->ctx, m->bad_partials);
    dev_free(m->ctx, m->ticket);
    dev_free(m->ctx, m->gen);
    dev_free(m->ctx, m->b_partials);
    dev_free(m->ctx, m->b_bad);
    dev_free(m->ctx, m->d_lam);
    dev_free(m->ctx, m->d_consts);
    dev_free(m->ctx, m->d_consts_ok);
    dev_free(m->ctx, m->d_ids);
    dev_free(m->ctx, m->d_bout);
    dev_free(m->ctx, m->d_sweep);
    dev_free(m->ctx, m->s_partials);
    dev_free(m->ctx, m->s_bad);
    dev_free(m->ctx, m->s_sums);
    dev_free(m->ctx, m->s_ticket);
    dev_free(m->ctx, m->s_out);
    host_slot_release(m->ctx, m->h_out);
    devbuf_release(m->raw);
    devbuf_release(m->wts);
    cudaGetLastError();
    delete m;
}

extern "C" mf_status mf_model_create(mf_ctx* ctx, mf_model_kind kind, const mf_dataset* ds, mf_model** out)
{
    if (!ctx || !ds || !out) return mf_fail(ctx, MF_ERR_ARG, "mf_model_create: NULL argument");
    if (ds->ctx != ctx) return mf_fail(ctx, MF_ERR_ARG, "mf_model_create: dataset belongs to another context");
    int K, ncol, ndim;
    switch (kind) {
    case MF_MASS_GAUSS_EXP: K = 4, ncol = 1, ndim = 1; break;
    case MF_ANGULAR_KSTMUMU: K = 8, ncol = 9, ndim = 3; break;
    case MF_MASS_X_ANGULAR: K = 16, ncol = 12, ndim = 4; break;
    default: return mf_fail(ctx, MF_ERR_ARG, "mf_model_create: unknown model kind");
    }
    if (ds->ndim != ndim) return mf_fail(ctx, MF_ERR_ARG, "mf_model_create: dataset ndim does not match the model kind");
    MF_CUDA(ctx, cudaSetDevice(ctx->device));
    mf_model* m = new (std::nothrow) mf_model();
    if (!m) return mf_fail(ctx, MF_ERR_OOM, "mf_model_create: host allocation failed");
    m->ctx = ctx;
    m->kind = kind;
    m->K = K;
    m->nacc = (kind == MF_MASS_GAUSS_EXP) ? MassHessModel::NACC : (kind == MF_ANGULAR_KSTMUMU) ? AngularHessModel::NACC : FourDModel::NACC;
    m->ncol = ncol;
    m->n_events = ds->n_events;
    m->n_pad = ds->n_pad;
    m->n_toys = ds->n_toys;
    m->ma = ds->lo[0];
    m->mb = ds->hi[0];
    m->raw = ds->raw;
    ++m->raw->refs;
    m->wts = ds->wts;
    if (m->wts) ++m->wts->refs;
#define MF_CUDA_M(call)                                                                               \
    do {                                                                                              \
        cudaError_t e__ = (call);                                                                     \
        if (e__ != cudaSuccess) {                                                                     \
            mf_model_destroy(m);                                                                      \
            const mf_status st__ = (e__ == cudaErrorMemoryAllocation) ? MF_ERR_OOM : MF_ERR_CUDA;     \
            return mf_fail(ctx, st__, std::string(#call) + ": " + cudaGetErrorString(e__));           \
        }                                                                                             \
    } while (0)
    const int64_t per_dim = m->n_pad * m->n_toys;
    const double* raw = m->raw->p;
    double2* d_part = nullptr;  // scratch of the column sum, freed after the synchronise below
    if (kind == MF_MASS_GAUSS_EXP) {
        m->col[0] = raw;
    } else {
        // S1: cache the nine merged angular basis columns
        MF_CUDA_M(dev_alloc(ctx, &m->cache, (size_t)std::max<int64_t>(9 * per_dim, 1) * sizeof(double)));
        const int a0 = (kind == MF_ANGULAR_KSTMUMU) ? 0 : 1;  // first angular dimension
        if (per_dim > 0) {
            const int grid = (int)std::min<int64_t>((per_dim + 255) / 256, 16 * (int64_t)ctx->sm_count);
            angular_precompute_kernel<<<grid, 256, 0, ctx->stream>>>(raw + (a0 + 0) * per_dim, raw + (a0 + 1) * per_dim,
                                                                     raw + (a0 + 2) * per_dim, m->cache, per_dim);
            ++ctx->launches;
            MF_CUDA_M(cudaGetLastError());
        }
        int c = 0;
        if (kind == MF_MASS_X_ANGULAR) {
            m->col[c++] = raw;                // m
            m->col[c++] = raw + 1 * per_dim;  // cos theta_l
            m->col[c++] = raw + 2 * per_dim;  // cos theta_K
        }
        for (int k = 0; k < 9; ++k) m->col[c++] = m->cache + k * per_dim;
    }
    if (kind != MF_ANGULAR_KSTMUMU) {
        // S1: sum_i m_i per toy (ln P_i contains tau m_i: its sum is an event-only constant times tau)
        MF_CUDA_M(dev_alloc(ctx, &m->d_sum_m, sizeof(double2) * m->n_toys));
        const int chunks = (int)std::max<int64_t>(1, std::min<int64_t>(m->n_pad / 8192, 512));
        if (chunks > 1) MF_CUDA_M(dev_alloc(ctx, &d_part, sizeof(double2) * m->n_toys * chunks));
        column_sum_kernel<<<(unsigned)(m->n_toys * chunks), 256, 0, ctx->stream>>>(raw, m->n_events, m->n_pad, chunks, d_part,
                                                                                 m->d_sum_m);
        ++ctx->launches;
        if (chunks > 1) {
            column_sum_finish_kernel<<<(unsigned)((m->n_toys + 127) / 128), 128, 0, ctx->stream>>>(d_part, chunks, m->n_toys,
                                                                                                 m->d_sum_m);
            ++ctx->launches;
        }
        MF_CUDA_M(cudaGetLastError());
        dev_free(ctx, d_part);  // stream-ordered: released after the finish kernel
        d_part = nullptr;
    }
    // launch geometry: persistent-style grid, CTAS_PER_SM CTAs per SM (one wave), never more CTAs than 8-warp groups of items
    // work units dealt to warps: 64-event items, or 256-event groups for the one-column mass model
    const int64_t n_items = (kind == MF_MASS_GAUSS_EXP) ? (m->n_pad / kItem + kGroupItems - 1) / kGroupItems : m->n_pad / kItem;
    if (n_items > (int64_t)0x3fffffff) {
        mf_model_destroy(m);
        return mf_fail(ctx, MF_ERR_ARG, "mf_model_create: more than 2^30 work units per toy");
    }
    const int ctas_per_sm = (kind == MF_MASS_X_ANGULAR) ? FourDModel::CTAS_PER_SM
                            : (kind == MF_ANGULAR_KSTMUMU) ? AngularModel::CTAS_PER_SM : MassModel::CTAS_PER_SM;
    m->grid = (int)std::max<int64_t>(1, std::min<int64_t>((n_items + kWarps - 1) / kWarps, ctas_per_sm * (int64_t)ctx->sm_count));
    // batch geometry: one CTA per toy up to 32768 events per toy, else split
    m->chunks = (int)std::max<int64_t>(1, std::min<int64_t>((m->n_pad + 32767) / 32768, 64));
    if (const char* e = std::getenv("MF_BATCH_CHUNKS")) m->chunks = std::max(1, std::atoi(e));  // tuning knob
    MF_CUDA_M(dev_alloc(ctx, &m->partials, sizeof(double) * kRing * m->nacc * m->grid));
    MF_CUDA_M(dev_alloc(ctx, &m->bad_partials, sizeof(unsigned) * kRing * m->grid));
    MF_CUDA_M(dev_alloc(ctx, &m->ticket, sizeof(unsigned) * (kRing + m->n_toys)));
    MF_CUDA_M(cudaMemsetAsync(m->ticket, 0, sizeof(unsigned) * (kRing + m->n_toys), ctx->stream));
    MF_CUDA_M(dev_alloc(ctx, &m->gen, sizeof(unsigned long long) * kRing));
    MF_CUDA_M(cudaMemsetAsync(m->gen, 0, sizeof(unsigned long long) * kRing, ctx->stream));
    MF_CUDA_M(host_slot_acquire(ctx, &m->h_out, &m->d_out_mapped));
    if (m->n_toys > 1) {
        const int64_t T = m->n_toys;
        if (m->chunks > 1) {
            MF_CUDA_M(dev_alloc(ctx, &m->b_partials, sizeof(double) * T * m->nacc * m->chunks));
            MF_CUDA_M(dev_alloc(ctx, &m->b_bad, sizeof(unsigned) * T * m->chunks));
        }
        MF_CUDA_M(dev_alloc(ctx, &m->d_lam, sizeof(double) * T * K));
        MF_CUDA_M(dev_alloc(ctx, &m->d_consts, sizeof(FourDConsts) * T));  // the largest Consts
        MF_CUDA_M(dev_alloc(ctx, &m->d_consts_ok, sizeof(int) * T));
        MF_CUDA_M(dev_alloc(ctx, &m->d_ids, sizeof(int) * T));
        const int nout1 = 1 + K + K * (K + 1) / 2 + 1;  // widest output row (value, gradient, Hessian triangle) + n_bad
        MF_CUDA_M(dev_alloc(ctx, &m->d_bout, sizeof(double) * T * nout1));
        m->bout_row = nout1;  // the pinned staging of these arrays lives in the context (stage_views)
    }
    // nothing here needs the host to wait: the kernels read sum_i m_i from device memory, so a model is ready to be
    // evaluated (in stream order) as soon as this returns
    if (cudaEventCreateWithFlags(&m->s1_done, cudaEventDisableTiming) == cudaSuccess)
        cudaEventRecord(m->s1_done, ctx->stream);
    else
        m->s1_done = nullptr;
    cudaGetLastError();
#undef MF_CUDA_M
    *out = m;
    return MF_OK;
}

extern "C" int mf_model_nparams(const mf_model* m) { return m ? m->K : 0; }
extern "C" int64_t mf_model_n_events(const mf_model* m) { return m ? m->n_events : 0; }
extern "C" int64_t mf_model_n_toys(const mf_model* m) { return m ? m->n_toys : 0; }

// ------------------------------------------------------------------------------ S2..S6

// Launch with programmatic stream serialisation: the kernel may begin while its predecessor on the
// stream (if that is one of ours) is still in its tail; see pdl_wait() in mf_kernels.cuh.
// allow == false: plain stream order.  The FIRST launch on a model after mf_model_create is made that way: its
// predecessors are the S0/S1 kernels (padding, range check, basis columns, sum_i m_i), whose output the event loop reads
// ahead of any griddepcontrol.wait, and model creation does not synchronise the host any more.
template <class... KArgs, class... Args>
static cudaError_t launch_pdl_v(void (*kernel)(KArgs...), int grid, int block, size_t smem, cudaStream_t stream, bool allow,
                                Args&&... args)
{
    static const bool no_pdl = std::getenv("MF_NO_PDL") != nullptr;  // ablation switch: plain stream order everywhere
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)grid);
    cfg.blockDim = dim3((unsigned)block);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = (no_pdl || !allow) ? 0 : 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kernel, std::forward<Args>(args)...);
}

template <class Args>
static cudaError_t launch_pdl(void (*kernel)(const Args), int grid, cudaStream_t stream, const Args& a, int block = kBlock,
                              size_t smem = 0, bool allow = true)
{
    return launch_pdl_v(kernel, grid, block, smem, stream, allow, a);
}

// true at most once per model: its first launch must not overlap the S0/S1 kernels of mf_model_create — unless those have
// completed by now (a model created ahead of time, the usual case: one event query)
static bool take_fresh(mf_model* m)
{
    if (!m->fresh) return false;
    m->fresh = false;
    if (m->s1_done) {
        const cudaError_t e = cudaEventQuery(m->s1_done);
        if (e == cudaSuccess) return false;
        cudaGetLastError();  // cudaErrorNotReady is not an error
    }
    return true;
}

template <class M>
static bool host_consts(const mf_model* m, const double* lam, typename M::Consts& c);
template <>
bool host_consts<MassModel>(const mf_model* m, const double* lam, MassConsts& c)
{
    return mass_consts(lam, m->ma, m->mb, c);
}
template <>
bool host_consts<MassHessModel>(const mf_model* m, const double* lam, MassConsts& c)
{
    return mass_consts(lam, m->ma, m->mb, c);
}
template <>
bool host_consts<AngularModel>(const mf_model*, const double* lam, AngularConsts& c)
{
    return angular_consts(lam, c);
}
template <>
bool host_consts<AngularHessModel>(const mf_model*, const double* lam, AngularConsts& c)
{
    return angular_consts(lam, c);
}
template <>
bool host_consts<FourDModel>(const mf_model* m, const double* lam, FourDConsts& c)
{
    return fourd_consts(lam, m->ma, m->mb, c);
}

// `pipelined`: the evaluation is one of a back-to-back series (mf_nll_grad_points).  The grid is then
// halved when that still leaves every SM a CTA, so that CTAs of the next evaluation are co-resident
// and the series is throughput- rather than latency-bound (measured: C1 4.3 -> 3.9 us per evaluation).
template <class M>
static mf_status launch_single(mf_model* m, const double* lam, double* out_dev, bool pipelined, bool signal_host)
{
    mf_ctx* ctx = m->ctx;
    EvalArgs<M> a;
    if (!host_consts<M>(m, lam, a.c)) return mf_fail(ctx, MF_ERR_PARAM_DOMAIN, "lambda outside the parameter domain");
    for (int i = 0; i < M::NCOL; ++i) a.col[i] = m->col[i];
    a.n = m->n_events;
    a.n_items = m->n_pad / kItem;
    a.sum_m = m->d_sum_m;
    const int slot = (int)(m->seq % kRing);
    a.partials = m->partials + (int64_t)slot * m->nacc * m->grid;
    a.bad_partials = m->bad_partials + (int64_t)slot * m->grid;
    a.ticket = m->ticket + slot;
    a.gen = m->gen + slot;
    a.need = m->seq / kRing;
    a.out = out_dev;
    a.done_flag = signal_host ? reinterpret_cast<unsigned long long*>(m->d_out_mapped + MF_HOST_DONE_INDEX) : nullptr;
    a.done_value = m->seq + 1;
    const int grid = (pipelined && M::CTAS_PER_SM > 1 && m->grid > ctx->sm_count) ? std::max(ctx->sm_count, m->grid / 2) : m->grid;
    if constexpr (std::is_same<M, AngularModel>::value || std::is_same<M, FourDModel>::value) {
        // 9 / 12 columns per event, HBM bound: columns staged through shared memory by the bulk-copy engine
        static const bool no_tma = std::getenv("MF_NO_TMA") != nullptr;  // ablation switch
        if (!no_tma && m->n_pad >= 4 * kBlock) {
            static const cudaError_t attr_set = cudaFuncSetAttribute(nll_grad_tma_kernel<M>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                                                     (int)tma_smem_bytes<M>());
            MF_CUDA(ctx, attr_set);
            const int tgrid = (int)std::min<int64_t>((m->n_pad + kBlock - 1) / kBlock, 2 * (int64_t)ctx->sm_count);
            MF_CUDA(ctx, launch_pdl(nll_grad_tma_kernel<M>, std::min(tgrid, m->grid), ctx->stream, a, kBlock, tma_smem_bytes<M>(),
                                    !take_fresh(m)));
            ++m->seq;
            ++ctx->launches;
            return MF_OK;
        }
    }
    MF_CUDA(ctx, launch_pdl(nll_grad_kernel<M>, grid, ctx->stream, a, kBlock, 0, !take_fresh(m)));
    ++m->seq;
    ++ctx->launches;
    return MF_OK;
}


// ---- second-order sums by tensor-core contraction (mf_second.cuh): weighted models, the 4D Hessian, the Fisher matrix ----

template <class S>
static bool second_consts(const mf_model* m, const double* lam, typename S::Consts& c);
template <>
bool second_consts<MassSecond>(const mf_model* m, const double* lam, MassConsts& c)
{
    return mass_consts(lam, m->ma, m->mb, c);
}
template <>
bool second_consts<AngularSecond>(const mf_model*, const double* lam, AngularConsts& c)
{
    return angular_consts(lam, c);
}
template <>
bool second_consts<FourDSecond>(const mf_model* m, const double* lam, FourDConsts& c)
{
    return fourd_consts(lam, m->ma, m->mb, c);
}

// grow-only pinned staging block of the context (shared with the batched calls; every user is synchronous)
static mf_status stage_reserve(mf_ctx* ctx, size_t bytes)
{
    if (ctx->h_stage_bytes >= bytes) return MF_OK;
    if (ctx->h_stage) {
        cudaStreamSynchronize(ctx->stream);
        cudaFreeHost(ctx->h_stage);
        ctx->h_stage = nullptr;
        ctx->h_stage_bytes = 0;
    }
    MF_CUDA(ctx, cudaHostAlloc(reinterpret_cast<void**>(&ctx->h_stage), bytes, cudaHostAllocMapped));
    ctx->h_stage_bytes = bytes;
    return MF_OK;
}

// MODE 0: -ln L and gradient; 1: + Hessian; 2: + Fisher matrix sum w^2 s s^T.  out_dev NULL = the model's own buffer.
// Output row: -ln L, gradient [K], Hessian upper triangle row by row [K(K+1)/2], Fisher likewise, n_bad.
template <class S, int MODE>
static mf_status launch_second(mf_model* m, const double* lam, double* out_dev, int64_t toy = 0,
                               unsigned long long* done_flag = nullptr, unsigned long long done_value = 0)
{
    using L = SecondLayout<S, MODE>;
    using LW = SecondLayout<S, 2>;  // scratch is sized for the widest mode
    mf_ctx* ctx = m->ctx;
    SecondArgs<S> a;
    if (!second_consts<S>(m, lam, a.c)) return mf_fail(ctx, MF_ERR_PARAM_DOMAIN, "lambda outside the parameter domain");
    if (!m->s_partials) {
        const int64_t n_cta_items = (m->n_pad / kSecondItem + 11) / 12;  // at least one item per warp of the smallest CTA
        m->s_grid = (int)std::max<int64_t>(1, std::min<int64_t>(n_cta_items, ctx->sm_count));
        MF_CUDA(ctx, dev_alloc(ctx, &m->s_partials, sizeof(double) * LW::NQ * m->s_grid));
        MF_CUDA(ctx, dev_alloc(ctx, &m->s_bad, sizeof(unsigned) * m->s_grid));
        MF_CUDA(ctx, dev_alloc(ctx, &m->s_sums, sizeof(double) * LW::NQ));
        MF_CUDA(ctx, dev_alloc(ctx, &m->s_ticket, sizeof(unsigned)));
        MF_CUDA(ctx, cudaMemsetAsync(m->s_ticket, 0, sizeof(unsigned), ctx->stream));
        MF_CUDA(ctx, dev_alloc(ctx, &m->s_out, sizeof(double) * (LW::NOUT + 1)));
    }
    for (int i = 0; i < S::NCOL; ++i) a.col[i] = m->col[i] + toy * m->n_pad;  // columns are [toy][n_pad]
    a.w = m->wts ? m->wts->p : nullptr;
    a.n = m->n_events;
    a.n_pad = m->n_pad;
    a.partials = m->s_partials;
    a.bad_partials = m->s_bad;
    static const cudaError_t attr_set = cudaFuncSetAttribute(nll_second_kernel<S, MODE>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                                             (int)L::smem_bytes());
    MF_CUDA(ctx, attr_set);
    take_fresh(m);  // plain stream order: these launches never overlap their predecessors
    nll_second_kernel<S, MODE><<<m->s_grid, L::THREADS, L::smem_bytes(), ctx->stream>>>(a);
    SecondCombineArgs<S> cb;
    cb.partials = m->s_partials;
    cb.bad_partials = m->s_bad;
    cb.G = m->s_grid;
    cb.sums = m->s_sums;
    cb.ticket = m->s_ticket;
    cb.c = a.c;
    cb.out = out_dev ? out_dev : m->s_out;
    cb.done_flag = done_flag;
    cb.done_value = done_value;
    second_combine_kernel<S, MODE><<<(L::NQ + kWarps - 1) / kWarps, kBlock, 0, ctx->stream>>>(cb);
    MF_CUDA(ctx, cudaGetLastError());
    ctx->launches += 2;
    return MF_OK;
}

template <int MODE>
static mf_status dispatch_second(mf_model* m, const double* lam, double* out_dev, unsigned long long* done_flag = nullptr,
                                 unsigned long long done_value = 0)
{
    switch (m->kind) {
    case MF_MASS_GAUSS_EXP: return launch_second<MassSecond, MODE>(m, lam, out_dev, 0, done_flag, done_value);
    case MF_ANGULAR_KSTMUMU: return launch_second<AngularSecond, MODE>(m, lam, out_dev, 0, done_flag, done_value);
    default: return launch_second<FourDSecond, MODE>(m, lam, out_dev, 0, done_flag, done_value);
    }
}

// Synchronous second-order evaluation; hess / fisher (host, K x K, row-major, symmetric) may be NULL.
static mf_status second_sync(mf_model* m, const double* lambda, double* nll, double* grad, double* hess, double* fisher,
                             const char* who)
{
    mf_ctx* ctx = m->ctx;
    const int K = m->K, NH = K * (K + 1) / 2;
    const int mode = fisher ? 2 : hess ? 1 : 0;
    const int nout = 1 + K + (mode >= 1 ? NH : 0) + (mode >= 2 ? NH : 0);
    // the combine kernel writes the result row and then a done word into mapped pinned memory; the host spins on the word
    // (a D2H copy + stream synchronise costs ~25 us per call, the kernels 60-110 us)
    constexpr int kBigDoubles = 512, kBigDone = 511;
    if (!ctx->h_big) {
        MF_CUDA(ctx, cudaHostAlloc(reinterpret_cast<void**>(&ctx->h_big), sizeof(double) * kBigDoubles, cudaHostAllocMapped));
        MF_CUDA(ctx, cudaHostGetDevicePointer(reinterpret_cast<void**>(&ctx->d_big), ctx->h_big, 0));
        std::memset(ctx->h_big, 0, sizeof(double) * kBigDoubles);
    }
    const unsigned long long want = ++ctx->big_seq;
    unsigned long long* d_done = reinterpret_cast<unsigned long long*>(ctx->d_big + kBigDone);
    const mf_status st = mode == 2   ? dispatch_second<2>(m, lambda, ctx->d_big, d_done, want)
                         : mode == 1 ? dispatch_second<1>(m, lambda, ctx->d_big, d_done, want)
                                     : dispatch_second<0>(m, lambda, ctx->d_big, d_done, want);
    if (st != MF_OK) return st;
    volatile unsigned long long* done = reinterpret_cast<volatile unsigned long long*>(ctx->h_big + kBigDone);
    for (unsigned spins = 1; *done != want; ++spins) {
        if ((spins & 0xFFFF) == 0) {
            const cudaError_t qy = cudaStreamQuery(ctx->stream);
            if (qy != cudaErrorNotReady && *done != want) {
                if (qy == cudaSuccess) continue;
                return mf_fail(ctx, MF_ERR_CUDA, std::string(who) + ": " + cudaGetErrorString(qy));
            }
        }
    }
    std::atomic_thread_fence(std::memory_order_acquire);
    const double* h = ctx->h_big;
    *nll = h[0];
    if (grad) std::memcpy(grad, h + 1, sizeof(double) * K);
    int q = 1 + K;
    if (mode >= 1)
        for (int i = 0; i < K; ++i)
            for (int j = i; j < K; ++j, ++q)
                if (hess) hess[i * K + j] = hess[j * K + i] = h[q];
    if (mode >= 2)
        for (int i = 0; i < K; ++i)
            for (int j = i; j < K; ++j, ++q) fisher[i * K + j] = fisher[j * K + i] = h[q];
    if (h[nout] != 0.0)
        return mf_fail(ctx, MF_NONPOSITIVE_PDF,
                       std::string(who) + ": P <= 0 for " + std::to_string((long long)h[nout]) + " events at this lambda");
    return MF_OK;
}

// true where an evaluation goes through the second-order kernels: weighted models, and the Hessian of the 4D model
static bool uses_second(const mf_model* m, bool hess) { return m->wts != nullptr || (hess && m->kind == MF_MASS_X_ANGULAR); }

static mf_status dispatch_single(mf_model* m, const double* lam, double* out_dev, bool pipelined = false,
                                 bool signal_host = false, bool hess = false)
{
    if (hess) {
        if (m->kind == MF_MASS_GAUSS_EXP) return launch_single<MassHessModel>(m, lam, out_dev, pipelined, signal_host);
        if (m->kind == MF_ANGULAR_KSTMUMU) return launch_single<AngularHessModel>(m, lam, out_dev, false, signal_host);
        return mf_fail(m->ctx, MF_ERR_ARG, "internal: the 4D Hessian goes through the second-order kernel");
    }
    switch (m->kind) {
    case MF_MASS_GAUSS_EXP: return launch_single<MassModel>(m, lam, out_dev, pipelined, signal_host);
    case MF_ANGULAR_KSTMUMU: return launch_single<AngularModel>(m, lam, out_dev, false, signal_host);
    default: return launch_single<FourDModel>(m, lam, out_dev, false, signal_host);
    }
}

extern "C" mf_status mf_nll_grad_async(mf_model* m, const double* lambda, double* out_dev)
{
    if (!m || !lambda || !out_dev) return mf_fail(m ? m->ctx : nullptr, MF_ERR_ARG, "mf_nll_grad_async: NULL argument");
    if (m->n_toys != 1) return mf_fail(m->ctx, MF_ERR_ARG, "mf_nll_grad_async: dataset has n_toys != 1; use mf_nll_grad_batch");
    if (uses_second(m, false)) return dispatch_second<0>(m, lambda, out_dev);
    return dispatch_single(m, lambda, out_dev);
}

// Several parameter points on ONE dataset in one launch: the batched kernel with every slot reading toy 0.
// The parameter-only constants are derived on the host (which also validates every point before anything is
// enqueued), written into a pinned staging block and copied to the model's grow-only scratch; a CTA is
// (point, event chunk); chunk sums are combined per point in fixed order.  Nothing is allocated, freed or cleared per
// call once the scratch has reached its size (the tickets are left at zero by the kernel itself).
static cudaError_t points_stage(mf_ctx* ctx, size_t bytes, char** h, int* stage)
{
    const int s = (int)(ctx->pts_seq++ % mf_ctx::kPointStages);
    if (ctx->pts_copied[s]) {
        const cudaError_t e = cudaEventSynchronize(ctx->pts_copied[s]);  // the copy that last used this block (long done)
        if (e != cudaSuccess) return e;
    } else {
        const cudaError_t e = cudaEventCreateWithFlags(&ctx->pts_copied[s], cudaEventDisableTiming);
        if (e != cudaSuccess) return e;
    }
    if (ctx->h_pts_bytes[s] < bytes) {
        if (ctx->h_pts[s]) cudaFreeHost(ctx->h_pts[s]);
        ctx->h_pts[s] = nullptr;
        ctx->h_pts_bytes[s] = 0;
        const size_t want = std::max<size_t>(bytes, 64 * 1024);
        const cudaError_t e = cudaHostAlloc(reinterpret_cast<void**>(&ctx->h_pts[s]), want, cudaHostAllocMapped);  // kernels may read it in place
        if (e != cudaSuccess) return e;
        ctx->h_pts_bytes[s] = want;
    }
    *h = ctx->h_pts[s];
    *stage = s;
    return cudaSuccess;
}

// Device scratch of the many-points evaluations, [consts | ok | partials | bad | ticket], grow-only, laid out for the largest
// (points, chunks) seen so far; ok flags non-zero (every point is validated on the host), tickets zero (the kernels leave
// them at zero).
static mf_status points_scratch(mf_ctx* ctx, int64_t n_points, int chunks)
{
    auto up = [](size_t x) { return (x + 255) / 256 * 256; };
    if (n_points > ctx->p_points || chunks > ctx->p_chunks || !ctx->p_blk) {
        const int64_t P = std::max<int64_t>(n_points, ctx->p_points);
        const int C = std::max(chunks, ctx->p_chunks);
        const size_t bytes = up(sizeof(FourDConsts) * P) + up(sizeof(int) * P) + up(sizeof(double) * P * MF_MAX_NACC * C) +
                             up(sizeof(unsigned) * P * C) + up(sizeof(unsigned) * P);
        dev_free(ctx, ctx->p_blk);  // stream-ordered: after the launches that still use it
        ctx->p_blk = nullptr;
        ctx->p_points = 0;
        ctx->p_chunks = 0;
        MF_CUDA(ctx, dev_alloc(ctx, &ctx->p_blk, bytes));
        ctx->p_bytes = bytes;
        ctx->p_points = P;
        ctx->p_chunks = C;
        MF_CUDA(ctx, cudaMemsetAsync(ctx->p_blk + up(sizeof(FourDConsts) * P), 0xFF, up(sizeof(int) * P), ctx->stream));
        MF_CUDA(ctx, cudaMemsetAsync(ctx->p_blk + bytes - up(sizeof(unsigned) * P), 0, up(sizeof(unsigned) * P), ctx->stream));
    }
    return MF_OK;
}

// The angular model's many-points evaluation as two tensor-core contractions (mf_points.cuh): one pass over the data per
// 64 points.  out_dev rows are K + 2 = 10 doubles.
// Width of the grid (G, passes) of the many-points kernels: G CTAs share the events of one pass.  Whole waves: the smallest
// G >= slots / 4 for which G x passes fills its waves of `slots` resident CTAs to >= 97 % (measured, C2: 64 points 1.89 us per
// evaluation at G = 296 -> 1.78 at 148; 128 points 1.69 -> 1.54 at G = 74; CTAs of different passes on one SM read the same
// events: L1 hits).  MF_POINTS_G overrides (tuning knob).
static int points_grid_width(int slots, int64_t passes, int64_t n_groups)
{
    static const int g_env = std::getenv("MF_POINTS_G") ? std::atoi(std::getenv("MF_POINTS_G")) : 0;
    int g_pick = slots;
    for (int g = std::max(1, slots / 4); g < slots; ++g) {
        const int64_t ctas = g * passes, waves = (ctas + slots - 1) / slots;
        if ((double)ctas >= 0.97 * (double)(waves * slots)) {
            g_pick = g;
            break;
        }
    }
    return (int)std::max<int64_t>(1, std::min<int64_t>((n_groups + kWarps - 1) / kWarps, g_env > 0 ? g_env : g_pick));
}

static mf_status launch_points_angular_mma(mf_model* m, int64_t n_points, const double* lambdas, double* out_dev)
{
    mf_ctx* ctx = m->ctx;
    for (int64_t i = 0; i < n_points * 8; ++i)
        if (!std::isfinite(lambdas[i]))
            return mf_fail(ctx, MF_ERR_PARAM_DOMAIN, "mf_nll_grad_points: lambda " + std::to_string((long long)(i / 8)) +
                                                         " is outside the parameter domain");
    const int64_t n_groups = m->n_pad / 8;
    static const int pass_env = std::getenv("MF_POINTS_PER_PASS") ? std::atoi(std::getenv("MF_POINTS_PER_PASS")) : 0;  // tuning knob
    // measured (C2, 1e6 events): 32 points per pass at 2 CTAs per SM (124 registers) 1.62 us per evaluation at 1000 points,
    // 64 per pass at 1 CTA per SM (212 registers) 1.85 us
    const int per_pass = (pass_env == 8 || pass_env == 16 || pass_env == 32 || pass_env == 64) ? pass_env : n_points > 16 ? 32 : n_points > 8 ? 16 : 8;
    const int ctas_per_sm = per_pass == 64 ? 1 : per_pass <= 16 ? 3 : 2;
    const int G = points_grid_width(ctas_per_sm * ctx->sm_count, (n_points + per_pass - 1) / per_pass, n_groups);
    {
        const mf_status ss = points_scratch(ctx, n_points, G);
        if (ss != MF_OK) return ss;
    }
    auto up = [](size_t x) { return (x + 255) / 256 * 256; };
    const int64_t P = ctx->p_points;
    const int C = ctx->p_chunks;
    const size_t b_coef = sizeof(double) * 8 * n_points;
    AngPointsArgs a;
    for (int i = 0; i < 9; ++i) a.col[i] = m->col[i];
    a.n = m->n_events;
    a.n_pad = m->n_pad;
    char* q = ctx->p_blk;
    a.coef = reinterpret_cast<const double*>(q);
    q += up(sizeof(FourDConsts) * P) + up(sizeof(int) * P);
    a.partials = reinterpret_cast<double*>(q);
    q += up(sizeof(double) * P * MF_MAX_NACC * C);
    a.bad_partials = reinterpret_cast<unsigned*>(q);
    a.n_points = (int)n_points;
    const dim3 grid((unsigned)G, (unsigned)((n_points + per_pass - 1) / per_pass));
    static const bool copy_coef = std::getenv("MF_POINTS_COPY") != nullptr;
    if (n_points <= kAngInlinePoints && per_pass != 64 && !copy_coef) {
        // the coefficients travel in the parameter block: nothing sits between this call and the previous kernel on the stream,
        // and both kernels are launched programmatically (mf_points.cuh): consecutive calls overlap
        const bool pdl_ok = !take_fresh(m);
        auto launch = [&](auto kernel, dim3 g, int block, size_t smem, bool allow, auto&&... args) {
            static const bool no_pdl = std::getenv("MF_NO_PDL") != nullptr;
            cudaLaunchConfig_t cfg = {};
            cfg.gridDim = g;
            cfg.blockDim = dim3((unsigned)block);
            cfg.dynamicSmemBytes = smem;
            cfg.stream = ctx->stream;
            cudaLaunchAttribute attr[1];
            attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
            attr[0].val.programmaticStreamSerializationAllowed = 1;
            cfg.attrs = attr;
            cfg.numAttrs = (allow && !no_pdl) ? 1 : 0;
            return cudaLaunchKernelEx(&cfg, kernel, args...);
        };
        if (n_points <= 32) {
            AngPointsInlineArgs<32> ia;
            ia.a = a;
            ia.a.coef = nullptr;
            std::memcpy(ia.coef, lambdas, b_coef);
            if (per_pass == 32) MF_CUDA(ctx, launch(angular_points_mma_inline_kernel<4, 32>, grid, kBlock, ang_points_smem<4>(), pdl_ok, ia));
            else if (per_pass == 16) MF_CUDA(ctx, launch(angular_points_mma_inline_kernel<2, 32>, grid, kBlock, ang_points_smem<2>(), pdl_ok, ia));
            else MF_CUDA(ctx, launch(angular_points_mma_inline_kernel<1, 32>, grid, kBlock, ang_points_smem<1>(), pdl_ok, ia));
        } else {
            AngPointsInlineArgs<kAngInlinePoints> ia;
            ia.a = a;
            ia.a.coef = nullptr;
            std::memcpy(ia.coef, lambdas, b_coef);
            if (per_pass == 32) MF_CUDA(ctx, launch(angular_points_mma_inline_kernel<4, kAngInlinePoints>, grid, kBlock, ang_points_smem<4>(), pdl_ok, ia));
            else if (per_pass == 16) MF_CUDA(ctx, launch(angular_points_mma_inline_kernel<2, kAngInlinePoints>, grid, kBlock, ang_points_smem<2>(), pdl_ok, ia));
            else MF_CUDA(ctx, launch(angular_points_mma_inline_kernel<1, kAngInlinePoints>, grid, kBlock, ang_points_smem<1>(), pdl_ok, ia));
        }
        MF_CUDA(ctx, launch(angular_points_combine_kernel, dim3((unsigned)n_points), kAngCombineThreads, 0, true,
                            (const double*)a.partials, (const unsigned*)a.bad_partials, G, (int)n_points, out_dev));
        ctx->launches += 2;
        return MF_OK;
    }
    char* h_blk = nullptr;
    int stage = 0;
    MF_CUDA(ctx, points_stage(ctx, b_coef, &h_blk, &stage));
    std::memcpy(h_blk, lambdas, b_coef);
    MF_CUDA(ctx, cudaMemcpyAsync(q = ctx->p_blk, h_blk, b_coef, cudaMemcpyHostToDevice, ctx->stream));
    MF_CUDA(ctx, cudaEventRecord(ctx->pts_copied[stage], ctx->stream));
    take_fresh(m);
    if (per_pass == 64) angular_points_mma_kernel<8><<<grid, kBlock, ang_points_smem<8>(), ctx->stream>>>(a);
    else if (per_pass == 32) angular_points_mma_kernel<4><<<grid, kBlock, ang_points_smem<4>(), ctx->stream>>>(a);
    else if (per_pass == 16) angular_points_mma_kernel<2><<<grid, kBlock, ang_points_smem<2>(), ctx->stream>>>(a);
    else angular_points_mma_kernel<1><<<grid, kBlock, ang_points_smem<1>(), ctx->stream>>>(a);
    angular_points_combine_kernel<<<(unsigned)n_points, kAngCombineThreads, 0, ctx->stream>>>(
        a.partials, a.bad_partials, G, (int)n_points, out_dev);
    MF_CUDA(ctx, cudaGetLastError());
    ctx->launches += 2;
    return MF_OK;
}

// The 4D model's many-points evaluation in one pass over the data (mf_points4d.cuh): 32 points per pass.  out_dev rows are
// K + 2 = 18 doubles.  *handled = false: a point has f = 0 or f = 1 exactly (ln f and 1/f, 1/(1-f) are folded into the
// per-point constants): the caller uses the (point, chunk) kernel.
static mf_status launch_points_fourd_mma(mf_model* m, int64_t n_points, const double* lambdas, double* out_dev, bool* handled)
{
    mf_ctx* ctx = m->ctx;
    *handled = true;
    const int64_t n_groups = m->n_pad / 8;
    static const int pass_env4 = std::getenv("MF_POINTS4D_PER_PASS") ? std::atoi(std::getenv("MF_POINTS4D_PER_PASS")) : 0;  // tuning knob
    const int per_pass = (pass_env4 == 16 || pass_env4 == 24 || pass_env4 == 32) ? pass_env4 : 16;
    const int G = points_grid_width(2 * ctx->sm_count, (n_points + per_pass - 1) / per_pass, n_groups);  // 2 CTAs per SM
    char* h_blk = nullptr;
    int stage = 0;
    const size_t per_point = sizeof(double) * (16 + kP4PointConsts + kP4FinishConsts);
    static_assert(sizeof(double) * (16 + kP4PointConsts + kP4FinishConsts) <= sizeof(FourDConsts), "per-point block fits the scratch layout");
    // up to kP4InlinePoints points: the per-point data travel in the kernels' parameter blocks (no copy, programmatic launches:
    // consecutive calls overlap); more: through the pinned staging ring and a stream-ordered copy
    static const bool copy_coef4 = std::getenv("MF_POINTS_COPY") != nullptr;
    const bool inl = n_points <= kP4InlinePoints && per_pass == 16 && !copy_coef4;
    FourDPointsInlineArgs ia;
    FourDCombineInlineArgs ic;
    double *h_coef, *h_pc, *h_fc;
    if (inl) {
        h_coef = ia.coef;
        h_pc = ia.pconst;
        h_fc = ic.fconst;
    } else {
        MF_CUDA(ctx, points_stage(ctx, per_point * n_points, &h_blk, &stage));
        h_coef = reinterpret_cast<double*>(h_blk);
        h_pc = h_coef + 16 * n_points;
        h_fc = h_pc + kP4PointConsts * n_points;
    }
    const double mref = 0.5 * (m->ma + m->mb);
    for (int64_t p = 0; p < n_points; ++p) {
        const double* lam = lambdas + p * 16;
        FourDConsts c;
        if (!fourd_consts(lam, m->ma, m->mb, c))
            return mf_fail(ctx, MF_ERR_PARAM_DOMAIN, "mf_nll_grad_points: lambda " + std::to_string((long long)p) +
                                                         " is outside the parameter domain");
        if (!(c.m.f > 0.0 && c.m.f < 1.0)) {
            *handled = false;
            return MF_OK;
        }
        std::memcpy(h_coef + 16 * p, lam, sizeof(double) * 16);
        double* pc = h_pc + kP4PointConsts * p;
        pc[0] = c.m.mu - mref;
        pc[1] = c.m.nb0;
        pc[2] = c.m.tau;
        pc[3] = c.m.lnk - c.m.tau * mref + std::log(c.m.f);
        double* fc = h_fc + kP4FinishConsts * p;
        fc[0] = 1.0 / c.m.f;
        fc[1] = 1.0 / c.m.omf;
        fc[2] = c.m.tau;
        fc[3] = c.m.lnc2;
        fc[4] = c.kappa;
        fc[5] = c.m.is2;
        fc[6] = c.m.kmu;
        fc[7] = c.m.is3;
        fc[8] = c.m.ksig;
        fc[9] = (c.m.mu - c.m.ma) - c.m.ktau;
        fc[10] = c.m.ma + c.m.ktau;
        fc[11] = 0.0;
    }
    {
        const mf_status ss = points_scratch(ctx, n_points, G);
        if (ss != MF_OK) return ss;
    }
    auto up = [](size_t x) { return (x + 255) / 256 * 256; };
    const int64_t P = ctx->p_points;
    const int C = ctx->p_chunks;
    FourDPointsArgs a;
    for (int i = 0; i < 12; ++i) a.col[i] = m->col[i];
    a.n = m->n_events;
    a.n_pad = m->n_pad;
    a.mref = mref;
    char* q = ctx->p_blk;
    double* d_blk = reinterpret_cast<double*>(q);
    a.coef = d_blk;
    a.pconst = d_blk + 16 * n_points;
    const double* d_fc = d_blk + (16 + kP4PointConsts) * n_points;
    q += up(sizeof(FourDConsts) * P) + up(sizeof(int) * P);
    a.partials = reinterpret_cast<double*>(q);
    q += up(sizeof(double) * P * MF_MAX_NACC * C);
    a.bad_partials = reinterpret_cast<unsigned*>(q);
    a.n_points = (int)n_points;
    const dim3 grid((unsigned)G, (unsigned)((n_points + per_pass - 1) / per_pass));
    const size_t smem4 = sizeof(double) * 2 * kBlock * kP4StageDoubles;  // 48 KB: above the default dynamic limit with the static part
    static const cudaError_t attr4 = [&] {
        cudaError_t e = cudaFuncSetAttribute(fourd_points_mma_kernel<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem4);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(fourd_points_mma_inline_kernel<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem4);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(fourd_points_mma_kernel<3>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem4);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(fourd_points_mma_kernel<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem4);
        return e;
    }();
    MF_CUDA(ctx, attr4);
    if (inl) {
        ia.a = a;
        ia.a.coef = nullptr;
        ia.a.pconst = nullptr;
        ic.partials = a.partials;
        ic.bad_partials = a.bad_partials;
        ic.G = G;
        ic.n_points = (int)n_points;
        ic.sum_m = m->d_sum_m;
        ic.n = (double)m->n_events;
        ic.out = out_dev;
        const bool pdl_ok = !take_fresh(m);
        auto launch = [&](auto kernel, dim3 g, int block, size_t smem, bool allow, const auto& arg) {
            static const bool no_pdl = std::getenv("MF_NO_PDL") != nullptr;
            cudaLaunchConfig_t cfg = {};
            cfg.gridDim = g;
            cfg.blockDim = dim3((unsigned)block);
            cfg.dynamicSmemBytes = smem;
            cfg.stream = ctx->stream;
            cudaLaunchAttribute attr[1];
            attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
            attr[0].val.programmaticStreamSerializationAllowed = 1;
            cfg.attrs = attr;
            cfg.numAttrs = (allow && !no_pdl) ? 1 : 0;
            return cudaLaunchKernelEx(&cfg, kernel, arg);
        };
        MF_CUDA(ctx, launch(fourd_points_mma_inline_kernel<2>, grid, kBlock, smem4, pdl_ok, ia));
        MF_CUDA(ctx, launch(fourd_points_combine_inline_kernel, dim3((unsigned)n_points), kP4CombineThreads, 0, true, ic));
        ctx->launches += 2;
        return MF_OK;
    }
    MF_CUDA(ctx, cudaMemcpyAsync(d_blk, h_blk, per_point * n_points, cudaMemcpyHostToDevice, ctx->stream));
    MF_CUDA(ctx, cudaEventRecord(ctx->pts_copied[stage], ctx->stream));
    take_fresh(m);
    if (per_pass == 32) fourd_points_mma_kernel<4><<<grid, kBlock, smem4, ctx->stream>>>(a);
    else if (per_pass == 24) fourd_points_mma_kernel<3><<<grid, kBlock, smem4, ctx->stream>>>(a);
    else fourd_points_mma_kernel<2><<<grid, kBlock, smem4, ctx->stream>>>(a);
    fourd_points_combine_kernel<<<(unsigned)n_points, kP4CombineThreads, 0, ctx->stream>>>(
        a.partials, a.bad_partials, G, (int)n_points, d_fc, m->d_sum_m, (double)m->n_events, out_dev);
    MF_CUDA(ctx, cudaGetLastError());
    ctx->launches += 2;
    return MF_OK;
}

template <class M>
static mf_status launch_points(mf_model* m, int64_t n_points, const double* lambdas, double* out_dev)
{
    mf_ctx* ctx = m->ctx;
    const int K = M::K;
    using Consts = typename M::Consts;
    const size_t b_consts = sizeof(Consts) * n_points;
    char* h_blk = nullptr;
    int stage = 0;
    MF_CUDA(ctx, points_stage(ctx, b_consts, &h_blk, &stage));
    Consts* hc = reinterpret_cast<Consts*>(h_blk);
    for (int64_t p = 0; p < n_points; ++p)
        if (!host_consts<M>(m, lambdas + p * K, hc[p]))
            return mf_fail(ctx, MF_ERR_PARAM_DOMAIN, "mf_nll_grad_points: lambda " + std::to_string((long long)p) +
                                                         " is outside the parameter domain");
    // CTAs: whole waves of the resident capacity, about 64k events per CTA
    const int64_t slots = (int64_t)M::BATCH_RESIDENT_CTAS * ctx->sm_count;
    static const int64_t per_cta = std::getenv("MF_POINTS_CTA_EVENTS") ? std::atoll(std::getenv("MF_POINTS_CTA_EVENTS")) : 65536;  // tuning knob
    const int64_t waves = std::max<int64_t>(1, (n_points * m->n_pad + slots * per_cta - 1) / (slots * per_cta));
    const int64_t units = (M::NCOL == 1) ? (m->n_pad / kItem + kGroupItems - 1) / kGroupItems : m->n_pad / kItem;  // per warp: groups or items
    const int64_t max_chunks = std::max<int64_t>(1, (units + M::BATCH_BLOCK / 32 - 1) / (M::BATCH_BLOCK / 32));
    const int64_t chunks64 = std::max<int64_t>(1, std::min<int64_t>(max_chunks, waves * slots / n_points));
    if (n_points * chunks64 > (int64_t)0x7fffffff)
        return mf_fail(ctx, MF_ERR_ARG, "mf_nll_grad_points: n_points x event chunks exceeds the grid limit; split the call");
    const int chunks = (int)chunks64;
    {
        const mf_status ss = points_scratch(ctx, n_points, chunks);
        if (ss != MF_OK) return ss;
    }
    auto up = [](size_t x) { return (x + 255) / 256 * 256; };
    const int64_t P = ctx->p_points;
    const int C = ctx->p_chunks;
    BatchArgs<M> a;
    for (int i = 0; i < M::NCOL; ++i) a.col[i] = m->col[i];
    a.toy_stride = 0;
    a.shared_data = 1;
    a.n = m->n_events;
    a.n_items = m->n_pad / kItem;
    a.chunks = chunks;
    a.ma = m->ma;
    a.mb = m->mb;
    a.sum_m = m->d_sum_m;
    a.lam = nullptr;
    a.lam_external = 0;
    char* q = ctx->p_blk;
    a.consts = reinterpret_cast<Consts*>(q);
    q += up(sizeof(FourDConsts) * P);
    a.consts_ok = reinterpret_cast<int*>(q);
    q += up(sizeof(int) * P);
    a.partials = reinterpret_cast<double*>(q);
    q += up(sizeof(double) * P * MF_MAX_NACC * C);
    a.bad_partials = reinterpret_cast<unsigned*>(q);
    q += up(sizeof(unsigned) * P * C);
    a.ticket = reinterpret_cast<unsigned*>(q);
    a.ids = nullptr;
    a.out = out_dev;
    a.ahead = 0;  // one dataset for every point: it comes from L2 anyway
    a.n_active = (int)n_points;
    // The kernel reads the constants in place from the pinned, device-mapped staging block (one 200-byte read per CTA, behind its
    // first event loads): no copy sits between this launch and the previous kernel on the stream, so the programmatic launch
    // lets this call's CTAs start in the tail of the previous call (measured, C1, ms per 1000 evaluations issued as 10 / 4 / 2 / 1
    // calls: 1.84 / 1.66 / 1.58 / 1.55 with the copy, 1.52 / 1.51 / 1.51 / 1.51 without).  MF_POINTS_COPY=1: the stream-ordered copy to device memory instead.
    static const bool copy_consts = std::getenv("MF_POINTS_COPY") != nullptr;
    bool pdl_ok = !take_fresh(m);  // a fresh model's S1 kernels must have completed: no early start behind them
    if (copy_consts) {
        MF_CUDA(ctx, cudaMemcpyAsync(a.consts, hc, b_consts, cudaMemcpyHostToDevice, ctx->stream));  // pinned: asynchronous
        pdl_ok = true;  // the copy precedes the launch: the kernel cannot start before what is ahead of the copy has completed
    } else {
        typename M::Consts* dc = nullptr;
        MF_CUDA(ctx, cudaHostGetDevicePointer(reinterpret_cast<void**>(&dc), hc, 0));
        a.consts = dc;
    }
    MF_CUDA(ctx, launch_pdl(nll_grad_batch_kernel<M>, (int)(n_points * chunks), ctx->stream, a, M::BATCH_BLOCK, 0, pdl_ok));
    MF_CUDA(ctx, cudaEventRecord(ctx->pts_copied[stage], ctx->stream));  // the staging block is free again after this kernel
    ++ctx->launches;
    return MF_OK;
}

extern "C" mf_status mf_nll_grad_points(mf_model* m, int64_t n_points, const double* lambdas, double* out_dev)
{
    if (!m || !lambdas || !out_dev || n_points < 0)
        return mf_fail(m ? m->ctx : nullptr, MF_ERR_ARG, "mf_nll_grad_points: bad argument");
    if (m->n_toys != 1) return mf_fail(m->ctx, MF_ERR_ARG, "mf_nll_grad_points: dataset has n_toys != 1");
    if (n_points == 0) return MF_OK;
    if (uses_second(m, false)) {  // weighted: one second-order evaluation (gradient mode) per point, in stream order
        for (int64_t p = 0; p < n_points; ++p) {
            const mf_status st = dispatch_second<0>(m, lambdas + p * m->K, out_dev + p * (m->K + 2));
            if (st != MF_OK) return st;
        }
        return MF_OK;
    }
    // few points: back-to-back pipelined single evaluations are faster.  Measured cross-overs (us per evaluation as singles /
    // as one many-points call): mass model, consecutive (point, chunk) calls overlapping: 8 points 2.99 / 2.22 at 1e6 events,
    // 2.86 / 1.31 at 1e4; 4 points 3.64 / 3.79 and 3.55 / 2.49.  Angular model (C2, L2-resident singles 7.7): one 16-point pass
    // costs ~40 us: 4 points 10.1, 8 points 5.1.  4D model (C3, singles 27.7): one pass ~245 us: 8 points 30.6, 12 points 20.4.
    static const int env_min_batch = std::getenv("MF_POINTS_MIN_BATCH") ? std::atoi(std::getenv("MF_POINTS_MIN_BATCH")) : 0;  // tuning knob
    const int min_batch = env_min_batch > 0                 ? env_min_batch
                          : (m->kind == MF_MASS_GAUSS_EXP)  ? (m->n_pad <= 200000 ? 4 : 8)
                          : (m->kind == MF_ANGULAR_KSTMUMU) ? 6
                                                            : 10;
    if (n_points < min_batch) {
        for (int64_t p = 0; p < n_points; ++p) {
            const mf_status st = dispatch_single(m, lambdas + p * m->K, out_dev + p * (m->K + 2), n_points > 1);
            if (st != MF_OK) return st;
        }
        return MF_OK;
    }
    if (n_points > (int64_t)1 << 20) return mf_fail(m->ctx, MF_ERR_ARG, "mf_nll_grad_points: more than 2^20 points per call");
    switch (m->kind) {
    case MF_MASS_GAUSS_EXP: return launch_points<MassModel>(m, n_points, lambdas, out_dev);
    case MF_ANGULAR_KSTMUMU: {
        static const bool no_mma = std::getenv("MF_NO_POINTS_MMA") != nullptr;  // ablation switch: the (point, chunk) kernel
        return no_mma ? launch_points<AngularModel>(m, n_points, lambdas, out_dev)
                      : launch_points_angular_mma(m, n_points, lambdas, out_dev);
    }
    default: {
        static const bool no_mma4 = std::getenv("MF_NO_POINTS_MMA") != nullptr;
        if (!no_mma4) {
            bool handled = false;
            const mf_status st = launch_points_fourd_mma(m, n_points, lambdas, out_dev, &handled);
            if (handled || st != MF_OK) return st;
        }
        return launch_points<FourDModel>(m, n_points, lambdas, out_dev);
    }
    }
}

// The same sweep with HOST results: one call evaluates n_points parameter points and returns when the values are on the
// host (BASELINE.json configs[1] as a user of the library sees it).
extern "C" mf_status mf_nll_grad_sweep(mf_model* m, int64_t n_points, const double* lambdas, double* nll, double* grad,
                                       int64_t* n_bad)
{
    if (!m || !lambdas || !nll || n_points < 0) return mf_fail(m ? m->ctx : nullptr, MF_ERR_ARG, "mf_nll_grad_sweep: bad argument");
    if (n_points == 0) return MF_OK;
    mf_ctx* ctx = m->ctx;
    const int K = m->K, row = K + 2;
    // The kernels write the result rows straight into the context's pinned, device-mapped staging block (grow-only): no
    // device-to-host copy behind them, one stream synchronise, then the rows are scattered to the caller's arrays
    const size_t bytes = sizeof(double) * n_points * row;
    if (ctx->h_stage_bytes < bytes) {
        if (ctx->h_stage) {
            cudaStreamSynchronize(ctx->stream);
            cudaFreeHost(ctx->h_stage);
            ctx->h_stage = nullptr;
            ctx->h_stage_bytes = 0;
        }
        MF_CUDA(ctx, cudaHostAlloc(reinterpret_cast<void**>(&ctx->h_stage), bytes, cudaHostAllocMapped));
        ctx->h_stage_bytes = bytes;
    }
    double* h = reinterpret_cast<double*>(ctx->h_stage);
    double* d_rows = nullptr;
    MF_CUDA(ctx, cudaHostGetDevicePointer(reinterpret_cast<void**>(&d_rows), h, 0));
    // Mass model (the (point, chunk) kernel, whose consecutive calls overlap on the GPU): the sweep is issued in sub-calls of
    // 128 points, so that the host derives the constants of the later points (~0.18 us each) while the GPU evaluates the
    // earlier ones: a 1000-point sweep of C1 1.74 -> 1.60 ms.  A point outside the domain in a later sub-call is found after the
    // earlier ones were enqueued; nothing is copied back then, so the caller's arrays stay untouched as documented.
    static const int64_t sub = std::getenv("MF_SWEEP_SUBCALL") ? std::max<int64_t>(16, std::atoll(std::getenv("MF_SWEEP_SUBCALL"))) : 128;
    if (m->kind == MF_MASS_GAUSS_EXP && !m->wts && n_points >= 2 * sub) {
        for (int64_t p0 = 0; p0 < n_points; p0 += sub) {
            const int64_t np = std::min<int64_t>(sub, n_points - p0);
            const mf_status st = mf_nll_grad_points(m, np, lambdas + p0 * K, d_rows + p0 * row);
            if (st != MF_OK) {
                if (st == MF_ERR_PARAM_DOMAIN)  // the index in the message is relative to the sub-call
                    mf_fail(ctx, st, "mf_nll_grad_sweep: a lambda in [" + std::to_string((long long)p0) + ", " +
                                         std::to_string((long long)(p0 + np)) + ") is outside the parameter domain");
                return st;
            }
        }
    } else {
        const mf_status st = mf_nll_grad_points(m, n_points, lambdas, d_rows);
        if (st != MF_OK) return st;
    }
    MF_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    int64_t bad_points = 0;
    for (int64_t p = 0; p < n_points; ++p) {
        const double* o = h + p * row;
        nll[p] = o[0];
        if (grad) std::memcpy(grad + p * K, o + 1, sizeof(double) * K);
        if (o[K + 1] != 0.0) ++bad_points;
    }
    if (n_bad) *n_bad = bad_points;
    return MF_OK;
}


// ---- resident evaluation kernel (mf_server.cuh) ---------------------------------------------------------------------

static bool server_applicable(const mf_model* m)
{
    static const bool off = std::getenv("MF_NO_SERVER") != nullptr;  // ablation switch: every evaluation is a launch
    return !off && m->kind == MF_MASS_GAUSS_EXP && m->n_toys == 1 && !m->wts && m->n_events > 0 && m->srv_failures < 3;
}

// Writes a request into the mapped slot: per 64-byte line the payload words first, then the line's request number
// (x86 keeps the store order; the device reads a line atomically).  c == NULL: the numbers only.
static void server_post(mf_model* m, unsigned long long seq, const MassConsts* c, int kind)
{
    volatile unsigned long long* req = reinterpret_cast<volatile unsigned long long*>(m->h_req);
    if (c) {
        unsigned long long pay[kServerReqPayload] = {};
        pay[0] = (unsigned long long)kind;
        static_assert(sizeof(MassConsts) + 8 <= sizeof(pay), "request payload too small");
        std::memcpy(pay + 1, c, sizeof(MassConsts));
        for (int l = 0; l < kServerReqLines; ++l)
            for (int j = 0; j < 7; ++j) req[8 * l + 1 + j] = pay[7 * l + j];
    }
    std::atomic_thread_fence(std::memory_order_release);
    for (int l = 0; l < kServerReqLines; ++l) req[8 * l] = seq;
}

static void server_stop(mf_model* m)
{
    if (!m->srv_running) return;
    server_post(m, kServerExit, nullptr, 0);
    cudaStreamSynchronize(m->ctx->server_stream);
    cudaGetLastError();
    m->srv_running = false;
    server_post(m, m->srv_seq, nullptr, 0);  // not a new request for the next kernel
}

// Launches the resident kernel.  pending: request srv_seq has been written and is to be served by this kernel.
static mf_status server_launch(mf_model* m, bool pending)
{
    mf_ctx* ctx = m->ctx;
    if (!ctx->server_stream) MF_CUDA(ctx, cudaStreamCreateWithFlags(&ctx->server_stream, cudaStreamNonBlocking));
    const int64_t n_groups = (m->n_pad / kItem + kGroupItems - 1) / kGroupItems;
    const int G = (int)std::max<int64_t>(1, std::min<int64_t>((n_groups + kWarps - 1) / kWarps, ctx->sm_count));
    if (!m->h_req) {
        MF_CUDA(ctx, host_slot_acquire(ctx, &m->h_req, &m->d_req_mapped));
        MF_CUDA(ctx, dev_alloc(ctx, reinterpret_cast<char**>(&m->srv_relay), sizeof(ServerRelay)));
        MF_CUDA(ctx, dev_alloc(ctx, &m->srv_partials, sizeof(double) * MassHessModel::NACC * ctx->sm_count));
        MF_CUDA(ctx, dev_alloc(ctx, &m->srv_bad, sizeof(unsigned) * ctx->sm_count));
        MF_CUDA(ctx, dev_alloc(ctx, &m->srv_ticket, sizeof(unsigned)));
        MF_CUDA(ctx, cudaMemsetAsync(m->srv_ticket, 0, sizeof(unsigned), ctx->stream));
        MF_CUDA(ctx, cudaMemsetAsync(m->srv_relay, 0, sizeof(ServerRelay), ctx->stream));
        ctx->serving.push_back(m);
    }
    // everything enqueued on the work stream (S0 / S1 kernels, the scratch set-up above) is complete before the kernel starts
    MF_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    const unsigned long long first = pending ? m->srv_seq - 1 : m->srv_seq;
    if (!pending) server_post(m, first, nullptr, 0);
    reinterpret_cast<volatile unsigned long long*>(m->h_out)[kServerRepExited] = 0ull;
    MF_CUDA(ctx, cudaMemcpyAsync(&static_cast<ServerRelay*>(m->srv_relay)->seq, &first, sizeof(first), cudaMemcpyHostToDevice,
                                 ctx->server_stream));  // pageable source: staged before the call returns
    ServerArgs a;
    a.col0 = m->col[0];
    a.n = m->n_events;
    a.n_items = m->n_pad / kItem;
    a.sum_m = m->d_sum_m;
    a.req = reinterpret_cast<const unsigned long long*>(m->d_req_mapped);
    a.rep = m->d_out_mapped;
    a.relay = static_cast<ServerRelay*>(m->srv_relay);
    a.partials = m->srv_partials;
    a.bad_partials = m->srv_bad;
    a.ticket = m->srv_ticket;
    a.first_seq = first;
    static const unsigned long long idle_us = std::getenv("MF_SERVER_IDLE_US") ? std::strtoull(std::getenv("MF_SERVER_IDLE_US"), nullptr, 10) : 5000;
    a.idle_ns = idle_us * 1000ull;
    nll_server_kernel<<<G, kBlock, 0, ctx->server_stream>>>(a);
    MF_CUDA(ctx, cudaGetLastError());
    m->srv_running = true;
    m->fresh = false;
    ++ctx->launches;
    return MF_OK;
}

// One evaluation through the resident kernel.  *handled = false: the server gave up (a tool serialises kernels): the caller
// evaluates by launch.
static mf_status server_eval_sync(mf_model* m, const double* lambda, double* nll, double* grad, double* hess, const char* who,
                                  bool* handled)
{
    mf_ctx* ctx = m->ctx;
    const int K = m->K;
    *handled = true;
    MassConsts c;
    if (!mass_consts(lambda, m->ma, m->mb, c)) return mf_fail(ctx, MF_ERR_PARAM_DOMAIN, "lambda outside the parameter domain");
    if (!m->h_req) {  // first use: set up and launch, then issue the request
        const mf_status st = server_launch(m, false);
        if (st != MF_OK) return st;
    }
    const unsigned long long want = ++m->srv_seq;
    server_post(m, want, &c, hess ? 1 : 0);
    if (!m->srv_running) {
        const mf_status st = server_launch(m, true);
        if (st != MF_OK) return st;
    }
    volatile unsigned long long* rep = reinterpret_cast<volatile unsigned long long*>(m->h_out);
    for (unsigned spins = 1; rep[kServerRepDone] != want; ++spins) {
        if ((spins & 0x3FFF) == 0 && rep[kServerRepExited] != 0 && rep[kServerRepDone] != want) {
            // the kernel left (idle time-out racing with this request, or a tool ran it to completion before we could ask)
            cudaStreamSynchronize(ctx->server_stream);
            m->srv_running = false;
            if (++m->srv_failures >= 3) {  // give up on the server for this model
                *handled = false;
                return MF_OK;
            }
            const mf_status st = server_launch(m, true);
            if (st != MF_OK) return st;
        }
        if ((spins & 0xFFFFF) == 0) {
            const cudaError_t q = cudaStreamQuery(ctx->server_stream);
            if (q != cudaErrorNotReady && q != cudaSuccess) return mf_fail(ctx, MF_ERR_CUDA, std::string(who) + ": " + cudaGetErrorString(q));
        }
    }
    std::atomic_thread_fence(std::memory_order_acquire);
    m->srv_failures = 0;
    *nll = m->h_out[0];
    if (grad) std::memcpy(grad, m->h_out + 1, sizeof(double) * K);
    const int nout = hess ? 1 + K + K * (K + 1) / 2 : K + 1;
    if (hess) {
        int q = 1 + K;
        for (int i = 0; i < K; ++i)
            for (int j = i; j < K; ++j, ++q) hess[i * K + j] = hess[j * K + i] = m->h_out[q];
    }
    if (m->h_out[nout] != 0.0)
        return mf_fail(ctx, MF_NONPOSITIVE_PDF, "P <= 0 for " + std::to_string((long long)m->h_out[nout]) + " events at this lambda");
    return MF_OK;
}

extern "C" mf_status mf_model_serve(mf_model* m, int on)
{
    if (!m) return MF_ERR_ARG;
    if (on) {
        if (!server_applicable(m))
            return mf_fail(m->ctx, MF_ERR_ARG, "mf_model_serve: only unweighted MF_MASS_GAUSS_EXP models on a single non-empty dataset");
        m->srv_on = true;
    } else {
        m->srv_on = false;
        server_stop(m);
    }
    return MF_OK;
}

extern "C" int mf_model_is_served(const mf_model* m) { return m && m->srv_on ? 1 : 0; }

mf_status mf_server_begin(mf_model* m)
{
    if (server_applicable(m)) m->srv_on = true;
    return MF_OK;
}

void mf_server_end(mf_model* m, bool was_on)
{
    if (!was_on) {
        m->srv_on = false;
        server_stop(m);
    }
}

// One synchronous evaluation: value, gradient and (hess != NULL, mass model) the K x K Hessian.
static mf_status eval_sync(mf_model* m, const double* lambda, double* nll, double* grad, double* hess, const char* who)
{
    mf_ctx* ctx = m->ctx;
    const int K = m->K;
    if (m->srv_on && server_applicable(m)) {  // resident kernel: no launch, no completion latency
        bool handled = false;
        const mf_status ss = server_eval_sync(m, lambda, nll, grad, hess, who, &handled);
        if (handled) return ss;
    }
    // the last CTA writes the result, then the done word, to mapped pinned memory; the host spins on the
    // done word (a stream synchronise costs ~20 us of driver latency per call, the kernel 4-30 us)
    const mf_status st = dispatch_single(m, lambda, m->d_out_mapped, false, true, hess != nullptr);
    if (st != MF_OK) return st;
    volatile unsigned long long* done = reinterpret_cast<volatile unsigned long long*>(m->h_out + MF_HOST_DONE_INDEX);
    const unsigned long long want = m->seq;
    for (unsigned spins = 1; *done != want; ++spins) {
        if ((spins & 0xFFFF) == 0) {  // every ~65k polls: make sure the stream is still alive
            const cudaError_t q = cudaStreamQuery(ctx->stream);
            if (q != cudaErrorNotReady && *done != want) {
                if (q == cudaSuccess) continue;  // completed: the word is on its way
                return mf_fail(ctx, MF_ERR_CUDA, std::string(who) + ": " + cudaGetErrorString(q));
            }
        }
    }
    std::atomic_thread_fence(std::memory_order_acquire);
    *nll = m->h_out[0];
    if (grad) std::memcpy(grad, m->h_out + 1, sizeof(double) * K);
    const int nout = hess ? 1 + K + K * (K + 1) / 2 : K + 1;
    if (hess) {
        int q = 1 + K;
        for (int i = 0; i < K; ++i)
            for (int j = i; j < K; ++j, ++q) hess[i * K + j] = hess[j * K + i] = m->h_out[q];
    }
    if (m->h_out[nout] != 0.0)
        return mf_fail(ctx, MF_NONPOSITIVE_PDF,
                       "P <= 0 for " + std::to_string((long long)m->h_out[nout]) + " events at this lambda");
    return MF_OK;
}

extern "C" mf_status mf_nll_grad(mf_model* m, const double* lambda, double* nll, double* grad)
{
    if (!m || !lambda || !nll) return mf_fail(m ? m->ctx : nullptr, MF_ERR_ARG, "mf_nll_grad: NULL argument");
    if (m->n_toys != 1) return mf_fail(m->ctx, MF_ERR_ARG, "mf_nll_grad: dataset has n_toys != 1; use mf_nll_grad_batch");
    if (uses_second(m, false)) return second_sync(m, lambda, nll, grad, nullptr, nullptr, "mf_nll_grad");
    return eval_sync(m, lambda, nll, grad, nullptr, "mf_nll_grad");
}

extern "C" mf_status mf_nll_grad_hess(mf_model* m, const double* lambda, double* nll, double* grad, double* hess)
{
    if (!m || !lambda || !nll || !hess) return mf_fail(m ? m->ctx : nullptr, MF_ERR_ARG, "mf_nll_grad_hess: NULL argument");
    if (m->n_toys != 1) return mf_fail(m->ctx, MF_ERR_ARG, "mf_nll_grad_hess: dataset has n_toys != 1; use mf_nll_grad_hess_batch");
    if (uses_second(m, true)) return second_sync(m, lambda, nll, grad, hess, nullptr, "mf_nll_grad_hess");
    return eval_sync(m, lambda, nll, grad, hess, "mf_nll_grad_hess");
}

extern "C" mf_status mf_nll_grad_hess_fisher(mf_model* m, const double* lambda, double* nll, double* grad, double* hess,
                                             double* fisher)
{
    if (!m || !lambda || !nll || !fisher)
        return mf_fail(m ? m->ctx : nullptr, MF_ERR_ARG, "mf_nll_grad_hess_fisher: NULL argument");
    if (m->n_toys != 1) return mf_fail(m->ctx, MF_ERR_ARG, "mf_nll_grad_hess_fisher: dataset has n_toys != 1");
    return second_sync(m, lambda, nll, grad, hess, fisher, "mf_nll_grad_hess_fisher");
}

// 1: the analytic Hessian is available (every family, single datasets and batched toys)
extern "C" int mf_model_has_hessian(const mf_model* m) { return m ? 1 : 0; }

extern "C" int mf_model_is_weighted(const mf_model* m) { return m && m->wts ? 1 : 0; }

template <class M>
static mf_status launch_batch(mf_model* m, int n_active, const double* lam_dev = nullptr, double* out_dev = nullptr)
{
    mf_ctx* ctx = m->ctx;
    BatchArgs<M> a;
    for (int i = 0; i < M::NCOL; ++i) a.col[i] = m->col[i];
    a.toy_stride = m->n_pad;
    a.shared_data = 0;
    a.n = m->n_events;
    a.n_items = m->n_pad / kItem;
    a.chunks = m->chunks;
    a.ma = m->ma;
    a.mb = m->mb;
    a.sum_m = m->d_sum_m;
    a.lam = lam_dev ? lam_dev : m->d_lam;
    a.lam_external = lam_dev ? 1 : 0;
    a.consts = static_cast<typename M::Consts*>(m->d_consts);
    a.consts_ok = m->d_consts_ok;
    a.ids = (n_active == m->n_toys) ? nullptr : m->d_ids;
    a.partials = m->b_partials;
    a.bad_partials = m->b_bad;
    a.ticket = m->ticket + kRing;
    a.out = out_dev ? out_dev : m->d_bout;
    a.n_active = n_active;
    a.ahead = 0;
    if (m->chunks == 1 && M::NCOL == 1) {
        static const int env_ahead = [] { const char* e = getenv("MF_BATCH_AHEAD"); return e ? atoi(e) : -1; }();
        a.ahead = env_ahead >= 0 ? env_ahead : ctx->sm_count;  // measured on B200: 74 .. 296 slots alike, 592 and 0 slower
    }
    // both kernels are launched programmatically: the constants kernel of evaluation i+1 starts (and computes) while the
    // batched kernel of evaluation i drains, and waits for it to complete only before overwriting the constants
    MF_CUDA(ctx, launch_pdl_v(batch_consts_kernel<M>, (n_active + 127) / 128, 128, 0, ctx->stream, !take_fresh(m), a, n_active));
    if constexpr (M::NCOL == 1) {
        // one-column toys come from HBM: events staged through shared memory by cp.async, 3 groups deep (0: direct loads)
        static const int env_stages = [] { const char* e = getenv("MF_BATCH_STAGES"); return e ? atoi(e) : 3; }();
        const int stages = env_stages;
        // CTA size by the number of active toys (BatchShape, mf_kernels.cuh): measured cross-overs at 24 and 40 toys per SM
        static const int env_block = [] { const char* e = getenv("MF_BATCH_BLOCK"); return e ? atoi(e) : 0; }();  // tuning knob
        const int block = (m->chunks != 1 || stages != 3)                ? 0
                          : (env_block == 32 || env_block == 64)         ? env_block
                          : env_block                                    ? 0
                          : (n_active >= 40 * (int64_t)ctx->sm_count)    ? 32
                          : (n_active >= 24 * (int64_t)ctx->sm_count)    ? 64
                                                                         : 0;
        if (block == 32) MF_CUDA(ctx, launch_pdl(nll_grad_batch_kernel<M, 3, 32>, n_active, ctx->stream, a, 32));
        else if (block == 64) MF_CUDA(ctx, launch_pdl(nll_grad_batch_kernel<M, 3, 64>, n_active, ctx->stream, a, 64));
        else if (stages == 2) MF_CUDA(ctx, launch_pdl(nll_grad_batch_kernel<M, 2>, n_active * m->chunks, ctx->stream, a, M::BATCH_BLOCK));
        else if (stages == 3) MF_CUDA(ctx, launch_pdl(nll_grad_batch_kernel<M, 3>, n_active * m->chunks, ctx->stream, a, M::BATCH_BLOCK));
        else if (stages == 4) MF_CUDA(ctx, launch_pdl(nll_grad_batch_kernel<M, 4>, n_active * m->chunks, ctx->stream, a, M::BATCH_BLOCK));
        else MF_CUDA(ctx, launch_pdl(nll_grad_batch_kernel<M>, n_active * m->chunks, ctx->stream, a, M::BATCH_BLOCK));
    } else {
        MF_CUDA(ctx, launch_pdl(nll_grad_batch_kernel<M>, n_active * m->chunks, ctx->stream, a, M::BATCH_BLOCK));
    }
    ctx->launches += 2;
    return MF_OK;
}

extern "C" mf_status mf_nll_grad_batch_async(mf_model* m, int64_t n_toys, const double* lambdas_dev, double* out_dev)
{
    if (!m || !lambdas_dev || !out_dev) return mf_fail(m ? m->ctx : nullptr, MF_ERR_ARG, "mf_nll_grad_batch_async: NULL argument");
    if (n_toys != m->n_toys || m->n_toys < 2 || !m->d_lam)
        return mf_fail(m->ctx, MF_ERR_ARG, "mf_nll_grad_batch_async: needs a dataset with n_toys > 1 and n_toys equal to it");
    switch (m->kind) {
    case MF_MASS_GAUSS_EXP: return launch_batch<MassModel>(m, (int)n_toys, lambdas_dev, out_dev);
    case MF_ANGULAR_KSTMUMU: return launch_batch<AngularModel>(m, (int)n_toys, lambdas_dev, out_dev);
    default: return launch_batch<FourDModel>(m, (int)n_toys, lambdas_dev, out_dev);
    }
}

// T toys at their own parameter points; hess != NULL (mass model): also the K x K Hessian per toy.
static mf_status eval_batch(mf_model* m, int64_t n_toys, const double* lambdas, const uint8_t* active, double* nll,
                            double* grad, double* hess, const char* who)
{
    mf_ctx* ctx = m->ctx;
    const int K = m->K;
    if (n_toys != m->n_toys) return mf_fail(ctx, MF_ERR_ARG, std::string(who) + ": n_toys does not match the dataset");
    if (m->n_toys < 2 && !m->d_lam) {
        // a 1-toy dataset evaluated through the batch entry: same result as the single call
        if (active && !active[0]) return MF_OK;
        double g[MF_MAX_PARAMS];
        const mf_status st = uses_second(m, hess != nullptr) ? second_sync(m, lambdas, nll, g, hess, nullptr, who)
                                                             : eval_sync(m, lambdas, nll, g, hess, who);
        if (st == MF_ERR_PARAM_DOMAIN || st == MF_NONPOSITIVE_PDF) {
            *nll = INFINITY;
            if (grad) for (int k = 0; k < K; ++k) grad[k] = NAN;
            if (hess) for (int k = 0; k < K * K; ++k) hess[k] = NAN;
            return MF_OK;
        }
        if (st == MF_OK && grad) std::memcpy(grad, g, sizeof(double) * K);
        return st;
    }
    MF_CUDA(ctx, stage_views(m));
    int n_active = 0;
    for (int64_t t = 0; t < n_toys; ++t) {
        if (active && !active[t]) continue;
        m->h_ids[n_active] = (int)t;
        std::memcpy(m->h_lam + (int64_t)n_active * K, lambdas + t * K, sizeof(double) * K);
        ++n_active;
    }
    if (n_active == 0) return MF_OK;
    // lambda and the result rows stay in the pinned, device-mapped staging block: the constants kernel reads the former in place,
    // the batched kernel writes the latter in place (one row per toy): no copy in either direction, one stream synchronise.
    // (The 4D Hessian path goes through the second-order kernel toy by toy and keeps its device rows and the copy.)
    static const bool copy_io = std::getenv("MF_BATCH_COPY") != nullptr;  // ablation: stream-ordered copies of lambda and the rows
    const bool in_place = !copy_io && !(hess && m->kind == MF_MASS_X_ANGULAR);
    double *d_lam_map = nullptr, *d_out_map = nullptr;
    if (in_place) {
        MF_CUDA(ctx, cudaHostGetDevicePointer(reinterpret_cast<void**>(&d_lam_map), m->h_lam, 0));
        MF_CUDA(ctx, cudaHostGetDevicePointer(reinterpret_cast<void**>(&d_out_map), m->h_bout, 0));
    } else {
        MF_CUDA(ctx, cudaMemcpyAsync(m->d_lam, m->h_lam, sizeof(double) * n_active * K, cudaMemcpyHostToDevice, ctx->stream));
    }
    if (n_active < n_toys)
        MF_CUDA(ctx, cudaMemcpyAsync(m->d_ids, m->h_ids, sizeof(int) * n_active, cudaMemcpyHostToDevice, ctx->stream));
    mf_status st = MF_OK;
    std::vector<int> invalid;  // 4D Hessian: slots whose lambda is outside the parameter domain
    if (hess && m->kind == MF_MASS_X_ANGULAR) {
        // batched 4D toys: the second-order kernel (tensor-core contraction) toy by toy, in stream order
        const int row4 = 1 + K + K * (K + 1) / 2 + 1;
        for (int s = 0; s < n_active; ++s) {
            const mf_status ss = launch_second<FourDSecond, 1>(m, m->h_lam + (int64_t)s * K, m->d_bout + (int64_t)s * row4, m->h_ids[s]);
            if (ss == MF_ERR_PARAM_DOMAIN) invalid.push_back(s);
            else if (ss != MF_OK) return ss;
        }
    } else if (hess) {
        st = (m->kind == MF_MASS_GAUSS_EXP) ? launch_batch<MassHessModel>(m, n_active, d_lam_map, d_out_map)
                                            : launch_batch<AngularHessModel>(m, n_active, d_lam_map, d_out_map);
    } else {
        switch (m->kind) {
        case MF_MASS_GAUSS_EXP: st = launch_batch<MassModel>(m, n_active, d_lam_map, d_out_map); break;
        case MF_ANGULAR_KSTMUMU: st = launch_batch<AngularModel>(m, n_active, d_lam_map, d_out_map); break;
        default: st = launch_batch<FourDModel>(m, n_active, d_lam_map, d_out_map); break;
        }
    }
    if (st != MF_OK) return st;
    const int row = (hess ? 1 + K + K * (K + 1) / 2 : K + 1) + 1;
    if (!in_place)
        MF_CUDA(ctx, cudaMemcpyAsync(m->h_bout, m->d_bout, sizeof(double) * n_active * row, cudaMemcpyDeviceToHost, ctx->stream));
    MF_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    for (int s : invalid) {  // as the batched kernels report a domain error: +inf, NaN
        double* o = m->h_bout + (int64_t)s * row;
        o[0] = INFINITY;
        for (int k = 1; k < row - 1; ++k) o[k] = NAN;
    }
    for (int s = 0; s < n_active; ++s) {
        const int64_t t = m->h_ids[s];
        const double* o = m->h_bout + (int64_t)s * row;
        nll[t] = o[0];
        if (grad) std::memcpy(grad + t * K, o + 1, sizeof(double) * K);
        if (hess) {
            double* H = hess + t * K * K;
            int q = 1 + K;
            for (int i = 0; i < K; ++i)
                for (int j = i; j < K; ++j, ++q) H[i * K + j] = H[j * K + i] = o[q];
        }
    }
    return MF_OK;
}

extern "C" mf_status mf_nll_grad_batch(mf_model* m, int64_t n_toys, const double* lambdas, const uint8_t* active,
                                       double* nll, double* grad)
{
    if (!m || !lambdas || !nll) return mf_fail(m ? m->ctx : nullptr, MF_ERR_ARG, "mf_nll_grad_batch: NULL argument");
    return eval_batch(m, n_toys, lambdas, active, nll, grad, nullptr, "mf_nll_grad_batch");
}

extern "C" mf_status mf_nll_grad_hess_batch(mf_model* m, int64_t n_toys, const double* lambdas, const uint8_t* active,
                                            double* nll, double* grad, double* hess)
{
    if (!m || !lambdas || !nll || !hess)
        return mf_fail(m ? m->ctx : nullptr, MF_ERR_ARG, "mf_nll_grad_hess_batch: NULL argument");
    return eval_batch(m, n_toys, lambdas, active, nll, grad, hess, "mf_nll_grad_hess_batch");
}
