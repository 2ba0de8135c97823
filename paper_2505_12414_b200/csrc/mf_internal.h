// mf_internal.h — host-side objects behind the opaque handles of include/morefit_b200.h.
#pragma once
#include <cuda_runtime.h>

#include <cstdint>
#include <string>
#include <vector>

#include "../../include/morefit_b200.h"

struct mf_ctx {
    int device = 0;
    cudaStream_t stream = nullptr;
    int sm_count = 0;
    int64_t launches = 0;
    std::string err;
    // pinned + mapped slab of per-model result slots (MF_MAX_PARAMS + 2 doubles and the done word)
    double* h_slab = nullptr;
    double* d_slab = nullptr;
    std::vector<int> free_slots;
    // pinned staging of the batched (synchronous) calls, shared by all models of the context, grow-only
    char* h_stage = nullptr;
    size_t h_stage_bytes = 0;
    // pinned staging of the parameter-only constants of mf_nll_grad_points: a ring of blocks, each guarded by an event
    // recorded after its host-to-device copy, so that successive calls never wait for one another's copies
    static constexpr int kPointStages = 4;
    char* h_pts[kPointStages] = {};
    size_t h_pts_bytes[kPointStages] = {};
    cudaEvent_t pts_copied[kPointStages] = {};
    unsigned pts_seq = 0;
    // device scratch of the many-points evaluation (mf_nll_grad_points / mf_nll_grad_sweep), shared by all models of the
    // context (every launch is ordered on the one stream, and the kernel touches the scratch only after its programmatic
    // wait): grow-only, laid out as [consts | ok | partials | bad | ticket] for the largest (points, chunks) seen so far
    // mapped pinned result row of the synchronous second-order calls (up to 1 + 16 + 136 + 136 + 1 doubles) and its done word
    double* h_big = nullptr;
    double* d_big = nullptr;
    unsigned long long big_seq = 0;
    cudaStream_t server_stream = nullptr;  // resident evaluation kernels (mf_model_serve) run here, beside the work stream
    std::vector<struct mf_model*> serving;  // models whose resident kernel may be running
    char* p_blk = nullptr;
    size_t p_bytes = 0;
    int64_t p_points = 0;
    int p_chunks = 0;
};

constexpr int MF_HOST_SLOT_DOUBLES = 64;  // widest output row (angular Hessian: 45 + n_bad) and the done word
constexpr int MF_HOST_DONE_INDEX = 63;    // the 64-bit done word of a synchronous call
constexpr int MF_HOST_SLOTS = 4096;

// Reference-counted device buffer so that a model can outlive the dataset handle.
struct mf_devbuf {
    cudaStream_t stream = nullptr;  // freed in the order of this stream
    double* p = nullptr;
    size_t bytes = 0;
    int refs = 1;
};

struct mf_dataset {
    mf_ctx* ctx = nullptr;
    int ndim = 0;
    int64_t n_events = 0;  // per toy
    int64_t n_pad = 0;     // per toy, multiple of 64
    int64_t n_toys = 1;
    double lo[MF_MAX_DIMS] = {0, 0, 0, 0}, hi[MF_MAX_DIMS] = {0, 0, 0, 0};
    mf_devbuf* raw = nullptr;  // [ndim][n_toys][n_pad]
    mf_devbuf* wts = nullptr;  // [n_pad] event weights (padding 0), or NULL: unweighted (mf_dataset_set_weights)
};

constexpr int MF_MAX_COLS = 12;
constexpr int MF_MAX_NACC = 17;  // accumulators of the widest value+gradient model (points-mode scratch layout)

struct mf_model {
    mf_ctx* ctx = nullptr;
    mf_model_kind kind = MF_MASS_GAUSS_EXP;
    int K = 0, nacc = 0, ncol = 0;
    int64_t n_events = 0, n_pad = 0, n_toys = 1;
    double ma = 0, mb = 0;            // mass normalisation range [m_a, m_b]
    mf_devbuf* raw = nullptr;         // shared with the dataset
    double* cache = nullptr;          // [9][n_toys][n_pad] angular basis columns (S1), or NULL
    double2* d_sum_m = nullptr;       // device [n_toys]: event-only constants sum_i m_i as (hi, lo) (S1), NULL without a mass dimension
    const double* col[MF_MAX_COLS] = {};  // column base pointers, stride between toys = n_pad
    // single-dataset evaluation
    int grid = 1;                     // CTAs of the fused kernel
    double* partials = nullptr;       // device [kRing][nacc][grid]
    unsigned* bad_partials = nullptr; // device [kRing][grid]
    unsigned* ticket = nullptr;       // device, kRing (single) + n_toys (batch)
    unsigned long long* gen = nullptr;  // device [kRing]: evaluations completed per scratch slot
    unsigned long long seq = 0;       // evaluations enqueued so far (evaluation e uses slot e % kRing)
    bool fresh = true;                // no kernel of this model launched yet: its first launch is made in plain stream order
    cudaEvent_t s1_done = nullptr;    // recorded behind the S0/S1 kernels of mf_model_create: once it has completed, `fresh` no longer matters
    double* h_out = nullptr;          // pinned + mapped host slot: the output row, the 64-bit done word at MF_HOST_DONE_INDEX
    double* d_out_mapped = nullptr;   // device alias of h_out
    // batched evaluation
    int chunks = 1;                   // CTAs per toy
    double* b_partials = nullptr;     // device [n_toys][nacc][chunks] (chunks > 1 only)
    unsigned* b_bad = nullptr;        // device [n_toys][chunks]
    void* d_consts = nullptr;         // device [n_toys] parameter-only constants of the batch kernel
    int* d_consts_ok = nullptr;       // device [n_toys]
    double* d_lam = nullptr;          // device [n_toys][K]
    int* d_ids = nullptr;             // device [n_toys]
    double* d_bout = nullptr;         // device [n_toys][K+2]
    double* h_lam = nullptr;          // views into the context's pinned staging block, set by every batched call:
    int* h_ids = nullptr;             //   [n_toys][K], [n_toys], [n_toys][widest output row]
    double* h_bout = nullptr;
    int bout_row = 0;                 // widest output row + n_bad (doubles)
    double* d_sweep = nullptr;        // device [p_sweep_rows][K+2] results of mf_nll_grad_sweep (grow-only)
    int64_t p_sweep_rows = 0;
    // second-order sums by tensor-core contraction (mf_second.cuh): weighted models, the 4D Hessian, the Fisher matrix
    mf_devbuf* wts = nullptr;         // shared with the dataset; NULL = unweighted
    int s_grid = 0;                   // CTAs of nll_second_kernel
    double* s_partials = nullptr;     // device [NQ of the widest mode][s_grid]
    unsigned* s_bad = nullptr;        // device [s_grid]
    double* s_sums = nullptr;         // device [NQ]
    unsigned* s_ticket = nullptr;     // device, one word, zero between launches
    double* s_out = nullptr;          // device [NOUT + 1] of the widest mode
    // resident evaluation kernel (mf_server.cuh; mass model, n_toys == 1, unweighted)
    bool srv_on = false;              // requested (mf_model_serve, or for the duration of mf_fit)
    bool srv_running = false;         // a kernel has been launched and has not been seen to leave
    int srv_failures = 0;             // relaunches that did not produce an answer (tools that serialise kernels): then disabled
    unsigned long long srv_seq = 0;   // last request number issued
    double* h_req = nullptr;          // mapped pinned request slot (64 words) and its device alias
    double* d_req_mapped = nullptr;
    void* srv_relay = nullptr;        // device: ServerRelay
    double* srv_partials = nullptr;   // device [13][grid]
    unsigned* srv_bad = nullptr;
    unsigned* srv_ticket = nullptr;
};

// mf_api.cu: resident evaluation kernel
mf_status mf_server_begin(mf_model* m);  // used by mf_fit: serve for the duration of the fit (no-op where not applicable)
void mf_server_end(mf_model* m, bool was_on);

// Sets ctx->err and returns st (mf_api.cu).
mf_status mf_fail(mf_ctx* ctx, mf_status st, const std::string& msg);
