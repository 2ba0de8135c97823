// mf_dist.cpp — S5 across GPUs (Eq. 1: the events of one likelihood are independent, so
// shards of them may be summed on different GPUs).  Each rank evaluates its event shard with mf_nll_grad; the K+1 partial
// sums of all ranks are gathered (torch.distributed, plumbing) and combined HERE, identically on every rank: a two-sum
// compensated accumulation in RANK ORDER, so that all ranks hold bit-identical totals and the result does not depend on a
// collective's reduction tree.  Host arithmetic only: <= 17 doubles per rank.
#include <cmath>

#include "mf_internal.h"

extern "C" mf_status mf_combine_partials(int n_ranks, int width, const double* rows, double* out)
{
    if (n_ranks < 1 || width < 1 || !rows || !out) return MF_ERR_ARG;
    for (int k = 0; k < width; ++k) {
        double s = 0.0, lo = 0.0, plain = 0.0;
        bool finite = true;
        for (int r = 0; r < n_ranks; ++r) {
            const double b = rows[(size_t)r * width + k];
            finite = finite && std::isfinite(b);
            plain += b;
            const double t = s + b;  // two-sum: t + e == s + b exactly
            const double bb = t - s;
            const double e = (s - (t - bb)) + (b - bb);
            lo += e;
            s = t;
        }
        out[k] = finite ? s + lo : plain;  // +inf (P <= 0 on a shard) and NaN propagate as a plain sum would
    }
    return MF_OK;
}
