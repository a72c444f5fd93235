/*
 * ts_sched.cu -- host-side batch scheduling primitives of libts (8(e);
 * 8(f) NEXT-1).  Plain host code, no device needed:
 *   ts_sched_fill      : InFlightAutobatcher admission -- "samples systems from the stream until
 *                        memory is full" (section 3)
 *   ts_sched_max_scaler: Figure 2 step 4 -- "max memory scaler = min(n systems * memory scaler)"
 *
 *   ts_sched_binpack   : BinningAutobatcher -- "the systems are optimally packed into bins of length
 *                        equal to the maximum memory of the model"; first-fit
 *                        decreasing (reading R26: exact optimum only claimed on tiny inputs)
 *   ts_sched_partition : multi-GPU sharding by system, longest-processing-time first
 */
#include <stdlib.h>

#include <algorithm>
#include <numeric>
#include <vector>

#include "ts.h"

extern "C" ts_status ts_sched_fill(const double *cost, int64_t n, double budget, int64_t *n_taken, double *used)
{
    if (!cost || !n_taken || n < 0 || !(budget >= 0.0)) return TS_ERR_INVALID_ARG;
    double u = 0.0;
    int64_t k = 0;
    for (; k < n; ++k) {
        if (!(cost[k] >= 0.0)) return TS_ERR_INVALID_ARG;
        if (u + cost[k] > budget) break;
        u += cost[k];
    }
    *n_taken = k;
    if (used) *used = u;
    return TS_OK;
}

extern "C" ts_status ts_sched_max_scaler(const int64_t *n_systems, const double *scaler, int32_t n_probes, double *out)
{
    if (!n_systems || !scaler || !out || n_probes < 1) return TS_ERR_INVALID_ARG;
    double m = 0.0;
    for (int32_t k = 0; k < n_probes; ++k) {
        if (n_systems[k] < 1 || !(scaler[k] > 0.0)) return TS_ERR_INVALID_ARG;
        double v = (double)n_systems[k] * scaler[k];
        m = (k == 0 || v < m) ? v : m;
    }
    *out = m;
    return TS_OK;
}

extern "C" ts_status ts_sched_binpack(const double *cost, int64_t n, double capacity, int32_t *bin_of, int32_t *n_bins)
{
    if (!cost || !bin_of || !n_bins || n < 0 || !(capacity > 0.0)) return TS_ERR_INVALID_ARG;
    std::vector<int64_t> order((size_t)n);
    std::iota(order.begin(), order.end(), (int64_t)0);
    for (int64_t k = 0; k < n; ++k)
        if (!(cost[k] >= 0.0) || cost[k] > capacity) return TS_ERR_INVALID_ARG;   /* a system that fits no bin */
    std::stable_sort(order.begin(), order.end(), [&](int64_t a, int64_t b) { return cost[a] > cost[b]; });
    std::vector<double> room;
    for (int64_t k : order) {
        size_t b = 0;
        while (b < room.size() && room[b] < cost[k]) ++b;
        if (b == room.size()) room.push_back(capacity);
        room[b] -= cost[k];
        bin_of[k] = (int32_t)b;
    }
    *n_bins = (int32_t)room.size();
    return TS_OK;
}

extern "C" ts_status ts_sched_partition(const double *cost, int64_t n, int32_t n_ranks, int32_t *rank_of, double *load)
{
    if (!cost || !rank_of || n < 0 || n_ranks < 1) return TS_ERR_INVALID_ARG;
    std::vector<int64_t> order((size_t)n);
    std::iota(order.begin(), order.end(), (int64_t)0);
    for (int64_t k = 0; k < n; ++k)
        if (!(cost[k] >= 0.0)) return TS_ERR_INVALID_ARG;
    std::stable_sort(order.begin(), order.end(), [&](int64_t a, int64_t b) { return cost[a] > cost[b]; });
    std::vector<double> l((size_t)n_ranks, 0.0);
    for (int64_t k : order) {
        int32_t r = (int32_t)(std::min_element(l.begin(), l.end()) - l.begin());   /* first minimum: deterministic */
        l[(size_t)r] += cost[k];
        rank_of[k] = r;
    }
    if (load) std::copy(l.begin(), l.end(), load);
    return TS_OK;
}
