// Controller logic of LUMEN (include/lumen_kv.h): checkpoint placement Eq. (1)
// (PAPER.md:137-143), recovery dispatch and greedy load rebalancing.
// Scalar host code, request granularity ("the controller operates at request granularity
// rather than token granularity"); no CUDA.
#include <cstdint>
#include <vector>

#include "lumen_kv.h"

extern "C" {

int lumen_kv_choose_holder(const double* q, const int64_t* held, const int32_t* held_begin,
                           const int64_t* available, int32_t W, int32_t serving,
                           int64_t footprint, double lambda, double bandwidth, int32_t* holder) {
    if (!holder) return LUMEN_KV_EINVAL;
    *holder = -1;
    if (W < 1 || !q || !held_begin || !available || footprint < 0 || !(bandwidth > 0.0) ||
        (held_begin[W] > 0 && !held))
        return LUMEN_KV_EINVAL;
    double best = 0.0;
    for (int32_t w = 0; w < W; ++w) {
        if (w == serving || available[w] < footprint) continue;          // F(r)
        int64_t sum = footprint;
        const int64_t count = held_begin[w + 1] - held_begin[w] + 1;
        if (count < 1) return LUMEN_KV_EINVAL;
        for (int32_t i = held_begin[w]; i < held_begin[w + 1]; ++i) sum += held[i];
        const double p = static_cast<double>(sum) / static_cast<double>(count) / bandwidth;
        const double score = q[w] + lambda * p;
        if (*holder < 0 || score < best) {                                // ties: lowest id
            *holder = w;
            best = score;
        }
    }
    return LUMEN_KV_OK;
}

int lumen_kv_recover(const int64_t* load, const uint8_t* alive, int32_t W, const int32_t* holder,
                     const int64_t* ckpt_size, int32_t n, int32_t* assign, uint8_t* reuse,
                     int64_t* final_load) {
    if (W < 1 || n < 0 || !load || !alive || !final_load ||
        (n > 0 && (!holder || !ckpt_size || !assign || !reuse)))
        return LUMEN_KV_EINVAL;
    std::vector<int32_t> surv;
    for (int32_t w = 0; w < W; ++w) {
        final_load[w] = alive[w] ? load[w] : 0;
        if (alive[w]) {
            if (load[w] < 0) return LUMEN_KV_EINVAL;
            surv.push_back(w);
        }
    }
    if (surv.empty()) return LUMEN_KV_EINVAL;
    int64_t* cur = final_load;
    auto least_loaded = [&](int32_t exclude) {
        int32_t best = -1;
        for (int32_t w : surv)
            if (w != exclude && (best < 0 || cur[w] < cur[best])) best = w;
        return best;
    };
    // dispatch: locality first
    for (int32_t i = 0; i < n; ++i) {
        if (ckpt_size[i] < 0) return LUMEN_KV_EINVAL;
        if (holder[i] >= 0 && holder[i] < W && alive[holder[i]]) {
            assign[i] = holder[i];
            reuse[i] = 1;
        } else {
            assign[i] = least_loaded(-1);
            reuse[i] = 0;
        }
        ++cur[assign[i]];
    }
    if (surv.size() < 2) return LUMEN_KV_OK;
    int64_t total = 0;
    for (int32_t w : surv) total += cur[w];
    const int64_t S = static_cast<int64_t>(surv.size());
    const int64_t limit = (total + S - 1) / S;                            // ceil(average)
    std::vector<int64_t> movable(static_cast<size_t>(W), 0);              // reusable requests per worker
    for (int32_t i = 0; i < n; ++i)
        if (reuse[i]) ++movable[assign[i]];
    for (;;) {
        int32_t src = -1;                                                 // most congested first
        for (int32_t w : surv)
            if (cur[w] > limit && movable[w] > 0 && (src < 0 || cur[w] > cur[src])) src = w;
        if (src < 0) break;
        int32_t pick = -1;                                                // smallest checkpoint
        for (int32_t i = 0; i < n; ++i)
            if (reuse[i] && assign[i] == src && (pick < 0 || ckpt_size[i] < ckpt_size[pick]))
                pick = i;
        const int32_t dst = least_loaded(src);
        assign[pick] = dst;
        reuse[pick] = 0;                                                  // forfeits its checkpoint
        --movable[src];
        --cur[src];
        ++cur[dst];
    }
    return LUMEN_KV_OK;
}

}  // extern "C"
