// bm_salc.cu -- SLO-aware latency controller (PAPER.md 4.5): host logic only, see include/bm.h.
// multiplicative decrease of the threshold when the recent P90 latency exceeds the SLO, linear increase
// when it falls below a warning line.  Constants are the caller's (reading A21).
#include <algorithm>
#include <cmath>
#include <vector>

#include "../../include/bm.h"

extern "C" {

int bm_salc_init(bm_salc *c, double slo, double warn_frac, double decrease, double increase, int window) {
    if (!c) return BM_ERR_NULL;
    if (!(slo > 0.0) || !(warn_frac > 0.0 && warn_frac <= 1.0) || !(decrease > 0.0 && decrease < 1.0) ||
        !(increase > 0.0) || window < 1 || window > BM_SALC_MAX_WINDOW)
        return BM_ERR_SHAPE;
    c->slo = slo; c->warn_frac = warn_frac; c->decrease = decrease; c->increase = increase;
    c->threshold = 1.0;
    c->window = window; c->count = 0; c->head = 0;
    for (int i = 0; i < BM_SALC_MAX_WINDOW; ++i) c->lat[i] = 0.0;
    return BM_OK;
}

double bm_salc_p90(const bm_salc *c) {
    if (!c || c->count <= 0) return 0.0;
    std::vector<double> v(c->lat, c->lat + c->count);
    const int rank = (int)std::ceil(0.9 * c->count);              // nearest-rank percentile, 1-based
    std::nth_element(v.begin(), v.begin() + (rank - 1), v.end());
    return v[rank - 1];
}

double bm_salc_observe(bm_salc *c, double latency) {
    if (!c) return (double)BM_ERR_NULL;
    if (!(latency == latency)) return (double)BM_ERR_SHAPE;
    c->lat[c->head] = latency;                                    // while count < window the ring is a prefix
    c->head = (c->head + 1) % c->window;
    if (c->count < c->window) ++c->count;
    const double p90 = bm_salc_p90(c);
    if (p90 > c->slo) c->threshold *= c->decrease;
    else if (p90 < c->warn_frac * c->slo) c->threshold = std::min(1.0, c->threshold + c->increase);
    return c->threshold;
}

int bm_salc_cold_mask(const int32_t *w, int E, double threshold, int32_t *cold_mask) {
    if (!w || !cold_mask) return BM_ERR_NULL;
    if (E < 1 || E > BM_MAX_E || !(threshold >= 0.0 && threshold <= 1.0)) return BM_ERR_SHAPE;
    const int n_cold = (int)std::lround((1.0 - threshold) * E);
    std::vector<int> order(E);
    for (int e = 0; e < E; ++e) order[e] = e;
    std::stable_sort(order.begin(), order.end(), [&](int a, int b) { return w[a] < w[b]; });   // ties: lower index colder
    for (int e = 0; e < E; ++e) cold_mask[e] = 0;
    for (int i = 0; i < n_cold && i < E; ++i) cold_mask[order[i]] = 1;
    return BM_OK;
}

}  // extern "C"
