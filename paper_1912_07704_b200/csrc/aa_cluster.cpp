/*
 * aa_cluster.cpp — candidate clustering (reading C10): friends-of-friends over the candidate list.
 * Host-side post-processing of a small list (PAPER.md:47 step 8: results are copied to the host and owned by the API);
 * nothing here touches the GPU.
 *
 * Linked: |dm_a - dm_b| <= dm_tol  and  sample_a <= sample_b + width_b + gap  and  sample_b <= sample_a + width_a + gap.
 * Clusters = connected components; representative = highest SNR, first in canonical order (range, dm_index, sample) on ties.
 */
#include <algorithm>
#include <cmath>
#include <numeric>
#include <vector>

#include "aa_internal.h"

namespace {

struct Dsu {
    std::vector<uint32_t> p;
    explicit Dsu(size_t n) : p(n) { std::iota(p.begin(), p.end(), 0u); }
    uint32_t find(uint32_t x) { while (p[x] != x) { p[x] = p[p[x]]; x = p[x]; } return x; }
    void unite(uint32_t a, uint32_t b) { a = find(a); b = find(b); if (a != b) p[std::max(a, b)] = std::min(a, b); }
};

bool canon_less(const aa_candidate& a, const aa_candidate& b) {
    if (a.range != b.range) return a.range < b.range;
    if (a.dm_index != b.dm_index) return a.dm_index < b.dm_index;
    return a.sample < b.sample;
}

/* clusters of in[0..n) into out (capacity n); returns their number */
size_t cluster(const aa_candidate* in, size_t n, double dm_tol, uint64_t gap, aa_cluster* out) {
    if (n == 0) return 0;
    std::vector<uint32_t> order(n);
    std::iota(order.begin(), order.end(), 0u);
    std::sort(order.begin(), order.end(), [&](uint32_t a, uint32_t b) {
        if (in[a].sample != in[b].sample) return in[a].sample < in[b].sample;
        return a < b;
    });
    Dsu dsu(n);
    /* sweep by boxcar start: b can only be linked to an earlier-starting a if start_b <= end_a + gap; keep the running
     * maximum of end + gap so the inner scan stops as soon as no earlier candidate can reach */
    for (size_t i = 0; i < n; ++i) {
        const aa_candidate& a = in[order[i]];
        const uint64_t reach = a.sample + (uint64_t)a.width + gap;
        for (size_t j = i + 1; j < n; ++j) {
            const aa_candidate& b = in[order[j]];
            if (b.sample > reach) break;                                   /* sorted by start: nobody later can be reached by a */
            if (std::fabs((double)a.dm - (double)b.dm) <= dm_tol) dsu.unite(order[i], order[j]);   /* a.sample <= b.sample holds */
        }
    }
    std::vector<int64_t> slot(n, -1);
    size_t nc = 0;
    for (size_t q = 0; q < n; ++q) {
        const uint32_t r = dsu.find((uint32_t)q);
        const aa_candidate& c = in[q];
        if (slot[r] < 0) {
            slot[r] = (int64_t)nc;
            aa_cluster& k = out[nc++];
            k.best = c; k.members = 1; k.dm_min = k.dm_max = c.dm; k.sample_min = c.sample; k.sample_end = c.sample + c.width;
        } else {
            aa_cluster& k = out[(size_t)slot[r]];
            ++k.members;
            if (c.snr > k.best.snr || (c.snr == k.best.snr && canon_less(c, k.best))) k.best = c;
            k.dm_min = std::min(k.dm_min, c.dm); k.dm_max = std::max(k.dm_max, c.dm);
            k.sample_min = std::min(k.sample_min, c.sample); k.sample_end = std::max(k.sample_end, c.sample + (uint64_t)c.width);
        }
    }
    std::sort(out, out + nc, [](const aa_cluster& a, const aa_cluster& b) { return canon_less(a.best, b.best); });
    return nc;
}

}  // namespace

extern "C" aa_status aa_cluster_candidates(const aa_candidate* in, size_t n, double dm_tol, uint64_t gap, aa_cluster* out, size_t* nout) {
    using aa::set_error;
    if (!nout || (n && (!in || !out))) { set_error("aa_cluster_candidates: NULL argument"); return AA_ERR_INVALID_ARG; }
    if (!(dm_tol >= 0.0) || !std::isfinite(dm_tol)) { set_error("aa_cluster_candidates: dm_tol = %g must be finite and >= 0", dm_tol); return AA_ERR_INVALID_ARG; }
    *nout = cluster(in, n, dm_tol, gap, out);
    return AA_OK;
}

extern "C" aa_status aa_get_clusters(aa_strategy* h, double dm_tol, uint64_t gap, const aa_cluster** out, size_t* n) {
    using aa::set_error;
    if (!out || !n) { set_error("aa_get_clusters: NULL output argument"); return AA_ERR_INVALID_ARG; }
    if (!(dm_tol >= 0.0) || !std::isfinite(dm_tol)) { set_error("aa_get_clusters: dm_tol = %g must be finite and >= 0", dm_tol); return AA_ERR_INVALID_ARG; }
    const aa_candidate* c = nullptr; size_t nc = 0;
    const aa_status st = aa_get_candidates(h, &c, &nc);
    if (st != AA_OK && st != AA_ERR_CANDIDATE_OVERFLOW) return st;
    aa::Strategy& s = h->s;
    s.clusters.resize(nc);
    s.clusters.resize(cluster(c, nc, dm_tol, gap, s.clusters.data()));
    *out = s.clusters.data();
    *n = s.clusters.size();
    return st;
}
