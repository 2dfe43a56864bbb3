// NEXT-4 / SURVEY 8(e): receiver-range sharding of one graph over the ranks of a node (host-side planning, no device work).
// PAPER.md L82 ("scale model deployment to larger systems"); reading N2: rank k owns a contiguous range of atoms
// [b_k, b_{k+1}) chosen so that the ranks hold about equal numbers of EDGES, and all in-edges of its atoms (their weights,
// SH rows and `out` rows never leave the rank).  The senders it does not own are its halo: their feature rows are fetched once
// per forward pass and their grad_feats rows are returned once per backward pass (one exchange each way, nothing else).
#include <algorithm>
#include <vector>

#include "e3_internal.h"

using namespace e3;

// boundaries b[0..world]: b[k] = receivers[floor(k*E/world)] (n_nodes when that index is E), made non-decreasing
extern "C" int e3_shard_ranges(const int32_t *receivers_h, int64_t n_edges, int32_t n_nodes, int world, int32_t *bounds /*[world+1]*/)
{
    if (world < 1 || n_edges < 0 || n_nodes < 0 || !bounds || (n_edges > 0 && !receivers_h)) { set_error("e3_shard_ranges: bad arguments"); return E3_ERR_INVALID_ARG; }
    for (int64_t e = 1; e < n_edges; ++e)
        if (receivers_h[e] < receivers_h[e - 1]) { set_error("e3_shard_ranges: receivers are not sorted ascending (edge %lld)", (long long)e); return E3_ERR_UNSORTED; }
    if (n_edges > 0 && (receivers_h[0] < 0 || receivers_h[n_edges - 1] >= n_nodes)) { set_error("e3_shard_ranges: receiver index out of range"); return E3_ERR_INVALID_ARG; }
    bounds[0] = 0;
    for (int k = 1; k < world; ++k) {
        const int64_t t = (int64_t)(((__int128)k * n_edges) / world);
        const int32_t v = t < n_edges ? receivers_h[t] : n_nodes;
        bounds[k] = std::max(bounds[k - 1], v);
    }
    bounds[world] = n_nodes;
    return E3_OK;
}

// local problem of the rank owning [lo, hi): edge range [e_lo, e_hi), halo (ascending global ids of the senders outside the range),
// local sender ids (owned atoms 0..hi-lo-1 in order, then the halo) and local receiver ids (r - lo) of its edges.
// halo / senders_local / receivers_local need room for e_hi - e_lo entries (query the range first with the three of them NULL).
extern "C" int e3_shard_localize(const int32_t *senders_h, const int32_t *receivers_h, int64_t n_edges, int32_t n_nodes, int32_t lo, int32_t hi,
                                 int64_t *e_lo, int64_t *e_hi, int32_t *halo, int32_t *n_halo, int32_t *senders_local, int32_t *receivers_local)
{
    if (n_edges < 0 || lo < 0 || hi < lo || hi > n_nodes || !e_lo || !e_hi || (n_edges > 0 && (!senders_h || !receivers_h))) {
        set_error("e3_shard_localize: bad arguments");
        return E3_ERR_INVALID_ARG;
    }
    const int32_t *rb = receivers_h, *re = receivers_h + n_edges;
    *e_lo = std::lower_bound(rb, re, lo) - rb;
    *e_hi = std::lower_bound(rb, re, hi) - rb;
    if (!halo || !n_halo || !senders_local || !receivers_local) return E3_OK;
    const int64_t n = *e_hi - *e_lo;
    std::vector<int32_t> h;
    for (int64_t i = 0; i < n; ++i) {
        const int32_t s = senders_h[*e_lo + i];
        if (s < 0 || s >= n_nodes) { set_error("e3_shard_localize: sender index out of range (edge %lld)", (long long)(*e_lo + i)); return E3_ERR_INVALID_ARG; }
        if (s < lo || s >= hi) h.push_back(s);
    }
    std::sort(h.begin(), h.end());
    h.erase(std::unique(h.begin(), h.end()), h.end());
    *n_halo = (int32_t)h.size();
    std::copy(h.begin(), h.end(), halo);
    for (int64_t i = 0; i < n; ++i) {
        const int32_t s = senders_h[*e_lo + i];
        senders_local[i] = (s >= lo && s < hi) ? s - lo : (hi - lo) + (int32_t)(std::lower_bound(h.begin(), h.end(), s) - h.begin());
        receivers_local[i] = receivers_h[*e_lo + i] - lo;
    }
    return E3_OK;
}
