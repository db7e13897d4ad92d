// bc_align_batch_best: the best-stratum mode short-read aligners use in production --
// per read, the hits of the exhaustive set with d <= min(d_min + stratum_plus, z), where d_min is the read's
// smallest difference count over both strands.  Most reads match well (~85 % match uniquely) and
// never pay for the deep budgets.
//
// Round 2: the mode lives INSIDE the persistent search kernel (bc_search.cu, "best-stratum mode"): every read is
// searched with its own budget, 0, 1, 2, ... by the warp that drew it, until its first hits appear (they all
// have d = that budget = d_min), then once more with min(d_min + plus, z).  One launch of the hot path, no host
// round trip between budgets (round 1 ran the whole path z+1 times with a synchronise and a D2H read per
// pass).  The states carry the differences still affordable (budget - d), so the search itself is the same
// code for both modes; the per-query records with the D / Ds thresholds are prepared once for all budgets.
#include "bc_ws.cuh"

int bc_align_impl(const bc_index *ix, const bc_reads *reads, const bc_opts *o, bc_result *res, void *d_workspace,
                  size_t ws_bytes, void *cuda_stream, int best_plus);

extern "C" int bc_align_best_workspace_bytes(const bc_index *ix, uint32_t n_reads, uint32_t max_len, const bc_opts *o,
                                             uint32_t raw_hits_per_read, uint64_t hits_capacity, size_t *bytes) {
    (void)hits_capacity;                         // (round 1 staged per-pass results; nothing is staged any more)
    return bc_align_workspace_bytes(ix, n_reads, max_len, o, raw_hits_per_read, bytes);
}

extern "C" int bc_align_batch_best(const bc_index *ix, const bc_reads *reads, const bc_opts *o, int32_t stratum_plus,
                                   bc_result *res, void *d_workspace, size_t ws_bytes, void *cuda_stream) {
    if (stratum_plus < 0 || stratum_plus > 255) return BC_E_INVAL;
    return bc_align_impl(ix, reads, o, res, d_workspace, ws_bytes, cuda_stream, stratum_plus);
}
