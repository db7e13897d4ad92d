// bc_align_batch_best: the best-stratum mode short-read aligners use in
// production -- per read, the hits of the exhaustive set with d <= d_min + stratum_plus, where d_min
// is the read's smallest difference count over both strands.  Computed by iterative deepening over
// the difference budget with the exhaustive hot path (bc_align_batch) as the inner step: pass z' =
// 0, 1, .. z aligns the still-active reads with budget z'; a read is final at the first pass
// z' >= min(d_min + stratum_plus, z) (d_min = the first pass that gave it a hit), or at z' = z if it
// never hits.  At that pass its hits are exactly {d <= min(d_min + stratum_plus, z)}, so nothing
// has to be filtered.  Reads that match well -- most reads (~85 % match uniquely) --
// never pay for the deep budgets.  Everything runs on the device; the host reads two counters per pass.
#include "bc_ws.cuh"

namespace {

inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

constexpr uint64_t SCAN_TILE = 256 * 8;

struct BestLayout {
    size_t off_inner, inner_bytes, off_sub_off, off_sub_len, off_act0, off_act1, off_fh, off_flag, off_fcnt, off_keep,
        off_fscan, off_kscan, off_blk, off_tmp_off, off_tmp_hits, off_needed, off_cnt, off_start, off_totals, off_arena, total;
    uint64_t tmp_cap, arena_cap;
};

int make_best_layout(const bc_index *ix, uint32_t n, uint32_t max_len, const bc_opts *o, uint32_t raw_hits_per_read,
                     uint64_t hits_capacity, BestLayout &L) {
    size_t inner = 0;
    int rc = bc_align_workspace_bytes(ix, n, max_len, o, raw_hits_per_read, &inner);
    if (rc) return rc;
    L.tmp_cap = hits_capacity;                        // one pass can return at most what the caller can take
    L.arena_cap = hits_capacity;
    size_t x = 0;
    L.off_inner = x;    L.inner_bytes = align_up(inner, 256); x += L.inner_bytes;
    L.off_sub_off = x;  x = align_up(x + (size_t)n * 8, 256);
    L.off_sub_len = x;  x = align_up(x + (size_t)n * 2, 256);
    L.off_act0 = x;     x = align_up(x + (size_t)n * 4, 256);
    L.off_act1 = x;     x = align_up(x + (size_t)n * 4, 256);
    L.off_fh = x;       x = align_up(x + (size_t)n, 256);
    L.off_flag = x;     x = align_up(x + (size_t)n * 4, 256);
    L.off_fcnt = x;     x = align_up(x + (size_t)n * 4, 256);
    L.off_keep = x;     x = align_up(x + (size_t)n * 4, 256);
    L.off_fscan = x;    x = align_up(x + ((size_t)n + 1) * 8, 256);
    L.off_kscan = x;    x = align_up(x + ((size_t)n + 1) * 8, 256);
    L.off_blk = x;      x = align_up(x + ((size_t)n / SCAN_TILE + 2) * 8, 256);
    L.off_tmp_off = x;  x = align_up(x + ((size_t)n + 1) * 8, 256);
    L.off_tmp_hits = x; x = align_up(x + (size_t)L.tmp_cap * sizeof(bc_hit), 256);
    L.off_needed = x;   x = align_up(x + 16, 256);
    L.off_cnt = x;      x = align_up(x + (size_t)n * 4, 256);
    L.off_start = x;    x = align_up(x + (size_t)n * 8, 256);
    L.off_totals = x;   x = align_up(x + 16, 256);
    L.off_arena = x;    x = align_up(x + (size_t)L.arena_cap * sizeof(bc_hit), 256);
    L.total = x;
    return BC_OK;
}

__global__ void best_init(uint32_t *act, uint8_t *fh, uint32_t *cnt, uint32_t n) {
    uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) { act[i] = i; fh[i] = 255; cnt[i] = 0; }
}

__global__ void best_gather(const uint64_t *off, const uint16_t *len, const uint32_t *act, uint32_t n_act,
                            uint64_t *sub_off, uint16_t *sub_len) {
    uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n_act) { uint32_t r = act[i]; sub_off[i] = off[r]; sub_len[i] = len[r]; }
}

// per active read: final at this pass?  fcnt = hits it contributes if final, keep = 1 if it stays active
__global__ void best_classify(const uint64_t *tmp_off, const uint32_t *act, uint32_t n_act, uint8_t *fh, int zp, int z,
                              int plus, uint32_t *flag, uint32_t *fcnt, uint32_t *keep) {
    uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_act) return;
    const uint32_t r = act[i];
    const uint32_t c = (uint32_t)(tmp_off[i + 1] - tmp_off[i]);
    bool fin;
    if (c > 0) {
        if (fh[r] == 255) fh[r] = (uint8_t)zp;            // first pass with a hit: d_min = zp
        int lim = (int)fh[r] + plus;
        if (lim > z) lim = z;
        fin = zp >= lim;
    } else fin = zp >= z;
    flag[i] = fin ? 1u : 0u;
    fcnt[i] = fin ? c : 0u;
    keep[i] = fin ? 0u : 1u;
}

__global__ void best_commit(const uint64_t *tmp_off, const bc_hit *tmp_hits, const uint32_t *act, uint32_t n_act,
                            const uint32_t *flag, const uint64_t *fscan, const uint64_t *kscan, uint64_t arena_base,
                            bc_hit *arena, uint64_t arena_cap, uint32_t *cnt, uint64_t *start, uint32_t *act_next) {
    uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_act) return;
    const uint32_t r = act[i];
    if (!flag[i]) { act_next[kscan[i]] = r; return; }
    const uint64_t b = tmp_off[i], c = tmp_off[i + 1] - b, dst = arena_base + fscan[i];
    cnt[r] = (uint32_t)c;
    start[r] = dst;
    for (uint64_t j = 0; j < c; ++j)
        if (dst + j < arena_cap) arena[dst + j] = tmp_hits[b + j];
}

__global__ void best_write(const uint32_t *cnt, const uint64_t *start, const uint64_t *offs, const bc_hit *arena,
                           bc_hit *hits, uint64_t hits_capacity, uint32_t n) {
    uint32_t r = blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= n) return;
    const uint64_t o = offs[r], s = start[r];
    const uint32_t c = cnt[r];
    for (uint32_t j = 0; j < c; ++j)
        if (o + j < hits_capacity) hits[o + j] = arena[s + j];
}

inline unsigned grid_for(uint64_t n) { return (unsigned)((n + 255) / 256); }

}  // namespace

extern "C" int bc_align_best_workspace_bytes(const bc_index *ix, uint32_t n_reads, uint32_t max_len, const bc_opts *o,
                                             uint32_t raw_hits_per_read, uint64_t hits_capacity, size_t *bytes) {
    if (!ix || !o || !bytes) return BC_E_INVAL;
    BestLayout L;
    int rc = make_best_layout(ix, n_reads, max_len, o, raw_hits_per_read, hits_capacity, L);
    if (rc) return rc;
    *bytes = L.total;
    return BC_OK;
}

extern "C" int bc_align_batch_best(const bc_index *ix_c, const bc_reads *reads, const bc_opts *o, int32_t stratum_plus,
                                   bc_result *res, void *d_workspace, size_t ws_bytes, void *cuda_stream) {
    bc_index *ix = const_cast<bc_index *>(ix_c);
    if (!ix || !reads || !o || !res || !d_workspace || ((uintptr_t)d_workspace & 255) || stratum_plus < 0 ||
        stratum_plus > 255 || o->z < 0 || o->z > 255)
        return BC_E_INVAL;
    if (!res->hit_offsets || !res->n_hits_needed || (res->hits_capacity && !res->hits)) return BC_E_INVAL;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const uint32_t n = reads->n_reads;
    if (n == 0) return bc_align_batch(ix, reads, o, res, d_workspace, ws_bytes, cuda_stream);
    if (!reads->off || !reads->len) return BC_E_INVAL;
    // lay out for the smallest inner arena; whatever the caller gave beyond that goes to the inner call
    BestLayout L;
    int rc = make_best_layout(ix, n, reads->max_len, o, 1, res->hits_capacity, L);
    if (rc) return rc;
    if (ws_bytes < L.total) return BC_E_NOMEM;
    {
        const size_t grow = (ws_bytes - L.total) & ~(size_t)255;
        L.inner_bytes += grow;
        size_t *offs[] = {&L.off_sub_off, &L.off_sub_len, &L.off_act0, &L.off_act1, &L.off_fh, &L.off_flag, &L.off_fcnt,
                          &L.off_keep, &L.off_fscan, &L.off_kscan, &L.off_blk, &L.off_tmp_off, &L.off_tmp_hits,
                          &L.off_needed, &L.off_cnt, &L.off_start, &L.off_totals, &L.off_arena};
        for (size_t *q : offs) *q += grow;
        L.total += grow;
    }

    char *base = (char *)d_workspace;
    uint64_t *sub_off = (uint64_t *)(base + L.off_sub_off);
    uint16_t *sub_len = (uint16_t *)(base + L.off_sub_len);
    uint32_t *act = (uint32_t *)(base + L.off_act0), *act_next = (uint32_t *)(base + L.off_act1);
    uint8_t *fh = (uint8_t *)(base + L.off_fh);
    uint32_t *flag = (uint32_t *)(base + L.off_flag), *fcnt = (uint32_t *)(base + L.off_fcnt);
    uint32_t *keep = (uint32_t *)(base + L.off_keep), *cnt = (uint32_t *)(base + L.off_cnt);
    uint64_t *fscan = (uint64_t *)(base + L.off_fscan), *kscan = (uint64_t *)(base + L.off_kscan);
    uint64_t *blk = (uint64_t *)(base + L.off_blk), *start = (uint64_t *)(base + L.off_start);
    uint64_t *totals = (uint64_t *)(base + L.off_totals);
    bc_hit *arena = (bc_hit *)(base + L.off_arena);
    bc_result tmp;
    tmp.hit_offsets = (uint64_t *)(base + L.off_tmp_off);
    tmp.hits = (bc_hit *)(base + L.off_tmp_hits);
    tmp.hits_capacity = L.tmp_cap;
    tmp.n_hits_needed = (uint64_t *)(base + L.off_needed);

    best_init<<<grid_for(n), 256, 0, st>>>(act, fh, cnt, n);
    if (cudaMemsetAsync(start, 0, (size_t)n * 8, st) != cudaSuccess) return BC_E_CUDA;
    uint64_t sum[16] = {0};
    uint32_t n_act = n;
    uint64_t arena_used = 0;
    int passes = 0;
    for (int zp = 0; zp <= o->z && n_act > 0; ++zp, ++passes) {
        best_gather<<<grid_for(n_act), 256, 0, st>>>(reads->off, reads->len, act, n_act, sub_off, sub_len);
        bc_reads sub = *reads;
        sub.off = sub_off; sub.len = sub_len; sub.n_reads = n_act;
        bc_opts oz = *o;
        oz.z = zp;
        rc = bc_align_batch(ix, &sub, &oz, &tmp, base + L.off_inner, L.inner_bytes, cuda_stream);
        for (int i = 0; i < 16; ++i) if (i != 5 && i != 7) sum[i] += ix->stats[i];
        if (ix->stats[5] > sum[5]) sum[5] = ix->stats[5];
        sum[7] = ix->stats[7];
        if (rc == BC_E_OVERFLOW) {                                 // report the failing pass's needs
            if (cudaMemcpyAsync(res->n_hits_needed, tmp.n_hits_needed, 16, cudaMemcpyDeviceToDevice, st) != cudaSuccess ||
                cudaStreamSynchronize(st) != cudaSuccess)
                return BC_E_CUDA;
            return BC_E_OVERFLOW;
        }
        if (rc) return rc;
        best_classify<<<grid_for(n_act), 256, 0, st>>>(tmp.hit_offsets, act, n_act, fh, zp, o->z, stratum_plus, flag, fcnt, keep);
        cudaError_t e = bc_exclusive_scan(fcnt, n_act, blk, fscan, totals, st);
        if (e == cudaSuccess) e = bc_exclusive_scan(keep, n_act, blk, kscan, totals + 1, st);
        if (e != cudaSuccess) return BC_E_CUDA;
        best_commit<<<grid_for(n_act), 256, 0, st>>>(tmp.hit_offsets, tmp.hits, act, n_act, flag, fscan, kscan, arena_used,
                                                      arena, L.arena_cap, cnt, start, act_next);
        uint64_t t2[2];
        if (cudaMemcpyAsync(t2, totals, 16, cudaMemcpyDeviceToHost, st) != cudaSuccess ||
            cudaStreamSynchronize(st) != cudaSuccess)
            return BC_E_CUDA;
        arena_used += t2[0];
        n_act = (uint32_t)t2[1];
        uint32_t *sw = act; act = act_next; act_next = sw;
    }
    // CSR in read order
    cudaError_t e = bc_exclusive_scan(cnt, n, blk, res->hit_offsets, totals, st);
    if (e != cudaSuccess) return BC_E_CUDA;
    best_write<<<grid_for(n), 256, 0, st>>>(cnt, start, res->hit_offsets, arena, res->hits, res->hits_capacity, n);
    uint64_t needed[2] = {arena_used, sum[3]};
    if (cudaGetLastError() != cudaSuccess ||
        cudaMemcpyAsync(res->n_hits_needed, needed, 16, cudaMemcpyHostToDevice, st) != cudaSuccess ||
        cudaStreamSynchronize(st) != cudaSuccess)
        return BC_E_CUDA;
    for (int i = 0; i < 16; ++i) ix->stats[i] = sum[i];
    ix->stats[15] = (uint64_t)passes;
    if (arena_used > res->hits_capacity) return BC_E_OVERFLOW;
    return BC_OK;
}
