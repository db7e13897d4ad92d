// bc_align_batch / bc_align_workspace_bytes: host orchestration of the hot path.
// Carves the caller's workspace, launches prepare -> search -> post on the caller's stream, reads
// the counter block back and turns it into a status code.  No device allocation, no CPU fallback.
#include "bc_ws.cuh"

namespace {

inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

constexpr uint64_t SCAN_TILE = 256 * 8;            // must match bc_post.cu
constexpr size_t RAW_BYTES = sizeof(BcRawHit) + sizeof(uint64_t) + sizeof(uint32_t);   // arena + seg_key + seg_d

struct WsLayout {
    size_t off_qrec, off_qz, off_spill, off_qcnt, off_qfill, off_seg_off, off_uoff, off_blk, off_big, off_sqf, off_ctr, off_sqb, fixed;
    uint32_t qstride, q_soff, q_boff, q_noff, nq, spill_blocks;
};

// the query record of bc_ws.cuh: thresholds | bases | N bits, 16-byte multiple
void qrec_layout(const bc_opts *o, uint32_t max_len, bool with_n, WsLayout &L) {
    const bool small = o->z <= BC_QREC_SMALL_Z && o->seed_z <= BC_QREC_SMALL_SZ;
    L.q_soff = small ? 8u : (uint32_t)o->z + 1u;
    L.q_boff = small ? 16u : (uint32_t)align_up((size_t)o->z + o->seed_z + 2, 16);
    const uint32_t nb = (max_len / 16u + 1u) * 4u, nn = (max_len / 32u + 1u) * 4u;
    L.q_noff = with_n ? L.q_boff + nb : 0u;
    L.qstride = (uint32_t)align_up((size_t)L.q_boff + nb + (with_n ? nn : 0u), 16);
}

// the workspace is sized for a batch WITH an N mask (bc_align_workspace_bytes does not see the reads);
// a batch without one uses the shorter records
int make_ws_layout(uint32_t n_reads, uint32_t max_len, const bc_opts *o, bool with_n, uint32_t grid_warps,
                   uint32_t spill_blocks, WsLayout &L) {
    if (max_len < 1 || max_len > BC_MAX_READ_LEN || n_reads > 0x7FFFFFF0u) return BC_E_INVAL;
    L.nq = 2 * n_reads;
    L.spill_blocks = spill_blocks;
    qrec_layout(o, max_len, true, L);
    const size_t qrec_bytes = (size_t)L.nq * L.qstride;
    if (qrec_bytes >= ((size_t)1 << 34)) return BC_E_INVAL;      // the kernel indexes record words with 32 bits
    qrec_layout(o, max_len, with_n, L);
    size_t x = 0;
    L.off_qrec = x;    x = align_up(x + qrec_bytes, 256);
    L.off_qz = x;      x = align_up(x + (size_t)n_reads, 256);
    L.off_spill = x;   x = align_up(x + (size_t)grid_warps * spill_blocks * 32 * BC_POOL_ENTRY_BYTES, 256);
    L.off_qcnt = x;    x = align_up(x + (size_t)L.nq * 4, 256);
    L.off_qfill = x;   x = align_up(x + (size_t)L.nq * 4, 256);
    L.off_seg_off = x; x = align_up(x + ((size_t)L.nq + 1) * 8, 256);
    L.off_uoff = x;    x = align_up(x + ((size_t)L.nq + 1) * 8, 256);
    L.off_blk = x;     x = align_up(x + ((size_t)L.nq / SCAN_TILE + 2) * 8, 256);
    L.off_big = x;     x = align_up(x + (size_t)L.nq * 4, 256);
    L.off_sqf = x;     x = align_up(x + BC_STEAL_SLOTS * 4, 256);
    L.off_ctr = x;     x = align_up(x + BC_CTR_COUNT * 8, 256);
    L.off_sqb = x;     x = align_up(x + (size_t)BC_STEAL_SLOTS * 32 * BC_POOL_ENTRY_BYTES, 256);
    L.fixed = x;
    return BC_OK;
}

struct Geometry { uint32_t ctas, warps, bcap, ccap, spill_blocks; };

// geometry of the persistent kernel: CTAs per SM, warps per CTA, per-warp branch ring (power of two)
// and run-stack sizes that fill the shared memory given to the pools
int choose_geometry(const bc_index *ix, Geometry &g) {
    g.warps = ix->warps_per_cta ? ix->warps_per_cta : 7;      // 4 CTAs x 7 warps: see the launch bounds in bc_search.cu
    g.ctas = ix->ctas_per_sm ? ix->ctas_per_sm : 4;
    g.spill_blocks = ix->spill_blocks ? ix->spill_blocks : BC_SPILL_BLOCKS;
    for (;; --g.ctas) {
        // pool bytes per SM; what is left of the shared memory / L1 array stays L1 (query records).  The autotuner's
        // tables with 4 x 7 warps (profiles/r02_autotune_config2.json, _config4.json): 16 MB index 192 / 208 KB ->
        // 85.1 / 83.4 ms; 1.5 GB index 160 / 176 / 208 KB -> 254.3 / 248.8 / 256.3 ms (L2 misses make L1 count there)
        const size_t total_kb = ix->pool_kb ? ix->pool_kb : (ix->bytes > ((size_t)64 << 20) ? 176 : 208);
        size_t budget = total_kb * 1024 / g.ctas;
        if (budget > 200 * 1024) budget = 200 * 1024;
        uint32_t per_warp = (uint32_t)(budget / ((size_t)g.warps * BC_POOL_ENTRY_BYTES));
        if (per_warp > 4096) per_warp = 4096;
        // the ring only has to hold the hot top of the branch stack (its bottom spills to global memory in
        // blocks of 32, kept >= 64 slots free): 128 entries; the rest goes to the two run stacks, which take
        // most of the children of a 32-wide branch step
        if (per_warp >= 128 + 96) { g.bcap = 128; g.ccap = per_warp - 128; return BC_OK; }
        if (g.ctas == 1) return BC_E_UNSUPPORTED;     // too many warps per CTA for the on-chip pools
    }
}

int check_opts(const bc_opts *o) {
    if (!o) return BC_E_INVAL;
    if (o->z < 0 || o->z > 255 || o->max_gap_open < 0 || o->max_gap_open > 255 || o->max_gap_ext < 0 ||
        o->max_gap_ext > 255 || o->seed_len < 0 || o->seed_len > BC_MAX_READ_LEN || o->seed_z < 0 || o->seed_z > 255 ||
        o->indel_end_skip < 0 || o->indel_end_skip > BC_MAX_READ_LEN)
        return BC_E_INVAL;
    return BC_OK;
}

}  // namespace

extern "C" int bc_align_workspace_bytes(const bc_index *ix, uint32_t n_reads, uint32_t max_len, const bc_opts *o,
                                        uint32_t raw_hits_per_read, size_t *bytes) {
    if (!ix || !bytes) return BC_E_INVAL;
    int rc = check_opts(o);
    if (rc) return rc;
    Geometry g;
    rc = choose_geometry(ix, g);
    if (rc) return rc;
    WsLayout L;
    rc = make_ws_layout(n_reads, max_len, o, true, (uint32_t)ix->sm_count * g.ctas * g.warps, g.spill_blocks, L);
    if (rc) return rc;
    if (raw_hits_per_read == 0) raw_hits_per_read = 16;
    uint64_t cap = (uint64_t)raw_hits_per_read * n_reads + 1024;
    *bytes = L.fixed + 3 * 256 + cap * RAW_BYTES;
    return BC_OK;
}

// the hot path; best_plus < 0: exhaustive (bc_align_batch), else the best-stratum mode with that `plus`
int bc_align_impl(const bc_index *ix_c, const bc_reads *reads, const bc_opts *o, bc_result *res,
                  void *d_workspace, size_t ws_bytes, void *cuda_stream, int best_plus) {
    bc_index *ix = const_cast<bc_index *>(ix_c);    // statistics live in the handle
    if (!ix || !reads || !res || !d_workspace || ((uintptr_t)d_workspace & 255)) return BC_E_INVAL;
    int rc = check_opts(o);
    if (rc) return rc;
    if (!res->hit_offsets || !res->n_hits_needed || (res->hits_capacity && !res->hits)) return BC_E_INVAL;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    for (int i = 0; i < 16; ++i) ix->stats[i] = 0;
    if (reads->n_reads == 0) {
        uint64_t zero[3] = {0, 0, 0};
        if (cudaMemcpyAsync(res->hit_offsets, zero, 8, cudaMemcpyHostToDevice, st) != cudaSuccess ||
            cudaMemcpyAsync(res->n_hits_needed, zero + 1, 16, cudaMemcpyHostToDevice, st) != cudaSuccess ||
            cudaStreamSynchronize(st) != cudaSuccess)
            return BC_E_CUDA;
        return BC_OK;
    }
    if (!reads->bases2 || !reads->off || !reads->len) return BC_E_INVAL;
    Geometry g;
    rc = choose_geometry(ix, g);
    if (rc) return rc;
    WsLayout L;
    rc = make_ws_layout(reads->n_reads, reads->max_len, o, reads->nmask != nullptr, (uint32_t)ix->sm_count * g.ctas * g.warps,
                        g.spill_blocks, L);
    if (rc) return rc;
    if (ws_bytes < L.fixed + 3 * 256 + RAW_BYTES) return BC_E_NOMEM;

    char *base = (char *)d_workspace;
    BcSearchParams p;
    p.ix = ix->dev;
    p.reads = *reads;
    p.o = *o;
    BcWorkspace &ws = p.ws;
    ws.nq = L.nq;
    ws.qz = (uint8_t *)(base + L.off_qz);
    ws.qrec = (uint8_t *)(base + L.off_qrec);
    ws.qstride = L.qstride; ws.q_soff = L.q_soff; ws.q_boff = L.q_boff; ws.q_noff = L.q_noff;
    ws.qcnt = (uint32_t *)(base + L.off_qcnt);
    ws.qfill = (uint32_t *)(base + L.off_qfill);
    ws.seg_off = (uint64_t *)(base + L.off_seg_off);
    ws.uoff = (uint64_t *)(base + L.off_uoff);
    ws.blk = (uint64_t *)(base + L.off_blk);
    ws.big = (uint32_t *)(base + L.off_big);
    ws.ctr = (uint64_t *)(base + L.off_ctr);
    uint64_t cap = (ws_bytes - L.fixed - 3 * 256) / RAW_BYTES;
    ws.arena_cap = cap;
    size_t o_arena = L.fixed;
    size_t o_key = align_up(o_arena + cap * sizeof(BcRawHit), 256);
    size_t o_d = align_up(o_key + cap * sizeof(uint64_t), 256);
    ws.arena = (BcRawHit *)(base + o_arena);
    ws.seg_key = (uint64_t *)(base + o_key);
    ws.seg_d = (uint32_t *)(base + o_d);

    const uint32_t ctas = g.ctas, warps = g.warps;
    p.bcap = g.bcap;
    p.ccap = g.ccap;
    p.best = best_plus >= 0 ? 1u : 0u;
    p.plus = best_plus >= 0 ? (uint32_t)best_plus : 0u;
    p.ld_policy = ix->ld_policy ? ix->ld_policy - 1u : 1u;     // autotuner: no L1 allocation wins at every index size
    ws.spill = (uint2 *)(base + L.off_spill);
    ws.spill_blocks = L.spill_blocks;

    ws.sq_flag = (uint32_t *)(base + L.off_sqf);
    ws.sq_buf = (uint2 *)(base + L.off_sqb);
    ws.sq_n = ix->no_exchange ? 0u : BC_STEAL_SLOTS;
    cudaError_t e = cudaMemsetAsync(base + L.off_qcnt, 0, L.off_sqb - L.off_qcnt, st);   // qcnt .. ctr
    if (e == cudaSuccess) e = bc_launch_prepare(p, st);
    if (e == cudaSuccess && ix->ev[0]) e = cudaEventRecord(ix->ev[0], st);
    if (e == cudaSuccess) e = bc_launch_search(p, ix->sm_count, ctas, warps, st);
    if (e == cudaSuccess && ix->ev[1]) e = cudaEventRecord(ix->ev[1], st);
    if (e == cudaSuccess) e = bc_launch_post(p, *res, st);
    uint64_t *ctr = ix->h_ctr;                       // pinned: one asynchronous D2H, one synchronize per call
    if (e == cudaSuccess) e = cudaMemcpyAsync(ctr, ws.ctr, BC_CTR_COUNT * sizeof(uint64_t), cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) { cudaGetLastError(); return BC_E_CUDA; }

    float ms = 0.f;
    if (ix->ev[0] && ix->ev[1] && cudaEventElapsedTime(&ms, ix->ev[0], ix->ev[1]) != cudaSuccess) { ms = 0.f; cudaGetLastError(); }
    ix->stats[0] = ctr[BC_CTR_NODES];
    ix->stats[1] = ctr[BC_CTR_LOOKUPS];
    ix->stats[2] = ctr[BC_CTR_LINES];
    ix->stats[3] = ctr[BC_CTR_ARENA];
    ix->stats[4] = ctr[BC_CTR_DLOOKUPS];
    ix->stats[5] = ctr[BC_CTR_POOLMAX];
    ix->stats[6] = (uint64_t)((double)ms * 1e6);
    ix->stats[7] = (uint64_t)ctas << 32 | (uint64_t)warps << 16 | (uint64_t)ix->dev.bwt[0].layout << 15 | (g.bcap + g.ccap);
    ix->stats[8] = ctr[BC_CTR_BSTEPS];
    ix->stats[9] = ctr[BC_CTR_BNODES];
    ix->stats[10] = ctr[BC_CTR_CSTEPS];
    ix->stats[11] = ctr[BC_CTR_NODES] - ctr[BC_CTR_BNODES];
    ix->stats[12] = ctr[BC_CTR_CANCEL];
    ix->stats[13] = ctr[BC_CTR_SPILL];
    ix->stats[14] = ctr[BC_CTR_SPILLMAX];
    ix->stats[15] = best_plus >= 0 ? ctr[BC_CTR_PASSES] : ctr[BC_CTR_STEALS];

    if (ctr[BC_CTR_ERROR] & 1ull) return BC_E_INVAL;        // a read length outside 1..max_len
    if (ctr[BC_CTR_ERROR] & 2ull) return BC_E_CUDA;         // pool discipline violated: a bug, never silent
    if (ctr[BC_CTR_ERROR] & 4ull) return BC_E_NOMEM;        // a warp's spill area ran full: bc_set_tuning(more blocks)
    // n_hits_needed[0..1] were written by the device (write_hits): {hits after dedup | 0 on arena overflow, raw hits}
    if (ctr[BC_CTR_ARENA] > cap) return BC_E_OVERFLOW;
    if (ctr[BC_CTR_TOTAL] > res->hits_capacity) return BC_E_OVERFLOW;
    return BC_OK;
}

extern "C" int bc_align_batch(const bc_index *ix, const bc_reads *reads, const bc_opts *o, bc_result *res,
                              void *d_workspace, size_t ws_bytes, void *cuda_stream) {
    return bc_align_impl(ix, reads, o, res, d_workspace, ws_bytes, cuda_stream, -1);
}
