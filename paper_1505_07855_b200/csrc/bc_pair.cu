// bc_pair_batch: the step after the hot path -- pairing the two ends of a
// fragment "by plausible distance" (what `sampe` does on the CPU).  Input is
// the CSR result of bc_align_batch / bc_align_batch_best for a batch whose reads 2i, 2i+1 are the
// ends of pair i.  Definition: every hit with at most max_occ occurrences is located
// (A7) into placements (pos, strand, d); a proper pair = one end placed on strand 0 at pf, the other
// on strand 1 at pr >= pf, with fragment length pr + len(reverse end) - pf in [min_frag, max_frag].
// Output per pair: records {pos1, pos2, frag, d1, d2, strand1} sorted by (pos1, pos2, strand1), one
// per key with the smallest d1+d2 (then d1).  Integer work only; deterministic.
#include "bc_ws.cuh"

namespace {

inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }
constexpr uint64_t SCAN_TILE = 256 * 8;
inline unsigned grid_for(uint64_t n) { return (unsigned)((n + 255) / 256); }

struct PairLayout {
    size_t off_pcnt, off_poff, off_blk, off_rows, off_pos, off_meta, off_rcnt, off_roff, off_ucnt, off_tot, off_tmp, total;
};

void make_pair_layout(uint32_t n_reads, uint64_t max_place, uint64_t max_raw, PairLayout &L) {
    const size_t n = n_reads, np = n_reads / 2;
    size_t x = 0;
    L.off_pcnt = x; x = align_up(x + n * 4, 256);
    L.off_poff = x; x = align_up(x + (n + 1) * 8, 256);
    L.off_blk = x;  x = align_up(x + (n / SCAN_TILE + 2) * 8, 256);
    L.off_rows = x; x = align_up(x + max_place * 4, 256);
    L.off_pos = x;  x = align_up(x + max_place * 4, 256);
    L.off_meta = x; x = align_up(x + max_place * 4, 256);
    L.off_rcnt = x; x = align_up(x + np * 4, 256);
    L.off_roff = x; x = align_up(x + (np + 1) * 8, 256);
    L.off_ucnt = x; x = align_up(x + np * 4, 256);
    L.off_tot = x;  x = align_up(x + 32, 256);
    L.off_tmp = x;  x = align_up(x + max_raw * sizeof(bc_pair), 256);
    L.total = x;
}

__global__ void pair_count_place(const uint64_t *ho, const bc_hit *hits, uint32_t n_reads, uint32_t max_occ, uint32_t *pcnt,
                                 unsigned long long *skipped) {
    uint32_t r = blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= n_reads) return;
    uint32_t c = 0, sk = 0;
    for (uint64_t h = ho[r]; h < ho[r + 1]; ++h) {
        const uint32_t occ = hits[h].l - hits[h].k + 1u;
        if (occ <= max_occ) c += occ; else ++sk;
    }
    pcnt[r] = c;
    if (sk) atomicAdd(skipped, (unsigned long long)sk);
}

__global__ void pair_expand(const uint64_t *ho, const bc_hit *hits, uint32_t n_reads, uint32_t max_occ, const uint64_t *poff,
                            uint32_t *rows, uint32_t *meta) {
    uint32_t r = blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= n_reads) return;
    uint64_t o = poff[r];
    for (uint64_t h = ho[r]; h < ho[r + 1]; ++h) {
        const bc_hit x = hits[h];
        if (x.l - x.k + 1u > max_occ) continue;
        for (uint32_t j = x.k; j <= x.l; ++j) { rows[o] = j; meta[o] = (uint32_t)x.d | ((uint32_t)x.strand << 8); ++o; }
    }
}

// is (placement a of read 2i, placement b of read 2i+1) a proper pair?  frag out.
__device__ __forceinline__ bool proper(uint32_t pa, uint32_t sa, uint32_t la, uint32_t pb, uint32_t sb, uint32_t lb,
                                       uint32_t min_frag, uint32_t max_frag, uint32_t &frag) {
    if (sa == sb) return false;
    const uint32_t pf = sa == 0 ? pa : pb, pr = sa == 0 ? pb : pa, lr = sa == 0 ? lb : la;
    if (pr < pf) return false;
    frag = pr + lr - pf;
    return frag >= min_frag && frag <= max_frag;
}

__global__ void pair_count(const uint64_t *poff, const uint32_t *pos, const uint32_t *meta, const uint16_t *len, uint32_t n_pairs,
                           bc_pair_opts o, uint32_t *rcnt) {
    uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_pairs) return;
    const uint64_t a0 = poff[2 * i], a1 = poff[2 * i + 1], b1 = poff[2 * i + 2];
    const uint32_t la = len[2 * i], lb = len[2 * i + 1];
    uint32_t c = 0, frag;
    for (uint64_t a = a0; a < a1; ++a)
        for (uint64_t b = a1; b < b1; ++b)
            c += proper(pos[a], (meta[a] >> 8) & 1u, la, pos[b], (meta[b] >> 8) & 1u, lb, o.min_frag, o.max_frag, frag) ? 1u : 0u;
    rcnt[i] = c;
}

__device__ __forceinline__ bool pair_less(const bc_pair &x, const bc_pair &y) {
    if (x.pos1 != y.pos1) return x.pos1 < y.pos1;
    if (x.pos2 != y.pos2) return x.pos2 < y.pos2;
    if (x.strand1 != y.strand1) return x.strand1 < y.strand1;
    const uint32_t sx = (uint32_t)x.d1 + x.d2, sy = (uint32_t)y.d1 + y.d2;
    if (sx != sy) return sx < sy;
    return x.d1 < y.d1;
}

// generate the candidates of pair i into its raw segment, insertion-sort them, keep the first of every key
__global__ void pair_fill(const uint64_t *poff, const uint32_t *pos, const uint32_t *meta, const uint16_t *len, uint32_t n_pairs,
                          bc_pair_opts o, const uint64_t *roff, bc_pair *tmp, uint32_t *ucnt) {
    uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_pairs) return;
    const uint64_t a0 = poff[2 * i], a1 = poff[2 * i + 1], b1 = poff[2 * i + 2];
    const uint32_t la = len[2 * i], lb = len[2 * i + 1];
    bc_pair *seg = tmp + roff[i];
    uint32_t n = 0, frag;
    for (uint64_t a = a0; a < a1; ++a)
        for (uint64_t b = a1; b < b1; ++b) {
            const uint32_t sa = (meta[a] >> 8) & 1u, sb = (meta[b] >> 8) & 1u;
            if (!proper(pos[a], sa, la, pos[b], sb, lb, o.min_frag, o.max_frag, frag)) continue;
            bc_pair x;
            x.pos1 = pos[a]; x.pos2 = pos[b]; x.frag = frag; x.d1 = (uint8_t)(meta[a] & 255u); x.d2 = (uint8_t)(meta[b] & 255u);
            x.strand1 = (uint8_t)sa; x.zero = 0;
            uint32_t j = n++;
            while (j > 0 && pair_less(x, seg[j - 1])) { seg[j] = seg[j - 1]; --j; }
            seg[j] = x;
        }
    uint32_t u = 0;
    for (uint32_t j = 0; j < n; ++j)
        if (j == 0 || seg[j].pos1 != seg[u - 1].pos1 || seg[j].pos2 != seg[u - 1].pos2 || seg[j].strand1 != seg[u - 1].strand1)
            seg[u++] = seg[j];
    ucnt[i] = u;
}

__global__ void pair_write(const uint64_t *roff, const uint32_t *ucnt, const uint64_t *uoff, const bc_pair *tmp, bc_pair *out,
                           uint64_t cap, uint32_t n_pairs) {
    uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_pairs) return;
    const bc_pair *seg = tmp + roff[i];
    const uint64_t o = uoff[i];
    for (uint32_t j = 0; j < ucnt[i]; ++j)
        if (o + j < cap) out[o + j] = seg[j];
}

}  // namespace

extern "C" int bc_pair_workspace_bytes(uint32_t n_reads, uint64_t max_placements, uint64_t max_raw_pairs, size_t *bytes) {
    if (!bytes || (n_reads & 1u)) return BC_E_INVAL;
    PairLayout L;
    make_pair_layout(n_reads, max_placements, max_raw_pairs, L);
    *bytes = L.total;
    return BC_OK;
}

extern "C" int bc_pair_batch(const bc_index *ix, const uint64_t *d_hit_offsets, const bc_hit *d_hits, const uint16_t *d_len,
                             uint32_t n_reads, const bc_pair_opts *o, uint64_t max_placements, uint64_t max_raw_pairs,
                             bc_pair_result *res, void *d_workspace, size_t ws_bytes, void *cuda_stream) {
    if (!ix || !d_hit_offsets || !d_len || !o || !res || !res->pair_offsets || !res->n_needed || !d_workspace ||
        ((uintptr_t)d_workspace & 255) || (n_reads & 1u) || o->min_frag > o->max_frag || o->max_occ == 0 ||
        (res->pairs_capacity && !res->pairs))
        return BC_E_INVAL;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    PairLayout L;
    make_pair_layout(n_reads, max_placements, max_raw_pairs, L);
    if (ws_bytes < L.total) return BC_E_NOMEM;
    const uint32_t n_pairs = n_reads / 2;
    char *base = (char *)d_workspace;
    uint32_t *pcnt = (uint32_t *)(base + L.off_pcnt), *rows = (uint32_t *)(base + L.off_rows);
    uint32_t *pos = (uint32_t *)(base + L.off_pos), *meta = (uint32_t *)(base + L.off_meta);
    uint32_t *rcnt = (uint32_t *)(base + L.off_rcnt), *ucnt = (uint32_t *)(base + L.off_ucnt);
    uint64_t *poff = (uint64_t *)(base + L.off_poff), *blk = (uint64_t *)(base + L.off_blk);
    uint64_t *roff = (uint64_t *)(base + L.off_roff), *tot = (uint64_t *)(base + L.off_tot);
    bc_pair *tmp = (bc_pair *)(base + L.off_tmp);
    uint64_t needed[4] = {0, 0, 0, 0};             // pairs after dedup, raw candidates, placements, skipped hits
    auto fail = [&](int code) {
        if (cudaMemcpyAsync(res->n_needed, needed, 32, cudaMemcpyHostToDevice, st) != cudaSuccess ||
            cudaStreamSynchronize(st) != cudaSuccess)
            return (int)BC_E_CUDA;
        return code;
    };
    if (n_pairs == 0) {
        if (cudaMemsetAsync(res->pair_offsets, 0, 8, st) != cudaSuccess) return BC_E_CUDA;
        return fail(BC_OK);
    }
    if (cudaMemsetAsync(tot, 0, 32, st) != cudaSuccess) return BC_E_CUDA;
    // placements
    pair_count_place<<<grid_for(n_reads), 256, 0, st>>>(d_hit_offsets, d_hits, n_reads, o->max_occ, pcnt,
                                                        (unsigned long long *)(tot + 3));
    if (bc_exclusive_scan(pcnt, n_reads, blk, poff, tot + 2, st) != cudaSuccess) return BC_E_CUDA;
    uint64_t h[4];
    if (cudaMemcpyAsync(h, tot, 32, cudaMemcpyDeviceToHost, st) != cudaSuccess || cudaStreamSynchronize(st) != cudaSuccess)
        return BC_E_CUDA;
    needed[2] = h[2]; needed[3] = h[3];
    if (h[2] > max_placements) return fail(BC_E_OVERFLOW);
    if (h[2] > 0) {
        pair_expand<<<grid_for(n_reads), 256, 0, st>>>(d_hit_offsets, d_hits, n_reads, o->max_occ, poff, rows, meta);
        int rc = bc_locate(ix, rows, h[2], pos, cuda_stream);
        if (rc) return rc;
    }
    // candidates
    pair_count<<<grid_for(n_pairs), 256, 0, st>>>(poff, pos, meta, d_len, n_pairs, *o, rcnt);
    if (bc_exclusive_scan(rcnt, n_pairs, blk, roff, tot + 1, st) != cudaSuccess) return BC_E_CUDA;
    if (cudaMemcpyAsync(h, tot, 32, cudaMemcpyDeviceToHost, st) != cudaSuccess || cudaStreamSynchronize(st) != cudaSuccess)
        return BC_E_CUDA;
    needed[1] = h[1];
    if (h[1] > max_raw_pairs) return fail(BC_E_OVERFLOW);
    pair_fill<<<grid_for(n_pairs), 256, 0, st>>>(poff, pos, meta, d_len, n_pairs, *o, roff, tmp, ucnt);
    if (bc_exclusive_scan(ucnt, n_pairs, blk, res->pair_offsets, tot, st) != cudaSuccess) return BC_E_CUDA;
    pair_write<<<grid_for(n_pairs), 256, 0, st>>>(roff, ucnt, res->pair_offsets, tmp, res->pairs, res->pairs_capacity, n_pairs);
    if (cudaGetLastError() != cudaSuccess || cudaMemcpyAsync(h, tot, 32, cudaMemcpyDeviceToHost, st) != cudaSuccess ||
        cudaStreamSynchronize(st) != cudaSuccess)
        return BC_E_CUDA;
    needed[0] = h[0];
    return fail(h[0] > res->pairs_capacity ? BC_E_OVERFLOW : BC_OK);
}
