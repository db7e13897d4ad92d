// A6: per-query sort + dedup of the raw hits and the CSR output.
//   scan(qcnt) -> segments; scatter raw records into their query's segment; sort every segment by
//   (k, l, d) -- one thread for short segments, one CTA (padding-safe bitonic network in global
//   memory) for long ones; keep the first record of every (k,l) (= minimum d); scan the unique
//   counts; write bc_hit records and hit_offsets.  The result is a pure function of the SET of raw
//   records, so it does not depend on the order in which warps emitted them.
#include "bc_ws.cuh"

namespace {

constexpr int SCAN_THREADS = 256, SCAN_ITEMS = 8, SCAN_TILE = SCAN_THREADS * SCAN_ITEMS;
constexpr uint32_t SMALL_SEG = 32;
constexpr uint32_t INVALID_Q = 0xFFFFFFFFu;

__device__ __forceinline__ unsigned long long block_reduce_sum(unsigned long long v, unsigned long long *sh) {
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = v;
    __syncthreads();
    unsigned long long t = 0;
    if (threadIdx.x == 0) for (int w = 0; w < (int)(blockDim.x >> 5); ++w) t += sh[w];
    return t;   // valid in thread 0
}

__global__ void scan_tile_sums(const uint32_t *__restrict__ in, uint64_t n, uint64_t *__restrict__ blk) {
    __shared__ unsigned long long sh[SCAN_THREADS / 32];
    uint64_t base = (uint64_t)blockIdx.x * SCAN_TILE + (uint64_t)threadIdx.x * SCAN_ITEMS;
    unsigned long long v = 0;
    for (int i = 0; i < SCAN_ITEMS; ++i) if (base + i < n) v += in[base + i];
    unsigned long long t = block_reduce_sum(v, sh);
    if (threadIdx.x == 0) blk[blockIdx.x] = t;
}

// exclusive scan of the tile sums in place, single block; blk[n_tiles] = total
__global__ void scan_block_sums(uint64_t *blk, uint64_t n_tiles) {
    __shared__ unsigned long long sh[1024];
    __shared__ unsigned long long carry;
    if (threadIdx.x == 0) carry = 0;
    __syncthreads();
    for (uint64_t base = 0; base < n_tiles; base += blockDim.x) {
        uint64_t i = base + threadIdx.x;
        unsigned long long v = i < n_tiles ? blk[i] : 0;
        sh[threadIdx.x] = v;
        __syncthreads();
        for (unsigned o = 1; o < blockDim.x; o <<= 1) {
            unsigned long long x = threadIdx.x >= o ? sh[threadIdx.x - o] : 0;
            __syncthreads();
            sh[threadIdx.x] += x;
            __syncthreads();
        }
        if (i < n_tiles) blk[i] = carry + sh[threadIdx.x] - v;
        __syncthreads();
        if (threadIdx.x == 0) carry += sh[blockDim.x - 1];
        __syncthreads();
    }
    if (threadIdx.x == 0) blk[n_tiles] = carry;
}

__global__ void scan_apply(const uint32_t *__restrict__ in, uint64_t n, const uint64_t *__restrict__ blk,
                           uint64_t *__restrict__ out, uint64_t *total_out) {
    __shared__ unsigned long long sh[SCAN_THREADS];
    uint64_t base = (uint64_t)blockIdx.x * SCAN_TILE + (uint64_t)threadIdx.x * SCAN_ITEMS;
    uint32_t v[SCAN_ITEMS];
    unsigned long long s = 0;
    for (int i = 0; i < SCAN_ITEMS; ++i) { v[i] = base + i < n ? in[base + i] : 0; s += v[i]; }
    sh[threadIdx.x] = s;
    __syncthreads();
    for (unsigned o = 1; o < SCAN_THREADS; o <<= 1) {
        unsigned long long x = threadIdx.x >= o ? sh[threadIdx.x - o] : 0;
        __syncthreads();
        sh[threadIdx.x] += x;
        __syncthreads();
    }
    unsigned long long run = blk[blockIdx.x] + sh[threadIdx.x] - s;
    for (int i = 0; i < SCAN_ITEMS; ++i) { if (base + i < n) out[base + i] = run; run += v[i]; }
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        uint64_t n_tiles = (n + SCAN_TILE - 1) / SCAN_TILE;
        out[n] = blk[n_tiles];
        if (total_out) *total_out = blk[n_tiles];
    }
}

cudaError_t exclusive_scan(const uint32_t *in, uint64_t n, uint64_t *blk, uint64_t *out, uint64_t *total_out, cudaStream_t st) {
    uint64_t n_tiles = (n + SCAN_TILE - 1) / SCAN_TILE;
    scan_tile_sums<<<(unsigned)n_tiles, SCAN_THREADS, 0, st>>>(in, n, blk);
    scan_block_sums<<<1, 1024, 0, st>>>(blk, n_tiles);
    scan_apply<<<(unsigned)n_tiles, SCAN_THREADS, 0, st>>>(in, n, blk, out, total_out);
    return cudaGetLastError();
}

__global__ void scatter_raw(BcWorkspace ws) {
    uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    uint64_t total = ws.ctr[BC_CTR_ARENA];
    if (total > ws.arena_cap) return;                // arena overflowed: the host reports it
    if (i >= total) return;
    BcRawHit h = ws.arena[i];
    uint64_t pos = ws.seg_off[h.qid] + atomicAdd(&ws.qfill[h.qid], 1u);
    ws.seg_key[pos] = ((uint64_t)h.k << 32) | h.l;
    ws.seg_d[pos] = h.d;
}

__device__ __forceinline__ bool rec_less(uint64_t ka, uint32_t da, uint64_t kb, uint32_t db) {
    return ka < kb || (ka == kb && da < db);
}

// short segments: one thread sorts (insertion), dedups and stages {qid,k,l,d} back into the arena
// at the segment's own slots; unused slots get INVALID_Q.  Long segments are queued for sort_big.
__global__ void sort_small(BcWorkspace ws) {
    uint32_t q = blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= ws.nq || ws.ctr[BC_CTR_ARENA] > ws.arena_cap) return;
    uint32_t n = ws.qcnt[q];
    if (n == 0) { ws.qfill[q] = 0; return; }
    if (n > SMALL_SEG) {
        uint32_t slot = (uint32_t)atomicAdd((unsigned long long *)&ws.ctr[BC_CTR_NBIG], 1ull);
        ws.big[slot] = q;
        return;
    }
    uint64_t o = ws.seg_off[q];
    uint64_t *key = ws.seg_key + o;
    uint32_t *dd = ws.seg_d + o;
    for (uint32_t i = 1; i < n; ++i) {
        uint64_t kx = key[i]; uint32_t dx = dd[i];
        uint32_t j = i;
        while (j > 0 && rec_less(kx, dx, key[j - 1], dd[j - 1])) { key[j] = key[j - 1]; dd[j] = dd[j - 1]; --j; }
        key[j] = kx; dd[j] = dx;
    }
    uint32_t u = 0;
    for (uint32_t i = 0; i < n; ++i)
        if (i == 0 || key[i] != key[i - 1])
            ws.arena[o + u++] = BcRawHit{q, (uint32_t)(key[i] >> 32), (uint32_t)key[i], dd[i]};
    for (uint32_t i = u; i < n; ++i) ws.arena[o + i].qid = INVALID_Q;
    ws.qfill[q] = u;
}

// long segments: one CTA each.  Bitonic network in which every compare-exchange leaves the minimum
// at the lower index (first stage of a merge mirrors, i ^ (k-1)); virtual +inf padding beyond n is
// then never moved, so any n works in place.
__global__ void sort_big(BcWorkspace ws) {
    __shared__ uint32_t sh_cnt[1024];
    uint64_t n_big = ws.ctr[BC_CTR_NBIG];
    if (ws.ctr[BC_CTR_ARENA] > ws.arena_cap) return;
    for (uint64_t bi = blockIdx.x; bi < n_big; bi += gridDim.x) {
        uint32_t q = ws.big[bi];
        uint32_t n = ws.qcnt[q];
        uint64_t o = ws.seg_off[q];
        uint64_t *key = ws.seg_key + o;
        uint32_t *dd = ws.seg_d + o;
        uint32_t n2 = 1; while (n2 < n) n2 <<= 1;
        for (uint32_t k = 2; k <= n2; k <<= 1) {
            for (uint32_t j = k >> 1; j > 0; j >>= 1) {
                for (uint32_t i = threadIdx.x; i < n; i += blockDim.x) {
                    uint32_t l = (j == (k >> 1)) ? (i ^ (k - 1)) : (i ^ j);
                    if (l > i && l < n) {
                        uint64_t ka = key[i], kb = key[l]; uint32_t da = dd[i], db = dd[l];
                        if (rec_less(kb, db, ka, da)) { key[i] = kb; dd[i] = db; key[l] = ka; dd[l] = da; }
                    }
                }
                __syncthreads();
            }
        }
        // dedup: chunk per thread, count heads, scan, stage
        uint32_t per = (n + blockDim.x - 1) / blockDim.x;
        uint32_t b = threadIdx.x * per, e = b + per < n ? b + per : n, heads = 0;
        for (uint32_t i = b; i < e; ++i) heads += (i == 0 || key[i] != key[i - 1]);
        sh_cnt[threadIdx.x] = heads;
        __syncthreads();
        for (unsigned s = 1; s < blockDim.x; s <<= 1) {
            uint32_t x = threadIdx.x >= s ? sh_cnt[threadIdx.x - s] : 0;
            __syncthreads();
            sh_cnt[threadIdx.x] += x;
            __syncthreads();
        }
        uint32_t u = sh_cnt[threadIdx.x] - heads, total_u = sh_cnt[blockDim.x - 1];
        for (uint32_t i = b; i < e; ++i)
            if (i == 0 || key[i] != key[i - 1])
                ws.arena[o + u++] = BcRawHit{q, (uint32_t)(key[i] >> 32), (uint32_t)key[i], dd[i]};
        __syncthreads();
        for (uint32_t i = total_u + threadIdx.x; i < n; i += blockDim.x) ws.arena[o + i].qid = INVALID_Q;
        if (threadIdx.x == 0) ws.qfill[q] = total_u;
        __syncthreads();
    }
}

__global__ void write_hits(BcWorkspace ws, bc_result res, uint32_t n_reads) {
    uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    uint64_t raw = ws.ctr[BC_CTR_ARENA], total = ws.uoff[ws.nq];
    if (i == 0) res.n_hits_needed[1] = raw;
    if (raw > ws.arena_cap) { if (i == 0) res.n_hits_needed[0] = 0; return; }   // arena overflowed: nothing was sorted
    if (i == 0) { res.n_hits_needed[0] = total; ws.ctr[BC_CTR_TOTAL] = total; }
    if (i <= n_reads) res.hit_offsets[i] = ws.uoff[i < n_reads ? 2 * i : ws.nq];
    if (total > res.hits_capacity || i >= raw) return;
    BcRawHit h = ws.arena[i];
    if (h.qid == INVALID_Q) return;
    uint64_t j = i - ws.seg_off[h.qid];
    bc_hit out;
    out.k = h.k; out.l = h.l; out.d = (uint8_t)h.d; out.strand = (uint8_t)(h.qid & 1u); out.zero = 0;
    res.hits[ws.uoff[h.qid] + j] = out;
}

}  // namespace

// exclusive scan of n uint32 counts into uint64 offsets (out[n] = total); blk: n/2048 + 2 uint64 of scratch
cudaError_t bc_exclusive_scan(const uint32_t *in, uint64_t n, uint64_t *blk, uint64_t *out, uint64_t *total_out,
                              cudaStream_t st) {
    return exclusive_scan(in, n, blk, out, total_out, st);
}

cudaError_t bc_launch_post(const BcSearchParams &p, bc_result res, cudaStream_t st) {
    const BcWorkspace &ws = p.ws;
    if (ws.nq == 0) return cudaSuccess;
    cudaError_t e = exclusive_scan(ws.qcnt, ws.nq, ws.blk, ws.seg_off, nullptr, st);
    if (e != cudaSuccess) return e;
    uint64_t slots = ws.arena_cap > (uint64_t)p.reads.n_reads + 1 ? ws.arena_cap : (uint64_t)p.reads.n_reads + 1;
    unsigned grid_slots = (unsigned)((slots + 255) / 256);
    scatter_raw<<<grid_slots, 256, 0, st>>>(ws);
    sort_small<<<(ws.nq + 127) / 128, 128, 0, st>>>(ws);
    sort_big<<<592, 512, 0, st>>>(ws);
    e = exclusive_scan(ws.qfill, ws.nq, ws.blk, ws.uoff, nullptr, st);
    if (e != cudaSuccess) return e;
    write_hits<<<grid_slots, 256, 0, st>>>(ws, res, p.reads.n_reads);
    return cudaGetLastError();
}
