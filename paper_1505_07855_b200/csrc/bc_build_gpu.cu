// bc_index_build_gpu: the step BEFORE the hot path -- index construction
// (the offline `index` command) -- on the GPU.  Suffix array of T$ and reverse(T)$
// by prefix doubling (Manber-Myers): rank the suffixes by their first 21 symbols, then repeatedly
// sort by (rank[i], rank[i+h]) and double h until all ranks are distinct.  The sorts and scans are
// CUB library primitives (DeviceRadixSort / DeviceScan); the keys, the re-ranking, the BWT, the Occ
// checkpoints and the SA sample are kernels below.  Produces exactly the transport arrays of
// bc_index_build_host (bit-identical; tests compare both with the oracle's naive suffix sort).
// Untimed helper, not part of the hot path.
#include <cub/cub.cuh>

#include <algorithm>
#include <new>

#include "bc_host_index.h"

namespace {

inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }
inline unsigned grid_for(uint64_t n) { return (unsigned)((n + 255) / 256); }

struct GpuLayout {
    size_t off_text, off_keyA, off_keyB, off_valA, off_valB, off_rank, off_flag, off_sym, off_cnt4, off_occ, off_bwt2, off_sa,
        off_misc, off_cub, cub_bytes, total;
};

struct Add4 {
    __host__ __device__ uint4 operator()(const uint4 &a, const uint4 &b) const {
        return make_uint4(a.x + b.x, a.y + b.y, a.z + b.z, a.w + b.w);
    }
};

size_t cub_temp_bytes(uint64_t N, uint64_t n_chunks) {
    size_t a = 0, b = 0, c = 0;
    cub::DeviceRadixSort::SortPairs(nullptr, a, (const uint64_t *)nullptr, (uint64_t *)nullptr, (const uint32_t *)nullptr,
                                    (uint32_t *)nullptr, (int64_t)N, 0, 64);
    cub::DeviceScan::InclusiveSum(nullptr, b, (const uint32_t *)nullptr, (uint32_t *)nullptr, (int64_t)N);
    cub::DeviceScan::ExclusiveScan(nullptr, c, (const uint4 *)nullptr, (uint4 *)nullptr, Add4(), make_uint4(0, 0, 0, 0),
                                   (int64_t)n_chunks);
    return std::max(a, std::max(b, c));
}

void make_layout(uint64_t n, uint32_t occ_interval, uint32_t sa_interval, GpuLayout &L) {
    const uint64_t N = n + 1, n_chunks = n / occ_interval + 1;
    size_t x = 0;
    L.off_text = x; x = align_up(x + n + 64, 256);
    L.off_keyA = x; x = align_up(x + N * 8, 256);
    L.off_keyB = x; x = align_up(x + N * 8, 256);
    L.off_valA = x; x = align_up(x + N * 4, 256);
    L.off_valB = x; x = align_up(x + N * 4, 256);
    L.off_rank = x; x = align_up(x + N * 4, 256);
    L.off_flag = x; x = align_up(x + N * 4, 256);
    L.off_sym = x;  x = align_up(x + n + 64, 256);
    L.off_cnt4 = x; x = align_up(x + n_chunks * 16, 256);
    L.off_occ = x;  x = align_up(x + n_chunks * 16, 256);
    L.off_bwt2 = x; x = align_up(x + (n / 32 + 1) * 8, 256);
    L.off_sa = x;   x = align_up(x + (n / sa_interval + 1) * 4, 256);
    L.off_misc = x; x = align_up(x + 64, 256);
    L.cub_bytes = align_up(cub_temp_bytes(N, n_chunks), 256);
    L.off_cub = x;  x += L.cub_bytes;
    L.total = x;
}

// key of suffix i from its first 21 symbols, 3 bits each (code+1; 0 = past the end, so that a
// suffix that is a prefix of another sorts first: '$' is the smallest symbol)
__global__ void k_init_keys(const uint8_t *text, uint64_t n, uint64_t *key, uint32_t *val) {
    uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i > n) return;
    uint64_t k = 0;
#pragma unroll
    for (int j = 0; j < 21; ++j) {
        const uint64_t p = i + j;
        k = (k << 3) | (p < n ? (uint64_t)text[p] + 1u : 0u);
    }
    key[i] = k;
    val[i] = (uint32_t)i;
}

__global__ void k_flag(const uint64_t *key, uint64_t N, uint32_t *flag) {
    uint64_t j = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (j < N) flag[j] = (j == 0 || key[j] != key[j - 1]) ? 1u : 0u;
}

__global__ void k_scatter_rank(const uint32_t *val, const uint32_t *r, uint64_t N, uint32_t *rank) {
    uint64_t j = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (j < N) rank[val[j]] = r[j];                       // 1-based rank of the group suffix val[j] is in
}

__global__ void k_pair_keys(const uint32_t *rank, uint64_t N, uint64_t h, uint64_t *key, uint32_t *val) {
    uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const uint64_t second = i + h < N ? rank[i + h] : 0u;
    key[i] = ((uint64_t)rank[i] << 32) | second;
    val[i] = (uint32_t)i;
}

__global__ void k_find_primary(const uint32_t *sa, uint64_t N, uint64_t *primary) {
    uint64_t j = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (j < N && sa[j] == 0) *primary = j;
}

__global__ void k_bwt_symbols(const uint8_t *text, const uint32_t *sa, uint64_t N, const uint64_t *primary, uint8_t *sym) {
    uint64_t j = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= N) return;
    const uint32_t p = sa[j];
    if (p == 0) return;                                   // the '$' row is removed
    const uint64_t pr = *primary;
    sym[j - (j > pr ? 1u : 0u)] = text[p - 1];
}

__global__ void k_pack_bwt(const uint8_t *sym, uint64_t n, uint64_t n_words, uint64_t *bwt2) {
    uint64_t w = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (w >= n_words) return;
    uint64_t x = 0;
    for (int b = 0; b < 32; ++b) {
        const uint64_t j = w * 32 + b;
        if (j < n) x |= (uint64_t)sym[j] << (2 * b);
    }
    bwt2[w] = x;
}

__global__ void k_chunk_counts(const uint8_t *sym, uint64_t n, uint32_t occ_interval, uint64_t n_chunks, uint4 *cnt4) {
    uint64_t t = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= n_chunks) return;
    uint32_t c[4] = {0, 0, 0, 0};
    const uint64_t b = t * occ_interval, e = b + occ_interval < n ? b + occ_interval : n;
    for (uint64_t j = b; j < e; ++j) c[sym[j] & 3]++;
    cnt4[t] = make_uint4(c[0], c[1], c[2], c[3]);
}

__global__ void k_sample_sa(const uint32_t *sa, uint64_t n_samples, uint32_t sa_interval, uint32_t *out) {
    uint64_t t = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t < n_samples) out[t] = sa[t * sa_interval];
}

#define CK(x) do { if ((x) != cudaSuccess) { cudaGetLastError(); return BC_E_CUDA; } } while (0)

// one direction: text (HOST) -> transport arrays in `out` / `pub`; fills sa_out if asked
int build_one(const uint8_t *text, uint64_t n, uint32_t occ_interval, uint32_t sa_interval, char *base, const GpuLayout &L,
              cudaStream_t st, BcBwtArrays &out, bc_bwt_host &pub, std::vector<uint32_t> *sa_out) {
    const uint64_t N = n + 1, n_chunks = n / occ_interval + 1, n_words = n / 32 + 1, n_samples = n / sa_interval + 1;
    uint8_t *d_text = (uint8_t *)(base + L.off_text), *d_sym = (uint8_t *)(base + L.off_sym);
    uint64_t *keyA = (uint64_t *)(base + L.off_keyA), *keyB = (uint64_t *)(base + L.off_keyB);
    uint32_t *valA = (uint32_t *)(base + L.off_valA), *valB = (uint32_t *)(base + L.off_valB);
    uint32_t *rank = (uint32_t *)(base + L.off_rank), *flag = (uint32_t *)(base + L.off_flag);
    uint4 *cnt4 = (uint4 *)(base + L.off_cnt4), *occ = (uint4 *)(base + L.off_occ);
    uint64_t *bwt2 = (uint64_t *)(base + L.off_bwt2), *misc = (uint64_t *)(base + L.off_misc);
    uint32_t *d_sa = (uint32_t *)(base + L.off_sa);
    void *cub_tmp = base + L.off_cub;
    size_t cub_bytes = L.cub_bytes;

    CK(cudaMemcpyAsync(d_text, text, n, cudaMemcpyHostToDevice, st));
    k_init_keys<<<grid_for(N), 256, 0, st>>>(d_text, n, keyA, valA);
    for (uint64_t h = 21;; h *= 2) {
        CK(cub::DeviceRadixSort::SortPairs(cub_tmp, cub_bytes, keyA, keyB, valA, valB, (int64_t)N, 0, 64, st));
        k_flag<<<grid_for(N), 256, 0, st>>>(keyB, N, flag);
        CK(cub::DeviceScan::InclusiveSum(cub_tmp, cub_bytes, flag, flag, (int64_t)N, st));
        k_scatter_rank<<<grid_for(N), 256, 0, st>>>(valB, flag, N, rank);
        uint32_t groups = 0;
        CK(cudaMemcpyAsync(&groups, flag + (N - 1), 4, cudaMemcpyDeviceToHost, st));
        CK(cudaStreamSynchronize(st));
        if (groups == N) break;                           // every suffix has its own rank: valB is the suffix array
        if (h > 2 * N) return BC_E_CUDA;                  // cannot happen: all suffixes of T$ are distinct
        k_pair_keys<<<grid_for(N), 256, 0, st>>>(rank, N, h, keyA, valA);
    }
    const uint32_t *sa = valB;
    k_find_primary<<<grid_for(N), 256, 0, st>>>(sa, N, misc);
    k_bwt_symbols<<<grid_for(N), 256, 0, st>>>(d_text, sa, N, misc, d_sym);
    k_pack_bwt<<<grid_for(n_words), 256, 0, st>>>(d_sym, n, n_words, bwt2);
    k_chunk_counts<<<grid_for(n_chunks), 256, 0, st>>>(d_sym, n, occ_interval, n_chunks, cnt4);
    CK(cub::DeviceScan::ExclusiveScan(cub_tmp, cub_bytes, cnt4, occ, Add4(), make_uint4(0, 0, 0, 0), (int64_t)n_chunks, st));
    out.bwt2.resize(n_words);
    out.occ.resize(n_chunks * 4);
    uint64_t primary = 0;
    CK(cudaMemcpyAsync(out.bwt2.data(), bwt2, n_words * 8, cudaMemcpyDeviceToHost, st));
    CK(cudaMemcpyAsync(out.occ.data(), occ, n_chunks * 16, cudaMemcpyDeviceToHost, st));
    CK(cudaMemcpyAsync(&primary, misc, 8, cudaMemcpyDeviceToHost, st));
    if (sa_out) {
        k_sample_sa<<<grid_for(n_samples), 256, 0, st>>>(sa, n_samples, sa_interval, d_sa);
        sa_out->resize(n_samples);
        CK(cudaMemcpyAsync(sa_out->data(), d_sa, n_samples * 4, cudaMemcpyDeviceToHost, st));
    }
    CK(cudaStreamSynchronize(st));
    CK(cudaGetLastError());
    uint64_t cnt[4] = {0, 0, 0, 0};
    for (uint64_t i = 0; i < n; ++i) cnt[text[i]]++;
    pub.n = n; pub.primary = primary; pub.bwt2 = out.bwt2.data(); pub.occ_interval = occ_interval; pub.occ = out.occ.data();
    pub.C[0] = 0;
    for (int c = 0; c < 4; ++c) pub.C[c + 1] = pub.C[c] + cnt[c];
    return BC_OK;
}

}  // namespace

extern "C" int bc_index_build_gpu_bytes(uint64_t n, uint32_t occ_interval, uint32_t sa_interval, size_t *bytes) {
    if (!bytes || n < 1 || n >= 0xFFFFFFFFull || occ_interval == 0 || occ_interval % 32 || sa_interval == 0) return BC_E_INVAL;
    GpuLayout L;
    make_layout(n, occ_interval, sa_interval, L);
    *bytes = L.total;
    return BC_OK;
}

extern "C" int bc_index_build_gpu(const uint8_t *text, uint64_t n, uint32_t occ_interval, uint32_t sa_interval,
                                  void *d_scratch, size_t scratch_bytes, void *cuda_stream, bc_index_host **out) {
    if (!text || !out || !d_scratch || ((uintptr_t)d_scratch & 255) || n < 1 || n >= 0xFFFFFFFFull || occ_interval == 0 ||
        occ_interval % 32 || sa_interval == 0)
        return BC_E_INVAL;
    for (uint64_t i = 0; i < n; ++i) if (text[i] > 3) return BC_E_INVAL;
    GpuLayout L;
    make_layout(n, occ_interval, sa_interval, L);
    if (scratch_bytes < L.total) return BC_E_NOMEM;
    BcHostIndexOwner *h = new (std::nothrow) BcHostIndexOwner();
    if (!h) return BC_E_NOMEM;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int rc;
    try {
        rc = build_one(text, n, occ_interval, sa_interval, (char *)d_scratch, L, st, h->fwd, h->pub.fwd, &h->sa);
        if (rc == BC_OK) {
            std::vector<uint8_t> rt(text, text + n);
            std::reverse(rt.begin(), rt.end());
            rc = build_one(rt.data(), n, occ_interval, sa_interval, (char *)d_scratch, L, st, h->rev, h->pub.rev, nullptr);
        }
    } catch (const std::bad_alloc &) { rc = BC_E_NOMEM; }
    if (rc) { delete h; return rc; }
    h->pub.sa_interval = sa_interval;
    h->pub.sa = h->sa.data();
    *out = &h->pub;
    return BC_OK;
}
