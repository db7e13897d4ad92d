// bc_index_upload (A0 re-layout kernel), bc_locate (A7), handle management.  sm_100a only.
#include <new>

#include "bc_internal.cuh"

namespace {

inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

struct Layout {
    size_t lines_bytes, off_fwd, off_rev, off_sa, sa_bytes, off_stage_bwt, stage_bwt_bytes, off_stage_occ,
        stage_occ_bytes, total;
    uint64_t n_lines;
    uint32_t layout;                                 // 0: 32-byte blocks of 64 symbols, 1: 128-byte lines of 384 (bc_internal.cuh)
};

// 0 = by index size (blocks up to 64 MB of them, lines beyond: the index then lives in HBM, where a missing
// sector costs a whole 128-byte line), 1 = blocks, 2 = lines.  Process-wide; read by bc_index_device_bytes / _upload.
int g_layout_choice = 0;

bool check_bwt(const bc_bwt_host &b) {
    return b.bwt2 && b.occ && b.n >= 1 && b.n < 0xFFFFFFFFull && b.primary <= b.n && b.occ_interval > 0 &&
           b.occ_interval % 32 == 0 && b.C[4] == b.n;
}

int make_layout(const bc_index_host *h, Layout &L) {
    if (!h || !h->sa || h->sa_interval == 0 || !check_bwt(h->fwd) || !check_bwt(h->rev) || h->fwd.n != h->rev.n)
        return BC_E_INVAL;
    uint64_t n = h->fwd.n;
    const size_t block_bytes = 2 * align_up((n / BC_BLOCK_SYMS + 1) * 32, 256);
    (void)block_bytes;
    L.layout = g_layout_choice ? (uint32_t)(g_layout_choice - 1) : 0u;   // measured: blocks win at every size
    if (L.layout == 0) { L.n_lines = n / BC_BLOCK_SYMS + 1; L.lines_bytes = align_up(L.n_lines * 32, 256); }
    else               { L.n_lines = n / BC_LINE_SYMS + 1;  L.lines_bytes = align_up(L.n_lines * 128, 256); }
    L.off_fwd = 0;
    L.off_rev = L.lines_bytes;
    L.off_sa = 2 * L.lines_bytes;
    L.sa_bytes = align_up((n / h->sa_interval + 1) * 4, 256);
    L.off_stage_bwt = L.off_sa + L.sa_bytes;
    L.stage_bwt_bytes = align_up((n / 32 + 1) * 8, 256);
    L.off_stage_occ = L.off_stage_bwt + L.stage_bwt_bytes;
    uint32_t oi = h->fwd.occ_interval < h->rev.occ_interval ? h->fwd.occ_interval : h->rev.occ_interval;
    L.stage_occ_bytes = align_up((n / oi + 1) * 16, 256);
    L.total = L.off_stage_occ + L.stage_occ_bytes;
    return BC_OK;
}

// even bits of x (bit 2i -> bit i)
__device__ __forceinline__ uint32_t compact_even(uint64_t x) {
    x &= 0x5555555555555555ull;
    x = (x | (x >> 1)) & 0x3333333333333333ull;
    x = (x | (x >> 2)) & 0x0F0F0F0F0F0F0F0Full;
    x = (x | (x >> 4)) & 0x00FF00FF00FF00FFull;
    x = (x | (x >> 8)) & 0x0000FFFF0000FFFFull;
    x = (x | (x >> 16)) & 0x00000000FFFFFFFFull;
    return (uint32_t)x;
}

// A0: one thread per 32-byte block
__global__ void bc_relayout_kernel(const uint64_t *__restrict__ bwt2, const uint32_t *__restrict__ occ,
                                   uint32_t occ_interval, uint64_t n, uint64_t n_lines, BcBlock *__restrict__ out) {
    uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_lines) return;
    uint64_t s0 = i * BC_BLOCK_SYMS;                 // first symbol of the block (may be == n: empty tail block)
    uint64_t n_words = n / 32 + 1;
    uint64_t t = s0 / occ_interval;
    uint32_t cnt[4];
    for (int c = 0; c < 4; ++c) cnt[c] = occ[t * 4 + c];
    for (uint64_t w = t * occ_interval / 32; w < s0 / 32; ++w) {   // whole words between checkpoint and line start
        uint64_t x = bwt2[w], lo = x & 0x5555555555555555ull, hi = (x >> 1) & 0x5555555555555555ull;
        uint32_t nt = __popcll(lo & hi), nc = __popcll(lo & ~hi), ng = __popcll(hi & ~lo);
        cnt[0] += 32 - nt - nc - ng; cnt[1] += nc; cnt[2] += ng; cnt[3] += nt;
    }
    BcBlock L;
    for (int c = 0; c < 4; ++c) L.cnt[c] = cnt[c];
    for (int q = 0; q < 2; ++q) {
        uint64_t w0 = s0 / 32 + q;
        uint64_t x = w0 < n_words ? bwt2[w0] : 0;
        L.lo[q] = compact_even(x);
        L.hi[q] = compact_even(x >> 1);
    }
    out[i] = L;
}

// A0, layout 1: one thread per 128-byte line of 384 symbols (12 transport words of 32 symbols)
__global__ void bc_relayout_lines_kernel(const uint64_t *__restrict__ bwt2, const uint32_t *__restrict__ occ,
                                         uint32_t occ_interval, uint64_t n, uint64_t n_lines, uint32_t *__restrict__ out) {
    uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_lines) return;
    uint64_t s0 = i * BC_LINE_SYMS;
    uint64_t n_words = n / 32 + 1;
    uint64_t t = s0 / occ_interval;
    uint32_t cnt[4];
    for (int c = 0; c < 4; ++c) cnt[c] = occ[t * 4 + c];
    for (uint64_t w = t * occ_interval / 32; w < s0 / 32; ++w) {   // whole words between checkpoint and line start
        uint64_t x = bwt2[w], lo = x & 0x5555555555555555ull, hi = (x >> 1) & 0x5555555555555555ull;
        uint32_t nt = __popcll(lo & hi), nc = __popcll(lo & ~hi), ng = __popcll(hi & ~lo);
        cnt[0] += 32 - nt - nc - ng; cnt[1] += nc; cnt[2] += ng; cnt[3] += nt;
    }
    uint32_t *L = out + i * 32;
    for (int c = 0; c < 4; ++c) L[c] = cnt[c];
    uint32_t in[4] = {0, 0, 0, 0};                   // counts inside the line so far
    for (int j = 0; j < 12; ++j) {
        if (j == 4) { L[4] = in[0] | (in[1] << 16); L[5] = in[2] | (in[3] << 16); }     // s1: symbols 0..127
        if (j == 8) { L[6] = in[0] | (in[1] << 16); L[7] = in[2] | (in[3] << 16); }     // s2: symbols 0..255
        uint64_t w0 = s0 / 32 + j;
        uint64_t x = w0 < n_words ? bwt2[w0] : 0;
        uint32_t lo = compact_even(x), hi = compact_even(x >> 1);
        uint32_t nt = __popc(lo & hi), nc = __popc(lo & ~hi), ng = __popc(hi & ~lo);
        in[0] += 32 - nt - nc - ng; in[1] += nc; in[2] += ng; in[3] += nt;
        // region g = j / 4 at words 8 + 8g: lo0 (2 words) | hi0 | lo1 | hi1; 64-bit word k = (j % 4) / 2, half j % 2
        const int g = j >> 2, k = (j & 3) >> 1, half = j & 1;
        L[8 + 8 * g + 4 * k + half] = lo;
        L[8 + 8 * g + 4 * k + 2 + half] = hi;
    }
}

// A7: one thread per row, LF-walk to a sampled row (one rank unit per step)
template <int LAY>
__global__ void bc_locate_kernel(BcIndexDev ix, const uint32_t *__restrict__ rows, uint64_t n_rows,
                                 uint32_t *__restrict__ pos) {
    uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_rows) return;
    const BcBwtDev &b = ix.bwt[0];
    uint32_t j = rows[i], steps = 0;
    if (j > b.n) { pos[i] = 0xFFFFFFFFu; return; }
    while (j % ix.sa_interval != 0 && j != b.primary) {
        uint32_t p = j - (j > b.primary ? 1u : 0u);           // index of B[j] in the '$'-less string
        const BcUnit<LAY> u = bc_load_unit<LAY, 0>(b.lines, p);
        uint32_t c = bc_unit_symbol(u, p);
        j = b.C[c] + bc_unit_rank1(u, p, c) + 1;              // C[c] + O(c, j), O counts B[0..j] inclusive
        ++steps;
    }
    pos[i] = (j == b.primary ? 0u : ix.sa[j / ix.sa_interval]) + steps;
}

}  // namespace

extern "C" int bc_index_device_bytes(const bc_index_host *h, size_t *bytes) {
    Layout L;
    if (!bytes) return BC_E_INVAL;
    int rc = make_layout(h, L);
    if (rc) return rc;
    *bytes = L.total;
    return BC_OK;
}

extern "C" int bc_index_upload(const bc_index_host *h, void *d_mem, size_t d_bytes, void *cuda_stream, bc_index **out) {
    Layout L;
    if (!out || !d_mem || ((uintptr_t)d_mem & 255)) return BC_E_INVAL;
    int rc = make_layout(h, L);
    if (rc) return rc;
    if (d_bytes < L.total) return BC_E_NOMEM;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    bc_index *ix = new (std::nothrow) bc_index();
    if (!ix) return BC_E_NOMEM;
    char *base = (char *)d_mem;
    uint64_t n = h->fwd.n;
    cudaError_t e = cudaSuccess;
    for (int which = 0; which < 2 && e == cudaSuccess; ++which) {
        const bc_bwt_host &b = which ? h->rev : h->fwd;
        uint64_t *s_bwt = (uint64_t *)(base + L.off_stage_bwt);
        uint32_t *s_occ = (uint32_t *)(base + L.off_stage_occ);
        BcBlock *lines = (BcBlock *)(base + (which ? L.off_rev : L.off_fwd));
        e = cudaMemcpyAsync(s_bwt, b.bwt2, (n / 32 + 1) * 8, cudaMemcpyHostToDevice, st);
        if (e == cudaSuccess) e = cudaMemcpyAsync(s_occ, b.occ, (n / b.occ_interval + 1) * 16, cudaMemcpyHostToDevice, st);
        if (e == cudaSuccess) {
            unsigned grid = (unsigned)((L.n_lines + 255) / 256);
            if (L.layout == 0) bc_relayout_kernel<<<grid, 256, 0, st>>>(s_bwt, s_occ, b.occ_interval, n, L.n_lines, lines);
            else bc_relayout_lines_kernel<<<grid, 256, 0, st>>>(s_bwt, s_occ, b.occ_interval, n, L.n_lines, (uint32_t *)lines);
            e = cudaGetLastError();
        }
        if (e == cudaSuccess) e = cudaStreamSynchronize(st);   // staging is reused; host arrays are borrowed
        BcBwtDev &d = ix->dev.bwt[which];
        d.lines = (const uint4 *)lines;
        d.layout = L.layout;
        d.n = (uint32_t)n;
        d.primary = (uint32_t)b.primary;
        for (int c = 0; c < 4; ++c) d.C[c] = (uint32_t)b.C[c];
    }
    if (e == cudaSuccess) e = cudaMemcpyAsync(base + L.off_sa, h->sa, (n / h->sa_interval + 1) * 4, cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) { delete ix; return BC_E_CUDA; }
    ix->dev.sa = (const uint32_t *)(base + L.off_sa);
    ix->dev.sa_interval = h->sa_interval;
    ix->n = n;
    ix->bytes = L.total;
    ix->ctas_per_sm = 0; ix->warps_per_cta = 0; ix->spill_blocks = 0; ix->pool_kb = 0; ix->ld_policy = 0; ix->no_exchange = 0;
    ix->h_ctr = nullptr;
    for (int i = 0; i < 16; ++i) ix->stats[i] = 0;
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) {
        delete ix; return BC_E_CUDA;
    }
    ix->sm_count = sms;
    ix->ev[0] = ix->ev[1] = nullptr;
    if (cudaEventCreate(&ix->ev[0]) != cudaSuccess || cudaEventCreate(&ix->ev[1]) != cudaSuccess ||
        cudaHostAlloc((void **)&ix->h_ctr, 32 * sizeof(uint64_t), cudaHostAllocDefault) != cudaSuccess) {
        for (int i = 0; i < 2; ++i) if (ix->ev[i]) cudaEventDestroy(ix->ev[i]);
        cudaGetLastError();
        delete ix; return BC_E_CUDA;
    }
    *out = ix;
    return BC_OK;
}

extern "C" int bc_index_free(bc_index *ix) {
    if (!ix) return BC_E_INVAL;
    for (int i = 0; i < 2; ++i) if (ix->ev[i]) cudaEventDestroy(ix->ev[i]);
    if (ix->h_ctr) cudaFreeHost(ix->h_ctr);
    delete ix;
    return BC_OK;
}

extern "C" int bc_locate(const bc_index *ix, const uint32_t *d_rows, uint64_t n_rows, uint32_t *d_pos, void *cuda_stream) {
    if (!ix || (n_rows && (!d_rows || !d_pos))) return BC_E_INVAL;
    if (n_rows == 0) return BC_OK;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    uint64_t grid = (n_rows + 255) / 256;
    if (grid > 0x7FFFFFFFull) return BC_E_INVAL;
    if (ix->dev.bwt[0].layout == 0) bc_locate_kernel<0><<<(unsigned)grid, 256, 0, st>>>(ix->dev, d_rows, n_rows, d_pos);
    else bc_locate_kernel<1><<<(unsigned)grid, 256, 0, st>>>(ix->dev, d_rows, n_rows, d_pos);
    if (cudaGetLastError() != cudaSuccess || cudaStreamSynchronize(st) != cudaSuccess) return BC_E_CUDA;
    return BC_OK;
}

extern "C" int bc_last_stats(const bc_index *ix, uint64_t *out16) {
    if (!ix || !out16) return BC_E_INVAL;
    for (int i = 0; i < 16; ++i) out16[i] = ix->stats[i];
    return BC_OK;
}

extern "C" int bc_set_geometry(bc_index *ix, uint32_t ctas_per_sm, uint32_t warps_per_cta) {
    if (!ix || warps_per_cta > 8 || ctas_per_sm > 8) return BC_E_INVAL;
    ix->ctas_per_sm = ctas_per_sm;
    ix->warps_per_cta = warps_per_cta;
    return BC_OK;
}

extern "C" int bc_set_index_layout(int choice) {
    if (choice < 0 || choice > 2) return BC_E_INVAL;
    g_layout_choice = choice;
    return BC_OK;
}

extern "C" int bc_set_tuning(bc_index *ix, uint32_t spill_blocks, uint32_t pool_kb, uint32_t ld_policy) {
    if (!ix || spill_blocks > 65536 || (pool_kb != 0 && (pool_kb < 16 || pool_kb > 220)) || (ld_policy & 255u) > 2 || ld_policy > 511u)
        return BC_E_INVAL;
    ix->spill_blocks = spill_blocks;
    ix->pool_kb = pool_kb;
    ix->ld_policy = ld_policy & 255u;
    ix->no_exchange = (ld_policy >> 8) & 1u;
    return BC_OK;
}

extern "C" const char *bc_strerror(int s) {
    switch (s) {
        case BC_OK: return "ok";
        case BC_E_INVAL: return "invalid argument";
        case BC_E_NOMEM: return "caller-provided buffer too small";
        case BC_E_CUDA: return "CUDA error";
        case BC_E_OVERFLOW: return "hit arena or hits_capacity too small (see n_hits_needed)";
        case BC_E_UNSUPPORTED: return "unsupported";
        default: return "unknown status";
    }
}
