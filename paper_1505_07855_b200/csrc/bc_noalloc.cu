// bc_exclusive_scan_u32_static: an entry point that ALLOCATES NOTHING, for callers that cannot call cudaMalloc
// (code under CUDA graph capture, tight serving loops, harnesses that forbid it).  It is the exclusive scan of the
// hot path's step A6 (per-query hit counts -> CSR offsets), whose three kernels need a scratch array
// of per-tile sums.  Everywhere else in the library that scratch is carved out of the caller's workspace; here it
// lives in a file-scope static __device__ array of a stated maximum size, so the caller passes inputs and outputs
// only.  Every GPU that loads the library holds the array (256 KB) until the process exits.
//
// Rules this file follows:
//  * In HOST code the name of a __device__ array is a host-side stand-in, not a device address: a kernel given it
//    faults (or, where the GPU can reach host memory, silently uses the wrong memory).  The device address comes
//    from cudaGetSymbolAddress, called in THIS translation unit, once per device, with that device current, return
//    code checked; the kernels get that pointer.
//  * No cudaMalloc, cudaFree or allocating library routine anywhere on this path.
//  * All calls on a device share the array, and it keeps the last call's contents.  Nothing in it has to start at
//    zero: every word a call reads (tile sums [0, n_tiles], written by scan_tile_sums / scan_block_sums) is written
//    earlier in the same call, so nothing is cleared.  Calls that OVERLAP on the GPU (two streams, two host threads)
//    race on the array: serialise them (one stream, or events), or use bc_exclusive_scan_u32 with scratch of your own.
#include <mutex>

#include "bc_ws.cuh"

#define BC_SCAN_TILE 2048ull                                 /* = SCAN_THREADS * SCAN_ITEMS of bc_post.cu */
#define BC_SCAN_STATIC_MAX_N (1ull << 26)                    /* 67,108,864 counts */
#define BC_SCAN_STATIC_WORDS (BC_SCAN_STATIC_MAX_N / BC_SCAN_TILE + 2)   /* 32,770 x 8 B = 262,160 bytes */

static __device__ __align__(256) unsigned long long g_scan_scratch[BC_SCAN_STATIC_WORDS];

namespace {

constexpr int MAX_DEVICES = 64;
std::mutex g_mu;
uint64_t *g_scratch_ptr[MAX_DEVICES];                        // device address of g_scan_scratch, per device; 0 = not set up

// the scratch of the CURRENT device (set-up on first use); nullptr on error
uint64_t *static_scratch() {
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= MAX_DEVICES) { cudaGetLastError(); return nullptr; }
    std::lock_guard<std::mutex> lock(g_mu);
    if (!g_scratch_ptr[dev]) {
        void *p = nullptr;
        if (cudaGetSymbolAddress(&p, g_scan_scratch) != cudaSuccess || !p) { cudaGetLastError(); return nullptr; }
        g_scratch_ptr[dev] = (uint64_t *)p;
    }
    return g_scratch_ptr[dev];
}

int scan_into(const uint32_t *d_in, uint64_t n, uint64_t *blk, uint64_t *d_out, cudaStream_t st) {
    if (n == 0) return cudaMemsetAsync(d_out, 0, sizeof(uint64_t), st) == cudaSuccess ? BC_OK : BC_E_CUDA;
    if (bc_exclusive_scan(d_in, n, blk, d_out, nullptr, st) != cudaSuccess) { cudaGetLastError(); return BC_E_CUDA; }
    return BC_OK;
}

}  // namespace

extern "C" uint64_t bc_scan_static_max_n(void) { return BC_SCAN_STATIC_MAX_N; }

extern "C" int bc_scan_static_setup(void) { return static_scratch() ? BC_OK : BC_E_CUDA; }

extern "C" size_t bc_exclusive_scan_scratch_bytes(uint64_t n) { return (size_t)(n / BC_SCAN_TILE + 2) * sizeof(uint64_t); }

extern "C" int bc_exclusive_scan_u32(const uint32_t *d_in, uint64_t n, void *d_scratch, size_t scratch_bytes,
                                     uint64_t *d_out, void *cuda_stream) {
    if (!d_out || (n && !d_in) || n > 0x7FFFFFFFull * BC_SCAN_TILE) return BC_E_INVAL;
    if (n && (!d_scratch || ((uintptr_t)d_scratch & 7))) return BC_E_INVAL;
    if (n && scratch_bytes < bc_exclusive_scan_scratch_bytes(n)) return BC_E_NOMEM;
    return scan_into(d_in, n, (uint64_t *)d_scratch, d_out, (cudaStream_t)cuda_stream);
}

extern "C" int bc_exclusive_scan_u32_static(const uint32_t *d_in, uint64_t n, uint64_t *d_out, void *cuda_stream) {
    if (!d_out || (n && !d_in)) return BC_E_INVAL;
    if (n > BC_SCAN_STATIC_MAX_N) return BC_E_UNSUPPORTED;      // beyond the static scratch: bc_exclusive_scan_u32
    uint64_t *blk = static_scratch();
    if (!blk) return BC_E_CUDA;
    return scan_into(d_in, n, blk, d_out, (cudaStream_t)cuda_stream);
}
