// bc_measure_random_sectors: the measured denominator of the metric "Occ lookups/s vs the
// random-sector roofline".  Every thread issues independent, uniformly random,
// 32-byte-aligned 256-bit loads (the access a rank query makes: one index block = one sector) over a
// caller-provided table; the kernel is timed with CUDA events on the caller's stream.  A table far
// larger than the 126 MB L2 gives the HBM random-sector rate, a table that fits L2 the on-chip one.
#include "bc_internal.cuh"

namespace {

__device__ __forceinline__ uint64_t mix64(uint64_t x) {
    x += 0x9E3779B97F4A7C15ull;
    x = (x ^ (x >> 30)) * 0xBF58476D1CE4E5B9ull;
    x = (x ^ (x >> 27)) * 0x94D049BB133111EBull;
    return x ^ (x >> 31);
}

template <int LD>
__global__ void __launch_bounds__(256) bc_random_sector_kernel(const uint4 *table, uint64_t n_sectors, uint32_t iters,
                                                               uint32_t *sink) {
    const uint64_t tid = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    uint32_t acc = 0;
    uint64_t h = mix64(tid);
    for (uint32_t i = 0; i < iters; i += 4) {
        uint32_t v[4][8];
#pragma unroll
        for (int u = 0; u < 4; ++u) {                    // four independent loads in flight per thread
            h = mix64(h + u);
            const uint4 *q = table + __umul64hi(h, n_sectors) * 2;   // uniform in [0, n_sectors) without a 64-bit division
            if (LD == 1)      // the search kernel's default policy: no L1 allocation, 64-byte L2 prefetch size
                asm volatile("ld.global.nc.L1::no_allocate.L2::64B.v8.u32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                             : "=r"(v[u][0]), "=r"(v[u][1]), "=r"(v[u][2]), "=r"(v[u][3]), "=r"(v[u][4]), "=r"(v[u][5]),
                               "=r"(v[u][6]), "=r"(v[u][7])
                             : "l"(q));
            else
                asm volatile("ld.global.nc.v8.u32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                             : "=r"(v[u][0]), "=r"(v[u][1]), "=r"(v[u][2]), "=r"(v[u][3]), "=r"(v[u][4]), "=r"(v[u][5]),
                               "=r"(v[u][6]), "=r"(v[u][7])
                             : "l"(q));
        }
#pragma unroll
        for (int u = 0; u < 4; ++u)
#pragma unroll
            for (int w = 0; w < 8; ++w) acc ^= v[u][w];
    }
    if (acc == 0x9E3779B9u) sink[0] = acc;               // keeps the loads alive; practically never taken
}

}  // namespace

extern "C" int bc_measure_random_sectors2(const void *d_table, size_t table_bytes, uint32_t loads_per_thread,
                                          int ld_policy, void *d_sink, void *cuda_stream, double *sectors_per_second) {
    if (ld_policy < 0 || ld_policy > 1) return BC_E_INVAL;
    if (!d_table || ((uintptr_t)d_table & 31) || table_bytes < 64 || !d_sink || !sectors_per_second ||
        loads_per_thread < 4)
        return BC_E_INVAL;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess)
        return BC_E_CUDA;
    const uint32_t iters = loads_per_thread & ~3u;
    const unsigned grid = (unsigned)sms * 8u;            // 8 CTAs x 256 threads = 64 warps per SM
    cudaEvent_t e0, e1;
    if (cudaEventCreate(&e0) != cudaSuccess) return BC_E_CUDA;
    if (cudaEventCreate(&e1) != cudaSuccess) { cudaEventDestroy(e0); return BC_E_CUDA; }
    const uint64_t n_sectors = table_bytes / 32;
    if (ld_policy == 1) {
        bc_random_sector_kernel<1><<<grid, 256, 0, st>>>((const uint4 *)d_table, n_sectors, 8, (uint32_t *)d_sink);   // warm-up
        cudaEventRecord(e0, st);
        bc_random_sector_kernel<1><<<grid, 256, 0, st>>>((const uint4 *)d_table, n_sectors, iters, (uint32_t *)d_sink);
    } else {
        bc_random_sector_kernel<0><<<grid, 256, 0, st>>>((const uint4 *)d_table, n_sectors, 8, (uint32_t *)d_sink);   // warm-up
        cudaEventRecord(e0, st);
        bc_random_sector_kernel<0><<<grid, 256, 0, st>>>((const uint4 *)d_table, n_sectors, iters, (uint32_t *)d_sink);
    }
    cudaEventRecord(e1, st);
    float ms = 0.f;
    cudaError_t e = cudaGetLastError();
    if (e == cudaSuccess) e = cudaEventSynchronize(e1);
    if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    if (e != cudaSuccess || ms <= 0.f) { cudaGetLastError(); return BC_E_CUDA; }
    *sectors_per_second = (double)grid * 256.0 * iters / (ms * 1e-3);
    return BC_OK;
}

extern "C" int bc_measure_random_sectors(const void *d_table, size_t table_bytes, uint32_t loads_per_thread,
                                         void *d_sink, void *cuda_stream, double *sectors_per_second) {
    return bc_measure_random_sectors2(d_table, table_bytes, loads_per_thread, 0, d_sink, cuda_stream, sectors_per_second);
}
