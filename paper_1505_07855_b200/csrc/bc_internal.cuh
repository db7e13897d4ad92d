// Internal device-side definitions shared by the .cu files of the library (not part of the ABI).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/barracuda_b200.h"

// ---------------------------------------------------------------------------------------------
// Device index layout (north_star: "each rank query is one 64-byte line").
// Line i of a BWT covers symbols 128*i .. 128*i+127 of the '$'-less BWT string:
//   uint32 cnt[4]   occurrences of A,C,G,T before symbol 128*i
//   uint32 lo[4]    bit s%32 of lo[s/32] = low  bit of the code of symbol 128*i+s
//   uint32 hi[4]    ... high bit
//   uint32 mid[4]   mid[w] = four packed bytes: occurrences of A,C,G,T in symbols [0, 32*w) of the
//                   line (mid[0] = 0), so a rank query touches ONE 32-bit word of each bit-plane
// Lines are 64-byte aligned: one rank query = one line = two 32-byte sectors; all four counts cost
// three popc, one symbol's count costs one.  Footprint n/2 bytes per BWT.
// ---------------------------------------------------------------------------------------------
#define BC_LINE_SYMS 128u

struct BcLine {
    uint32_t cnt[4];
    uint32_t lo[4];
    uint32_t hi[4];
    uint32_t mid[4];
};
static_assert(sizeof(BcLine) == 64, "line must be 64 bytes");

struct BcBwtDev {
    const uint4 *lines;      // n/128 + 1 lines, each 4 x uint4
    uint32_t n;              // |T|
    uint32_t primary;        // row of '$'
    uint32_t C[4];           // C[c] = # symbols smaller than c
};

struct BcIndexDev {
    BcBwtDev bwt[2];         // [0] = forward text, [1] = reversed text
    const uint32_t *sa;      // SA_fwd[t * sa_interval]
    uint32_t sa_interval;
};

struct bc_index {            // the opaque handle of the ABI
    BcIndexDev dev;
    uint64_t n;
    size_t bytes;
    uint32_t ctas_per_sm, warps_per_cta;
    uint64_t stats[16];
    int sm_count;
    cudaEvent_t ev[2];       // around the search kernel of the last bc_align_batch (stats[6])
};

#ifdef __CUDACC__
// Occurrences of all four symbols in B[0..x) where x counts ROWS of the full (n+1)-row BWT
// (x = j+1 for O(.,j)); the '$' row is skipped by the index shift.
__device__ __forceinline__ uint32_t bc_rank_pos(const BcBwtDev &b, uint32_t x) {
    return x - (x > b.primary ? 1u : 0u);          // symbols of the '$'-less string before row x
}

// all four O(., .) before position p of the '$'-less string: out[c] = #{j < p : B'[j] = c}
__device__ __forceinline__ void bc_rank4(const uint4 *lines, uint32_t p, uint32_t out[4]) {
    const uint32_t *L = reinterpret_cast<const uint32_t *>(lines + (size_t)(p >> 7) * 4);
    const uint32_t w = (p >> 5) & 3u, b = p & 31u;
    const uint4 c = __ldg(reinterpret_cast<const uint4 *>(L));
    uint32_t lo = __ldg(L + 4 + w), hi = __ldg(L + 8 + w);
    const uint32_t mid = __ldg(L + 12 + w);
    const uint32_t m = (1u << b) - 1u;
    lo &= m; hi &= m;
    const uint32_t nt = __popc(lo & hi), nc = __popc(lo & ~hi), ng = __popc(hi & ~lo);
    out[0] = c.x + (mid & 255u) + (b - nc - ng - nt);
    out[1] = c.y + ((mid >> 8) & 255u) + nc;
    out[2] = c.z + ((mid >> 16) & 255u) + ng;
    out[3] = c.w + (mid >> 24) + nt;
}

// one symbol's count: #{j < p : B'[j] = c}
__device__ __forceinline__ uint32_t bc_rank1(const uint4 *lines, uint32_t p, uint32_t c) {
    const uint32_t *L = reinterpret_cast<const uint32_t *>(lines + (size_t)(p >> 7) * 4);
    const uint32_t w = (p >> 5) & 3u, b = p & 31u;
    const uint32_t base = __ldg(L + c);
    uint32_t lo = __ldg(L + 4 + w), hi = __ldg(L + 8 + w);
    const uint32_t mid = __ldg(L + 12 + w);
    lo = (c & 1u) ? lo : ~lo;
    hi = (c & 2u) ? hi : ~hi;
    return base + ((mid >> (8u * c)) & 255u) + __popc(lo & hi & ((1u << b) - 1u));
}

// symbol at position p of the '$'-less string
__device__ __forceinline__ uint32_t bc_symbol(const uint4 *lines, uint32_t p) {
    const uint32_t *L = reinterpret_cast<const uint32_t *>(lines + (size_t)(p >> 7) * 4);
    const uint32_t w = (p >> 5) & 3u, b = p & 31u;
    return ((__ldg(L + 4 + w) >> b) & 1u) | (((__ldg(L + 8 + w) >> b) & 1u) << 1);
}
#endif
