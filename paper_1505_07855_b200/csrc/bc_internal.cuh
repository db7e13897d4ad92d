// Internal device-side definitions shared by the .cu files of the library (not part of the ABI).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/barracuda_b200.h"

// ---------------------------------------------------------------------------------------------
// Device index layout (north_star: "each rank query is one 64-byte line").
// Line i of a BWT covers symbols 192*i .. 192*i+191 of the '$'-less BWT string:
//   uint32 cnt[4]   occurrences of A,C,G,T before symbol 192*i
//   uint64 lo[3]    bit s%64 of lo[s/64] = low  bit of the code of symbol 192*i+s
//   uint64 hi[3]    ... high bit
// Lines are 64-byte aligned, so one rank query = one line = two 32-byte DRAM sectors.
// ---------------------------------------------------------------------------------------------
#define BC_LINE_SYMS 192u

struct BcLine {
    uint32_t cnt[4];
    uint64_t lo[3];
    uint64_t hi[3];
};
static_assert(sizeof(BcLine) == 64, "line must be 64 bytes");

struct BcBwtDev {
    const uint4 *lines;      // n/192 + 1 lines, each 4 x uint4
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
    uint64_t stats[8];
    int sm_count;
    cudaEvent_t ev[2];       // around the search kernel of the last bc_align_batch (stats[6])
};

#ifdef __CUDACC__
// Occurrences of all four symbols in B[0..x) where x counts ROWS of the full (n+1)-row BWT
// (x = j+1 for O(.,j)); the '$' row is skipped by the index shift.
// `line_id` of the line the query falls in is returned so callers can detect shared lines.
__device__ __forceinline__ uint32_t bc_rank_pos(const BcBwtDev &b, uint32_t x) {
    return x - (x > b.primary ? 1u : 0u);          // symbols of the '$'-less string before row x
}

struct BcLineRegs { uint4 a, b, c, d; };

__device__ __forceinline__ BcLineRegs bc_load_line(const uint4 *lines, uint32_t line_id) {
    const uint4 *p = lines + (size_t)line_id * 4;
    BcLineRegs r;
    r.a = __ldg(p); r.b = __ldg(p + 1); r.c = __ldg(p + 2); r.d = __ldg(p + 3);
    return r;
}

// counts of A,C,G,T in the first r (0..191) symbols of the line, added to the line's checkpoint
__device__ __forceinline__ void bc_line_rank4(const BcLineRegs &L, uint32_t r, uint32_t out[4]) {
    const uint64_t lo[3] = {((uint64_t)L.b.y << 32) | L.b.x, ((uint64_t)L.b.w << 32) | L.b.z,
                            ((uint64_t)L.c.y << 32) | L.c.x};
    const uint64_t hi[3] = {((uint64_t)L.c.w << 32) | L.c.z, ((uint64_t)L.d.y << 32) | L.d.x,
                            ((uint64_t)L.d.w << 32) | L.d.z};
    uint32_t nc = 0, ng = 0, nt = 0;
#pragma unroll
    for (int w = 0; w < 3; ++w) {
        int nb = (int)r - 64 * w;
        uint64_t m = nb >= 64 ? ~0ull : (nb <= 0 ? 0ull : ((1ull << nb) - 1ull));
        uint64_t l = lo[w] & m, h = hi[w] & m;
        nt += __popcll(l & h);
        nc += __popcll(l & ~h);
        ng += __popcll(h & ~l);
    }
    out[0] = L.a.x + (r - nc - ng - nt);
    out[1] = L.a.y + nc;
    out[2] = L.a.z + ng;
    out[3] = L.a.w + nt;
}

// symbol s (0..191) of the line
__device__ __forceinline__ uint32_t bc_line_symbol(const BcLineRegs &L, uint32_t s) {
    const uint32_t lo[6] = {L.b.x, L.b.y, L.b.z, L.b.w, L.c.x, L.c.y};
    const uint32_t hi[6] = {L.c.z, L.c.w, L.d.x, L.d.y, L.d.z, L.d.w};
    uint32_t w = s >> 5, bit = s & 31, l = 0, h = 0;
#pragma unroll
    for (int i = 0; i < 6; ++i) if (w == (uint32_t)i) { l = lo[i]; h = hi[i]; }
    return ((l >> bit) & 1u) | (((h >> bit) & 1u) << 1);
}
#endif
