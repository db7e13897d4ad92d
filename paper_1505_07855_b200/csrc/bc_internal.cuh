// Internal device-side definitions shared by the .cu files of the library (not part of the ABI).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/barracuda_b200.h"

// ---------------------------------------------------------------------------------------------
// Device index layouts (north_star: "each rank query is one 64-byte line").  The '$'-less BWT
// string is stored as bit-planes (lo / hi bit of the 2-bit codes) with occurrence counts in front, in one of two
// layouts chosen at upload by the index size (bc_index_upload; an autotuner gene):
//
// LAY 0 -- 32-byte BLOCKS of 64 symbols (index up to 64 MB: it lives in L2, the kernel is issue-bound):
//   uint32 cnt[4] (A,C,G,T before symbol 64*i) | uint64 lo | uint64 hi.  A rank query O(.,j) = ONE 256-bit load
//   (LDG.E.256, one 32-byte sector): all four counts cost three 64-bit popc, one symbol's count one.
//   Footprint n/2 bytes per BWT.
//
// LAY 1 -- 128-byte LINES of 384 symbols (index beyond L2).  Measured on B200: a missing 32-byte sector costs the
//   WHOLE 128-byte line in DRAM (profiles/r02_random_line_ncu.md), so the line is made the unit of the layout:
//   sector 0: uint32 cnt[4] before symbol 384*i | uint16 s1[4] (counts in symbols 0..127) | uint16 s2[4] (0..255)
//   sector 1+g, g = 0..2 ("region" of 128 symbols): uint64 lo0 | hi0 | lo1 | hi1
//   A rank query = TWO 256-bit loads from ONE line (header + region) and at most two 64-bit words per plane to
//   count.  Footprint n/3 bytes per BWT (a third less: more of it stays in L2), and both ends of an interval
//   share their loads up to 128 rows apart instead of 64.
// (Round-1 history: 192-symbol lines with 64-bit planes were ALU-bound, 128-symbol lines read with four narrow
// loads were L1-request-bound; profiles/r01_*.)
// ---------------------------------------------------------------------------------------------
#define BC_BLOCK_SYMS 64u
#define BC_LINE_SYMS 384u

struct BcBlock {
    uint32_t cnt[4];
    uint32_t lo[2];
    uint32_t hi[2];
};
static_assert(sizeof(BcBlock) == 32, "block must be 32 bytes");

struct BcBwtDev {
    const uint4 *lines;      // LAY 0: n/64 + 1 blocks of 2 x uint4; LAY 1: n/384 + 1 lines of 8 x uint4
    uint32_t layout;         // 0 or 1 (above)
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
    uint32_t ctas_per_sm, warps_per_cta;   // 0 = chosen by the library (bc_set_geometry)
    uint32_t spill_blocks;   // per-warp spill area of the branch rings, blocks of 32 states (bc_set_tuning)
    uint32_t pool_kb;        // shared memory per SM given to the state pools, 0 = by index size (bc_set_tuning)
    uint32_t ld_policy;      // cache policy of the index loads: 0 = library default, 1..2 = LD 0..1 of bc_ld256
    uint32_t no_exchange;    // 1 = warps keep their states to themselves (bc_set_tuning ld_policy bit 8: A/B measurements)
    uint64_t stats[16];
    int sm_count;
    cudaEvent_t ev[2];       // around the search kernel of the last bc_align_batch (stats[6])
    uint64_t *h_ctr;         // pinned host copy of the device counter block (one D2H per call)
};

#ifdef __CUDACC__
// Occurrences of all four symbols in B[0..x) where x counts ROWS of the full (n+1)-row BWT
// (x = j+1 for O(.,j)); the '$' row is skipped by the index shift.
__device__ __forceinline__ uint32_t bc_rank_pos(const BcBwtDev &b, uint32_t x) {
    return x - (x > b.primary ? 1u : 0u);          // symbols of the '$'-less string before row x
}

// one 256-bit read-only load with one of two cache policies (bc_set_tuning; the default is the autotuner's result,
// profiles/r02_autotune_*):
//   LD = 0  default policies
//   LD = 1  no L1 allocation, 64-byte L2 prefetch size (index lines hit L1 9 % of the time; not allocating them
//           leaves L1 to the query records: -9 % time on config 2, -3..5 % on config 4)
template <int LD>
__device__ __forceinline__ void bc_ld256(const uint4 *q, uint32_t (&v)[8]) {
    if (LD == 1)
        asm("ld.global.nc.L1::no_allocate.L2::64B.v8.u32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
            : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]) : "l"(q));
    else
        asm("ld.global.nc.v8.u32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
            : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]) : "l"(q));
}

// A loaded RANK UNIT: what one rank query reads.  Positions with the same bc_unit_id are answered from the same
// loaded unit (both ends of a narrow interval usually are).
template <int LAY> struct BcUnit;
template <> struct BcUnit<0> { uint32_t c0, c1, c2, c3; uint64_t lo, hi; };                  // one 32-byte block
template <> struct BcUnit<1> { uint32_t c0, c1, c2, c3; uint64_t lo0, hi0, lo1, hi1; };      // counts up to the region + its 128 symbols

template <int LAY> __device__ __forceinline__ uint32_t bc_unit_id(uint32_t p) { return LAY == 0 ? p >> 6 : p >> 7; }
template <int LAY> __device__ __forceinline__ uint32_t bc_unit_sectors() { return LAY == 0 ? 1u : 2u; }

template <int LAY, int LD>
__device__ __forceinline__ BcUnit<LAY> bc_load_unit(const uint4 *lines, uint32_t p);

template <>
__device__ __forceinline__ BcUnit<0> bc_load_unit<0, 0>(const uint4 *lines, uint32_t p) {
    uint32_t v[8];
    bc_ld256<0>(lines + (size_t)(p >> 6) * 2, v);
    BcUnit<0> u; u.c0 = v[0]; u.c1 = v[1]; u.c2 = v[2]; u.c3 = v[3];
    u.lo = ((uint64_t)v[5] << 32) | v[4]; u.hi = ((uint64_t)v[7] << 32) | v[6];
    return u;
}
template <>
__device__ __forceinline__ BcUnit<0> bc_load_unit<0, 1>(const uint4 *lines, uint32_t p) {
    uint32_t v[8];
    bc_ld256<1>(lines + (size_t)(p >> 6) * 2, v);
    BcUnit<0> u; u.c0 = v[0]; u.c1 = v[1]; u.c2 = v[2]; u.c3 = v[3];
    u.lo = ((uint64_t)v[5] << 32) | v[4]; u.hi = ((uint64_t)v[7] << 32) | v[6];
    return u;
}
template <int LD>
__device__ __forceinline__ BcUnit<1> bc_load_line(const uint4 *lines, uint32_t p) {
    const uint32_t q = p >> 7, b = __umulhi(q, 0xAAAAAAABu) >> 1, g = q - 3u * b;     // line b, region g = 0..2
    const uint4 *L = lines + (size_t)b * 8;
    uint32_t h[8], r[8];
    bc_ld256<LD>(L, h);
    bc_ld256<LD>(L + 2 + 2 * g, r);
    const uint32_t sa = g == 1u ? h[4] : h[6], sb = g == 1u ? h[5] : h[7];              // s1 or s2, two uint16 per word
    BcUnit<1> u;
    u.c0 = h[0] + (g ? (sa & 0xFFFFu) : 0u); u.c1 = h[1] + (g ? (sa >> 16) : 0u);
    u.c2 = h[2] + (g ? (sb & 0xFFFFu) : 0u); u.c3 = h[3] + (g ? (sb >> 16) : 0u);
    u.lo0 = ((uint64_t)r[1] << 32) | r[0]; u.hi0 = ((uint64_t)r[3] << 32) | r[2];
    u.lo1 = ((uint64_t)r[5] << 32) | r[4]; u.hi1 = ((uint64_t)r[7] << 32) | r[6];
    return u;
}
template <> __device__ __forceinline__ BcUnit<1> bc_load_unit<1, 0>(const uint4 *lines, uint32_t p) { return bc_load_line<0>(lines, p); }
template <> __device__ __forceinline__ BcUnit<1> bc_load_unit<1, 1>(const uint4 *lines, uint32_t p) { return bc_load_line<1>(lines, p); }

// all four counts from a loaded unit: out[c] = #{j < p : B'[j] = c}
__device__ __forceinline__ void bc_unit_rank4(const BcUnit<0> &r, uint32_t p, uint32_t out[4]) {
    const uint32_t b = p & 63u;
    const uint64_t m = (1ull << b) - 1ull;
    const uint64_t lo = r.lo & m, hi = r.hi & m;
    const uint32_t nt = __popcll(lo & hi), nc = __popcll(lo & ~hi), ng = __popcll(hi & ~lo);
    out[0] = r.c0 + (b - nc - ng - nt);
    out[1] = r.c1 + nc;
    out[2] = r.c2 + ng;
    out[3] = r.c3 + nt;
}
__device__ __forceinline__ void bc_unit_rank4(const BcUnit<1> &r, uint32_t p, uint32_t out[4]) {
    const uint32_t rr = p & 127u, b = rr & 63u;
    const uint64_t lowm = (1ull << b) - 1ull;
    const uint64_t m0 = rr >= 64u ? ~0ull : lowm, m1 = rr >= 64u ? lowm : 0ull;
    const uint64_t l0 = r.lo0 & m0, h0 = r.hi0 & m0, l1 = r.lo1 & m1, h1 = r.hi1 & m1;
    const uint32_t nt = __popcll(l0 & h0) + __popcll(l1 & h1), nc = __popcll(l0 & ~h0) + __popcll(l1 & ~h1),
                   ng = __popcll(h0 & ~l0) + __popcll(h1 & ~l1);
    out[0] = r.c0 + (rr - nc - ng - nt);
    out[1] = r.c1 + nc;
    out[2] = r.c2 + ng;
    out[3] = r.c3 + nt;
}

// one symbol's count from a loaded unit: #{j < p : B'[j] = c}  (c > 3 gives a don't-care value)
__device__ __forceinline__ uint32_t bc_unit_rank1(const BcUnit<0> &r, uint32_t p, uint32_t c) {
    const uint32_t b = p & 63u;
    const uint64_t lo = (c & 1u) ? r.lo : ~r.lo, hi = (c & 2u) ? r.hi : ~r.hi;
    const uint32_t base = (c & 2u) ? ((c & 1u) ? r.c3 : r.c2) : ((c & 1u) ? r.c1 : r.c0);
    return base + __popcll(lo & hi & ((1ull << b) - 1ull));
}
__device__ __forceinline__ uint32_t bc_unit_rank1(const BcUnit<1> &r, uint32_t p, uint32_t c) {
    const uint32_t rr = p & 127u, b = rr & 63u;
    const uint64_t lowm = (1ull << b) - 1ull;
    const uint64_t m0 = rr >= 64u ? ~0ull : lowm, m1 = rr >= 64u ? lowm : 0ull;
    const uint64_t xl = (c & 1u) ? 0ull : ~0ull, xh = (c & 2u) ? 0ull : ~0ull;
    const uint32_t base = (c & 2u) ? ((c & 1u) ? r.c3 : r.c2) : ((c & 1u) ? r.c1 : r.c0);
    return base + __popcll((r.lo0 ^ xl) & (r.hi0 ^ xh) & m0) + __popcll((r.lo1 ^ xl) & (r.hi1 ^ xh) & m1);
}

// symbol at position p (must lie in the unit)
__device__ __forceinline__ uint32_t bc_unit_symbol(const BcUnit<0> &r, uint32_t p) {
    const uint32_t b = p & 63u;
    return (uint32_t)((r.lo >> b) & 1ull) | ((uint32_t)((r.hi >> b) & 1ull) << 1);
}
__device__ __forceinline__ uint32_t bc_unit_symbol(const BcUnit<1> &r, uint32_t p) {
    const uint32_t rr = p & 127u, b = rr & 63u;
    const uint64_t lo = rr >= 64u ? r.lo1 : r.lo0, hi = rr >= 64u ? r.hi1 : r.hi0;
    return (uint32_t)((lo >> b) & 1ull) | ((uint32_t)((hi >> b) & 1ull) << 1);
}

// one symbol's count: #{j < p : B'[j] = c}  (helpers outside the search kernel; default cache policy)
template <int LAY>
__device__ __forceinline__ uint32_t bc_rank1(const uint4 *lines, uint32_t p, uint32_t c) {
    return bc_unit_rank1(bc_load_unit<LAY, 0>(lines, p), p, c);
}
#endif
