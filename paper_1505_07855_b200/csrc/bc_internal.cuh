// Internal device-side definitions shared by the .cu files of the library (not part of the ABI).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/barracuda_b200.h"

// ---------------------------------------------------------------------------------------------
// Device index layout (north_star: "each rank query is one 64-byte line").
// The '$'-less BWT string is cut into 32-byte BLOCKS of 64 symbols; two blocks share a 64-byte line:
//   uint32 cnt[4]   occurrences of A,C,G,T before symbol 64*i
//   uint32 lo[2]    bit s of the 64-bit word lo = low  bit of the code of symbol 64*i+s
//   uint32 hi[2]    ... high bit
// A rank query O(.,j) reads ONE block = one aligned 32-byte sector with ONE 256-bit load
// (LDG.E.256), i.e. half a line: all four counts cost three 64-bit popc, one symbol's count one.
// Footprint n/2 bytes per BWT.  (Round-1 history: 192-symbol lines with 64-bit planes were ALU-bound,
// 128-symbol lines read with four narrow loads were L1-request-bound; profiles/r01_*.)
// ---------------------------------------------------------------------------------------------
#define BC_BLOCK_SYMS 64u

struct BcBlock {
    uint32_t cnt[4];
    uint32_t lo[2];
    uint32_t hi[2];
};
static_assert(sizeof(BcBlock) == 32, "block must be 32 bytes");

struct BcBwtDev {
    const uint4 *lines;      // n/64 + 1 blocks of 2 x uint4 (32-byte aligned)
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
    uint32_t ld_policy;      // cache policy of the index loads: 0 = library default, 1..3 = LD 0..2 of bc_load_block
    uint32_t wide_shift;     // LD 2: intervals of >= n >> wide_shift rows count as the top of the trees (0 = 16)
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

struct BcBlockRegs { uint32_t c0, c1, c2, c3; uint64_t lo, hi; };

// The one load that carries the whole search, with three cache policies (bc_set_tuning; the defaults are the
// autotuner's result, profiles/r02_autotune_*):
//   LD = 0  read-only path, default policies
//   LD = 1  read-only path, no L1 allocation, 64-byte L2 prefetch size (index lines hit L1 9 % of the time; not
//           allocating them leaves L1 to the query records: -9 % time on config 2, -3..5 % on config 4)
//   LD = 2  as 1, plus an L2 eviction priority by interval width: `wide` (the top of the search trees, which every
//           query walks) evict-last, the rest evict-first -- random deep lines turn the 126 MB L2 over every ~25 us
//           and would otherwise push the shared top levels out
// one 256-bit read-only load of the block that holds position p of the '$'-less string
template <int LD = 0>
__device__ __forceinline__ BcBlockRegs bc_load_block(const uint4 *lines, uint32_t p, bool wide = false) {
    const uint4 *q = lines + (size_t)(p >> 6) * 2;
    BcBlockRegs r;
    uint32_t l0, l1, h0, h1;
    if (LD == 2) {
        if (wide)
            asm("ld.global.nc.L1::no_allocate.L2::evict_last.L2::64B.v8.u32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                : "=r"(r.c0), "=r"(r.c1), "=r"(r.c2), "=r"(r.c3), "=r"(l0), "=r"(l1), "=r"(h0), "=r"(h1)
                : "l"(q));
        else
            asm("ld.global.nc.L1::no_allocate.L2::evict_first.L2::64B.v8.u32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                : "=r"(r.c0), "=r"(r.c1), "=r"(r.c2), "=r"(r.c3), "=r"(l0), "=r"(l1), "=r"(h0), "=r"(h1)
                : "l"(q));
    } else if (LD == 1)
        asm("ld.global.nc.L1::no_allocate.L2::64B.v8.u32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
            : "=r"(r.c0), "=r"(r.c1), "=r"(r.c2), "=r"(r.c3), "=r"(l0), "=r"(l1), "=r"(h0), "=r"(h1)
            : "l"(q));
    else
        asm("ld.global.nc.v8.u32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
            : "=r"(r.c0), "=r"(r.c1), "=r"(r.c2), "=r"(r.c3), "=r"(l0), "=r"(l1), "=r"(h0), "=r"(h1)
            : "l"(q));
    r.lo = ((uint64_t)l1 << 32) | l0;
    r.hi = ((uint64_t)h1 << 32) | h0;
    return r;
}

// all four counts from a loaded block: out[c] = #{j < p : B'[j] = c}
__device__ __forceinline__ void bc_block_rank4(const BcBlockRegs &r, uint32_t p, uint32_t out[4]) {
    const uint32_t b = p & 63u;
    const uint64_t m = (1ull << b) - 1ull;
    const uint64_t lo = r.lo & m, hi = r.hi & m;
    const uint32_t nt = __popcll(lo & hi), nc = __popcll(lo & ~hi), ng = __popcll(hi & ~lo);
    out[0] = r.c0 + (b - nc - ng - nt);
    out[1] = r.c1 + nc;
    out[2] = r.c2 + ng;
    out[3] = r.c3 + nt;
}

// all four O(., .) before position p of the '$'-less string
template <int LD = 0>
__device__ __forceinline__ void bc_rank4(const uint4 *lines, uint32_t p, uint32_t out[4], bool wide = false) {
    bc_block_rank4(bc_load_block<LD>(lines, p, wide), p, out);
}

// one symbol's count from a loaded block: #{j < p : B'[j] = c}  (c > 3 gives a don't-care value)
__device__ __forceinline__ uint32_t bc_block_rank1(const BcBlockRegs &r, uint32_t p, uint32_t c) {
    const uint32_t b = p & 63u;
    const uint64_t lo = (c & 1u) ? r.lo : ~r.lo, hi = (c & 2u) ? r.hi : ~r.hi;
    const uint32_t base = (c & 2u) ? ((c & 1u) ? r.c3 : r.c2) : ((c & 1u) ? r.c1 : r.c0);
    return base + __popcll(lo & hi & ((1ull << b) - 1ull));
}

// one symbol's count: #{j < p : B'[j] = c}
__device__ __forceinline__ uint32_t bc_rank1(const uint4 *lines, uint32_t p, uint32_t c) {
    return bc_block_rank1(bc_load_block(lines, p), p, c);
}

// symbol at position p of the '$'-less string
__device__ __forceinline__ uint32_t bc_symbol(const uint4 *lines, uint32_t p) {
    const uint32_t *L = reinterpret_cast<const uint32_t *>(lines + (size_t)(p >> 6) * 2);
    const uint32_t w = (p >> 5) & 1u, b = p & 31u;
    return ((__ldg(L + 4 + w) >> b) & 1u) | (((__ldg(L + 6 + w) >> b) & 1u) << 1);
}
#endif
