// Workspace layout and launch interfaces between bc_align.cu (host orchestration), bc_search.cu
// (A1-A5) and bc_post.cu (A6).  Internal.
#pragma once
#include "bc_internal.cuh"

// prepared query entry (uint16) for consumption step t of query q = 2*read + strand:
//   bits 0-2  base consumed at step t (strand 1: complemented), 4 = N
//   bits 3-8  D[t]  = lower bound on differences needed for W[t..m-1], clamped to 63
//   bits 9-14 Ds[t] = same for the unconsumed seed part W[t..seed_len-1] (0 outside the seed)
#define BC_PREP_BASE(p) ((p) & 7u)
#define BC_PREP_D(p) (((p) >> 3) & 63u)
#define BC_PREP_DS(p) (((p) >> 9) & 63u)

enum {                      // indices into the uint64 counter block
    BC_CTR_TICKET = 0,      // next query to hand to a warp
    BC_CTR_ARENA = 1,       // raw hits produced (cursor; may exceed the capacity)
    BC_CTR_NODES = 2,
    BC_CTR_LOOKUPS = 3,
    BC_CTR_LINES = 4,
    BC_CTR_ERROR = 5,       // bit 0: bad read length, bit 1: pool overflow (must never happen)
    BC_CTR_DLOOKUPS = 6,
    BC_CTR_POOLMAX = 7,
    BC_CTR_NBIG = 8,        // queries whose raw segment is sorted by a whole CTA
    BC_CTR_TOTAL = 9,       // hits after dedup
    BC_CTR_BSTEPS = 10,     // warp-level branch steps
    BC_CTR_BNODES = 11,     // states expanded in branch steps
    BC_CTR_CSTEPS = 12,     // warp-level chain iterations
    BC_CTR_CANCEL = 13,     // branch states popped and put back because their children did not fit
    BC_CTR_SPILL = 14,      // 32-entry blocks moved from the branch rings to global memory
    BC_CTR_COUNT = 16
};

struct BcRawHit { uint32_t qid, k, l, d; };

struct BcWorkspace {        // device pointers into the caller's workspace
    uint16_t *prep;         // [nq][stride]
    uint32_t stride;
    uint32_t *qcnt;         // [nq] raw hits per query
    uint32_t *qfill;        // [nq] scatter cursors, later: unique hits per query
    uint64_t *seg_off;      // [nq+1] exclusive scan of qcnt
    uint64_t *uoff;         // [nq+1] exclusive scan of unique counts
    uint64_t *blk;          // scan block sums
    uint32_t *big;          // [nq] list of big segments
    uint64_t *ctr;          // [BC_CTR_COUNT]
    BcRawHit *arena;        // [arena_cap]
    uint64_t *seg_key;      // [arena_cap] (k<<32 | l), grouped by query
    uint32_t *seg_d;        // [arena_cap]
    uint64_t arena_cap;
    uint2 *spill;           // [warps in the grid][spill_blocks][32 entries][3] overflow of the branch rings
    uint32_t spill_blocks;  // blocks of 32 entries per warp
    uint32_t nq;
};

struct BcSearchParams {
    BcIndexDev ix;
    bc_reads reads;
    bc_opts o;
    BcWorkspace ws;
    uint32_t bcap;          // branch ring entries per warp (power of two)
    uint32_t ccap;          // chain stack entries per warp
};

// launchers (return cudaError_t of the launch)
cudaError_t bc_launch_prepare(const BcSearchParams &p, cudaStream_t st);
cudaError_t bc_launch_search(const BcSearchParams &p, int sm_count, uint32_t ctas_per_sm, uint32_t warps_per_cta,
                             cudaStream_t st);
cudaError_t bc_launch_post(const BcSearchParams &p, bc_result res, cudaStream_t st);
cudaError_t bc_exclusive_scan(const uint32_t *in, uint64_t n, uint64_t *blk, uint64_t *out, uint64_t *total_out,
                              cudaStream_t st);
// smem bytes one pool entry takes; used by the host to size pools
#define BC_POOL_ENTRY_BYTES 24u
#define BC_SPILL_BLOCKS 128u          // per warp: 128 x 32 entries x 24 B = 96 KB of workspace
