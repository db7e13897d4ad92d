// Workspace layout and launch interfaces between bc_align.cu (host orchestration), bc_search.cu
// (A1-A5) and bc_post.cu (A6).  Internal.
#pragma once
#include "bc_internal.cuh"

// Prepared query RECORD (one per query q = 2*read + strand, `qstride` bytes, 16-byte aligned), written by
// bc_prepare_kernel and read by the search kernel -- everything a search node needs to know about its
// query, compact enough to stay cache-resident beside an index far larger than L2:
//   [0 .. q_soff)        thrD[r], r = 0..z   (bytes): smallest t with D[t] <= r, clamped to 255
//   [q_soff .. q_boff)   thrS[r], r = 0..seed_z      : the same for Ds[] (0 when the seed is off)
//   [q_boff .. q_noff)   the query's bases, 2 bits each, base t at bits 2*(t%16) of word t/16
//                        (strand 1: already complemented), max_len/16 + 1 words
//   [q_noff .. qstride)  1 bit per base: N (only when the batch carries an N mask)
// D[t] = lower bound on the differences W[t..m-1] needs, Ds[t] the same for the unconsumed
// seed part; both never increase with t, so a budget check "D[t] <= r" is "t >= thrD[r]".  A threshold
// that is rounded DOWN (the clamp, m = 256 only) weakens the prune, never the result.
// Small budgets (z <= 7, seed_z <= 3): thrD in bytes 0-7, thrS in bytes 8-11, q_boff = 16, so that one
// 128-bit load brings every threshold into registers (BC_QREC_SMALL).
#define BC_QREC_SMALL_Z 7
#define BC_QREC_SMALL_SZ 3

enum {                      // indices into the uint64 counter block
    BC_CTR_TICKET = 0,      // next query to hand to a warp
    BC_CTR_ARENA = 1,       // raw hits produced (cursor; may exceed the capacity)
    BC_CTR_NODES = 2,
    BC_CTR_LOOKUPS = 3,
    BC_CTR_LINES = 4,
    BC_CTR_ERROR = 5,       // bit 0: bad read length, bit 1: pool overflow (must never happen), bit 2: spill area exhausted
    BC_CTR_DLOOKUPS = 6,
    BC_CTR_POOLMAX = 7,
    BC_CTR_NBIG = 8,        // queries whose raw segment is sorted by a whole CTA
    BC_CTR_TOTAL = 9,       // hits after dedup
    BC_CTR_BSTEPS = 10,     // warp-level branch steps
    BC_CTR_BNODES = 11,     // states expanded in branch steps
    BC_CTR_CSTEPS = 12,     // warp-level chain iterations
    BC_CTR_CANCEL = 13,     // branch states popped and put back because their children did not fit
    BC_CTR_SPILL = 14,      // 32-entry blocks moved from the branch rings to global memory
    BC_CTR_SPILLMAX = 15,   // deepest per-warp spill stack seen (blocks)
    BC_CTR_PASSES = 16,     // best-stratum mode: largest per-read budget searched + 1
    BC_CTR_GIDLE = 17,      // warps that are out of work (state exchange between warps)
    BC_CTR_QREADY = 18,     // donated blocks waiting in the exchange
    BC_CTR_STEALS = 19,     // blocks of 32 states that changed warps
    BC_CTR_STARTED = 20,    // warps that have started (the exchange waits for these, not for the whole grid)
    BC_CTR_COUNT = 24
};

struct BcRawHit { uint32_t qid, k, l, d; };

struct BcWorkspace {        // device pointers into the caller's workspace
    uint8_t *qz;            // [n_reads] best-stratum mode: the budget each read is being searched with
    uint8_t *qrec;          // [nq][qstride] prepared query records (layout above)
    uint32_t qstride, q_soff, q_boff, q_noff;
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
    uint32_t *sq_flag;      // [sq_n] state exchange between warps: slot states (zeroed per call)
    uint2 *sq_buf;          // [sq_n][32 entries][3]
    uint32_t sq_n;          // slots (multiple of 32; 0 = exchange off)
    uint32_t nq;
};

struct BcSearchParams {
    BcIndexDev ix;
    bc_reads reads;
    bc_opts o;
    BcWorkspace ws;
    uint32_t bcap;          // branch ring entries per warp (power of two)
    uint32_t ccap;          // run stack entries per warp (both strands)
    uint32_t best, plus;    // best-stratum mode (bc_align_batch_best): per read only the hits with d <= min(d_min + plus, z)
    uint32_t ld_policy;     // LD of bc_ld256: cache policy of the index loads
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
#define BC_STEAL_SLOTS 256u           // blocks in flight between warps (768 B each)
#define BC_SPILL_BLOCKS 128u          // per warp: 128 x 32 entries x 24 B = 96 KB of workspace
