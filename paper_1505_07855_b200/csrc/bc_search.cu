// A1 query preparation + A2 D[] bounds (bc_prepare_kernel), A3-A5 inexact search with per-warp
// state pools in shared memory (bc_search_kernel).  sm_100a only; integer arithmetic only.
//
// Orientation: BOTH strands consume the read 5'->3' (step t consumes W[t]),
// so that the seed, with its tighter limit, bounds the fully-branching top of the tree:
//   strand 1 (query revcomp(W)): prepending comp(W[t]) on the FORWARD index; [k, k+s-1] is the hit.
//   strand 0 (query W):          prepending W[t] on the REVERSE index extends the forward string to
//                                the right; the forward interval start k2 is carried along
//                                (bidirectional extension).
// The D[] lower bound for the unconsumed part W[t..m-1] comes from the index of the opposite
// direction (strand 1: reverse index -- north_star's "D[] prune from the reverse-BWT index").
#include "bc_ws.cuh"

namespace {

__device__ __forceinline__ uint32_t read_base(const bc_reads &rd, uint64_t pos) {
    uint32_t c = (rd.bases2[pos >> 4] >> (2 * (pos & 15))) & 3u;
    if (rd.nmask && ((rd.nmask[pos >> 5] >> (pos & 31)) & 1u)) c = 4;
    return c;
}

// ---------------------------------------------------------------------------------------------
// A1 + A2: one thread per query (read, strand).  SURVEY C7 loop, in W coordinates: pieces are
// grown from W[m-1] leftwards by prepending on the opposite-direction index.
// ---------------------------------------------------------------------------------------------
__global__ void bc_prepare_kernel(BcSearchParams p) {
    uint32_t q = blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= p.ws.nq) return;
    uint32_t r = q >> 1, strand = q & 1;
    uint32_t m = p.reads.len[r];
    uint16_t *out = p.ws.prep + (size_t)q * p.ws.stride;
    if (m < 1 || m > p.reads.max_len) {
        atomicOr((unsigned long long *)&p.ws.ctr[BC_CTR_ERROR], 1ull);
        return;
    }
    uint64_t off = p.reads.off[r];
    const BcBwtDev &Y = p.ix.bwt[strand ? 1 : 0];       // opposite direction of the search index
    const uint32_t full = Y.n + 1;
    const bool seed_on = p.o.seed_len > 0 && (uint32_t)p.o.seed_len < m;
    uint64_t lookups = 0;
    // pass 1: Ds over the seed part (entries outside the seed get 0 in pass 2)
    if (seed_on) {
        uint32_t cnt = 0, k = 0, s = full;
        for (int a = p.o.seed_len - 1; a >= 0; --a) {
            uint32_t c = read_base(p.reads, off + a);
            if (c < 4 && strand) c = 3 - c;
            if (c > 3) { cnt++; k = 0; s = full; }
            else {
                uint32_t olo = bc_rank1(Y.lines, bc_rank_pos(Y, k), c), ohi = bc_rank1(Y.lines, bc_rank_pos(Y, k + s), c);
                lookups += 2;
                uint32_t s2 = ohi - olo;
                if (s2 == 0) { cnt++; k = 0; s = full; } else { k = Y.C[c] + olo + 1; s = s2; }
            }
            out[a] = (uint16_t)((cnt < 63 ? cnt : 63) << 9);
        }
    }
    // pass 2: D over the whole read + the consumed base
    {
        uint32_t cnt = 0, k = 0, s = full;
        for (int a = (int)m - 1; a >= 0; --a) {
            uint32_t c = read_base(p.reads, off + a);
            if (c < 4 && strand) c = 3 - c;
            if (c > 3) { cnt++; k = 0; s = full; }
            else {
                uint32_t olo = bc_rank1(Y.lines, bc_rank_pos(Y, k), c), ohi = bc_rank1(Y.lines, bc_rank_pos(Y, k + s), c);
                lookups += 2;
                uint32_t s2 = ohi - olo;
                if (s2 == 0) { cnt++; k = 0; s = full; } else { k = Y.C[c] + olo + 1; s = s2; }
            }
            uint32_t ds = (seed_on && a < p.o.seed_len) ? (out[a] & (63u << 9)) : 0u;
            out[a] = (uint16_t)(c | ((cnt < 63 ? cnt : 63) << 3) | ds);
        }
        out[m] = 0;
    }
    atomicAdd((unsigned long long *)&p.ws.ctr[BC_CTR_DLOOKUPS], (unsigned long long)lookups);
}

}  // namespace

cudaError_t bc_launch_prepare(const BcSearchParams &p, cudaStream_t st) {
    if (p.ws.nq == 0) return cudaSuccess;
    bc_prepare_kernel<<<(p.ws.nq + 127) / 128, 128, 0, st>>>(p);
    return cudaGetLastError();
}


namespace {

__device__ __forceinline__ uint32_t sel4(uint32_t a0, uint32_t a1, uint32_t a2, uint32_t a3, uint32_t b) {
    const uint32_t lo = (b & 1) ? a1 : a0, hi = (b & 1) ? a3 : a2;
    return (b & 2) ? hi : lo;
}

// Pool entry = 24 bytes, array-of-structures, moved with three 64-bit shared-memory accesses:
//   {qid, k} {s, k2} {mlo, mhi}
//   mlo = t (bits 0-8) | st (9-10; 0 = M, 1 = I, 2 = D) | n_go (11-18) | n_ge (19-26)
//   mhi = seed_d (0-7) | d (8-15) | m-1 (16-23);  chain entries also carry their next base in mlo bits 27-29
// Per warp: a RING of BRANCH states (budget left, d < z), whose cold bottom spills to global memory in
// blocks of 32, and a stack of CHAIN states (budget exhausted, d == z: only exact matching follows).
#ifndef BC_SEARCH_MAX_THREADS
#define BC_SEARCH_MAX_THREADS 256
#endif
#ifndef BC_SEARCH_MIN_CTAS
#define BC_SEARCH_MIN_CTAS 3
#endif

__device__ __forceinline__ void ent_store(uint2 *P, uint32_t idx, uint32_t qid, uint32_t k, uint32_t s, uint32_t k2,
                                          uint32_t mlo, uint32_t mhi) {
    uint2 *e = P + idx * 3u;
    e[0] = make_uint2(qid, k); e[1] = make_uint2(s, k2); e[2] = make_uint2(mlo, mhi);
}

// warp-aggregated append of raw hits (A5); called by all 32 lanes
__device__ __noinline__ void emit_hits(BcRawHit *arena, unsigned long long arena_cap, uint32_t *qcnt,
                                       unsigned long long *ctr, bool emit, uint32_t qid, uint32_t kf, uint32_t s, uint32_t d) {
    const uint32_t lane = threadIdx.x & 31u;
    uint32_t emask = __ballot_sync(0xffffffffu, emit);
    if (emask == 0) return;
    unsigned long long base = 0;
    int leader = __ffs(emask) - 1;
    if ((int)lane == leader) base = atomicAdd(&ctr[BC_CTR_ARENA], (unsigned long long)__popc(emask));
    base = __shfl_sync(0xffffffffu, base, leader);
    if (emit) {
        unsigned long long pos = base + __popc(emask & ((1u << lane) - 1u));
        if (pos < arena_cap) arena[pos] = BcRawHit{qid, kf, kf + s - 1u, d};
        atomicAdd(&qcnt[qid], 1u);
    }
}

// per-warp statistics: n_xsect is per lane (second sectors of a rank pair), the rest warp-uniform
__device__ __noinline__ void flush_stats(unsigned long long *ctr, uint32_t lane, uint32_t n_cnodes, uint32_t n_xsect,
                                         uint32_t n_bsteps, uint32_t n_bnodes, uint32_t n_csteps, uint32_t n_cancel,
                                         uint32_t n_spill) {
    uint32_t x = n_xsect;
    for (int o = 16; o > 0; o >>= 1) x += __shfl_down_sync(0xffffffffu, x, o);
    if (lane == 0) {
        const unsigned long long nodes = (unsigned long long)n_cnodes + n_bnodes;
        atomicAdd(&ctr[BC_CTR_NODES], nodes);
        atomicAdd(&ctr[BC_CTR_LOOKUPS], 2ull * nodes);
        atomicAdd(&ctr[BC_CTR_LINES], nodes + x);          // one sector per node + the pairs that straddle two
        atomicAdd(&ctr[BC_CTR_BSTEPS], (unsigned long long)n_bsteps);
        atomicAdd(&ctr[BC_CTR_BNODES], (unsigned long long)n_bnodes);
        atomicAdd(&ctr[BC_CTR_CSTEPS], (unsigned long long)n_csteps);
        atomicAdd(&ctr[BC_CTR_CANCEL], (unsigned long long)n_cancel);
        atomicAdd(&ctr[BC_CTR_SPILL], (unsigned long long)n_spill);
    }
}

struct SearchConsts {            // warp-uniform values the phases share; suffix = strand
    const uint4 *lines0, *lines1;   // index the strand's query is matched on (strand 0: reverse index)
    uint32_t primary0, primary1;
};

// ---------------------------------------------------------------------------------------------
// CHAIN steps (see the kernel's header comment): while the stack of strand S holds a warp's worth
// of chain states (or, when draining, anything at all), pop 32, extend each by ONE exactly matching
// base -- one symbol's rank at both interval ends -- and push the survivors back compacted.  Flat
// cost per node whatever the chain lengths; lanes are full whenever 32 states are pending.
// Strand 0 (searched on the reverse index) also advances the forward interval start k2 by the
// bidirectional update of SURVEY C7 (R): '$' + the symbols smaller than c inside the interval.
// Stack layout inside the chain area Cq[0..CCAP): strand 1 grows up from 0, strand 0 down from CCAP-1.
// ---------------------------------------------------------------------------------------------
template <bool S0>
__device__ __forceinline__ void chain_steps(const BcSearchParams &p, const uint4 *lines, uint32_t primary,
                                            const uint32_t *Cs, uint2 *Cq, uint32_t CCAP, uint32_t &cnt,
                                            bool drain, unsigned long long *ctr, uint32_t &n_nodes, uint32_t &n_xsect,
                                            uint32_t &n_steps) {
    const uint32_t lane = threadIdx.x & 31u, lt_mask = (1u << lane) - 1u;
    while (cnt >= 32u || (drain && cnt > 0u)) {
        const uint32_t a = cnt < 32u ? cnt : 32u;
        const bool act = lane < a;
        uint32_t qid = 0, k = 0, s = 0, k2 = 0, mlo = 0, mhi = 0;
        if (act) {
            const uint2 *e = Cq + (S0 ? CCAP - cnt + lane : cnt - 1u - lane) * 3u;
            const uint2 a0 = e[0], a1 = e[1], a2 = e[2];
            qid = a0.x; k = a0.y; s = a1.x; k2 = a1.y; mlo = a2.x; mhi = a2.y;
        }
        cnt -= a;
        __syncwarp();
        n_nodes += a; ++n_steps;
        uint32_t t = mlo & 511u;
        const uint32_t c = mlo >> 27, m = ((mhi >> 16) & 255u) + 1u;
        bool alive = false, emit = false;
        if (act) {
            const uint32_t x1 = k + s;
            const uint32_t plo = k - (k > primary ? 1u : 0u), phi = x1 - (x1 > primary ? 1u : 0u);
            const bool two = (plo >> 6) != (phi >> 6);
            const BcBlockRegs rlo = bc_load_block(lines, plo);
            n_xsect += two ? 1u : 0u;
            // strand 0 also needs one OTHER symbol's count for the forward start k2 (see below):
            // x = A when c is A or C, x = T when c is G or T
            const uint32_t x = c < 2u ? 0u : 3u;
            uint32_t olo = bc_block_rank1(rlo, plo, c), ohi, xlo = 0, xhi = 0;
            if (S0) xlo = bc_block_rank1(rlo, plo, x);
            if (two) {                                    // most narrow intervals sit in one sector
                const BcBlockRegs rhi = bc_load_block(lines, phi);
                ohi = bc_block_rank1(rhi, phi, c);
                if (S0) xhi = bc_block_rank1(rhi, phi, x);
            } else {
                ohi = bc_block_rank1(rlo, phi, c);
                if (S0) xhi = bc_block_rank1(rlo, phi, x);
            }
            if (c <= 3u && ohi != olo) {
                if (S0) {
                    // children split the forward interval in the order $,A,C,G,T:
                    //   A: k2 + dollar;  C: k2 + dollar + nA;  G: k2 + s - nT - nG;  T: k2 + s - nT
                    const uint32_t dollar = s - (phi - plo), nx = xhi - xlo, nc_ = ohi - olo;
                    k2 = c == 0u ? k2 + dollar : (c == 1u ? k2 + dollar + nx : (c == 2u ? k2 + s - nx - nc_ : k2 + s - nc_));
                }
                k = Cs[c] + olo + 1u; s = ohi - olo; ++t;
                emit = t == m; alive = !emit;
            }
        }
        uint32_t nb = 0;
        if (alive) nb = BC_PREP_BASE(p.ws.prep[(size_t)qid * p.ws.stride + t]);
        const uint32_t smask = __ballot_sync(0xffffffffu, alive);
        if (alive) {
            const uint32_t r = __popc(smask & lt_mask);
            ent_store(Cq, S0 ? CCAP - 1u - cnt - r : cnt + r, qid, k, s, k2, t | (nb << 27), mhi);
        }
        cnt += __popc(smask);
        if (__any_sync(0xffffffffu, emit))
            emit_hits(p.ws.arena, p.ws.arena_cap, p.ws.qcnt, ctr, emit, qid, S0 ? k2 : k, s, (mhi >> 8) & 255u);
        __syncwarp();
    }
}

// ---------------------------------------------------------------------------------------------
// A3 + A4 + A5.  Persistent kernel, one LIFO pool per warp, two kinds of step:
//  * BRANCH step: up to 32 branch states are popped, one per lane, and expanded in lock step:
//    all four child intervals from one rank4 pair (1-2 index sectors) -> match, <=3 mismatch,
//    <=4 deletion and 1 insertion children, pruned by the budgets and D/Ds.  Every lane counts its
//    surviving children, a warp scan assigns pool slots, and each lane writes its own children:
//    those that still have budget to the branch stack (match child deepest), those with d == z to
//    the chain stack; terminal children are emitted.
//  * CHAIN steps: whenever a strand's chain stack holds 32 states, 32 are popped, each is extended
//    by ONE exactly matching base (one symbol's rank at both interval ends) and the survivors are
//    pushed back compacted -- a flat cost per node, full lanes, whatever the chain lengths.
// New queries are drawn from a global ticket counter whenever fewer than 32 branch states are
// pending, so lanes stay busy and converged whatever the shape of the individual search trees.
// Pool bound: a multi-lane step keeps only the leading lanes whose children leave the
// ring at <= BCAP - R entries (R = 8z+9) and fit the chain stack; the others are un-popped.  Lane 0
// alone may fill the ring up to BCAP, and a run of single-lane steps from height P <= BCAP - R never
// exceeds P-1+R because the match child is explored last.  If even lane 0 does not fit, the chain
// stack (which only shrinks) is drained first.  Spilling the ring's bottom to global memory is an
// optimisation on top of that bound (it keeps steps 32 wide), not part of it.
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(BC_SEARCH_MAX_THREADS, BC_SEARCH_MIN_CTAS) bc_search_kernel(BcSearchParams p) {
    extern __shared__ uint2 pool_mem[];
    __shared__ __align__(16) uint32_t Ctab[8];                               // C[c] of the index each strand searches
    const uint32_t lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
    const uint32_t BCAP = p.bcap, CCAP = p.ccap, BM = p.bcap - 1u;
    uint2 *P = pool_mem + (size_t)warp * 3u * (BCAP + CCAP);     // branch ring: slots (bb + i) & BM
    uint2 *Cq = P + 3u * BCAP;                                    // chain area: strand 1 up from 0, strand 0 down from CCAP-1
    uint2 *G = p.ws.spill + ((size_t)blockIdx.x * (blockDim.x >> 5) + warp) * ((size_t)p.ws.spill_blocks * 96u);
    const uint32_t GB = p.ws.spill_blocks;
    const uint32_t lt_mask = (1u << lane) - 1u;
    const int z = p.o.z, E = p.o.indel_end_skip, max_go = p.o.max_gap_open, max_ge = p.o.max_gap_ext;
    const int seed_len = p.o.seed_len, seed_z = p.o.seed_z;
    const uint32_t R = 8u * (uint32_t)z + 9u;
    const uint32_t nq = p.ws.nq;
    const uint32_t full = p.ix.bwt[0].n + 1;
    unsigned long long *ctr = (unsigned long long *)p.ws.ctr;
    SearchConsts sc;
    sc.lines0 = p.ix.bwt[1].lines; sc.lines1 = p.ix.bwt[0].lines;          // strand 0 searches the reverse index
    sc.primary0 = p.ix.bwt[1].primary; sc.primary1 = p.ix.bwt[0].primary;

    if (threadIdx.x < 8) Ctab[threadIdx.x] = p.ix.bwt[threadIdx.x < 4 ? 1 : 0].C[threadIdx.x & 3];
    __syncthreads();
    uint32_t bb = 1u << 24, bcnt = 0, c0 = 0, c1 = 0, gsp = 0, pool_max = 0;   // ring bottom, counts (branch, chain per strand), spilled blocks
    bool more = true, force_drain = false;
    // 32-bit statistics, flushed to the 64-bit global counters at every intake and at the end
    uint32_t n_cnodes = 0, n_xsect = 0, n_bsteps = 0, n_bnodes = 0, n_csteps = 0, n_cancel = 0, n_spill = 0;

    for (;;) {
        // ---- ring <-> global: keep the hot top of the branch stack on chip --------------------------
        while (bcnt >= 64u && bcnt + 96u + R > BCAP && gsp < GB) {          // spill the bottom 32 entries
            const uint2 *src = P + ((bb + lane) & BM) * 3u;
            uint2 *dst = G + ((size_t)gsp * 32u + lane) * 3u;
            dst[0] = src[0]; dst[1] = src[1]; dst[2] = src[2];
            bb += 32u; bcnt -= 32u; ++gsp; ++n_spill;
            __syncwarp();
        }
        if (bcnt < 32u && gsp > 0u) {                                          // bring the last block back
            --gsp; bb -= 32u;
            const uint2 *src = G + ((size_t)gsp * 32u + lane) * 3u;
            uint2 *dst = P + ((bb + lane) & BM) * 3u;
            dst[0] = src[0]; dst[1] = src[1]; dst[2] = src[2];
            bcnt += 32u;
            __syncwarp();
        }
        // ---- intake: new root states while the branch stack is shallow ------------------------
        if (more && bcnt < 32u && gsp == 0u && c0 + c1 + 32u <= CCAP) {
            flush_stats(ctr, lane, n_cnodes, n_xsect, n_bsteps, n_bnodes, n_csteps, n_cancel, n_spill);
            n_cnodes = n_xsect = n_bsteps = n_bnodes = n_csteps = n_cancel = n_spill = 0;
            uint32_t need = 32u - bcnt;
            unsigned long long tk = 0;
            if (lane == 0) {
                // towards the end of the batch take fewer queries at a time, so that the last heavy
                // trees are spread over the warps instead of queueing behind one another
                const unsigned long long seen = *(volatile unsigned long long *)&ctr[BC_CTR_TICKET];
                const unsigned long long left = seen < nq ? nq - seen : 0ull;
                const unsigned long long fair = left / (4ull * gridDim.x * (blockDim.x >> 5)) + 1ull;
                if (fair < need) need = (uint32_t)fair;
                tk = atomicAdd(&ctr[BC_CTR_TICKET], (unsigned long long)need);
            }
            need = __shfl_sync(0xffffffffu, need, 0);
            tk = __shfl_sync(0xffffffffu, tk, 0);
            if (tk + need >= nq) more = false;
            unsigned long long q = tk + lane;
            bool ok = lane < need && q < nq;
            uint32_t m = 0, pr = 0;
            if (ok) {
                m = p.reads.len[q >> 1];
                pr = p.ws.prep[(size_t)q * p.ws.stride];
                ok = m >= 1 && m <= p.reads.max_len && (int)BC_PREP_D(pr) <= z && (int)BC_PREP_DS(pr) <= seed_z;
            }
            const bool odd = (q & 1ull) != 0;
            const uint32_t mask = __ballot_sync(0xffffffffu, ok);
            const uint32_t mask1 = __ballot_sync(0xffffffffu, ok && odd), mask0 = mask & ~mask1;
            if (ok) {
                if (z > 0) ent_store(P, (bb + bcnt + __popc(mask & lt_mask)) & BM, (uint32_t)q, 0u, full, 0u, 0u, (m - 1) << 16);
                else ent_store(Cq, odd ? c1 + __popc(mask1 & lt_mask) : CCAP - 1u - c0 - __popc(mask0 & lt_mask), (uint32_t)q,
                               0u, full, 0u, BC_PREP_BASE(pr) << 27, (m - 1) << 16);
            }
            if (z > 0) bcnt += __popc(mask); else { c1 += __popc(mask1); c0 += __popc(mask0); }
            __syncwarp();
        }
        if (bcnt == 0 && c0 + c1 == 0) { if (!more) break; continue; }
        pool_max = bcnt + c0 + c1 > pool_max ? bcnt + c0 + c1 : pool_max;

        if (c1 >= 32u || c0 >= 32u || ((bcnt == 0 || force_drain) && c0 + c1 > 0u)) {
            const bool drain = bcnt == 0 || force_drain;
            chain_steps<false>(p, sc.lines1, sc.primary1, Ctab + 4, Cq, CCAP, c1, drain, ctr, n_cnodes, n_xsect, n_csteps);
            chain_steps<true>(p, sc.lines0, sc.primary0, Ctab, Cq, CCAP, c0, drain, ctr, n_cnodes, n_xsect, n_csteps);
            force_drain = false;
            continue;
        }

        // ==== BRANCH step ========================================================================
        const uint32_t a = bcnt < 32u ? bcnt : 32u;
        bool act = lane < a;
        uint32_t qid = 0, k = 0, s = 0, k2 = 0, mlo = 0, mhi = 0;
        if (act) {
            const uint2 *e = P + ((bb + bcnt - 1u - lane) & BM) * 3u;
            const uint2 a0 = e[0], a1 = e[1], a2 = e[2];
            qid = a0.x; k = a0.y; s = a1.x; k2 = a1.y; mlo = a2.x; mhi = a2.y;
        }
        __syncwarp();

        const int t = mlo & 511, st = (mlo >> 9) & 3, go = (mlo >> 11) & 255, ge = (mlo >> 19) & 255;
        const int sd = mhi & 255, d = (mhi >> 8) & 255, m = (int)((mhi >> 16) & 255) + 1;
        const uint32_t strand = qid & 1u;
        const bool seed_on = seed_len > 0 && seed_len < m;
        const bool has_base = act && t < m;
        const bool del_ok = act && st != 1 && t >= E && m - t >= E;
        const bool ins_ok = has_base && st != 2 && t >= E && m - 1 - t >= E;
        uint32_t pr0 = 0, pr1 = 0;
        if (act) {
            const uint16_t *pp = p.ws.prep + (size_t)qid * p.ws.stride + t;
            pr0 = pp[0];
            if (has_base) pr1 = pp[1];
        }
        const uint32_t qb = BC_PREP_BASE(pr0);
        uint32_t nk[4] = {0, 0, 0, 0}, ns[4] = {0, 0, 0, 0}, nk2[4] = {0, 0, 0, 0};
        bool straddle = false;
        if (has_base || del_ok) {
            const uint4 *lines = strand ? sc.lines1 : sc.lines0;
            const uint32_t primary = strand ? sc.primary1 : sc.primary0;
            const uint32_t x1 = k + s;
            const uint32_t plo = k - (k > primary ? 1u : 0u), phi = x1 - (x1 > primary ? 1u : 0u);
            uint32_t olo[4], ohi[4];
            bc_rank4(lines, plo, olo);                    // two unconditional loads: predicating the second one on
            bc_rank4(lines, phi, ohi);                    // "other sector" was measured 3 % slower here (not in the chain step)
            straddle = (plo >> 6) != (phi >> 6);
            const uint4 Cv = *reinterpret_cast<const uint4 *>(Ctab + strand * 4u);
            const uint32_t Cc[4] = {Cv.x, Cv.y, Cv.z, Cv.w};
            uint32_t acc = k2 + s;                       // k2 + dollar + prefix, built below
#pragma unroll
            for (int b = 0; b < 4; ++b) { ns[b] = ohi[b] - olo[b]; nk[b] = Cc[b] + olo[b] + 1u; acc -= ns[b]; }
#pragma unroll
            for (int b = 0; b < 4; ++b) { nk2[b] = acc; acc += ns[b]; }
        }
        const int in_seed_base = (seed_on && t < seed_len) ? 1 : 0;
        const int in_seed_del = (seed_on && t > 0 && t < seed_len) ? 1 : 0;
        const uint32_t m_bits = mhi & 0x00FF0000u;
        // class-level validity and packed child state (same for every child of a class)
        const int nd1 = d + 1;
        const bool v_mm = has_base && nd1 <= z && sd + in_seed_base <= seed_z && z - nd1 >= (int)BC_PREP_D(pr1) &&
                          seed_z - (sd + in_seed_base) >= (int)BC_PREP_DS(pr1);
        const int d_go = go + (st != 2), d_ge = ge + (st == 2), i_go = go + (st != 1), i_ge = ge + (st == 1);
        const bool v_del = del_ok && nd1 <= z && d_go <= max_go && d_ge <= max_ge && sd + in_seed_del <= seed_z &&
                           z - nd1 >= (int)BC_PREP_D(pr0) && seed_z - (sd + in_seed_del) >= (int)BC_PREP_DS(pr0);
        const bool v_ins = ins_ok && nd1 <= z && i_go <= max_go && i_ge <= max_ge && sd + in_seed_base <= seed_z &&
                           z - nd1 >= (int)BC_PREP_D(pr1) && seed_z - (sd + in_seed_base) >= (int)BC_PREP_DS(pr1);
        const uint32_t tn = (uint32_t)t + 1u;
        const uint32_t ma_lo = tn | ((uint32_t)go << 11) | ((uint32_t)ge << 19);
        const uint32_t ma_hi = (uint32_t)sd | ((uint32_t)d << 8) | m_bits;
        const uint32_t mm_hi = (uint32_t)(sd + in_seed_base) | ((uint32_t)nd1 << 8) | m_bits;
        const uint32_t de_lo = (uint32_t)t | (2u << 9) | ((uint32_t)d_go << 11) | ((uint32_t)d_ge << 19);
        const uint32_t de_hi = (uint32_t)(sd + in_seed_del) | ((uint32_t)nd1 << 8) | m_bits;
        const uint32_t in_lo = tn | (1u << 9) | ((uint32_t)i_go << 11) | ((uint32_t)i_ge << 19);
        const uint32_t cb0 = qb << 27, cb1 = BC_PREP_BASE(pr1) << 27;   // first base of a chain child (bits 27-29)
        const bool last1 = nd1 == z;                     // children that cost a difference exhaust the budget
        const bool term_base = (int)tn == m;             // children that consume W[t] finish the read
        const bool term_del = t == m;

        // child bit masks: bit 0 match; 1-4 mismatch with symbol bit-1; 5-8 deletion of symbol bit-5; 9 insertion
        uint32_t vbits = 0;
#pragma unroll
        for (int b = 0; b < 4; ++b) {
            const bool ne = ns[b] > 0u;
            if (has_base && qb == (uint32_t)b && ne) vbits |= 1u;
            if (v_mm && qb != (uint32_t)b && ne) vbits |= 2u << b;
            if (v_del && ne) vbits |= 32u << b;
        }
        if (v_ins) vbits |= 512u;
        const uint32_t tbits = (term_base ? 0x21Fu : 0u) | (term_del ? 0x1E0u : 0u);   // terminal children
        uint32_t ebits = vbits & tbits;
        if (s == full) ebits &= ~512u;                   // the empty string is not a hit (C3)
        // a terminal state is expanded further only for trailing deletions (E == 0) with budget left
        const uint32_t keep_t = E == 0 ? (last1 ? 1u : 0x3FFu) : 0u;
        uint32_t pbits = vbits & (~tbits | keep_t);
        uint32_t cbits = last1 ? (pbits & 0x3FEu) : 0u;
        const uint32_t cshift = strand ? 10u : 20u;      // packed counters: branch (bits 0-9) | chain strand 1 (10-19) | strand 0 (20-29)

        // slots: warp scan of (branch pushes | chain pushes << 16); net growth decides who is kept
        const uint32_t mine = (uint32_t)__popc(pbits & ~cbits) | ((uint32_t)__popc(cbits) << cshift);
        uint32_t incl = mine;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t v = __shfl_up_sync(0xffffffffu, incl, o);
            if ((int)lane >= o) incl += v;
        }
        // lanes 0..lane kept, the lanes behind un-popped: ring and chain occupancy after the step
        const uint32_t ring_if = bcnt - (lane + 1u) + (incl & 1023u);
        const uint32_t chain_if = c0 + c1 + ((incl >> 10) & 1023u) + (incl >> 20);
        const bool fits = act && ring_if + R <= BCAP && chain_if <= CCAP;
        uint32_t keepmask = __ballot_sync(0xffffffffu, fits);
        uint32_t akeep = keepmask == 0xffffffffu ? 32u : (uint32_t)(__ffs(~keepmask) - 1);   // leading run
        if (akeep > a) akeep = a;
        if (akeep == 0) {                                 // lane 0 alone may use the whole ring
            const uint32_t r0 = __shfl_sync(0xffffffffu, ring_if, 0), c0 = __shfl_sync(0xffffffffu, chain_if, 0);
            if (r0 <= BCAP && c0 <= CCAP) akeep = 1;
        }
        if (akeep == 0) {
            if (c0 + c1 == 0) { if (lane == 0) atomicOr(&ctr[BC_CTR_ERROR], 2ull); break; }   // cannot happen (pool bound)
            force_drain = true;                           // nothing popped; make room first
            n_cancel += a;
            continue;
        }
        if (lane >= akeep) { act = false; pbits = 0; cbits = 0; ebits = 0; }
        n_cancel += a - akeep;
        const uint32_t tot = __shfl_sync(0xffffffffu, incl, akeep - 1u);
        const uint32_t excl = incl - mine;
        uint32_t bpos = bb + bcnt - akeep + (excl & 1023u);           // ring index (masked at the store)
        uint32_t cpos = strand ? c1 + ((excl >> 10) & 1023u) : CCAP - 1u - c0 - (excl >> 20);
        const uint32_t cstep = strand ? 1u : 0xFFFFFFFFu;             // strand 1 grows up, strand 0 down
        bcnt = bcnt - akeep + (tot & 1023u);
        c1 += (tot >> 10) & 1023u;
        c0 += tot >> 20;
        n_bnodes += akeep; ++n_bsteps;
        n_xsect += (act && straddle) ? 1u : 0u;

        if (pbits) {
            if (pbits & 1u) {
                ent_store(P, (bpos++) & BM, qid, sel4(nk[0], nk[1], nk[2], nk[3], qb), sel4(ns[0], ns[1], ns[2], ns[3], qb),
                          sel4(nk2[0], nk2[1], nk2[2], nk2[3], qb), ma_lo, ma_hi);
            }
#pragma unroll
            for (int b = 0; b < 4; ++b) {
                if (pbits & (2u << b)) {
                    if (last1) { ent_store(Cq, cpos, qid, nk[b], ns[b], nk2[b], ma_lo | cb1, mm_hi); cpos += cstep; }
                    else ent_store(P, (bpos++) & BM, qid, nk[b], ns[b], nk2[b], ma_lo, mm_hi);
                }
            }
#pragma unroll
            for (int b = 0; b < 4; ++b) {
                if (pbits & (32u << b)) {
                    if (last1) { ent_store(Cq, cpos, qid, nk[b], ns[b], nk2[b], de_lo | cb0, de_hi); cpos += cstep; }
                    else ent_store(P, (bpos++) & BM, qid, nk[b], ns[b], nk2[b], de_lo, de_hi);
                }
            }
            if (pbits & 512u) {
                if (last1) { ent_store(Cq, cpos, qid, k, s, k2, in_lo | cb1, mm_hi); cpos += cstep; }
                else ent_store(P, (bpos++) & BM, qid, k, s, k2, in_lo, mm_hi);
            }
        }
        if (__any_sync(0xffffffffu, ebits != 0u)) {
#pragma unroll 1
            for (int slot = 0; slot < 10; ++slot) {
                const bool em = (ebits >> slot) & 1u;
                if (!__any_sync(0xffffffffu, em)) continue;
                const uint32_t b = slot == 0 ? qb : (uint32_t)((slot - 1) & 3);
                uint32_t ck = sel4(nk[0], nk[1], nk[2], nk[3], b), cs = sel4(ns[0], ns[1], ns[2], ns[3], b);
                uint32_t ck2 = sel4(nk2[0], nk2[1], nk2[2], nk2[3], b);
                if (slot == 9) { ck = k; cs = s; ck2 = k2; }
                emit_hits(p.ws.arena, p.ws.arena_cap, p.ws.qcnt, ctr, em, qid, strand ? ck : ck2, cs,
                          (uint32_t)(slot == 0 ? d : nd1));
            }
        }
        __syncwarp();
    }
    flush_stats(ctr, lane, n_cnodes, n_xsect, n_bsteps, n_bnodes, n_csteps, n_cancel, n_spill);
    if (lane == 0) atomicMax(&ctr[BC_CTR_POOLMAX], (unsigned long long)pool_max);
}

}  // namespace

cudaError_t bc_launch_search(const BcSearchParams &p, int sm_count, uint32_t ctas_per_sm, uint32_t warps_per_cta,
                             cudaStream_t st) {
    if (p.ws.nq == 0) return cudaSuccess;
    size_t smem = (size_t)warps_per_cta * (p.bcap + p.ccap) * BC_POOL_ENTRY_BYTES;
    cudaError_t e = cudaFuncSetAttribute(bc_search_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    bc_search_kernel<<<sm_count * ctas_per_sm, warps_per_cta * 32, smem, st>>>(p);
    return cudaGetLastError();
}
