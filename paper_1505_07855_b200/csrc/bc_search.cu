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

// all four O(., j) for the two ends of the row interval [k, k+s-1]: olo = O(., k-1), ohi = O(., k+s-1).
// Returns the number of distinct 32-byte blocks (sectors) touched (1 or 2).
__device__ __forceinline__ uint32_t rank4_pair(const BcBwtDev &b, uint32_t k, uint32_t s, uint32_t olo[4], uint32_t ohi[4]) {
    const uint32_t plo = bc_rank_pos(b, k), phi = bc_rank_pos(b, k + s);
    bc_rank4(b.lines, plo, olo);
    bc_rank4(b.lines, phi, ohi);
    return 1u + ((plo >> 6) != (phi >> 6) ? 1u : 0u);
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

// pool entry, 6 words, stored field-major (SoA) per warp so that lanes hit distinct banks:
//   qid | k | s | k2 | mlo | mhi
//   mlo = t (bits 0-8) | st (9-10; 0 = M, 1 = I, 2 = D) | n_go (11-18) | n_ge (19-26)
//   mhi = seed_d (0-7) | d (8-15) | m-1 (16-23)
// One pool per warp holds two stacks: BRANCH states (budget left, d < z) grow up from slot 0,
// CHAIN states (budget exhausted, d == z: only exact matching can follow) grow down from CAP-1.
#define BC_SEARCH_MAX_THREADS 256

struct WarpCtx {
    uint32_t *P;
    uint32_t CAP, lane, lt_mask;
    unsigned long long *ctr;
};

// warp-aggregated append of raw hits (A5)
__device__ __forceinline__ void emit_hits(BcRawHit *arena, unsigned long long arena_cap, uint32_t *qcnt, const WarpCtx &w,
                                          bool emit, uint32_t qid, uint32_t kf, uint32_t s, uint32_t d) {
    uint32_t emask = __ballot_sync(0xffffffffu, emit);
    if (emask == 0) return;
    unsigned long long base = 0;
    int leader = __ffs(emask) - 1;
    if ((int)w.lane == leader) base = atomicAdd(&w.ctr[BC_CTR_ARENA], (unsigned long long)__popc(emask));
    base = __shfl_sync(0xffffffffu, base, leader);
    if (emit) {
        unsigned long long pos = base + __popc(emask & w.lt_mask);
        if (pos < arena_cap) arena[pos] = BcRawHit{qid, kf, kf + s - 1u, d};
        atomicAdd(&qcnt[qid], 1u);
    }
}

// Strand 0 only: forward-interval start after exactly matching W[t0..t1) from the state
// (k, s, k2) -- the bidirectional update of SURVEY C7 (R), replayed where a chain needs it.
__device__ __noinline__ uint32_t replay_k2(const uint4 *lines, uint32_t primary, uint4 Cv, const uint16_t *pp, uint32_t k,
                                           uint32_t s, uint32_t k2, uint32_t t0, uint32_t t1) {
    for (uint32_t t = t0; t < t1; ++t) {
        const uint32_t c = BC_PREP_BASE(pp[t]);
        uint32_t olo[4], ohi[4];
        bc_rank4(lines, k - (k > primary ? 1u : 0u), olo);
        bc_rank4(lines, k + s - (k + s > primary ? 1u : 0u), ohi);
        uint32_t acc = k2 + s;
#pragma unroll
        for (int b = 0; b < 4; ++b) acc -= ohi[b] - olo[b];           // k2 + (1 if '$' is in the interval)
#pragma unroll
        for (int b = 0; b < 4; ++b) if ((uint32_t)b < c) acc += ohi[b] - olo[b];
        k2 = acc;
        const uint32_t o = sel4(olo[0], olo[1], olo[2], olo[3], c);
        s = sel4(ohi[0], ohi[1], ohi[2], ohi[3], c) - o;
        k = sel4(Cv.x, Cv.y, Cv.z, Cv.w, c) + o + 1u;
    }
    return k2;
}

// ---------------------------------------------------------------------------------------------
// A3 + A4 + A5.  Persistent kernel, one LIFO pool per warp, two kinds of step:
//  * BRANCH step: the top `a` branch states are popped, one per lane, and expanded in lock step:
//    all four child intervals from one rank4 pair (1-2 index lines) -> match, <=3 mismatch,
//    <=4 deletion and 1 insertion children, pruned by the budgets and D/Ds.  Children that still
//    have budget go back to the branch stack (match child deepest), children with d == z go to
//    the chain stack, terminal children are emitted.
//  * CHAIN phase: lanes pull chain states and extend them by exact matching only (one symbol's
//    rank at both interval ends per step, no pool traffic), refilling from the chain stack as they
//    die, until the stack is dry and fewer than half the lanes are busy; survivors are parked.
// New queries are drawn from a global ticket counter whenever fewer than 32 branch states are
// pending, so lanes stay busy and converged whatever the shape of the individual search trees.
// Pool bound: with used = branch + chain entries, a = clamp((CAP - R - used)/8, .., 32)
// and R = 8z+9; when that is < 1 the chain stack is drained first (it only shrinks), and a run of
// single-state steps from height P never exceeds P-1+R because the match child is explored last.
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(BC_SEARCH_MAX_THREADS, 3) bc_search_kernel(BcSearchParams p) {
    extern __shared__ uint32_t pool_mem[];
    WarpCtx w;
    w.lane = threadIdx.x & 31u;
    const uint32_t warp = threadIdx.x >> 5;
    const uint32_t CAP = p.pool_cap;
    w.CAP = CAP;
    uint32_t *P = pool_mem + (size_t)warp * 6u * CAP;
    w.P = P;
    w.lt_mask = (1u << w.lane) - 1u;
    const uint32_t lane = w.lane, lt_mask = w.lt_mask;
    const int z = p.o.z, E = p.o.indel_end_skip, max_go = p.o.max_gap_open, max_ge = p.o.max_gap_ext;
    const int seed_len = p.o.seed_len, seed_z = p.o.seed_z;
    const int R = 8 * z + 9;
    const uint32_t nq = p.ws.nq;
    const uint32_t full = p.ix.bwt[0].n + 1;
    unsigned long long *ctr = (unsigned long long *)p.ws.ctr;
    w.ctr = ctr;

    const uint4 *rv_lines = p.ix.bwt[1].lines;
    const uint32_t rv_primary = p.ix.bwt[1].primary;
    const uint4 rv_C = make_uint4(p.ix.bwt[1].C[0], p.ix.bwt[1].C[1], p.ix.bwt[1].C[2], p.ix.bwt[1].C[3]);
    uint32_t bcnt = 0, ccnt = 0, pool_max = 0;
    bool more = true;
    unsigned long long n_nodes = 0, n_lines = 0, n_bsteps = 0, n_bnodes = 0, n_csteps = 0;

    for (;;) {
        // ---- intake: new root states while the branch stack is shallow ------------------------
        if (more && bcnt < 32u && bcnt + ccnt + 40u <= CAP) {
            uint32_t need = 32u - bcnt;
            unsigned long long tk = 0;
            if (lane == 0) tk = atomicAdd(&ctr[BC_CTR_TICKET], (unsigned long long)need);
            tk = __shfl_sync(0xffffffffu, tk, 0);
            if (tk + need >= nq) more = false;
            unsigned long long q = tk + lane;
            bool ok = lane < need && q < nq;
            uint32_t m = 0;
            if (ok) {
                m = p.reads.len[q >> 1];
                uint32_t pr = p.ws.prep[(size_t)q * p.ws.stride];
                ok = m >= 1 && m <= p.reads.max_len && (int)BC_PREP_D(pr) <= z && (int)BC_PREP_DS(pr) <= seed_z;
            }
            uint32_t mask = __ballot_sync(0xffffffffu, ok);
            if (ok) {
                uint32_t r = __popc(mask & lt_mask);
                uint32_t pos = z > 0 ? bcnt + r : CAP - 1u - ccnt - r;
                P[0 * CAP + pos] = (uint32_t)q; P[1 * CAP + pos] = 0; P[2 * CAP + pos] = full;
                P[3 * CAP + pos] = 0; P[4 * CAP + pos] = 0; P[5 * CAP + pos] = (m - 1) << 16;
            }
            if (z > 0) bcnt += __popc(mask); else ccnt += __popc(mask);
            __syncwarp();
        }
        if (bcnt == 0 && ccnt == 0) { if (!more) break; continue; }
        pool_max = bcnt + ccnt > pool_max ? bcnt + ccnt : pool_max;

        int a = ((int)CAP - R - (int)(bcnt + ccnt)) / 8;
        if (ccnt > 0 && (ccnt >= 32u || bcnt == 0 || a < 1)) {
            // ==== CHAIN phase ====================================================================
            const bool must_finish = (bcnt == 0 && !more) || a < 1;   // a < 1: the drain must make room
            bool act = false;
            uint32_t qid = 0, k = 0, s = 0, k2 = 0, t = 0, m = 0, dz = 0;
            uint32_t k0 = 0, s0 = 0, t0 = 0;                      // strand 0: state k2 belongs to
            for (;;) {
                uint32_t idle = __ballot_sync(0xffffffffu, !act);
                if (idle && ccnt) {
                    uint32_t r = __popc(idle & lt_mask);
                    if (!act && r < ccnt) {
                        uint32_t idx = CAP - ccnt + r;
                        qid = P[0 * CAP + idx]; k = P[1 * CAP + idx]; s = P[2 * CAP + idx]; k2 = P[3 * CAP + idx];
                        uint32_t mlo = P[4 * CAP + idx], mhi = P[5 * CAP + idx];
                        t = mlo & 511u; m = ((mhi >> 16) & 255u) + 1u; dz = (mhi >> 8) & 255u;
                        k0 = k; s0 = s; t0 = t;
                        act = true;
                    }
                    uint32_t take = __popc(idle);
                    ccnt -= take < ccnt ? take : ccnt;
                    __syncwarp();
                }
                uint32_t am = __ballot_sync(0xffffffffu, act);
                if (am == 0) break;
                if (!must_finish && ccnt == 0 && __popc(am) < 16) {
                    // park the survivors (strand 0 first brings k2 up to date)
                    if (act) {
                        if (!(qid & 1u) && t > t0) k2 = replay_k2(rv_lines, rv_primary, rv_C, p.ws.prep + (size_t)qid * p.ws.stride, k0, s0, k2, t0, t);
                        uint32_t idx = CAP - 1u - __popc(am & lt_mask);
                        P[0 * CAP + idx] = qid; P[1 * CAP + idx] = k; P[2 * CAP + idx] = s; P[3 * CAP + idx] = k2;
                        P[4 * CAP + idx] = t; P[5 * CAP + idx] = (dz << 8) | ((m - 1u) << 16);
                    }
                    ccnt = __popc(am);
                    __syncwarp();
                    break;
                }
                n_nodes += (unsigned long long)__popc(am);
                ++n_csteps;
                bool emit = false;
                if (act) {
                    const uint32_t strand = qid & 1u;
                    const uint32_t c = BC_PREP_BASE(p.ws.prep[(size_t)qid * p.ws.stride + t]);
                    if (c > 3u) act = false;
                    else {
                        const BcBwtDev &X = p.ix.bwt[strand ? 0 : 1];
                        const uint32_t plo = bc_rank_pos(X, k), phi = bc_rank_pos(X, k + s);
                        const uint32_t olo = bc_rank1(X.lines, plo, c), ohi = bc_rank1(X.lines, phi, c);
                        n_lines += 1u + ((plo >> 6) != (phi >> 6) ? 1u : 0u);
                        if (ohi == olo) act = false;
                        else {
                            k = X.C[c] + olo + 1u; s = ohi - olo; ++t;
                            if (t == m) { emit = true; act = false; }
                        }
                    }
                }
                if (__any_sync(0xffffffffu, emit)) {
                    uint32_t kf = k;
                    if (emit && !(qid & 1u)) kf = replay_k2(rv_lines, rv_primary, rv_C, p.ws.prep + (size_t)qid * p.ws.stride, k0, s0, k2, t0, t);
                    emit_hits(p.ws.arena, p.ws.arena_cap, p.ws.qcnt, w, emit, qid, kf, s, dz);
                }
            }
            continue;
        }

        // ==== BRANCH step ========================================================================
        a = a < 1 ? 1 : (a > 32 ? 32 : a);
        a = a > (int)bcnt ? (int)bcnt : a;
        const bool act = (int)lane < a;
        uint32_t qid = 0, k = 0, s = 0, k2 = 0, mlo = 0, mhi = 0;
        if (act) {
            uint32_t idx = bcnt - 1u - lane;
            qid = P[0 * CAP + idx]; k = P[1 * CAP + idx]; s = P[2 * CAP + idx];
            k2 = P[3 * CAP + idx]; mlo = P[4 * CAP + idx]; mhi = P[5 * CAP + idx];
        }
        __syncwarp();
        bcnt -= (uint32_t)a;
        n_nodes += (unsigned long long)a;
        n_bnodes += (unsigned long long)a;
        ++n_bsteps;

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
        if (has_base || del_ok) {
            const BcBwtDev &X = p.ix.bwt[strand ? 0 : 1];
            uint32_t olo[4], ohi[4];
            n_lines += rank4_pair(X, k, s, olo, ohi);
            uint32_t acc = k2 + s;                       // k2 + dollar + prefix, built below
#pragma unroll
            for (int b = 0; b < 4; ++b) { ns[b] = ohi[b] - olo[b]; nk[b] = X.C[b] + olo[b] + 1u; acc -= ns[b]; }
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
        const bool last1 = nd1 == z;                     // children that cost a difference exhaust the budget
        const bool term_base = (int)tn == m;             // children that consume W[t] finish the read
        const bool term_del = t == m;

#pragma unroll
        for (int slot = 0; slot < 10; ++slot) {
            // slot 0: match; 1-4: mismatch with symbol slot-1; 5-8: deletion of symbol slot-5; 9: insertion
            bool valid, terminal, chain;
            uint32_t ck = k, cs = s, ck2 = k2, clo, chi;
            if (slot == 0) {
                ck = sel4(nk[0], nk[1], nk[2], nk[3], qb); cs = sel4(ns[0], ns[1], ns[2], ns[3], qb);
                ck2 = sel4(nk2[0], nk2[1], nk2[2], nk2[3], qb);
                valid = has_base && qb < 4u && cs > 0u; terminal = term_base; chain = false;
                clo = ma_lo; chi = ma_hi;
            } else if (slot <= 4) {
                const int b = slot - 1;
                ck = nk[b]; cs = ns[b]; ck2 = nk2[b];
                valid = v_mm && qb != (uint32_t)b && cs > 0u; terminal = term_base; chain = last1;
                clo = ma_lo; chi = mm_hi;
            } else if (slot <= 8) {
                const int b = slot - 5;
                ck = nk[b]; cs = ns[b]; ck2 = nk2[b];
                valid = v_del && cs > 0u; terminal = term_del; chain = last1;
                clo = de_lo; chi = de_hi;
            } else {
                valid = v_ins; terminal = term_base; chain = last1;
                clo = in_lo; chi = mm_hi;
            }
            const bool emit = valid && terminal && cs != full;
            // a terminal state is expanded further only for trailing deletions (E == 0) with budget left
            const bool push = valid && (!terminal || (E == 0 && !chain));
            if (__any_sync(0xffffffffu, emit))
                emit_hits(p.ws.arena, p.ws.arena_cap, p.ws.qcnt, w, emit, qid, strand ? ck : ck2, cs, (chi >> 8) & 255u);
            const uint32_t bmask = __ballot_sync(0xffffffffu, push && !chain);
            const uint32_t cmask = __ballot_sync(0xffffffffu, push && chain);
            const bool room = bcnt + ccnt + (uint32_t)a <= CAP;   // always true (pool bound); never write outside
            if (push && room) {
                const uint32_t pos = chain ? CAP - 1u - ccnt - __popc(cmask & lt_mask) : bcnt + __popc(bmask & lt_mask);
                P[0 * CAP + pos] = qid; P[1 * CAP + pos] = ck; P[2 * CAP + pos] = cs; P[3 * CAP + pos] = ck2;
                P[4 * CAP + pos] = clo; P[5 * CAP + pos] = chi;
            }
            if (!room && (bmask | cmask)) {                       // cannot happen; never silent
                if (lane == 0) atomicOr(&ctr[BC_CTR_ERROR], 2ull);
            } else {
                bcnt += __popc(bmask);
                ccnt += __popc(cmask);
            }
        }
        __syncwarp();
    }
    // per-warp statistics
    for (int o = 16; o > 0; o >>= 1) n_lines += __shfl_down_sync(0xffffffffu, n_lines, o);
    if (lane == 0) {
        atomicAdd(&ctr[BC_CTR_NODES], n_nodes);
        atomicAdd(&ctr[BC_CTR_LOOKUPS], 2ull * n_nodes);
        atomicAdd(&ctr[BC_CTR_LINES], n_lines);
        atomicMax(&ctr[BC_CTR_POOLMAX], (unsigned long long)pool_max);
        atomicAdd(&ctr[BC_CTR_BSTEPS], n_bsteps);
        atomicAdd(&ctr[BC_CTR_BNODES], n_bnodes);
        atomicAdd(&ctr[BC_CTR_CSTEPS], n_csteps);
    }
}

}  // namespace

cudaError_t bc_launch_search(const BcSearchParams &p, int sm_count, uint32_t ctas_per_sm, uint32_t warps_per_cta,
                             cudaStream_t st) {
    if (p.ws.nq == 0) return cudaSuccess;
    size_t smem = (size_t)warps_per_cta * p.pool_cap * BC_POOL_ENTRY_BYTES;
    cudaError_t e = cudaFuncSetAttribute(bc_search_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    bc_search_kernel<<<sm_count * ctas_per_sm, warps_per_cta * 32, smem, st>>>(p);
    return cudaGetLastError();
}
