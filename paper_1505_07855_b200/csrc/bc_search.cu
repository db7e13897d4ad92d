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

// greedy piece count of SURVEY C7 over W[lo..hi), grown from W[hi-1] leftwards on the opposite-direction
// index Y.  Whenever the count steps from c to c+1 at position a, D[a+1] = c is the last position with
// D <= c: thr[c] = a+1 (thresholds beyond `rmax` are not needed; thr[] was zeroed: D[lo] <= r => 0).
template <int LAY>
__device__ __forceinline__ void piece_thresholds(const bc_reads &rd, uint64_t off, uint32_t strand, const BcBwtDev &Y,
                                                 int lo, int hi, int rmax, uint8_t *thr, uint64_t &lookups) {
    const uint32_t full = Y.n + 1;
    uint32_t cnt = 0, k = 0, s = full;
    for (int a = hi - 1; a >= lo; --a) {
        uint32_t c = read_base(rd, off + a);
        if (c < 4 && strand) c = 3 - c;
        bool brk = c > 3;
        if (!brk) {
            const uint32_t olo = bc_rank1<LAY>(Y.lines, bc_rank_pos(Y, k), c), ohi = bc_rank1<LAY>(Y.lines, bc_rank_pos(Y, k + s), c);
            lookups += 2;
            if (ohi == olo) brk = true; else { k = Y.C[c] + olo + 1; s = ohi - olo; }
        }
        if (brk) {
            if ((int)cnt <= rmax) thr[cnt] = (uint8_t)(a + 1 < 255 ? a + 1 : 255);
            cnt++; k = 0; s = full;
        }
    }
}

// ---------------------------------------------------------------------------------------------
// A1 + A2: one thread per query (read, strand): writes the query record of bc_ws.cuh -- bases
// (complemented for strand 1), N bits, and the D / Ds bounds as thresholds.
// ---------------------------------------------------------------------------------------------
template <int LAY>
__global__ void bc_prepare_kernel(BcSearchParams p) {
    uint32_t q = blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= p.ws.nq) return;
    uint32_t r = q >> 1, strand = q & 1;
    uint32_t m = p.reads.len[r];
    uint8_t *rec = p.ws.qrec + (size_t)q * p.ws.qstride;
    for (uint32_t i = 0; i < p.ws.qstride; i += 16) *reinterpret_cast<uint4 *>(rec + i) = make_uint4(0, 0, 0, 0);
    if (m < 1 || m > p.reads.max_len) {
        atomicOr((unsigned long long *)&p.ws.ctr[BC_CTR_ERROR], 1ull);
        return;
    }
    uint64_t off = p.reads.off[r];
    // bases and N bits, re-aligned to bit 0 of the record's words
    uint32_t *bw = reinterpret_cast<uint32_t *>(rec + p.ws.q_boff);
    for (uint32_t w = 0; 16u * w < m; ++w) {
        const uint64_t pos = off + 16u * w, last = off + (16u * w + 15u < m ? 16u * w + 15u : m - 1u);
        const uint32_t lo = p.reads.bases2[pos >> 4], hi = (last >> 4) > (pos >> 4) ? p.reads.bases2[(pos >> 4) + 1] : 0u;
        const uint32_t v = __funnelshift_r(lo, hi, 2u * (uint32_t)(pos & 15));
        bw[w] = strand ? ~v : v;
    }
    if (p.ws.q_noff) {
        uint32_t *nw = reinterpret_cast<uint32_t *>(rec + p.ws.q_noff);
        for (uint32_t w = 0; 32u * w < m; ++w) {
            const uint64_t pos = off + 32u * w, last = off + (32u * w + 31u < m ? 32u * w + 31u : m - 1u);
            const uint32_t lo = p.reads.nmask[pos >> 5], hi = (last >> 5) > (pos >> 5) ? p.reads.nmask[(pos >> 5) + 1] : 0u;
            uint32_t v = __funnelshift_r(lo, hi, (uint32_t)(pos & 31));
            if (32u * w + 32u > m) v &= (1u << (m - 32u * w)) - 1u;   // bits past the read's end are not N
            nw[w] = v;
        }
    }
    const BcBwtDev &Y = p.ix.bwt[strand ? 1 : 0];       // opposite direction of the search index
    const bool seed_on = p.o.seed_len > 0 && (uint32_t)p.o.seed_len < m;
    uint64_t lookups = 0;
    if (seed_on) piece_thresholds<LAY>(p.reads, off, strand, Y, 0, p.o.seed_len, p.o.seed_z, rec + p.ws.q_soff, lookups);
    piece_thresholds<LAY>(p.reads, off, strand, Y, 0, (int)m, p.o.z, rec, lookups);
    atomicAdd((unsigned long long *)&p.ws.ctr[BC_CTR_DLOOKUPS], (unsigned long long)lookups);
}

}  // namespace

cudaError_t bc_launch_prepare(const BcSearchParams &p, cudaStream_t st) {
    if (p.ws.nq == 0) return cudaSuccess;
    if (p.ix.bwt[0].layout == 0) bc_prepare_kernel<0><<<(p.ws.nq + 127) / 128, 128, 0, st>>>(p);
    else bc_prepare_kernel<1><<<(p.ws.nq + 127) / 128, 128, 0, st>>>(p);
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
//   mhi = seed_d (0-7) | rem (8-15) | m-1 (16-23);  rem = the query's budget - d, the differences still affordable
//         (the kernel never needs d itself except when a hit is emitted: d = budget - rem)
//   run entries also carry the base they match next (mlo bits 27-29) and the end of their run - 1 (mhi 24-31)
//   mlo bit 30 (BC_FREE_BIT): this state may change warps (always in the exhaustive mode; best-stratum mode: only
//   states of a read's LAST round, whose outcome no verdict waits for)
// Per warp: a RING of BRANCH states (some difference is affordable at their position), whose cold bottom
// spills to global memory in blocks of 32, and two stacks of RUN states (see the kernel's comment).
#define BC_FREE_BIT 0x40000000u
#ifndef BC_POLLERS_PER_CTA
#define BC_POLLERS_PER_CTA 8u          /* idle warps per CTA that stay to take donated blocks (build-time gene; measured 1 / 3 / 8) */
#endif
#ifndef BC_FAIR_DIV
#define BC_FAIR_DIV 4                   /* intake draws at most (queries left) / (BC_FAIR_DIV x warps) + 1 at a time (build-time gene) */
#endif
#ifndef BC_POLL_NS
#define BC_POLL_NS 8000
#endif
// Launch bounds (build-time genes of the autotuner).  The default flavour is compiled for up to 7 warps per CTA and
// 4 CTAs per SM (28 warps per SM at 72 registers: measured -2.8 % time on config 2 and -2.0 % on config 4 against 3 x 8
// warps at 80 registers; 5 x 6 and 6 x 5 warps at 64 registers spill and lose 6-7 %); a second flavour (256 threads,
// 3 CTAs, 80 registers) serves geometries with 8 warps per CTA.
#ifndef BC_SEARCH_MAX_THREADS
#define BC_SEARCH_MAX_THREADS 224
#endif
#ifndef BC_SEARCH_MIN_CTAS
#define BC_SEARCH_MIN_CTAS 4
#endif

__device__ __forceinline__ void ent_store(uint2 *P, uint32_t idx, uint32_t qid, uint32_t k, uint32_t s, uint32_t k2,
                                          uint32_t mlo, uint32_t mhi) {
    uint2 *e = P + idx * 3u;
    e[0] = make_uint2(qid, k); e[1] = make_uint2(s, k2); e[2] = make_uint2(mlo, mhi);
}

// warp-aggregated append of raw hits (A5); called by all 32 lanes
// d = budget - rem: the batch's z, or the read's own current budget in the best-stratum mode (qz != nullptr)
__device__ __noinline__ void emit_hits(BcRawHit *arena, unsigned long long arena_cap, uint32_t *qcnt,
                                       unsigned long long *ctr, bool emit, uint32_t qid, uint32_t kf, uint32_t s, uint32_t rem,
                                       uint32_t z, const uint8_t *qz) {
    const uint32_t lane = threadIdx.x & 31u;
    uint32_t emask = __ballot_sync(0xffffffffu, emit);
    if (emask == 0) return;
    unsigned long long base = 0;
    int leader = __ffs(emask) - 1;
    if ((int)lane == leader) base = atomicAdd(&ctr[BC_CTR_ARENA], (unsigned long long)__popc(emask));
    base = __shfl_sync(0xffffffffu, base, leader);
    if (emit) {
        unsigned long long pos = base + __popc(emask & ((1u << lane) - 1u));
        const uint32_t d = (qz ? (uint32_t)__ldcg(qz + (qid >> 1)) : z) - rem;
        if (pos < arena_cap) arena[pos] = BcRawHit{qid, kf, kf + s - 1u, d};
        atomicAdd(&qcnt[qid], 1u);
    }
}

// per-warp statistics: n_xsect is per lane (second sectors of a rank pair), the rest warp-uniform
__device__ __noinline__ void flush_stats(unsigned long long *ctr, uint32_t lane, uint32_t n_cnodes, uint32_t n_xsect,
                                         uint32_t n_bsteps, uint32_t n_bnodes, uint32_t n_csteps, uint32_t n_cancel,
                                         uint32_t n_spill, uint32_t sect) {
    uint32_t x = n_xsect;
    for (int o = 16; o > 0; o >>= 1) x += __shfl_down_sync(0xffffffffu, x, o);
    if (lane == 0) {
        const unsigned long long nodes = (unsigned long long)n_cnodes + n_bnodes;
        atomicAdd(&ctr[BC_CTR_NODES], nodes);
        atomicAdd(&ctr[BC_CTR_LOOKUPS], 2ull * nodes);
        atomicAdd(&ctr[BC_CTR_LINES], (nodes + x) * sect);   // rank units read (one per node + the pairs that straddle two) x sectors per unit
        atomicAdd(&ctr[BC_CTR_BSTEPS], (unsigned long long)n_bsteps);
        atomicAdd(&ctr[BC_CTR_BNODES], (unsigned long long)n_bnodes);
        atomicAdd(&ctr[BC_CTR_CSTEPS], (unsigned long long)n_csteps);
        atomicAdd(&ctr[BC_CTR_CANCEL], (unsigned long long)n_cancel);
        atomicAdd(&ctr[BC_CTR_SPILL], (unsigned long long)n_spill);
    }
}

// ---- query record access (layout in bc_ws.cuh) ------------------------------------------------
struct QThr { uint32_t dlo, dhi, s; const uint8_t *rec; };

template <bool SMALL>
__device__ __forceinline__ QThr load_thr(const uint8_t *rec) {
    QThr q; q.rec = rec; q.dlo = q.dhi = q.s = 0;
    if (SMALL) { const uint4 v = __ldg(reinterpret_cast<const uint4 *>(rec)); q.dlo = v.x; q.dhi = v.y; q.s = v.z; }
    return q;
}
template <bool SMALL>
__device__ __forceinline__ uint32_t thr_d(const QThr &q, int r) {             // smallest t with D[t] <= r
    if (SMALL) return __byte_perm(q.dlo, q.dhi, (uint32_t)r) & 255u;
    return __ldg(q.rec + r);
}
template <bool SMALL>
__device__ __forceinline__ uint32_t thr_s(const QThr &q, int r, uint32_t soff) {   // ... with Ds[t] <= r
    if (SMALL) return (q.s >> (8u * (uint32_t)r)) & 255u;
    return __ldg(q.rec + soff + r);
}
template <bool HAS_N>
__device__ __forceinline__ uint32_t q_base(const uint8_t *rec, uint32_t boff, uint32_t noff, uint32_t t) {
    const uint32_t w = __ldg(reinterpret_cast<const uint32_t *>(rec + boff) + (t >> 4));
    uint32_t c = (w >> (2u * (t & 15u))) & 3u;
    if (HAS_N) {
        const uint32_t nm = __ldg(reinterpret_cast<const uint32_t *>(rec + noff) + (t >> 5));
        if ((nm >> (t & 31u)) & 1u) c = 4u;
    }
    return c;
}
// the same by query number, with 32-bit word arithmetic (the host refuses batches whose records exceed 2^34 bytes)
template <bool HAS_N>
__device__ __forceinline__ uint32_t q_base_at(const uint8_t *qrec, uint32_t qid, uint32_t qstride, uint32_t boff, uint32_t noff,
                                              uint32_t t) {
    const uint32_t *W = reinterpret_cast<const uint32_t *>(qrec);
    const uint32_t r = qid * (qstride >> 2);
    const uint32_t w = __ldg(W + (r + (boff >> 2) + (t >> 4)));
    uint32_t c = (w >> (2u * (t & 15u))) & 3u;
    if (HAS_N) {
        const uint32_t nm = __ldg(W + (r + (noff >> 2) + (t >> 5)));
        if ((nm >> (t & 31u)) & 1u) c = 4u;
    }
    return c;
}

// First position at which a state with `rem` differences left, seed differences sdc can afford ANY difference:
// before it the D / Ds bounds (or a spent seed budget) leave exact matching as the only move.  rem == 0: the
// read's end.  A value that is too SMALL only sends the state to a branch step early, which applies every rule itself.
//   mismatch / insertion at t need D[t+1] <= rem-1, i.e. t >= thrD[rem-1] - 1 (deletions one later);
//   inside the seed also sdc < seed_z and Ds[t+1] <= seed_z-sdc-1.
// With E == 0 a deletion may precede W[0] outside the seed rule and follow W[m-1]; runs are then used for
// spent budgets only (tests only; every config has E = 5).
template <bool SMALL>
__device__ __forceinline__ uint32_t run_end(const QThr &q, int rem, int sdc, int seed_z, bool seed_on,
                                            uint32_t seed_len, uint32_t m, bool e0, uint32_t soff) {
    if (rem <= 0) return m;
    if (e0) return 0u;
    uint32_t te = thr_d<SMALL>(q, rem - 1);
    te = te ? te - 1u : 0u;
    if (seed_on) {
        uint32_t ts = seed_len;
        if (sdc < seed_z) { ts = thr_s<SMALL>(q, seed_z - sdc - 1, soff); ts = ts ? ts - 1u : 0u; }
        te = te > ts ? te : ts;
    }
    return te;
}

// ---------------------------------------------------------------------------------------------
// RUN steps (see the kernel's header comment): while the stack of strand S holds a warp's worth of run
// states (or, when draining, anything at all), pop 32, extend each by ONE exactly matching base -- one
// symbol's rank at both interval ends -- and push the survivors back compacted.  A state whose run ends
// (t == its run end) is a hit if the read is consumed, else it moves to the branch ring.  Flat cost per
// node whatever the run lengths; lanes are full whenever 32 states are pending.
// Strand 0 (searched on the reverse index) also advances the forward interval start k2 by the
// bidirectional update of SURVEY C7 (R): '$' + the symbols smaller than c inside the interval.
// Stack layout inside the run area Cq[0..CCAP): strand 1 grows up from 0, strand 0 down from CCAP-1.
// The caller guarantees 32 free ring slots per iteration (the loop re-checks).
// ---------------------------------------------------------------------------------------------
template <bool S0, bool HAS_N, int LD, int LAY>
__device__ __forceinline__ void chain_steps(const BcSearchParams &p, const uint4 *lines, uint32_t primary,
                                            const uint32_t *Cs, uint2 *Cq, uint32_t CCAP, uint32_t &cnt,
                                            bool drain, uint2 *P, uint32_t bb, uint32_t &bcnt, uint32_t BCAP,
                                            unsigned long long *ctr, uint32_t z, const uint8_t *qz, uint32_t &n_nodes,
                                            uint32_t &n_xsect, uint32_t &n_steps) {
    const uint32_t lane = threadIdx.x & 31u, lt_mask = (1u << lane) - 1u, BM = BCAP - 1u;
    while ((cnt >= 32u || (drain && cnt > 0u)) && bcnt + 32u <= BCAP) {
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
        const uint32_t c = (mlo >> 27) & 7u, m = ((mhi >> 16) & 255u) + 1u, te = (mhi >> 24) + 1u;
        bool alive = false, emit = false, toring = false;
        if (act) {
            const uint32_t x1 = k + s;
            const uint32_t plo = k - (k > primary ? 1u : 0u), phi = x1 - (x1 > primary ? 1u : 0u);
            const bool two = bc_unit_id<LAY>(plo) != bc_unit_id<LAY>(phi);
            const BcUnit<LAY> rlo = bc_load_unit<LAY, LD>(lines, plo);
            n_xsect += two ? 1u : 0u;
            // strand 0 also needs one OTHER symbol's count for the forward start k2 (see below):
            // x = A when c is A or C, x = T when c is G or T
            const uint32_t x = c < 2u ? 0u : 3u;
            uint32_t olo = bc_unit_rank1(rlo, plo, c), ohi, xlo = 0, xhi = 0;
            if (S0) xlo = bc_unit_rank1(rlo, plo, x);
            if (two) {                                    // most narrow intervals sit in one unit
                const BcUnit<LAY> rhi = bc_load_unit<LAY, LD>(lines, phi);
                ohi = bc_unit_rank1(rhi, phi, c);
                if (S0) xhi = bc_unit_rank1(rhi, phi, x);
            } else {
                ohi = bc_unit_rank1(rlo, phi, c);
                if (S0) xhi = bc_unit_rank1(rlo, phi, x);
            }
            if (c <= 3u && ohi != olo) {
                if (S0) {
                    // children split the forward interval in the order $,A,C,G,T:
                    //   A: k2 + dollar;  C: k2 + dollar + nA;  G: k2 + s - nT - nG;  T: k2 + s - nT
                    const uint32_t dollar = s - (phi - plo), nx = xhi - xlo, nc_ = ohi - olo;
                    k2 = c == 0u ? k2 + dollar : (c == 1u ? k2 + dollar + nx : (c == 2u ? k2 + s - nx - nc_ : k2 + s - nc_));
                }
                k = p.ix.bwt[S0 ? 1 : 0].C[c] + olo + 1u; s = ohi - olo; ++t;
                const bool done = t == te;
                emit = done && t == m; toring = done && !emit; alive = !done;
            }
        }
        uint32_t nb = 0;
        if (alive) nb = q_base_at<HAS_N>(p.ws.qrec, qid, p.ws.qstride, p.ws.q_boff, p.ws.q_noff, t);
        const uint32_t smask = __ballot_sync(0xffffffffu, alive);
        if (alive) {
            const uint32_t r = __popc(smask & lt_mask);
            ent_store(Cq, S0 ? CCAP - 1u - cnt - r : cnt + r, qid, k, s, k2, (mlo & 0x47FFFE00u) | t | (nb << 27), mhi);
        }
        cnt += __popc(smask);
        const uint32_t rmask = __ballot_sync(0xffffffffu, toring);
        if (toring)      // a run consists of matches: gap state M, budgets unchanged
            ent_store(P, (bb + bcnt + __popc(rmask & lt_mask)) & BM, qid, k, s, k2, (mlo & 0x47FFF800u) | t, mhi & 0x00FFFFFFu);
        bcnt += __popc(rmask);
        if (__any_sync(0xffffffffu, emit))
            emit_hits(p.ws.arena, p.ws.arena_cap, p.ws.qcnt, ctr, emit, qid, S0 ? k2 : k, s, (mhi >> 8) & 255u, z, qz);
        __syncwarp();
    }
}

// Root states of up to 32 queries (one per lane, `want`), each with `budget` differences to spend: dropped if its
// D[0] / Ds[0] bounds already exceed the budgets, else pushed on the branch ring or -- when no
// difference is affordable at W[0] -- on its strand's run stack.  The caller guarantees room for 32 entries.
template <bool SMALL, bool HAS_N>
__device__ __forceinline__ void push_roots(const BcSearchParams &p, bool want, uint32_t q, int budget, uint2 *P, uint32_t bb,
                                           uint32_t &bcnt, uint32_t BM, uint2 *Cq, uint32_t CCAP, uint32_t &c0, uint32_t &c1,
                                           bool e0, bool free_state) {
    const uint32_t lane = threadIdx.x & 31u, lt_mask = (1u << lane) - 1u;
    const uint32_t full = p.ix.bwt[0].n + 1;
    const int seed_len = p.o.seed_len, seed_z = p.o.seed_z;
    bool ok = want;
    uint32_t m = 0, te = 0, b0 = 0;
    if (ok) {
        m = p.reads.len[q >> 1];
        ok = m >= 1 && m <= p.reads.max_len;
    }
    if (ok) {
        const uint8_t *rec = p.ws.qrec + (size_t)q * p.ws.qstride;
        const QThr th = load_thr<SMALL>(rec);
        const bool seed_on = seed_len > 0 && seed_len < (int)m;
        ok = thr_d<SMALL>(th, budget) == 0u && (!seed_on || thr_s<SMALL>(th, seed_z, p.ws.q_soff) == 0u);
        te = run_end<SMALL>(th, budget, 0, seed_z, seed_on, (uint32_t)seed_len, m, e0, p.ws.q_soff);
        b0 = q_base<HAS_N>(rec, p.ws.q_boff, p.ws.q_noff, 0u);
    }
    const bool odd = (q & 1u) != 0, run = ok && te > 0u;
    const uint32_t maskb = __ballot_sync(0xffffffffu, ok && !run);
    const uint32_t mask1 = __ballot_sync(0xffffffffu, run && odd), mask0 = __ballot_sync(0xffffffffu, run && !odd);
    const uint32_t hi = ((uint32_t)budget << 8) | ((m - 1u) << 16);
    if (ok) {
        const uint32_t fb = free_state ? BC_FREE_BIT : 0u;
        if (!run) ent_store(P, (bb + bcnt + __popc(maskb & lt_mask)) & BM, q, 0u, full, 0u, fb, hi);
        else ent_store(Cq, odd ? c1 + __popc(mask1 & lt_mask) : CCAP - 1u - c0 - __popc(mask0 & lt_mask), q,
                       0u, full, 0u, (b0 << 27) | fb, hi | ((te - 1u) << 24));
    }
    bcnt += __popc(maskb); c1 += __popc(mask1); c0 += __popc(mask0);
    __syncwarp();
}

// ---------------------------------------------------------------------------------------------
// A3 + A4 + A5.  Persistent kernel, one LIFO pool per warp, two kinds of state and of step:
//  * BRANCH step: up to 32 branch states are popped, one per lane, and expanded in lock step:
//    all four child intervals from one rank4 pair (1-2 index sectors) -> match, <=3 mismatch,
//    <=4 deletion and 1 insertion children, pruned by the budgets and D/Ds.  Every lane counts its
//    surviving children, a warp scan assigns pool slots, and each lane writes its own children.
//  * RUN steps: a state that can afford no difference before position `te` -- its budget is spent
//    (te = m), its seed budget is spent (te = seed_len), or the D / Ds bounds say so -- can only match
//    exactly until there.  Such states live on two stacks (one per strand); whenever a stack holds 32,
//    32 are popped and each is extended by ONE exactly matching base (one symbol's rank at both interval
//    ends); survivors go back compacted, finished runs are emitted (t == m) or become branch states.
//    Flat cost per node, full lanes, whatever the run lengths.
// New queries are drawn from a global ticket counter whenever fewer than 32 branch states are
// pending, so lanes stay busy and converged whatever the shape of the individual search trees.
// Pool discipline: a multi-lane branch step keeps only the leading lanes whose children fit the ring
// and the run stacks; the others are un-popped (their entries are still in place).  The ring's cold
// bottom moves to a per-warp area of the workspace in blocks of 32 whenever fewer than 64 slots are
// free and comes back when the ring runs low; if that area is ever full the warp raises error bit 2
// (BC_E_NOMEM: the caller passes a larger spill area), never a silent truncation.
// ---------------------------------------------------------------------------------------------
template <bool SMALL, bool HAS_N, int LD, int LAY, bool W8>
__global__ void __launch_bounds__(W8 ? 256 : BC_SEARCH_MAX_THREADS, W8 ? 3 : BC_SEARCH_MIN_CTAS) bc_search_kernel(BcSearchParams p) {
    extern __shared__ uint2 pool_mem[];
    __shared__ __align__(16) uint32_t Ctab[8];                               // C[c] of the index each strand searches
    __shared__ uint32_t cta_poller;                                          // warps of this CTA that have become pollers
    // rarely touched per-lane / per-warp variables live in shared memory, not in registers of the hot loop:
    __shared__ uint2 best_lane[256];                       // best mode: {read, budget | state << 8} of this lane's read
    __shared__ uint32_t warp_flags[8];              // bit 0 poller, 1 counted idle, 2 best mode done
    const uint32_t lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
    const uint32_t BCAP = p.bcap, CCAP = p.ccap, BM = p.bcap - 1u;
    uint2 *P = pool_mem + (size_t)warp * 3u * (BCAP + CCAP);     // branch ring: slots (bb + i) & BM
    uint2 *Cq = P + 3u * BCAP;                                    // run area: strand 1 up from 0, strand 0 down from CCAP-1
    uint2 *G = p.ws.spill + ((size_t)blockIdx.x * (blockDim.x >> 5) + warp) * ((size_t)p.ws.spill_blocks * 96u);
    const uint32_t GB = p.ws.spill_blocks;
    const uint32_t lt_mask = (1u << lane) - 1u;
    const int z = p.o.z, E = p.o.indel_end_skip, max_go = p.o.max_gap_open, max_ge = p.o.max_gap_ext;
    const int seed_len = p.o.seed_len, seed_z = p.o.seed_z;
    const bool e0 = E == 0;
    const uint32_t nq = p.ws.nq, n_reads = p.ws.nq >> 1;
    const uint32_t full = p.ix.bwt[0].n + 1;
    const bool best = p.best != 0;                  // best-stratum mode: per-read budgets in qz[]
    const uint8_t *qz = best ? p.ws.qz : nullptr;
    const uint32_t qstride = p.ws.qstride, soff = p.ws.q_soff, boff = p.ws.q_boff, noff = p.ws.q_noff;
    unsigned long long *ctr = (unsigned long long *)p.ws.ctr;
    const uint4 *lines0 = p.ix.bwt[1].lines, *lines1 = p.ix.bwt[0].lines;  // strand 0 searches the reverse index
    const uint32_t primary0 = p.ix.bwt[1].primary, primary1 = p.ix.bwt[0].primary;

    if (threadIdx.x < 8) Ctab[threadIdx.x] = p.ix.bwt[threadIdx.x < 4 ? 1 : 0].C[threadIdx.x & 3];
    if (threadIdx.x == 0) cta_poller = 0u;
    __syncthreads();
    // A4, state-level redistribution ACROSS warps: a busy warp that is about to spill the bottom of its ring gives that
    // block of 32 pending states away instead (through the exchange buffer of the workspace) if some warp has run out
    // of work; warps that are out of work stay behind as pollers and take such blocks (protocol and termination: the
    // "out of work" branch of the main loop, and DESIGN.md 6).  Only blocks whose 32 states all carry BC_FREE_BIT move.
#define QN (p.ws.sq_n)                                /* read from the parameter bank where needed: no register */
#define sq_flag ((volatile uint32_t *)p.ws.sq_flag)  /* per slot: 0 free, 3 being written, 1 ready, 2 being read */
    best_lane[threadIdx.x] = make_uint2(0u, 0u);     // state 0 free / 1 searching for the first hit / 2 final round
    if (lane == 0) warp_flags[warp] = 0u;
    __syncwarp();
#define WF_POLLER 1u
#define WF_COUNTED 2u
#define WF_BESTDONE 4u
    // warps that have STARTED: with more CTAs in the grid than fit on the machine the others start only when these
    // leave, so "everybody idle" must mean everybody who runs (a late CTA finds no tickets and no blocks, and leaves)
    if (lane == 0 && QN) atomicAdd(&ctr[BC_CTR_STARTED], 1ull);
    uint32_t bb = 1u << 24, bcnt = 0, c0 = 0, c1 = 0, gsp = 0, pool_max = 0;   // ring bottom, counts (branch, run per strand), spilled blocks
    bool more = true, force_drain = false;
    // 32-bit statistics, flushed to the 64-bit global counters at every intake and at the end
    uint32_t n_cnodes = 0, n_xsect = 0, n_bsteps = 0, n_bnodes = 0, n_csteps = 0, n_cancel = 0, n_spill = 0;

    for (;;) {
        // ---- ring <-> global: keep the hot top of the branch stack on chip, >= 64 slots free ----------
        while (bcnt >= 32u && bcnt + 64u > BCAP) {                             // move the bottom 32 entries out
            const uint2 *src = P + ((bb + lane) & BM) * 3u;
            uint32_t slot = 0xFFFFFFFFu;
            if (QN) {                                                          // somebody idle?  give the block away
                const bool all_free = __all_sync(0xffffffffu, (src[2].x & BC_FREE_BIT) != 0u);
                if (lane == 0 && all_free && *(volatile unsigned long long *)&ctr[BC_CTR_GIDLE] > 0ull)
                    for (uint32_t a = 0; a < 4u && slot == 0xFFFFFFFFu; ++a) {
                        const uint32_t s_ = ((blockIdx.x * 8u + warp) * 7u + a * 61u + n_spill + gsp + bb) % QN;
                        if (atomicCAS(const_cast<uint32_t *>(&sq_flag[s_]), 0u, 3u) == 0u) slot = s_;
                    }
                slot = __shfl_sync(0xffffffffu, slot, 0);
            }
            if (slot != 0xFFFFFFFFu) {
                uint2 *dst = p.ws.sq_buf + ((size_t)slot * 32u + lane) * 3u;
                dst[0] = src[0]; dst[1] = src[1]; dst[2] = src[2];
                __threadfence();
                __syncwarp();
                if (lane == 0) {
                    atomicExch(const_cast<uint32_t *>(&sq_flag[slot]), 1u);
                    atomicAdd(&ctr[BC_CTR_QREADY], 1ull);
                }
            } else {
                if (gsp >= GB) break;
                uint2 *dst = G + ((size_t)gsp * 32u + lane) * 3u;
                dst[0] = src[0]; dst[1] = src[1]; dst[2] = src[2];
                ++gsp; ++n_spill;
                if (lane == 0 && (gsp & 7u) == 0u) atomicMax(&ctr[BC_CTR_SPILLMAX], (unsigned long long)gsp);   // (to a multiple of 8)
            }
            bb += 32u; bcnt -= 32u;
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
        // ---- intake: new root states ---------------------------------------------------------------
        if (!best) {
            // exhaustive mode: new queries whenever the branch stack is shallow
            if (more && bcnt < 32u && gsp == 0u && c0 + c1 + 32u <= CCAP) {
                flush_stats(ctr, lane, n_cnodes, n_xsect, n_bsteps, n_bnodes, n_csteps, n_cancel, n_spill, bc_unit_sectors<LAY>());
                n_cnodes = n_xsect = n_bsteps = n_bnodes = n_csteps = n_cancel = n_spill = 0;
                uint32_t need = 32u - bcnt;
                unsigned long long tk = 0;
                if (lane == 0) {
                    // towards the end of the batch take fewer queries at a time, so that the last heavy
                    // trees are spread over the warps instead of queueing behind one another
                    const unsigned long long seen = *(volatile unsigned long long *)&ctr[BC_CTR_TICKET];
                    const unsigned long long left = seen < nq ? nq - seen : 0ull;
                    const unsigned long long fair = left / ((unsigned long long)BC_FAIR_DIV * gridDim.x * (blockDim.x >> 5)) + 1ull;
                    if (fair < need) need = (uint32_t)fair;
                    tk = atomicAdd(&ctr[BC_CTR_TICKET], (unsigned long long)need);
                }
                need = __shfl_sync(0xffffffffu, need, 0);
                tk = __shfl_sync(0xffffffffu, tk, 0);
                if (tk + need >= nq) more = false;
                const unsigned long long q = tk + lane;
                push_roots<SMALL, HAS_N>(p, lane < need && q < nq, (uint32_t)q, z, P, bb, bcnt, BM, Cq, CCAP, c0, c1, e0, true);
            }
        } else if (bcnt == 0u && c0 + c1 == 0u && gsp == 0u) {
            // best-stratum mode: one read per lane, searched with ITS OWN budget, round by round.  All of
            // the warp's trees are finished here, so each lane can judge its read by the raw hits counted so far:
            //   no hit yet  -> same read again with budget + 1 (up to z);
            //   first hits  -> they all have d = budget = d_min; one more round at min(d_min + plus, z) if that is
            //                  larger (its hits are exactly the wanted set; the earlier ones are in it: duplicates
            //                  with equal d, which the dedup of A6 removes), else done.
            // Free lanes draw new reads.  Nothing with d > d_min + plus is ever explored.
            flush_stats(ctr, lane, n_cnodes, n_xsect, n_bsteps, n_bnodes, n_csteps, n_cancel, n_spill, bc_unit_sectors<LAY>());
            n_cnodes = n_xsect = n_bsteps = n_bnodes = n_csteps = n_cancel = n_spill = 0;
            uint32_t my_read = best_lane[threadIdx.x].x, my_bud = best_lane[threadIdx.x].y & 255u, my_st = best_lane[threadIdx.x].y >> 8;
            if (my_st) {
                const uint32_t h = *(volatile uint32_t *)&p.ws.qcnt[2u * my_read] + *(volatile uint32_t *)&p.ws.qcnt[2u * my_read + 1u];
                if (my_st == 2u) my_st = 0u;
                else if (h > 0u) {
                    const uint32_t zf = my_bud + (uint32_t)p.plus < (uint32_t)z ? my_bud + (uint32_t)p.plus : (uint32_t)z;
                    if (zf > my_bud) { my_bud = zf; my_st = 2u; } else my_st = 0u;
                } else if (my_bud < (uint32_t)z) ++my_bud;
                else my_st = 0u;
            }
            const uint32_t freemask = __ballot_sync(0xffffffffu, my_st == 0u);
            if (more && freemask) {
                uint32_t need = __popc(freemask);
                unsigned long long tk = 0;
                if (lane == 0) {
                    const unsigned long long seen = *(volatile unsigned long long *)&ctr[BC_CTR_TICKET];
                    const unsigned long long left = seen < n_reads ? n_reads - seen : 0ull;
                    const unsigned long long fair = left / ((unsigned long long)BC_FAIR_DIV * gridDim.x * (blockDim.x >> 5)) + 1ull;
                    if (fair < need) need = (uint32_t)fair;
                    tk = atomicAdd(&ctr[BC_CTR_TICKET], (unsigned long long)need);     // tickets are READS in this mode
                }
                need = __shfl_sync(0xffffffffu, need, 0);
                tk = __shfl_sync(0xffffffffu, tk, 0);
                if (tk + need >= n_reads) more = false;
                const uint32_t rank = __popc(freemask & lt_mask);
                if (my_st == 0u && rank < need && tk + rank < n_reads) { my_read = (uint32_t)(tk + rank); my_bud = 0u; my_st = 1u; }
            }
            best_lane[threadIdx.x] = make_uint2(my_read, my_bud | (my_st << 8));
            if (!__any_sync(0xffffffffu, my_st != 0u)) { if (more) continue; if (lane == 0) warp_flags[warp] |= WF_BESTDONE; __syncwarp(); }
            else {
            if (my_st) __stcg(const_cast<uint8_t *>(qz) + my_read, (uint8_t)my_bud);
            { const uint32_t mb = __reduce_max_sync(0xffffffffu, my_st ? my_bud + 1u : 0u); if (lane == 0) atomicMax(&ctr[BC_CTR_PASSES], (unsigned long long)mb); }
            __syncwarp();
            // a round after which the read is done whatever it finds (its final round, or budget z) may share its states
            const bool last_round = my_st == 2u || my_bud >= (uint32_t)z;
            push_roots<SMALL, HAS_N>(p, my_st != 0u, 2u * my_read + 1u, (int)my_bud, P, bb, bcnt, BM, Cq, CCAP, c0, c1, e0, last_round);
            push_roots<SMALL, HAS_N>(p, my_st != 0u, 2u * my_read, (int)my_bud, P, bb, bcnt, BM, Cq, CCAP, c0, c1, e0, last_round);
            }
        }
        if (bcnt == 0 && c0 + c1 == 0) {
            if (more || (best && !(warp_flags[warp] & WF_BESTDONE))) continue;   // (best mode: the round logic above decides when the warp is done)
            if (!QN) break;
            // ---- out of work.  Count this warp idle; up to BC_POLLERS_PER_CTA idle warps of a CTA (default: all) stay as
            // pollers, further ones leave.
            flush_stats(ctr, lane, n_cnodes, n_xsect, n_bsteps, n_bnodes, n_csteps, n_cancel, n_spill, bc_unit_sectors<LAY>());
            n_cnodes = n_xsect = n_bsteps = n_bnodes = n_csteps = n_cancel = n_spill = 0;
            if (lane == 0) {
                if (!(warp_flags[warp] & WF_POLLER) && atomicAdd(&cta_poller, 1u) < BC_POLLERS_PER_CTA) warp_flags[warp] |= WF_POLLER;
                __threadfence();
                atomicAdd(&ctr[BC_CTR_GIDLE], 1ull);
                warp_flags[warp] |= WF_COUNTED;
            }
            __syncwarp();
            if (!(warp_flags[warp] & WF_POLLER)) break;
            // ---- poller: take donated blocks until every warp is idle and nothing is left in the exchange.
            // A thief un-counts itself BEFORE it tries to claim, so "all idle" (read first) followed by "nothing ready"
            // (read second) means every published block was claimed by a warp that will come back here.
            bool got = false;
            uint32_t spins = 0;
            for (;;) {
                unsigned long long idle = 0, ready = 0, err = 0, started = 0;
                if (lane == 0) {
                    started = *(volatile unsigned long long *)&ctr[BC_CTR_STARTED];
                    idle = *(volatile unsigned long long *)&ctr[BC_CTR_GIDLE];
                    __threadfence();
                    ready = *(volatile unsigned long long *)&ctr[BC_CTR_QREADY];
                    err = *(volatile unsigned long long *)&ctr[BC_CTR_ERROR];
                }
                idle = __shfl_sync(0xffffffffu, idle, 0); ready = __shfl_sync(0xffffffffu, ready, 0);
                err = __shfl_sync(0xffffffffu, err, 0); started = __shfl_sync(0xffffffffu, started, 0);
                if (err) break;
                if (++spins > (1u << 27)) { if (lane == 0) atomicOr(&ctr[BC_CTR_ERROR], 2ull); break; }   // ~18 min of polling: a bug, not a wait
                if (ready > 0ull) {
                    if (lane == 0) atomicAdd(&ctr[BC_CTR_GIDLE], ~0ull);                  // -1: not idle while claiming
                    uint32_t slot = 0xFFFFFFFFu;
                    for (uint32_t base = 0; base < QN && slot == 0xFFFFFFFFu; base += 32u) {
                        const uint32_t s_ = ((blockIdx.x * 8u + warp) * 13u + base + lane) % QN;
                        uint32_t mk = __ballot_sync(0xffffffffu, sq_flag[s_] == 1u);
                        while (mk && slot == 0xFFFFFFFFu) {
                            const int l = __ffs(mk) - 1;
                            mk &= mk - 1u;
                            const uint32_t cand = __shfl_sync(0xffffffffu, s_, l);
                            uint32_t ok = 0;
                            if (lane == 0) ok = atomicCAS(const_cast<uint32_t *>(&sq_flag[cand]), 1u, 2u) == 1u ? 1u : 0u;
                            if (__shfl_sync(0xffffffffu, ok, 0)) slot = cand;
                        }
                    }
                    if (slot != 0xFFFFFFFFu) {
                        if (lane == 0) atomicAdd(&ctr[BC_CTR_QREADY], ~0ull);
                        const uint2 *src = p.ws.sq_buf + ((size_t)slot * 32u + lane) * 3u;
                        uint2 *dst = P + ((bb + lane) & BM) * 3u;
                        dst[0] = __ldcg(src); dst[1] = __ldcg(src + 1); dst[2] = __ldcg(src + 2);
                        bcnt = 32u;
                        __syncwarp();
                        if (lane == 0) { __threadfence(); atomicExch(const_cast<uint32_t *>(&sq_flag[slot]), 0u); atomicAdd(&ctr[BC_CTR_STEALS], 1ull); }
                        if (lane == 0) warp_flags[warp] &= ~WF_COUNTED;
                        got = true;
                        break;
                    }
                    if (lane == 0) atomicAdd(&ctr[BC_CTR_GIDLE], 1ull);
                } else if (idle >= started) break;
                __nanosleep(BC_POLL_NS);
            }
            if (!got) break;
            continue;
        }
        pool_max = bcnt + c0 + c1 > pool_max ? bcnt + c0 + c1 : pool_max;

        if (c1 >= 32u || c0 >= 32u || ((bcnt == 0 || force_drain) && c0 + c1 > 0u)) {
            if (bcnt + 32u > BCAP) { if (lane == 0) atomicOr(&ctr[BC_CTR_ERROR], 4ull); break; }   // spill area exhausted
            const bool drain = bcnt == 0 || force_drain;
            chain_steps<false, HAS_N, LD, LAY>(p, lines1, primary1, Ctab + 4, Cq, CCAP, c1, drain, P, bb, bcnt, BCAP, ctr, (uint32_t)z, qz, n_cnodes, n_xsect, n_csteps);
            chain_steps<true, HAS_N, LD, LAY>(p, lines0, primary0, Ctab, Cq, CCAP, c0, drain, P, bb, bcnt, BCAP, ctr, (uint32_t)z, qz, n_cnodes, n_xsect, n_csteps);
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
        const int sd = mhi & 255, rem = (mhi >> 8) & 255, m = (int)((mhi >> 16) & 255) + 1;
        const uint32_t strand = qid & 1u;
        const bool seed_on = seed_len > 0 && seed_len < m;
        const bool has_base = act && t < m;
        const bool del_ok = act && st != 1 && t >= E && m - t >= E;
        const bool ins_ok = has_base && st != 2 && t >= E && m - 1 - t >= E;
        const uint8_t *rec = p.ws.qrec + (size_t)qid * qstride;
        QThr th = load_thr<SMALL>(act ? rec : p.ws.qrec);
        uint32_t qb = 4u, qb1 = 4u;                      // W[t], W[t+1] of the query (4 = N / none)
        if (has_base) {
            qb = q_base<HAS_N>(rec, boff, noff, (uint32_t)t);
            if (t + 1 < m) qb1 = q_base<HAS_N>(rec, boff, noff, (uint32_t)t + 1u);
        }
        uint32_t nk[4] = {0, 0, 0, 0}, ns[4] = {0, 0, 0, 0}, nk2[4] = {0, 0, 0, 0};
        bool straddle = false;
        if (has_base || del_ok) {
            const uint4 *lines = strand ? lines1 : lines0;
            const uint32_t primary = strand ? primary1 : primary0;
            const uint32_t x1 = k + s;
            const uint32_t plo = k - (k > primary ? 1u : 0u), phi = x1 - (x1 > primary ? 1u : 0u);
            uint32_t olo[4], ohi[4];
            straddle = bc_unit_id<LAY>(plo) != bc_unit_id<LAY>(phi);
            const BcUnit<LAY> ulo = bc_load_unit<LAY, LD>(lines, plo);
            bc_unit_rank4(ulo, plo, olo);
            if (LAY == 0) {                              // blocks: a second unconditional load (predicating it on "other
                bc_unit_rank4(bc_load_unit<LAY, LD>(lines, phi), phi, ohi);   // block" was measured 3 % slower here)
            } else if (straddle) {
                bc_unit_rank4(bc_load_unit<LAY, LD>(lines, phi), phi, ohi);
            } else bc_unit_rank4(ulo, phi, ohi);
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
        // class-level validity and packed child state (same for every child of a class).  A child that costs a
        // difference has rem-1 = nrem left and needs D <= nrem at ITS position: t+1 for mismatch / insertion, t for a
        // deletion; inside the seed the same with Ds and the seed budget (zero thresholds outside / seed off).
        const int nrem = rem - 1, sdb = sd + in_seed_base, sdd = sd + in_seed_del;
        const uint32_t tn = (uint32_t)t + 1u;
        const bool bud = act && rem >= 1;
        const uint32_t thD = bud ? thr_d<SMALL>(th, nrem) : 0u;
        const bool v_base = bud && has_base && sdb <= seed_z && tn >= thD && tn >= thr_s<SMALL>(th, sdb <= seed_z ? seed_z - sdb : 0, soff);
        const int d_go = go + (st != 2), d_ge = ge + (st == 2), i_go = go + (st != 1), i_ge = ge + (st == 1);
        const bool v_mm = v_base;
        const bool v_ins = v_base && ins_ok && i_go <= max_go && i_ge <= max_ge;
        const bool v_del = bud && del_ok && d_go <= max_go && d_ge <= max_ge && sdd <= seed_z && (uint32_t)t >= thD &&
                           (uint32_t)t >= thr_s<SMALL>(th, sdd <= seed_z ? seed_z - sdd : 0, soff);
        // where the children go: the end of the run a child starts with (te > its position: run stack)
        const uint32_t te_b = run_end<SMALL>(th, nrem, sdb, seed_z, seed_on, (uint32_t)seed_len, (uint32_t)m, e0, soff);
        const uint32_t te_d = in_seed_del == in_seed_base ? te_b
                              : run_end<SMALL>(th, nrem, sdd, seed_z, seed_on, (uint32_t)seed_len, (uint32_t)m, e0, soff);
        const bool run_b = te_b > tn, run_d = te_d > (uint32_t)t;
        const uint32_t nrem8 = (uint32_t)(nrem & 255) << 8;
        const uint32_t fb = mlo & BC_FREE_BIT;
        const uint32_t ma_lo = tn | ((uint32_t)go << 11) | ((uint32_t)ge << 19) | fb;
        const uint32_t ma_hi = (uint32_t)sd | ((uint32_t)rem << 8) | m_bits;
        const uint32_t mm_hi = (uint32_t)sdb | nrem8 | m_bits | (run_b ? (te_b - 1u) << 24 : 0u);
        const uint32_t de_lo = (uint32_t)t | (2u << 9) | ((uint32_t)d_go << 11) | ((uint32_t)d_ge << 19) | fb;
        const uint32_t de_hi = (uint32_t)sdd | nrem8 | m_bits | (run_d ? (te_d - 1u) << 24 : 0u);
        const uint32_t in_lo = tn | (1u << 9) | ((uint32_t)i_go << 11) | ((uint32_t)i_ge << 19) | fb;
        const uint32_t cb0 = run_d ? qb << 27 : 0u, cb1 = run_b ? qb1 << 27 : 0u;   // first base of a run child
        const bool last1 = nrem == 0;                    // children that cost a difference exhaust the budget
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
        const uint32_t keep_t = e0 ? (last1 ? 1u : 0x3FFu) : 0u;
        uint32_t pbits = vbits & (~tbits | keep_t);
        uint32_t cbits = pbits & ((run_b ? 0x21Eu : 0u) | (run_d ? 0x1E0u : 0u));
        const uint32_t cshift = strand ? 10u : 20u;      // packed counters: branch (bits 0-9) | run strand 1 (10-19) | strand 0 (20-29)

        // slots: warp scan of (branch pushes | run pushes << 10/20); net growth decides who is kept
        const uint32_t mine = (uint32_t)__popc(pbits & ~cbits) | ((uint32_t)__popc(cbits) << cshift);
        uint32_t incl = mine;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t v = __shfl_up_sync(0xffffffffu, incl, o);
            if ((int)lane >= o) incl += v;
        }
        // lanes 0..lane kept, the lanes behind un-popped: ring and run-stack occupancy after the step
        const uint32_t ring_if = bcnt - (lane + 1u) + (incl & 1023u);
        const uint32_t chain_if = c0 + c1 + ((incl >> 10) & 1023u) + (incl >> 20);
        const bool fits = act && ring_if <= BCAP && chain_if <= CCAP;
        uint32_t keepmask = __ballot_sync(0xffffffffu, fits);
        uint32_t akeep = keepmask == 0xffffffffu ? 32u : (uint32_t)(__ffs(~keepmask) - 1);   // leading run
        if (akeep > a) akeep = a;
        if (akeep == 0) {                                 // not even lane 0 fits
            const uint32_t ch0 = __shfl_sync(0xffffffffu, chain_if, 0);
            if (ch0 <= CCAP) { if (lane == 0) atomicOr(&ctr[BC_CTR_ERROR], 4ull); break; }   // ring full and nowhere to spill
            force_drain = true;                           // nothing popped; make room on the run stacks first
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
            if (pbits & 1u) {                             // the match child stays a branch state (same d, same bounds)
                ent_store(P, (bpos++) & BM, qid, sel4(nk[0], nk[1], nk[2], nk[3], qb), sel4(ns[0], ns[1], ns[2], ns[3], qb),
                          sel4(nk2[0], nk2[1], nk2[2], nk2[3], qb), ma_lo, ma_hi);
            }
#pragma unroll
            for (int b = 0; b < 4; ++b) {
                if (pbits & (2u << b)) {
                    if (run_b) { ent_store(Cq, cpos, qid, nk[b], ns[b], nk2[b], ma_lo | cb1, mm_hi); cpos += cstep; }
                    else ent_store(P, (bpos++) & BM, qid, nk[b], ns[b], nk2[b], ma_lo, mm_hi);
                }
            }
#pragma unroll
            for (int b = 0; b < 4; ++b) {
                if (pbits & (32u << b)) {
                    if (run_d) { ent_store(Cq, cpos, qid, nk[b], ns[b], nk2[b], de_lo | cb0, de_hi); cpos += cstep; }
                    else ent_store(P, (bpos++) & BM, qid, nk[b], ns[b], nk2[b], de_lo, de_hi);
                }
            }
            if (pbits & 512u) {
                if (run_b) { ent_store(Cq, cpos, qid, k, s, k2, in_lo | cb1, mm_hi); cpos += cstep; }
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
                          (uint32_t)(slot == 0 ? rem : nrem), (uint32_t)z, qz);
            }
        }
        __syncwarp();
    }
    flush_stats(ctr, lane, n_cnodes, n_xsect, n_bsteps, n_bnodes, n_csteps, n_cancel, n_spill, bc_unit_sectors<LAY>());
    if (QN && lane == 0 && !(warp_flags[warp] & WF_COUNTED)) atomicAdd(&ctr[BC_CTR_GIDLE], 1ull);    // error exits: pollers must not wait for this warp
    if (lane == 0) {
        atomicMax(&ctr[BC_CTR_POOLMAX], (unsigned long long)pool_max);
    }
#undef QN
#undef sq_flag
#undef WF_POLLER
#undef WF_COUNTED
#undef WF_BESTDONE
}

template <bool SMALL, bool HAS_N, int LD, int LAY, bool W8>
cudaError_t launch_search_w(const BcSearchParams &p, int grid, int threads, size_t smem, cudaStream_t st) {
    cudaError_t e = cudaFuncSetAttribute(bc_search_kernel<SMALL, HAS_N, LD, LAY, W8>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    bc_search_kernel<SMALL, HAS_N, LD, LAY, W8><<<grid, threads, smem, st>>>(p);
    return cudaGetLastError();
}

template <bool SMALL, bool HAS_N, int LD, int LAY>
cudaError_t launch_search(const BcSearchParams &p, int grid, int threads, size_t smem, cudaStream_t st) {
    if (threads > BC_SEARCH_MAX_THREADS) return launch_search_w<SMALL, HAS_N, LD, LAY, true>(p, grid, threads, smem, st);
    return launch_search_w<SMALL, HAS_N, LD, LAY, false>(p, grid, threads, smem, st);
}

template <bool SMALL, bool HAS_N>
cudaError_t launch_search_ld(const BcSearchParams &p, int grid, int threads, size_t smem, cudaStream_t st) {
    if (p.ix.bwt[0].layout == 0)
        return p.ld_policy ? launch_search<SMALL, HAS_N, 1, 0>(p, grid, threads, smem, st) : launch_search<SMALL, HAS_N, 0, 0>(p, grid, threads, smem, st);
    return p.ld_policy ? launch_search<SMALL, HAS_N, 1, 1>(p, grid, threads, smem, st) : launch_search<SMALL, HAS_N, 0, 1>(p, grid, threads, smem, st);
}

}  // namespace

cudaError_t bc_launch_search(const BcSearchParams &p, int sm_count, uint32_t ctas_per_sm, uint32_t warps_per_cta,
                             cudaStream_t st) {
    if (p.ws.nq == 0) return cudaSuccess;
    const size_t smem = (size_t)warps_per_cta * (p.bcap + p.ccap) * BC_POOL_ENTRY_BYTES;
    const int grid = sm_count * (int)ctas_per_sm, threads = (int)warps_per_cta * 32;
    const bool small = p.o.z <= BC_QREC_SMALL_Z && p.o.seed_z <= BC_QREC_SMALL_SZ, has_n = p.ws.q_noff != 0;
    if (small) return has_n ? launch_search_ld<true, true>(p, grid, threads, smem, st) : launch_search_ld<true, false>(p, grid, threads, smem, st);
    return has_n ? launch_search_ld<false, true>(p, grid, threads, smem, st) : launch_search_ld<false, false>(p, grid, threads, smem, st);
}
