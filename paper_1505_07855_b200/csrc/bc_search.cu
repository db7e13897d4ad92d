// A1 query preparation + A2 D[] bounds (bc_prepare_kernel), A3-A5 inexact search with a per-warp
// state pool in shared memory (bc_search_kernel).  sm_100a only; integer arithmetic only.
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

// all four O(., j) for the two ends of an interval [k, k+s-1]: olo = O(., k-1), ohi = O(., k+s-1)
__device__ __forceinline__ uint32_t rank_pair(const BcBwtDev &b, uint32_t k, uint32_t s, uint32_t olo[4], uint32_t ohi[4]) {
    uint32_t plo = bc_rank_pos(b, k), phi = bc_rank_pos(b, k + s);
    uint32_t llo = plo / BC_LINE_SYMS, lhi = phi / BC_LINE_SYMS;
    BcLineRegs L = bc_load_line(b.lines, llo);
    bc_line_rank4(L, plo - llo * BC_LINE_SYMS, olo);
    uint32_t n_lines = 1;
    if (lhi != llo) { L = bc_load_line(b.lines, lhi); n_lines = 2; }
    bc_line_rank4(L, phi - lhi * BC_LINE_SYMS, ohi);
    return n_lines;
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
                uint32_t olo[4], ohi[4];
                rank_pair(Y, k, s, olo, ohi); lookups += 2;
                uint32_t s2 = ohi[c] - olo[c];
                if (s2 == 0) { cnt++; k = 0; s = full; } else { k = Y.C[c] + olo[c] + 1; s = s2; }
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
                uint32_t olo[4], ohi[4];
                rank_pair(Y, k, s, olo, ohi); lookups += 2;
                uint32_t s2 = ohi[c] - olo[c];
                if (s2 == 0) { cnt++; k = 0; s = full; } else { k = Y.C[c] + olo[c] + 1; s = s2; }
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
    uint32_t lo = (b & 1) ? a1 : a0, hi = (b & 1) ? a3 : a2;
    return (b & 2) ? hi : lo;
}

// pool entry, 6 words, stored field-major (SoA) per warp so that lanes hit distinct banks:
//   qid | k | s | k2 | mlo | mhi
//   mlo = t (bits 0-8) | st (9-10; 0 = M, 1 = I, 2 = D) | n_go (11-18) | n_ge (19-26)
//   mhi = seed_d (0-7) | d (8-15) | m-1 (16-23)
#define BC_SEARCH_THREADS 512

// ---------------------------------------------------------------------------------------------
// A3 + A4 + A5.  Persistent kernel: every warp owns a LIFO pool of pending states (any read, any
// strand); each iteration the top `a` states are popped, one per lane, expanded in lock step
// (1-2 index lines -> <= 9 children), and the surviving children are compacted with ballots and
// pushed back, match children deepest.  New queries are drawn from a global ticket counter
// whenever fewer than 32 states are pending, so lanes stay busy and converged whatever the shape
// of the individual search trees.  Pool bound: a = clamp((CAP - R - cnt)/8, 1, 32)
// with R = 8z+9 keeps cnt < CAP for ever: a wide step ends at cnt <= CAP-R, and a run of
// single-state steps from height P never exceeds P-1+R because the match child is explored last.
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(BC_SEARCH_THREADS, 2) bc_search_kernel(BcSearchParams p) {
    extern __shared__ uint32_t pool_mem[];
    const uint32_t lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
    const uint32_t CAP = p.pool_cap;
    uint32_t *P = pool_mem + (size_t)warp * 6u * CAP;
    const uint32_t lt_mask = (1u << lane) - 1u;
    const int z = p.o.z, E = p.o.indel_end_skip, max_go = p.o.max_gap_open, max_ge = p.o.max_gap_ext;
    const int seed_len = p.o.seed_len, seed_z = p.o.seed_z;
    const int R = 8 * z + 9;
    const uint32_t nq = p.ws.nq;
    const uint32_t full = p.ix.bwt[0].n + 1;
    unsigned long long *ctr = (unsigned long long *)p.ws.ctr;

    uint32_t cnt = 0, pool_max = 0;
    bool more = true;
    unsigned long long n_nodes = 0, n_lookups = 0, n_lines = 0;

    for (;;) {
        // ---- intake: new root states while the pool is shallow --------------------------------
        if (cnt < 32u && more) {
            uint32_t need = 32u - cnt;
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
                uint32_t pos = cnt + __popc(mask & lt_mask);
                P[0 * CAP + pos] = (uint32_t)q; P[1 * CAP + pos] = 0; P[2 * CAP + pos] = full;
                P[3 * CAP + pos] = 0; P[4 * CAP + pos] = 0; P[5 * CAP + pos] = (m - 1) << 16;
            }
            cnt += __popc(mask);
            __syncwarp();
        }
        if (cnt == 0) { if (!more) break; continue; }
        pool_max = cnt > pool_max ? cnt : pool_max;

        // ---- pop ------------------------------------------------------------------------------
        int a = ((int)CAP - R - (int)cnt) / 8;
        a = a < 1 ? 1 : (a > 32 ? 32 : a);
        a = a > (int)cnt ? (int)cnt : a;
        const bool act = (int)lane < a;
        uint32_t qid = 0, k = 0, s = 0, k2 = 0, mlo = 0, mhi = 0;
        if (act) {
            uint32_t idx = cnt - 1u - lane;
            qid = P[0 * CAP + idx]; k = P[1 * CAP + idx]; s = P[2 * CAP + idx];
            k2 = P[3 * CAP + idx]; mlo = P[4 * CAP + idx]; mhi = P[5 * CAP + idx];
        }
        __syncwarp();
        cnt -= (uint32_t)a;
        n_nodes += (unsigned long long)a;

        // ---- expand ---------------------------------------------------------------------------
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
            n_lines += rank_pair(X, k, s, olo, ohi);
            n_lookups += 2;
            uint32_t acc = k2 + s;                       // k2 + dollar + prefix, built below
#pragma unroll
            for (int b = 0; b < 4; ++b) { ns[b] = ohi[b] - olo[b]; nk[b] = X.C[b] + olo[b] + 1u; acc -= ns[b]; }
#pragma unroll
            for (int b = 0; b < 4; ++b) { nk2[b] = acc; acc += ns[b]; }
        }
        const int in_seed_base = (seed_on && t < seed_len) ? 1 : 0;
        const int in_seed_del = (seed_on && t > 0 && t < seed_len) ? 1 : 0;

#pragma unroll
        for (int slot = 0; slot < 9; ++slot) {
            bool valid = false;
            uint32_t ck = k, cs = s, ck2 = k2;
            int nt = t + 1, nd = d + 1, ngo = go, nge = ge, nsd = sd, nst = 0;
            if (slot < 8) {
                const bool isdel = slot >= 4;
                uint32_t b;
                int cost = 1;
                if (isdel) b = (uint32_t)(slot - 4);
                else if (qb < 4) { b = (qb + (uint32_t)slot) & 3u; cost = slot == 0 ? 0 : 1; }
                else b = (uint32_t)slot;
                ck = sel4(nk[0], nk[1], nk[2], nk[3], b);
                cs = sel4(ns[0], ns[1], ns[2], ns[3], b);
                ck2 = sel4(nk2[0], nk2[1], nk2[2], nk2[3], b);
                if (isdel) {
                    nt = t; nst = 2; ngo = go + (st != 2); nge = ge + (st == 2); nsd = sd + in_seed_del;
                    valid = del_ok;
                } else {
                    nd = d + cost; nsd = sd + cost * in_seed_base;
                    valid = has_base;
                }
                valid = valid && cs > 0;
            } else {
                nst = 1; ngo = go + (st != 1); nge = ge + (st == 1); nsd = sd + in_seed_base;
                valid = ins_ok;
            }
            const uint32_t prn = (nt == t) ? pr0 : pr1;
            valid = valid && nd <= z && ngo <= max_go && nge <= max_ge && nsd <= seed_z &&
                    z - nd >= (int)BC_PREP_D(prn) && seed_z - nsd >= (int)BC_PREP_DS(prn);
            const bool terminal = nt == m;
            const bool emit = valid && terminal && cs != full;
            const bool push = valid && (!terminal || E == 0);

            uint32_t emask = __ballot_sync(0xffffffffu, emit);
            if (emask) {
                unsigned long long base = 0;
                int leader = __ffs(emask) - 1;
                if ((int)lane == leader) base = atomicAdd(&ctr[BC_CTR_ARENA], (unsigned long long)__popc(emask));
                base = __shfl_sync(0xffffffffu, base, leader);
                if (emit) {
                    unsigned long long pos = base + __popc(emask & lt_mask);
                    uint32_t kf = strand ? ck : ck2;
                    if (pos < p.ws.arena_cap) p.ws.arena[pos] = BcRawHit{qid, kf, kf + cs - 1u, (uint32_t)nd};
                    atomicAdd(&p.ws.qcnt[qid], 1u);
                }
            }
            uint32_t pmask = __ballot_sync(0xffffffffu, push);
            if (push) {
                uint32_t pos = cnt + __popc(pmask & lt_mask);
                if (pos < CAP) {
                    P[0 * CAP + pos] = qid; P[1 * CAP + pos] = ck; P[2 * CAP + pos] = cs; P[3 * CAP + pos] = ck2;
                    P[4 * CAP + pos] = (uint32_t)nt | ((uint32_t)nst << 9) | ((uint32_t)ngo << 11) | ((uint32_t)nge << 19);
                    P[5 * CAP + pos] = (uint32_t)nsd | ((uint32_t)nd << 8) | (mhi & 0x00FF0000u);
                } else {
                    atomicOr(&ctr[BC_CTR_ERROR], 2ull);   // cannot happen (pool bound); never silent
                }
            }
            cnt += __popc(pmask);
            if (cnt > CAP) cnt = CAP;
        }
        __syncwarp();
    }
    // per-warp statistics
    for (int o = 16; o > 0; o >>= 1) {
        n_lookups += __shfl_down_sync(0xffffffffu, n_lookups, o);
        n_lines += __shfl_down_sync(0xffffffffu, n_lines, o);
    }
    if (lane == 0) {
        atomicAdd(&ctr[BC_CTR_NODES], n_nodes);
        atomicAdd(&ctr[BC_CTR_LOOKUPS], n_lookups);
        atomicAdd(&ctr[BC_CTR_LINES], n_lines);
        atomicMax(&ctr[BC_CTR_POOLMAX], (unsigned long long)pool_max);
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
