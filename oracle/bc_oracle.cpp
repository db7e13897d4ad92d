// ORACLE -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
//
// Plain, slow, obviously-correct CPU implementation of what the hot path computes: per read and
// strand, the set of suffix-array intervals [k,l] of every reference substring that aligns to the
// query within the difference budgets, with the minimum difference count per interval.
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may
// call this.  It shares no code with paper_1505_07855_b200/ (the CUDA path) and neither imports
// the other.  Integer arithmetic only; nothing here is tuned.
//
// What it follows (PAPER.md gives the method only in prose, so the contract is SURVEY.md 8c):
//   * index: BWT by NAIVE SUFFIX SORT of T$ (north_star; beyond 150 M suffixes the sort is
//     bucketed by the first 12 bases and each bucket comparison-sorted, as C8 allows).  Two pointers k,l updated
//     per base from the index, l-k+1 = number of matches, crossing = absent.
//   * search: "carefully back up its search and start trying out alternatives" =
//     the recursion of SURVEY C4, written out in that order and notation, on the alignment
//     definition C2 and result definition C3.
//   * prunes: the D / Ds lower bounds of SURVEY C7 (optional; results must not depend on them).
//   * strand + "5'-first the plain way" (SURVEY C7 last bullet): search reverse(W) on the reverse
//     index carrying the matched string S, convert each hit by an exact backward search of S.
//
// Pins (tests/test_oracle_*.py, all -m "not gpu"): worked example tests/golden/worked_example.txt,
// exact-match counts vs naive scanning, brute-force enumeration + alignment DP on tiny genomes,
// Hamming / Levenshtein special cases, prune on/off, ban on/off, strand and reversal symmetry,
// locate = naive SA, BWT inversion.  Nothing is "parity unpinned".
#include <algorithm>
#include <cstdint>
#include <cstdlib>
#include <cstring>
#include <map>
#include <string>
#include <thread>
#include <utility>
#include <vector>

namespace {

// ---------------------------------------------------------------------------------------------
// C1. index of one text X = T$
// ---------------------------------------------------------------------------------------------
struct Index {
    uint64_t n = 0, primary = 0;
    std::vector<uint8_t> T;     // text, codes 0..3
    std::vector<uint32_t> SA;   // n+1 rows, SA[0] = n
    std::vector<uint8_t> B;     // n+1 symbols, B[primary] = 4 ('$')
    std::vector<uint32_t> ck;   // ck[t*4+c] = #{j < 64 t : B[j] = c}
    uint64_t C[5] = {0, 0, 0, 0, 0};

    // O(c, j) = #{j' <= j : B[j'] = c}, O(c,-1) = 0
    uint64_t O(int c, int64_t j) const {
        uint64_t p = (uint64_t)(j + 1);         // count over B[0..p)
        uint64_t t = p / 64;
        uint64_t r = ck[t * 4 + c];
        for (uint64_t q = t * 64; q < p; ++q) r += (B[q] == c);
        return r;
    }
    // prepend c to a string with interval [k,l]; returns false if empty
    bool prepend(int c, int64_t k, int64_t l, int64_t &k2, int64_t &l2) const {
        k2 = (int64_t)(C[c] + O(c, k - 1) + 1);
        l2 = (int64_t)(C[c] + O(c, l));
        return k2 <= l2;
    }
};

// suffix comparison on X = T$ ('$' smallest): literal definition
struct SufLess {
    const uint8_t *T; uint64_t n;
    bool operator()(uint32_t a, uint32_t b) const {
        if (a == b) return false;
        uint64_t la = n - a, lb = n - b, len = la < lb ? la : lb;
        int r = len ? memcmp(T + a, T + b, len) : 0;
        if (r != 0) return r < 0;
        return la < lb;                          // the shorter suffix hits '$' first
    }
};

// naive comparison sort of ALL suffixes; threads only split it into a merge sort
void sort_suffixes_literal(Index &ix, int nthreads) {
    const uint64_t n = ix.n;
    SufLess less{ix.T.data(), n};
    int parts = 1; while (parts * 2 <= nthreads && (n + 1) / (parts * 2) > 4096) parts *= 2;
    std::vector<uint64_t> cut(parts + 1);
    for (int p = 0; p <= parts; ++p) cut[p] = (n + 1) * (uint64_t)p / parts;
    {
        std::vector<std::thread> th;
        for (int p = 0; p < parts; ++p)
            th.emplace_back([&, p] { std::sort(ix.SA.begin() + cut[p], ix.SA.begin() + cut[p + 1], less); });
        for (auto &t : th) t.join();
    }
    for (int w = 1; w < parts; w *= 2) {
        std::vector<std::thread> th;
        for (int p = 0; p + w < parts; p += 2 * w)
            th.emplace_back([&, p, w] {
                int e = std::min(parts, p + 2 * w);
                std::inplace_merge(ix.SA.begin() + cut[p], ix.SA.begin() + cut[p + w], ix.SA.begin() + cut[e], less);
            });
        for (auto &t : th) t.join();
    }
}

// SURVEY C8, for genomes where the literal sort takes hours: "bucket suffixes by their first 12 bases
// (16.7 M buckets), then comparison-sort each bucket on the text in parallel -- still no clever
// construction algorithm".  Key of suffix i = its first 12 symbols, 2 bits each, padded with A (= 0) past
// the end of T.  The padding cannot misplace a suffix ACROSS buckets: at the first position where two
// padded prefixes differ, the suffix with the smaller symbol is the smaller suffix if that position lies
// inside both, and a padded position (A, the smallest base) can never be the larger one.  WITHIN a bucket
// the same literal comparator as above ('$' smallest) decides.  Pinned by equality with the literal sort
// (tests/test_oracle_pins2.py).
void sort_suffixes_bucketed(Index &ix, int nthreads) {
    const uint64_t n = ix.n;
    const int K = 12;
    const uint64_t NB = 1ull << (2 * K);
    const uint8_t *T = ix.T.data();
    auto key_at = [&](uint64_t i) {            // suffix i = T[i..n) $ ; i == n is the '$' suffix: all padding
        uint64_t key = 0;
        for (int j = 0; j < K; ++j) key = (key << 2) | (i + j < n ? T[i + j] : 0);
        return key;
    };
    std::vector<uint64_t> start(NB + 1, 0);
    for (uint64_t i = 0; i <= n; ++i) start[key_at(i) + 1]++;
    for (uint64_t b = 0; b < NB; ++b) start[b + 1] += start[b];
    if (nthreads < 1) nthreads = 1;
    // thread t owns the buckets [own[t], own[t+1]): about (n+1)/nthreads suffixes each
    std::vector<uint64_t> own(nthreads + 1, NB);
    own[0] = 0;
    for (int t = 1; t < nthreads; ++t) {
        const uint64_t want = (n + 1) * (uint64_t)t / nthreads;
        own[t] = (uint64_t)(std::lower_bound(start.begin(), start.end(), want) - start.begin());
        if (own[t] > NB) own[t] = NB;
        if (own[t] < own[t - 1]) own[t] = own[t - 1];
    }
    SufLess less{T, n};
    std::vector<std::thread> th;
    for (int t = 0; t < nthreads; ++t)
        th.emplace_back([&, t] {
            const uint64_t b0 = own[t], b1 = own[t + 1];
            if (b0 >= b1) return;
            std::vector<uint64_t> fill(start.begin() + b0, start.begin() + b1);   // next free slot of my buckets
            for (uint64_t i = 0; i <= n; ++i) {          // every thread scans the text, keeps what it owns
                const uint64_t key = key_at(i);
                if (key >= b0 && key < b1) ix.SA[fill[key - b0]++] = (uint32_t)i;
            }
            for (uint64_t b = b0; b < b1; ++b)
                if (start[b + 1] - start[b] > 1) std::sort(ix.SA.begin() + start[b], ix.SA.begin() + start[b + 1], less);
        });
    for (auto &t : th) t.join();
}

// mode: 0 = literal sort of all suffixes, 1 = bucketed (C8), -1 = literal up to 150 M suffixes, bucketed beyond
void build_index(Index &ix, const uint8_t *T, uint64_t n, int nthreads, int mode = 0) {
    ix.n = n; ix.T.assign(T, T + n);
    ix.SA.resize(n + 1);
    for (uint64_t i = 0; i <= n; ++i) ix.SA[i] = (uint32_t)i;
    if (mode == 1 || (mode < 0 && n > 150000000ull)) sort_suffixes_bucketed(ix, nthreads);
    else sort_suffixes_literal(ix, nthreads);
    ix.B.resize(n + 1);
    {                                            // B[j] = X[SA[j]-1]; threads only split the rows
        const int nt = nthreads < 1 ? 1 : nthreads;
        std::vector<std::thread> th;
        for (int t = 0; t < nt; ++t)
            th.emplace_back([&, t] {
                for (uint64_t j = (n + 1) * (uint64_t)t / nt; j < (n + 1) * (uint64_t)(t + 1) / nt; ++j) {
                    if (ix.SA[j] == 0) { ix.B[j] = 4; ix.primary = j; }
                    else ix.B[j] = ix.T[ix.SA[j] - 1];
                }
            });
        for (auto &t : th) t.join();
    }
    uint64_t cnt[4] = {0, 0, 0, 0};
    for (uint64_t i = 0; i < n; ++i) cnt[ix.T[i]]++;
    ix.C[0] = 0; for (int c = 0; c < 4; ++c) ix.C[c + 1] = ix.C[c] + cnt[c];
    uint64_t nck = (n + 1) / 64 + 2;
    ix.ck.assign(nck * 4, 0);
    uint32_t run[4] = {0, 0, 0, 0};
    for (uint64_t j = 0; j <= n; ++j) {
        if (j % 64 == 0) for (int c = 0; c < 4; ++c) ix.ck[(j / 64) * 4 + c] = run[c];
        if (ix.B[j] < 4) run[ix.B[j]]++;
    }
    if ((n + 1) % 64 == 0) for (int c = 0; c < 4; ++c) ix.ck[((n + 1) / 64) * 4 + c] = run[c];
}

struct Opts { int32_t z, max_gap_open, max_gap_ext, seed_len, seed_z, indel_end_skip; };

enum { FLAG_PRUNE = 1, FLAG_BAN_ID = 2, FLAG_PLUS_5P_FIRST = 4 };

// ---------------------------------------------------------------------------------------------
// C7. D lower bound: greedy piece count over Q[from..], growing each piece to the right by
// prepending on the index of the OPPOSITE direction (Y).  D[i] for i in [from, to).
// ---------------------------------------------------------------------------------------------
void compute_D(const Index &Y, const uint8_t *Q, int from, int to, std::vector<int> &D, uint64_t *lookups) {
    int cnt = 0; int64_t k = 0, l = (int64_t)Y.n;
    for (int i = from; i < to; ++i) {
        if (Q[i] > 3) { cnt++; k = 0; l = (int64_t)Y.n; }
        else {
            int64_t k2, l2;
            if (lookups) *lookups += 2;
            if (!Y.prepend(Q[i], k, l, k2, l2)) { cnt++; k = 0; l = (int64_t)Y.n; }
            else { k = k2; l = l2; }
        }
        D[i] = cnt;
    }
}

// ---------------------------------------------------------------------------------------------
// C4. the recursion (right-to-left over Q, prepending on index X)
// ---------------------------------------------------------------------------------------------
struct Search {
    const Index *X;            // index the query is matched on (prepend)
    const uint8_t *Q; int m;
    Opts o; int flags;
    int s0, s1; bool seed_on;  // seed range in Q indices
    std::vector<int> D, Ds;    // lower bounds (FLAG_PRUNE)
    bool carry;                // carry the matched string S (for the reverse-index mode)
    std::string S;             // S as matched so far, most recently prepended symbol LAST
    std::map<std::pair<uint32_t, uint32_t>, int> *out;   // (k,l) -> min d, in X coordinates
    const Index *conv;         // if carry: convert S to an interval on this index
    uint64_t nodes = 0, lookups = 0;

    void record(int64_t k, int64_t l, int d) {
        if (k == 0 && l == (int64_t)X->n) return;   // empty S (all-insertion alignment): C3 wants non-empty S
        if (carry) {
            // S holds reverse-text symbols in prepend order: S[0] was prepended first, i.e. it is
            // the LAST symbol of the matched substring S' of reverse(T); S' = reverse(S-buffer).
            // The forward string is reverse(S') = the buffer in order.  Exact backward search
            // consumes a string right-to-left.
            int64_t kk = 0, ll = (int64_t)conv->n;
            for (int p = (int)S.size() - 1; p >= 0; --p) {
                int64_t k2, l2; lookups += 2;
                bool ok = conv->prepend(S[p], kk, ll, k2, l2);
                if (!ok) abort();               // cannot happen: S occurs in T
                kk = k2; ll = l2;
            }
            k = kk; l = ll;
        }
        auto key = std::make_pair((uint32_t)k, (uint32_t)l);
        auto it = out->find(key);
        if (it == out->end()) (*out)[key] = d; else if (d < it->second) it->second = d;
    }

    // st: 0 = M, 1 = I, 2 = D
    void rec(int i, int64_t k, int64_t l, int st, int n_go, int n_ge, int seed_d, int d) {
        // budgets (C2-1, C2-4)
        if (d > o.z || n_go > o.max_gap_open || n_ge > o.max_gap_ext) return;
        if (seed_on && seed_d > o.seed_z) return;
        if (flags & FLAG_PRUNE) {
            if (i >= 0 && o.z - d < D[i]) return;
            if (seed_on && i >= s0) { int ii = i < s1 ? i : s1 - 1; if (o.seed_z - seed_d < Ds[ii]) return; }
        }
        nodes++;
        const int E = o.indel_end_skip;
        const int left = i + 1;
        const bool ban = flags & FLAG_BAN_ID;
        if (i < 0) {
            // the whole query is consumed.  Non-empty S only (C3): d deletions alone would give m = 0.
            record(k, l, d);
        }
        // insertion: Q[i] against nothing
        if (i >= 0 && !(ban && st == 2) && i >= E && m - 1 - i >= E) {
            int in_seed = seed_on && s0 <= i && i < s1;
            rec(i - 1, k, l, 1, n_go + (st != 1), n_ge + (st == 1), seed_d + in_seed, d + 1);
        }
        bool del_ok = !(ban && st == 1) && left >= E && m - left >= E;
        if (i < 0 && !del_ok) return;
        for (int b = 0; b < 4; ++b) {
            int64_t k2, l2; lookups += 2;
            if (!X->prepend(b, k, l, k2, l2)) continue;
            if (carry) S.push_back((char)b);
            if (del_ok) {
                int in_seed = seed_on && s0 < left && left < s1;
                rec(i, k2, l2, 2, n_go + (st != 2), n_ge + (st == 2), seed_d + in_seed, d + 1);
            }
            if (i >= 0) {
                int c = (Q[i] == b && Q[i] < 4) ? 0 : 1;
                int in_seed = seed_on && s0 <= i && i < s1;
                rec(i - 1, k2, l2, 0, n_go, n_ge, seed_d + c * in_seed, d + c);
            }
            if (carry) S.pop_back();
        }
    }
};

struct Hit { uint32_t k, l; uint8_t d, strand; uint16_t zero; };

struct Handle { Index fwd, rev; };

struct Result {
    std::vector<uint64_t> off;      // n_reads + 1
    std::vector<Hit> hits;
    uint64_t nodes = 0, lookups = 0;
};

// one (read, strand): fills `out` with forward-index intervals
void align_query(const Handle &h, const uint8_t *W, int m, const Opts &o, int flags, int strand,
                 std::map<std::pair<uint32_t, uint32_t>, int> &out, uint64_t &nodes, uint64_t &lookups) {
    std::vector<uint8_t> Q(m);
    Search s; s.o = o; s.flags = flags; s.m = m; s.out = &out;
    s.seed_on = o.seed_len > 0 && o.seed_len < m;
    const Index *Y;     // opposite-direction index for the D bound
    if (strand == 1) {                      // Q = revcomp(W) on the forward index; seed = last seed_len of Q
        for (int i = 0; i < m; ++i) { uint8_t c = W[m - 1 - i]; Q[i] = c < 4 ? 3 - c : 4; }
        s.X = &h.fwd; Y = &h.rev; s.carry = false; s.conv = nullptr;
        s.s0 = m - o.seed_len; s.s1 = m;
    } else if (flags & FLAG_PLUS_5P_FIRST) { // reverse(W) on the reverse index, S carried
        for (int i = 0; i < m; ++i) Q[i] = W[m - 1 - i];
        s.X = &h.rev; Y = &h.fwd; s.carry = true; s.conv = &h.fwd;
        s.s0 = m - o.seed_len; s.s1 = m;
    } else {                                // textbook: Q = W right-to-left on the forward index
        for (int i = 0; i < m; ++i) Q[i] = W[i];
        s.X = &h.fwd; Y = &h.rev; s.carry = false; s.conv = nullptr;
        s.s0 = 0; s.s1 = o.seed_len;
    }
    if (!s.seed_on) { s.s0 = 0; s.s1 = 0; }
    s.Q = Q.data();
    if (flags & FLAG_PRUNE) {
        s.D.assign(m, 0); compute_D(*Y, s.Q, 0, m, s.D, &s.lookups);
        s.Ds.assign(m, 0); if (s.seed_on) compute_D(*Y, s.Q, s.s0, s.s1, s.Ds, &s.lookups);
    }
    s.rec(m - 1, 0, (int64_t)s.X->n, 0, 0, 0, 0, 0);
    nodes += s.nodes; lookups += s.lookups;
}

}  // namespace

extern "C" {

void *orc_index_build2(const uint8_t *T, uint64_t n, int nthreads, int mode) {
    Handle *h = new Handle();
    build_index(h->fwd, T, n, nthreads, mode);
    std::vector<uint8_t> R(T, T + n); std::reverse(R.begin(), R.end());
    build_index(h->rev, R.data(), n, nthreads, mode);
    return h;
}
void *orc_index_build(const uint8_t *T, uint64_t n, int nthreads) { return orc_index_build2(T, n, nthreads, 0); }
void orc_index_free(void *h) { delete (Handle *)h; }

// which: 0 fwd, 1 rev.  Any out pointer may be NULL.
void orc_index_get(void *hv, int which, uint32_t *SA, uint8_t *B, uint64_t *C5, uint64_t *primary) {
    Handle *h = (Handle *)hv; const Index &ix = which ? h->rev : h->fwd;
    if (SA) memcpy(SA, ix.SA.data(), (ix.n + 1) * 4);
    if (B) memcpy(B, ix.B.data(), ix.n + 1);
    if (C5) for (int c = 0; c < 5; ++c) C5[c] = ix.C[c];
    if (primary) *primary = ix.primary;
}

// O(c, j) on either index (for pins)
uint64_t orc_occ(void *hv, int which, int c, int64_t j) {
    Handle *h = (Handle *)hv; return (which ? h->rev : h->fwd).O(c, j);
}

// D[] of SURVEY C7's loop for a query consumed right-to-left: D[i] over Q[0..i] on the REVERSE index
void orc_D(void *hv, const uint8_t *Q, int m, int32_t *D) {
    Handle *h = (Handle *)hv; std::vector<int> d(m, 0);
    compute_D(h->rev, Q, 0, m, d, nullptr);
    for (int i = 0; i < m; ++i) D[i] = d[i];
}

// Ds[] ("Ds is the same loop started at i = s0 with cnt = 0"): the loop of orc_D restricted to
// Q[from..to) -- an accessor for the pins, no arithmetic of its own.  Entries outside [from,to) are 0.
void orc_D_range(void *hv, const uint8_t *Q, int m, int from, int to, int32_t *D) {
    Handle *h = (Handle *)hv; std::vector<int> d(m, 0);
    compute_D(h->rev, Q, from, to, d, nullptr);
    for (int i = 0; i < m; ++i) D[i] = d[i];
}

// rows -> SA[row] (definition of locate)
void orc_locate(void *hv, const uint32_t *rows, uint64_t n_rows, uint32_t *pos) {
    Handle *h = (Handle *)hv;
    for (uint64_t i = 0; i < n_rows; ++i) pos[i] = h->fwd.SA[rows[i]];
}

// reads: flat codes (0..3, 4 = N), off[r], len[r].  opts6 = {z, go, ge, seed_len, seed_z, E}.
void *orc_align(void *hv, const uint8_t *codes, const uint64_t *off, const uint16_t *len,
                uint64_t n_reads, const int32_t *opts6, int flags, int nthreads) {
    Handle *h = (Handle *)hv;
    Opts o{opts6[0], opts6[1], opts6[2], opts6[3], opts6[4], opts6[5]};
    Result *res = new Result();
    std::vector<std::vector<Hit>> per(n_reads);
    if (nthreads < 1) nthreads = 1;
    std::vector<uint64_t> nodes(nthreads, 0), lookups(nthreads, 0);
    std::vector<std::thread> th;
    for (int t = 0; t < nthreads; ++t)
        th.emplace_back([&, t] {
            for (uint64_t r = t; r < n_reads; r += nthreads) {   // reads split across threads
                for (int strand = 0; strand < 2; ++strand) {
                    std::map<std::pair<uint32_t, uint32_t>, int> out;
                    align_query(*h, codes + off[r], len[r], o, flags, strand, out, nodes[t], lookups[t]);
                    for (auto &kv : out)                          // std::map iterates in (k,l) order
                        per[r].push_back(Hit{kv.first.first, kv.first.second, (uint8_t)kv.second, (uint8_t)strand, 0});
                }
            }
        });
    for (auto &t : th) t.join();
    res->off.assign(n_reads + 1, 0);
    for (uint64_t r = 0; r < n_reads; ++r) res->off[r + 1] = res->off[r] + per[r].size();
    res->hits.reserve(res->off[n_reads]);
    for (uint64_t r = 0; r < n_reads; ++r) res->hits.insert(res->hits.end(), per[r].begin(), per[r].end());
    for (int t = 0; t < nthreads; ++t) { res->nodes += nodes[t]; res->lookups += lookups[t]; }
    return res;
}
uint64_t orc_result_total(void *rv) { return ((Result *)rv)->hits.size(); }
uint64_t orc_result_nodes(void *rv) { return ((Result *)rv)->nodes; }
uint64_t orc_result_lookups(void *rv) { return ((Result *)rv)->lookups; }
void orc_result_copy(void *rv, uint64_t *off, void *hits12) {
    Result *r = (Result *)rv;
    memcpy(off, r->off.data(), r->off.size() * 8);
    if (!r->hits.empty()) memcpy(hits12, r->hits.data(), r->hits.size() * sizeof(Hit));
}
void orc_result_free(void *rv) { delete (Result *)rv; }

}  // extern "C"
