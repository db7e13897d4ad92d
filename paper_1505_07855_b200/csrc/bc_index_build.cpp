// Host-side index construction (untimed helper; SURVEY.md section 2 #4, 8a "A0 input").
// The paper builds its index offline with an `index` command; here the same
// role is played, for synthetic genomes, by a bucketed suffix sort: suffixes are grouped by their
// first 12 bases (counting sort) and every bucket is then comparison-sorted on the text with an
// 8-bytes-at-a-time comparator.  Product code: shares nothing with oracle/.
#include "bc_host_index.h"

#include <algorithm>
#include <atomic>
#include <cstdlib>
#include <cstring>
#include <new>
#include <thread>
#include <vector>

namespace {

constexpr int KPFX = 12;                       // bases in the bucket key (24 bits)
constexpr uint32_t NBUCKET = 1u << (2 * KPFX);

using BwtArrays = BcBwtArrays;
using HostIndexOwner = BcHostIndexOwner;

// lexicographic compare of suffixes a,b of text[0..n) ('$' = end of text is smallest)
struct SuffixCmp {
    const uint8_t *t;                           // padded with >= 8 zero bytes past n
    uint64_t n;
    bool operator()(uint32_t a, uint32_t b) const {
        if (a == b) return false;
        uint64_t la = n - a, lb = n - b, lim = la < lb ? la : lb, o = KPFX < lim ? KPFX : 0;
        // the first KPFX bases are equal inside a bucket when both suffixes are that long
        for (; o + 8 <= lim; o += 8) {
            uint64_t x, y;
            memcpy(&x, t + a + o, 8); memcpy(&y, t + b + o, 8);
            if (x != y) return __builtin_bswap64(x) < __builtin_bswap64(y);
        }
        for (; o < lim; ++o)
            if (t[a + o] != t[b + o]) return t[a + o] < t[b + o];
        return la < lb;
    }
};

uint32_t prefix_key(const uint8_t *t, uint64_t n, uint64_t i) {
    uint32_t key = 0;
    for (int j = 0; j < KPFX; ++j) key = (key << 2) | (i + j < n ? t[i + j] : 0);
    return key;
}

// suffix array of text$ into sa[0..n]
void suffix_sort(const uint8_t *text, uint64_t n, std::vector<uint32_t> &sa, int n_threads) {
    std::vector<uint8_t> pad(n + 16, 0);
    memcpy(pad.data(), text, n);
    const uint8_t *t = pad.data();
    sa.assign(n + 1, 0);
    std::vector<uint64_t> start((size_t)NBUCKET + 1, 0);
    {   // histogram of rolling keys
        uint32_t key = prefix_key(t, n, 0);
        for (uint64_t i = 0; i < n; ++i) {
            start[key + 1]++;
            key = ((key << 2) & (NBUCKET - 1)) | (i + KPFX < n ? t[i + KPFX] : 0);
        }
    }
    sa[0] = (uint32_t)n;                        // the empty suffix '$' is row 0
    start[0] = 1;
    for (uint32_t b = 0; b < NBUCKET; ++b) start[b + 1] += start[b];
    {
        std::vector<uint64_t> fill(start.begin(), start.end() - 1);
        uint32_t key = prefix_key(t, n, 0);
        for (uint64_t i = 0; i < n; ++i) {
            sa[fill[key]++] = (uint32_t)i;
            key = ((key << 2) & (NBUCKET - 1)) | (i + KPFX < n ? t[i + KPFX] : 0);
        }
    }
    SuffixCmp cmp{t, n};
    std::atomic<uint32_t> next(0);
    const uint32_t CH = 1024;
    auto work = [&] {
        for (;;) {
            uint32_t b0 = next.fetch_add(CH);
            if (b0 >= NBUCKET) break;
            uint32_t b1 = b0 + CH < NBUCKET ? b0 + CH : NBUCKET;
            for (uint32_t b = b0; b < b1; ++b)
                if (start[b + 1] - start[b] > 1) std::sort(sa.begin() + start[b], sa.begin() + start[b + 1], cmp);
        }
    };
    if (n_threads < 1) n_threads = 1;
    std::vector<std::thread> th;
    for (int i = 1; i < n_threads; ++i) th.emplace_back(work);
    work();
    for (auto &x : th) x.join();
}

void make_bwt(const uint8_t *text, uint64_t n, const std::vector<uint32_t> &sa, uint32_t occ_interval,
              BwtArrays &out, bc_bwt_host &pub) {
    out.bwt2.assign(n / 32 + 1, 0);
    out.occ.assign((n / occ_interval + 1) * 4, 0);
    uint32_t run[4] = {0, 0, 0, 0};
    uint64_t j = 0;                             // index in the '$'-less BWT
    for (uint64_t row = 0; row <= n; ++row) {
        if (sa[row] == 0) { pub.primary = row; continue; }
        if (j % occ_interval == 0) for (int c = 0; c < 4; ++c) out.occ[(j / occ_interval) * 4 + c] = run[c];
        uint64_t c = text[sa[row] - 1];
        out.bwt2[j >> 5] |= c << (2 * (j & 31));
        run[c]++; ++j;
    }
    if (n % occ_interval == 0) for (int c = 0; c < 4; ++c) out.occ[(n / occ_interval) * 4 + c] = run[c];
    pub.n = n;
    pub.bwt2 = out.bwt2.data();
    pub.occ_interval = occ_interval;
    pub.occ = out.occ.data();
    pub.C[0] = 0;
    for (int c = 0; c < 4; ++c) pub.C[c + 1] = pub.C[c] + run[c];
}

}  // namespace

extern "C" int bc_index_build_host(const uint8_t *text, uint64_t n, uint32_t occ_interval, uint32_t sa_interval,
                                   int n_threads, bc_index_host **out) {
    if (!text || !out || n < 1 || n >= 0xFFFFFFFFull || occ_interval == 0 || occ_interval % 32 || sa_interval == 0)
        return BC_E_INVAL;
    for (uint64_t i = 0; i < n; ++i) if (text[i] > 3) return BC_E_INVAL;
    HostIndexOwner *h = new (std::nothrow) HostIndexOwner();
    if (!h) return BC_E_NOMEM;
    try {
        std::vector<uint32_t> sa;
        suffix_sort(text, n, sa, n_threads);
        make_bwt(text, n, sa, occ_interval, h->fwd, h->pub.fwd);
        h->sa.resize(n / sa_interval + 1);
        for (uint64_t t = 0; t * sa_interval <= n; ++t) h->sa[t] = sa[t * sa_interval];
        std::vector<uint8_t> rt(text, text + n);
        std::reverse(rt.begin(), rt.end());
        suffix_sort(rt.data(), n, sa, n_threads);
        make_bwt(rt.data(), n, sa, occ_interval, h->rev, h->pub.rev);
    } catch (const std::bad_alloc &) {
        delete h;
        return BC_E_NOMEM;
    }
    h->pub.sa_interval = sa_interval;
    h->pub.sa = h->sa.data();
    *out = &h->pub;
    return BC_OK;
}

extern "C" int bc_index_host_free(bc_index_host *p) {
    if (!p) return BC_E_INVAL;
    delete reinterpret_cast<HostIndexOwner *>(p);
    return BC_OK;
}
