"""More pins for the oracle (round 2).  CPU only.

Added because the first set was thin in three places: (a) with E = 5 -- the end rule every gapped
config uses -- a gap needs m >= 11, which the first brute-force set almost never reached; (b) the
reversal symmetry compared only sums of interval widths; (c) Ds, the seed-restricted bound, was
pinned only through prune-on = prune-off.  Nothing here re-types the oracle's formulae: the
expected values come from the alignment DP over enumerated substrings (tests/bruteforce.py), from
naive substring containment (Python's `in`), from Sellers' DP and from position arithmetic."""
import random

import numpy as np
import pytest

import synthdata as sd
from oracle import Oracle, FLAG_PRUNE, FLAG_BAN_ID, FLAG_PLUS_5P_FIRST, DEFAULT_FLAGS
from tests.bruteforce import brute_align, revcomp
from tests.test_oracle_pins import hits_list, min_diffs_anywhere


# ------------------------------------------------------------------------------- P3, thick
def _long_case(rng):
    """reads of 11..14 bases with indels/mismatches planted in the middle, so that E = 5 admits gaps."""
    n = rng.randint(20, 34)
    alpha = rng.choice([[0, 1, 2, 3], [0, 1, 2, 3], [0, 0, 1, 2, 3], [0, 1]])
    T = [rng.choice(alpha) for _ in range(n)]
    if rng.random() < 0.4:                          # tandem / dispersed repeat
        a, L = rng.randint(0, n - 12), rng.randint(3, 7)
        b = rng.randint(0, n - L)
        T[b:b + L] = T[a:a + L]
    m = rng.randint(11, 14)
    p = rng.randint(0, n - m)
    W = T[p:p + m + 3]
    for _ in range(rng.randint(0, 2)):
        r = rng.random()
        q = rng.randint(4, 8)                       # the middle: >= 5 bases on either side is possible
        if r < 0.35 and len(W) > q + 1:
            del W[q:q + rng.randint(1, 2)]
        elif r < 0.70:
            for _ in range(rng.randint(1, 2)):
                W.insert(q, rng.randint(0, 3))
        elif r < 0.95:
            W[q] = (W[q] + rng.randint(1, 3)) & 3
        else:
            W[q] = 4
    W = W[:m]
    if len(W) < 11:
        W = W + [rng.randint(0, 3) for _ in range(11 - len(W))]
    if rng.random() < 0.5:
        W = revcomp(W)
    m = len(W)
    z = rng.randint(1, 3)
    go = rng.randint(0, 2)
    ge = rng.randint(0, 2)
    E = rng.choice([5, 5, 5, 4, 2])
    seed_len = rng.choice([0, rng.randint(4, m - 1), rng.randint(6, 9)])
    seed_z = rng.randint(0, 2)
    return T, W, (z, go, ge, seed_len, seed_z, E)


@pytest.mark.parametrize("chunk", range(10))
def test_p3_bruteforce_long_reads_with_end_rule(chunk):
    """1,000 cases, m = 11..14, E mostly 5: the gapped paths every config takes (C2-3)."""
    rng = random.Random(52000 + chunk)
    gapped = 0
    for _ in range(100):
        T, W, opts = _long_case(rng)
        want = brute_align(T, W, opts)
        want_nogap = brute_align(T, W, (opts[0], 0, 0) + opts[3:])
        gapped += want != want_nogap
        o = Oracle(np.asarray(T, dtype=np.uint8), nthreads=1)
        for flags in (0, DEFAULT_FLAGS, FLAG_PRUNE | FLAG_BAN_ID):
            got = hits_list(o, [np.asarray(W, dtype=np.uint8)], opts, flags)[0]
            assert got == want, (T, W, opts, flags)
    assert gapped >= 5            # the set does exercise gaps under the end rule


# deletions at, just inside and just outside the seed boundary (C2-4: "strictly inside")
def test_p3_seed_straddling_deletion():
    rng = random.Random(99)
    n_diff = 0
    for case in range(60):
        n = 30
        T = [rng.randint(0, 3) for _ in range(n)]
        m = 13
        p = rng.randint(0, n - m - 2)
        src = T[p:p + m + 2]
        cut = rng.randint(5, 8)                     # read = source with 1..2 reference bases deleted at `cut`
        gl = rng.randint(1, 2)
        W = (src[:cut] + src[cut + gl:])[:m]
        strand_flip = rng.random() < 0.5
        if strand_flip:
            W = revcomp(W)
        res = {}
        for seed_len in (cut - 1, cut, cut + 1, cut + 2):
            for seed_z in (0, 1):
                opts = (2, 1, 1, seed_len, seed_z, 5)
                want = brute_align(T, W, opts)
                o = Oracle(np.asarray(T, dtype=np.uint8), nthreads=1)
                for flags in (0, DEFAULT_FLAGS):
                    assert hits_list(o, [np.asarray(W, np.uint8)], opts, flags)[0] == want, (T, W, opts, flags)
                res[(seed_len, seed_z)] = want
        n_diff += len({tuple(v) for v in res.values()}) > 1
    assert n_diff >= 10           # the seed position relative to the gap does change the result


# ------------------------------------------------------------------------------- P5, reversal by positions
@pytest.fixture(scope="module")
def mid():
    cfg = sd.CONFIGS["2"].scaled(n=50_000, n_reads=60)
    g = sd.make_genome(cfg)
    return cfg, g, Oracle(g), Oracle(g[::-1].copy()), sd.make_reads(cfg, g)


def _positions_by_d(oracle, hits):
    out = {}
    for (s, k, l, d) in hits:
        if s == 0:
            out.setdefault(d, set()).update(int(x) for x in oracle.locate(np.arange(k, l + 1)))
    return out


def test_p5_reversal_symmetry_position_sets_gaps_off(mid):
    """mismatches only: every matched string has length m, so a hit of Q at p in T is a hit of
    reverse(Q) at n - p - m in reverse(T), with the same d -- compared as SETS per d."""
    cfg, g, o, o_rev, reads = mid
    n, m = len(g), reads.m
    R = reads.codes
    opts = (3, 0, 0, 0, 0, 5)
    a = hits_list(o, R, opts)
    b = hits_list(o_rev, np.ascontiguousarray(R[:, ::-1]), opts)
    seen = 0
    for x, y in zip(a, b):
        pa, pb = _positions_by_d(o, x), _positions_by_d(o_rev, y)
        assert sorted(pa) == sorted(pb)
        for d in pa:
            assert {n - p - m for p in pa[d]} == pb[d]
            seen += len(pa[d])
    assert seen >= 20


def test_p5_reversal_symmetry_position_sets_with_gaps(mid):
    """with gaps the matched length is m - del .. m + ins, so the mirrored START is known up to that
    window; the mirrored END of the reversed hit = n - p exactly for one admissible length."""
    cfg, g, o, o_rev, reads = mid
    n, m = len(g), reads.m
    R = reads.codes[:30]
    opts = (2, 1, 1, 0, 0, 5)
    a = hits_list(o, R, opts)
    b = hits_list(o_rev, np.ascontiguousarray(R[:, ::-1]), opts)
    for x, y in zip(a, b):
        pa, pb = _positions_by_d(o, x), _positions_by_d(o_rev, y)
        allb = set().union(*pb.values()) if pb else set()
        alla = set().union(*pa.values()) if pa else set()
        assert min(pa, default=None) == min(pb, default=None)           # same best stratum
        for p in alla:
            assert any((n - p - L) in allb for L in range(m - 2, m + 3)), (p,)
        for p in allb:
            assert any((n - p - L) in alla for L in range(m - 2, m + 3)), (p,)


# ------------------------------------------------------------------------------- C7 / P6: D and Ds directly
def _greedy_pieces(Q, Ts, lo, hi):
    """C7 in words: split Q[lo..hi) greedily from lo into the longest pieces that occur in T; count the
    pieces that fail (the failing base belongs to the failed piece; N always fails).  Naive `in`."""
    out = [0] * len(Q)
    cnt, piece = 0, ""
    for i in range(lo, hi):
        if Q[i] > 3:
            cnt, piece = cnt + 1, ""
        else:
            piece += "ACGT"[Q[i]]
            if piece not in Ts:
                cnt, piece = cnt + 1, ""
        out[i] = cnt
    return out


def test_c7_D_and_Ds_equal_naive_piece_count_and_are_admissible():
    rng = random.Random(4242)
    for _ in range(120):
        n = rng.randint(30, 200)
        T = [rng.choice([0, 1, 2, 3]) for _ in range(n)]
        Ts = sd.decode(T)
        m = rng.randint(6, 24)
        p = rng.randint(0, n - m)
        Q = T[p:p + m]
        for _ in range(rng.randint(0, 4)):
            Q[rng.randrange(m)] = rng.choice([0, 1, 2, 3, 4])
        o = Oracle(np.asarray(T, dtype=np.uint8), nthreads=1)
        Qa = np.asarray(Q, np.uint8)
        assert o.D(Qa).tolist() == _greedy_pieces(Q, Ts, 0, m)
        lo = rng.randint(0, m - 2)
        hi = rng.randint(lo + 1, m)
        Ds = o.D_range(Qa, lo, hi).tolist()
        assert Ds == _greedy_pieces(Q, Ts, lo, hi)
        assert Ds[lo:hi] == o.D(Qa[lo:hi]).tolist()                     # = the bound of the seed taken alone
        for i in range(lo, hi):                                         # admissible for the seed part alone
            assert Ds[i] <= min_diffs_anywhere(Q[lo:i + 1], T), (T, Q, lo, i)


def test_seed_limit_equals_filter_of_unseeded_alignments_gaps_off():
    """mismatches only: the seeded result = the unseeded Hamming ball filtered by the number of
    mismatches inside the read's first seed_len bases (either strand: the seed is the READ's 5' end)."""
    rng = random.Random(808)
    T = [rng.choice([0, 0, 1, 2, 3]) for _ in range(400)]
    o = Oracle(np.asarray(T, dtype=np.uint8))
    SA = o.index(0)[0]
    checked = 0
    for _ in range(60):
        m, z = rng.randint(8, 14), rng.randint(1, 3)
        seed_len, seed_z = rng.randint(2, m - 1), rng.randint(0, 1)
        p = rng.randint(0, len(T) - m)
        W = T[p:p + m]
        for _ in range(rng.randint(0, 3)):
            W[rng.randrange(m)] = rng.randint(0, 3)
        if rng.random() < 0.5:
            W = revcomp(W)
        got = hits_list(o, [np.asarray(W, np.uint8)], (z, 0, 0, seed_len, seed_z, 5))[0]
        want = set()
        for strand in (0, 1):
            Q = W if strand == 0 else revcomp(W)
            seedpos = range(0, seed_len) if strand == 0 else range(m - seed_len, m)
            for s in range(len(T) - m + 1):
                S = T[s:s + m]
                mm = [i for i in range(m) if Q[i] != S[i]]
                if len(mm) <= z and sum(1 for i in mm if i in seedpos) <= seed_z:
                    want.add((strand, s, len(mm)))
        have = set()
        for (s_, k, l, d) in got:
            for row in range(k, l + 1):
                have.add((s_, int(SA[row]), d))
        assert have == want
        checked += len(want)
    assert checked >= 30


# ------------------------------------------------------------------------------- C8: the bucketed suffix sort
@pytest.mark.parametrize("n,alpha", [(1, 4), (5, 1), (11, 2), (12, 4), (13, 4), (300, 1), (5000, 2), (200_000, 4)])
def test_c8_bucketed_suffix_sort_equals_literal_sort(n, alpha):
    """SURVEY C8 allows bucketing by the first 12 bases at sizes the literal sort cannot reach; both builds must
    give the same index (SA, BWT, C, primary) -- incl. texts shorter than the bucket key, runs of one base
    (every suffix in bucket 0 or padded into it) and suffixes that end inside the key."""
    rng = np.random.default_rng(n * 7 + alpha)
    T = rng.integers(0, alpha, size=n).astype(np.uint8)
    if n >= 5000:
        T[100:160] = T[1000:1060]                 # a repeat: deep comparisons inside one bucket
        T[-40:] = 0                               # a run of A at the end: suffixes that are all padding
    a, b = Oracle(T, nthreads=3, sort="literal"), Oracle(T, nthreads=3, sort="bucketed")
    for which in (0, 1):
        SA_a, B_a, C_a, p_a = a.index(which)
        SA_b, B_b, C_b, p_b = b.index(which)
        assert np.array_equal(SA_a, SA_b) and np.array_equal(B_a, B_b) and np.array_equal(C_a, C_b) and p_a == p_b
    if n <= 300:
        from tests.bruteforce import suffix_rows
        assert b.index(0)[0].tolist() == suffix_rows(T.tolist())
