"""Pins for the oracle.  CPU only.  None of these re-types the oracle's
formulae: they compare it with Python's sorted(), naive scanning, an alignment DP over enumerated
substrings (tests/bruteforce.py), Hamming / Wagner-Fischer textbook definitions and invariants."""
import os
import random
import re

import numpy as np
import pytest

import synthdata as sd
from oracle import Oracle, FLAG_PRUNE, FLAG_BAN_ID, FLAG_PLUS_5P_FIRST, DEFAULT_FLAGS
from tests.bruteforce import brute_align, suffix_rows, revcomp

GOLD = os.path.join(os.path.dirname(__file__), "golden", "worked_example.txt")


def hits_list(oracle, reads, opts, flags=DEFAULT_FLAGS):
    off, h = oracle.align(reads, opts, flags)
    out = []
    for r in range(len(reads)):
        out.append([(int(x["strand"]), int(x["k"]), int(x["l"]), int(x["d"])) for x in h[int(off[r]):int(off[r + 1])]])
    return out


def parse_gold():
    g = {"HIT": [], "D": []}
    for line in open(GOLD):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        tag, rest = line.split(" ", 1)
        if tag == "HIT":
            left, right = rest.split(":")
            f = left.split()
            read, (z, go, ge, E, sl, sz) = f[0], map(int, f[1:7])
            hits = []
            if right.strip() != "-":
                for rec in right.split(";"):
                    v = rec.strip().split(",")
                    pos = sorted(int(p) for p in v[4].split("|")) if len(v) > 4 else None
                    hits.append((int(v[0]), int(v[1]), int(v[2]), int(v[3]), pos))
            g["HIT"].append((read, (z, go, ge, sl, sz, E), hits))
        elif tag == "D":
            q, v = rest.split()
            g["D"].append((q, [int(x) for x in v.split(",")]))
        else:
            g[tag] = rest
    return g


# ------------------------------------------------------------------------------------------- P1
def test_p1_worked_example_index():
    g = parse_gold()
    T = sd.encode(g["T"])
    o = Oracle(T)
    SA, B, C, primary = o.index(0)
    assert SA.tolist() == [int(x) for x in g["SA"].split(",")]
    assert "".join("ACGT$"[b] for b in B) == g["B"]
    assert primary == int(g["PRIMARY"])
    assert C.tolist() == [int(x) for x in g["C"].split(",")]
    rSA, rB, rC, rprimary = o.index(1)
    assert sd.decode(T[::-1]) == g["RT"]
    assert rSA.tolist() == [int(x) for x in g["RSA"].split(",")]
    assert "".join("ACGT$"[b] for b in rB) == g["RB"]
    assert rprimary == int(g["RPRIMARY"])
    assert [o.occ(0, 0, j) for j in range(-1, 22)] == [int(x) for x in g["OA"].split(",")]
    # and the fixture's SA is what Python's sorted() says
    assert suffix_rows(T.tolist()) == SA.tolist()


@pytest.mark.parametrize("flags", [DEFAULT_FLAGS, FLAG_BAN_ID, FLAG_PRUNE | FLAG_BAN_ID, 0])
def test_p1_worked_example_hits(flags):
    g = parse_gold()
    T = sd.encode(g["T"])
    o = Oracle(T)
    for read, opts, want in g["HIT"]:
        got = hits_list(o, [sd.encode(read)], opts, flags)[0]
        assert got == [w[:4] for w in want], (read, opts)
        for (s, k, l, d, pos) in want:
            if pos is not None:
                assert sorted(o.locate(np.arange(k, l + 1)).tolist()) == pos


def test_p1_worked_example_hits_bruteforce():
    """the fixture itself agrees with the brute-force validator (so a typo in it cannot hide)."""
    g = parse_gold()
    T = sd.encode(g["T"]).tolist()
    for read, opts, want in g["HIT"]:
        assert brute_align(T, sd.encode(read).tolist(), opts) == [w[:4] for w in want], (read, opts)


def test_p1_D_arrays():
    g = parse_gold()
    o = Oracle(sd.encode(g["T"]))
    for q, want in g["D"]:
        assert o.D(sd.encode(q)).tolist() == want


# ------------------------------------------------------------------------------------------- P2
def naive_positions(Ts, Qs):
    return [mm.start() for mm in re.finditer("(?=" + Qs + ")", Ts)]


def test_p2_exact_match_equals_naive_count():
    rng = random.Random(11)
    T = np.asarray([rng.choice([0, 0, 1, 2, 3]) for _ in range(5000)], dtype=np.uint8)
    Ts = sd.decode(T)
    o = Oracle(T)
    reads = []
    for _ in range(300):
        m = rng.randint(1, 14)
        if rng.random() < 0.7:
            p = rng.randint(0, len(T) - m)
            w = T[p:p + m].copy()
            if rng.random() < 0.5:
                w = np.asarray(revcomp(w.tolist()), dtype=np.uint8)
        else:
            w = np.asarray([rng.randint(0, 3) for _ in range(m)], dtype=np.uint8)
        reads.append(w)
    res = hits_list(o, reads, (0, 0, 0, 0, 0, 1))
    for w, hits in zip(reads, res):
        for strand in (0, 1):
            q = w.tolist() if strand == 0 else revcomp(w.tolist())
            pos = naive_positions(Ts, sd.decode(q))
            mine = [h for h in hits if h[0] == strand]
            assert len(mine) == (1 if pos else 0)            # at most one hit per strand
            if pos:
                _, k, l, d = mine[0]
                assert d == 0 and l - k + 1 == len(pos)       # distance between the pointers
                assert sorted(o.locate(np.arange(k, l + 1)).tolist()) == pos


# ------------------------------------------------------------------------------------------- P3
def _rand_case(rng):
    n = rng.randint(12, 40)
    alpha = rng.choice([[0, 1], [0, 1, 2, 3], [0, 0, 0, 1, 2, 3], [0, 3]])
    T = [rng.choice(alpha) for _ in range(n)]
    if rng.random() < 0.5 and n > 20:           # plant a repeat
        a, L = rng.randint(0, n - 16), rng.randint(4, 8)
        b = rng.randint(0, n - L)
        T[b:b + L] = T[a:a + L]
    m = rng.randint(2, 9)
    p = rng.randint(0, n - m)
    W = T[p:p + m]
    for _ in range(rng.randint(0, 2)):          # a few edits so that inexact paths are exercised
        r = rng.random()
        q = rng.randrange(len(W))
        if r < 0.5:
            W[q] = rng.randint(0, 3)
        elif r < 0.7 and len(W) > 2:
            del W[q]
        elif r < 0.9:
            W.insert(q, rng.randint(0, 3))
        else:
            W[q] = 4
    if rng.random() < 0.5:
        W = revcomp(W)
    m = len(W)
    z = rng.randint(0, 3)
    go = rng.randint(0, 2)
    ge = rng.randint(0, 2)
    E = rng.choice([0, 1, 2, 5])
    seed_len = rng.choice([0, 0, rng.randint(1, max(1, m))])
    seed_z = rng.randint(0, 2)
    return T, W, (z, go, ge, seed_len, seed_z, E)


@pytest.mark.parametrize("chunk", range(6))
def test_p3_bruteforce_tiny_genomes(chunk):
    rng = random.Random(1000 + chunk)
    for _ in range(22):
        T, W, opts = _rand_case(rng)
        want = brute_align(T, W, opts)
        o = Oracle(np.asarray(T, dtype=np.uint8), nthreads=1)
        for flags in (0, FLAG_BAN_ID, DEFAULT_FLAGS, FLAG_PRUNE | FLAG_PLUS_5P_FIRST):
            got = hits_list(o, [np.asarray(W, dtype=np.uint8)], opts, flags)[0]
            assert got == want, (T, W, opts, flags)


def test_p3_ban_is_result_neutral_in_the_definition():
    """C2-2: the I/D adjacency ban does not change the result set (checked on the DP itself)."""
    rng = random.Random(77)
    for _ in range(25):
        T, W, opts = _rand_case(rng)
        assert brute_align(T, W, opts, ban=True) == brute_align(T, W, opts, ban=False)


# ------------------------------------------------------------------------------------------- P4
def _intervals_of_strings(T, strings_d):
    rows = suffix_rows(T)
    res = {}
    for S, d in strings_d.items():
        L = len(S)
        hit = [j for j, p in enumerate(rows) if tuple(T[p:p + L]) == S]
        kl = (hit[0], hit[-1])
        res[kl] = min(d, res.get(kl, 99))
    return sorted((k, l, d) for (k, l), d in res.items())


def test_p4_gaps_off_is_hamming():
    rng = random.Random(5)
    T = [rng.choice([0, 0, 1, 2, 3]) for _ in range(300)]
    o = Oracle(np.asarray(T, dtype=np.uint8))
    for _ in range(40):
        m, z = rng.randint(3, 10), rng.randint(0, 3)
        p = rng.randint(0, len(T) - m)
        W = T[p:p + m]
        for _ in range(rng.randint(0, 2)):
            W[rng.randrange(m)] = rng.choice([0, 1, 2, 3, 4])
        got = hits_list(o, [np.asarray(W, np.uint8)], (z, 0, 0, 0, 0, 5))[0]
        for strand in (0, 1):
            Q = W if strand == 0 else revcomp(W)
            sd_ = {}
            for s in range(len(T) - m + 1):
                S = tuple(T[s:s + m])
                ham = sum(1 for a, b in zip(Q, S) if a != b or a == 4)
                if ham <= z:
                    sd_[S] = ham
            want = _intervals_of_strings(T, sd_)
            assert [(k, l, d) for (s, k, l, d) in got if s == strand] == want


def levenshtein(a, b):
    prev = list(range(len(b) + 1))
    for i, ca in enumerate(a, 1):
        cur = [i]
        for j, cb in enumerate(b, 1):
            cur.append(min(prev[j] + 1, cur[j - 1] + 1, prev[j - 1] + (0 if (ca == cb and ca < 4) else 1)))
        prev = cur
    return prev[-1]


def test_p4_free_gaps_is_levenshtein():
    """E = 0, max_gap_open = max_gap_ext = z, no seed, m > z  =>  all substrings within edit distance z."""
    rng = random.Random(6)
    T = [rng.choice([0, 1, 2, 3]) for _ in range(60)]
    o = Oracle(np.asarray(T, dtype=np.uint8))
    for _ in range(12):
        z = rng.randint(1, 2)
        m = rng.randint(z + 2, 8)
        p = rng.randint(0, len(T) - m)
        W = T[p:p + m]
        if rng.random() < 0.7:
            W[rng.randrange(m)] = rng.randint(0, 3)
        got = hits_list(o, [np.asarray(W, np.uint8)], (z, z, z, 0, 0, 0))[0]
        for strand in (0, 1):
            Q = W if strand == 0 else revcomp(W)
            sd_ = {}
            for L in range(max(1, m - z), m + z + 1):
                for s in range(len(T) - L + 1):
                    S = tuple(T[s:s + L])
                    if S not in sd_:
                        d = levenshtein(Q, S)
                        if d <= z:
                            sd_[S] = d
            assert [(k, l, d) for (s, k, l, d) in got if s == strand] == _intervals_of_strings(T, sd_)


# ------------------------------------------------------------------------------------------- P5
@pytest.fixture(scope="module")
def mid():
    cfg = sd.CONFIGS["2"].scaled(n=60_000, n_reads=120)
    g = sd.make_genome(cfg)
    return cfg, g, Oracle(g), sd.make_reads(cfg, g)


def test_p5_flag_invariance_and_monotone_in_z(mid):
    cfg, g, o, reads = mid
    R = reads.codes[:60]
    opts = (2, 1, 2, 0, 0, 5)
    base = hits_list(o, R, opts)
    for flags in (0, FLAG_BAN_ID, FLAG_PRUNE, FLAG_PRUNE | FLAG_BAN_ID, FLAG_PLUS_5P_FIRST, FLAG_PRUNE | FLAG_PLUS_5P_FIRST):
        assert hits_list(o, R, opts, flags) == base
    seeded = (3, 1, 2, 20, 1, 5)
    a = hits_list(o, R, seeded)
    assert hits_list(o, R, seeded, FLAG_BAN_ID) == a            # textbook direction, no prune
    bigger = hits_list(o, R, (3, 1, 2, 0, 0, 5))
    for lo, hi in zip(base, bigger):                              # R(z) subset of R(z+1), d unchanged
        assert set(lo) <= set(hi)
    for s_, b_ in zip(a, bigger):                                 # a seed limit only removes hits
        assert {x[:3] for x in s_} <= {x[:3] for x in b_}
    assert sum(len(x) for x in base) >= 50                        # the reads do align


def test_p5_strand_and_reversal_symmetry(mid):
    cfg, g, o, reads = mid
    R = reads.codes[:40]
    opts = (2, 1, 2, 0, 0, 5)       # no seed: the seed is the READ's 5' end, which revcomp moves
    a = hits_list(o, R, opts)
    rc = np.asarray([revcomp(r.tolist()) for r in R], dtype=np.uint8)
    b = hits_list(o, rc, opts)
    for x, y in zip(a, b):
        # hits of W on strand + = hits of revcomp(W) on strand -
        assert [(k, l, d) for (s, k, l, d) in x if s == 0] == [(k, l, d) for (s, k, l, d) in y if s == 1]
        assert [(k, l, d) for (s, k, l, d) in x if s == 1] == [(k, l, d) for (s, k, l, d) in y if s == 0]
    # reversal: reverse(Q) against reverse(T) has the mirrored position sets (no seed, symmetric rules)
    opts = (2, 1, 2, 0, 0, 5)
    o_rev = Oracle(g[::-1].copy())
    a = hits_list(o, R[:15], opts)
    b = hits_list(o_rev, np.ascontiguousarray(R[:15, ::-1]), opts)
    n = len(g)
    for x, y in zip(a, b):
        wa = sorted(int(l - k + 1) for (s, k, l, d) in x if s == 0)
        wb = sorted(int(l - k + 1) for (s, k, l, d) in y if s == 0)
        assert sum(wa) == sum(wb)
        da = sorted(d for (s, k, l, d) in x if s == 0)
        db = sorted(d for (s, k, l, d) in y if s == 0)
        assert (min(da) if da else None) == (min(db) if db else None)


def test_p5_bwt_inversion_locate_and_totals(mid):
    cfg, g, o, reads = mid
    n = len(g)
    for which, text in ((0, g), (1, g[::-1])):
        SA, B, C, primary = o.index(which)
        assert sorted(SA.tolist()) == list(range(n + 1)) and SA[0] == n and SA[primary] == 0
        assert C.tolist() == [0] + np.cumsum(np.bincount(text, minlength=4)).tolist()
        for c in range(4):
            assert o.occ(which, c, n) == int((text == c).sum())
            assert o.occ(which, c, -1) == 0
        # LF-walk from `primary` spells T backwards:  j <- C[c] + O(c, j),  c = B[j]
        # start at the row of the whole text (SA = 0): its BWT symbol is '$'; begin from row 0 ('$' suffix)
        j, out = 0, []
        for _ in range(2000):
            c = int(B[j])
            out.append(c)
            j = int(C[c]) + o.occ(which, c, j)
        assert out == text[::-1][:2000].tolist()
    SA = o.index(0)[0]
    rows = np.asarray([0, 1, 5, n // 2, n - 1, n], dtype=np.uint32)
    assert o.locate(rows).tolist() == SA[rows].tolist()
    # spot-check SA order against direct suffix comparison
    rng = random.Random(3)
    gb = g.tobytes()
    for _ in range(300):
        j = rng.randint(0, n - 1)
        assert gb[SA[j]:] + b"" < gb[SA[j + 1]:] or gb[SA[j + 1]:].startswith(gb[SA[j]:])


# ------------------------------------------------------------------------------------------- P6
def min_diffs_anywhere(Q, T):
    """Sellers: min edit distance of Q to any substring of T (N never matches)."""
    prev = [0] * (len(T) + 1)
    for i, cq in enumerate(Q, 1):
        cur = [i]
        for j, ct in enumerate(T, 1):
            cur.append(min(prev[j] + 1, cur[j - 1] + 1, prev[j - 1] + (0 if (cq == ct and cq < 4) else 1)))
        prev = cur
    return min(prev)


def test_p6_D_is_admissible():
    rng = random.Random(9)
    for _ in range(30):
        T, W, _ = _rand_case(rng)
        o = Oracle(np.asarray(T, dtype=np.uint8), nthreads=1)
        D = o.D(np.asarray(W, np.uint8)).tolist()
        assert all(b - a in (0, 1) for a, b in zip([0] + D, D))
        for i in range(len(W)):
            assert D[i] <= min_diffs_anywhere(W[:i + 1], T), (T, W, i)
