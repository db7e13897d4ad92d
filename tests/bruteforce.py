"""Brute-force validator for the oracle.  No BWT, no backward search:
enumerate every distinct substring S of T, decide by an explicit alignment DP (definition C2)
whether the query aligns to it and at what minimum d, and map S to its suffix-array interval by
scanning the sorted suffixes.  Pure Python; tiny inputs only.  Shares nothing with oracle/ or the
CUDA path."""
from functools import lru_cache

INF = 10 ** 9


def suffix_rows(T):
    """sorted suffixes of T$ as a list of start positions ($ smallest)."""
    n = len(T)
    return sorted(range(n + 1), key=lambda i: tuple(T[i:]) + (-1,))


def interval_of(T, rows, S):
    """[k,l] = rows whose suffix starts with S (S occurs in T)."""
    L = len(S)
    hit = [j for j, p in enumerate(rows) if tuple(T[p:p + L]) == tuple(S)]
    assert hit and hit == list(range(hit[0], hit[-1] + 1))
    return hit[0], hit[-1]


def min_d(Q, S, opts, ban=True):
    """minimum d over valid alignments (C2) of Q to S, or None.  opts = (z, go, ge, seed_len, seed_z, E);
    the seed range [s0,s1) is passed in Q indices via opts[3] = (s0, s1) or None."""
    z, max_go, max_ge, seed, seed_z, E = opts
    m, L = len(Q), len(S)
    s0, s1 = seed if seed else (0, 0)
    seed_on = seed is not None

    @lru_cache(maxsize=None)
    def f(i, j, st, go, ge, sd):
        # i read bases and j reference bases consumed; st = type of the previous column
        if i == m and j == L:
            return 0
        best = INF
        if i < m and j < L:                                   # M(i)
            c = 0 if (Q[i] == S[j] and Q[i] < 4) else 1
            nsd = sd + (c if (seed_on and s0 <= i < s1) else 0)
            if not seed_on or nsd <= seed_z:
                best = min(best, c + f(i + 1, j + 1, 0, go, ge, nsd))
        if i < m and not (ban and st == 2) and i >= E and m - 1 - i >= E:   # I(i)
            ngo, nge = (go + 1, ge) if st != 1 else (go, ge + 1)
            nsd = sd + (1 if (seed_on and s0 <= i < s1) else 0)
            if ngo <= max_go and nge <= max_ge and (not seed_on or nsd <= seed_z):
                best = min(best, 1 + f(i + 1, j, 1, ngo, nge, nsd))
        if j < L and not (ban and st == 1) and i >= E and m - i >= E:       # D, i read bases to its left
            ngo, nge = (go + 1, ge) if st != 2 else (go, ge + 1)
            nsd = sd + (1 if (seed_on and s0 < i < s1) else 0)
            if ngo <= max_go and nge <= max_ge and (not seed_on or nsd <= seed_z):
                best = min(best, 1 + f(i, j + 1, 2, ngo, nge, nsd))
        return best

    d = f(0, 0, 0, 0, 0, 0)
    return d if d <= z else None


def revcomp(W):
    return [3 - c if c < 4 else 4 for c in reversed(W)]


def brute_align(T, W, opts6, ban=True):
    """Expected output for one read: list of (strand, k, l, d) sorted by (strand, k, l).
    opts6 = (z, go, ge, seed_len, seed_z, E) as in bc_opts."""
    z, go, ge, seed_len, seed_z, E = opts6
    T = list(T)
    n, m = len(T), len(W)
    rows = suffix_rows(T)
    out = []
    maxgap = min(z, go + ge)
    for strand in (0, 1):
        Q = list(W) if strand == 0 else revcomp(W)
        seed = None
        if 0 < seed_len < m:
            seed = (0, seed_len) if strand == 0 else (m - seed_len, m)
        res = {}
        seen = set()
        for L in range(max(1, m - maxgap), m + maxgap + 1):
            for p in range(0, n - L + 1):
                S = tuple(T[p:p + L])
                if S in seen:
                    continue
                seen.add(S)
                d = min_d(tuple(Q), S, (z, go, ge, seed, seed_z, E), ban)
                if d is None:
                    continue
                kl = interval_of(T, rows, S)
                if kl not in res or d < res[kl]:
                    res[kl] = d
        out += [(strand, k, l, d) for (k, l), d in sorted(res.items())]
    return out
