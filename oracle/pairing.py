"""ORACLE -- test infrastructure, not product code.  Brute-force pairing of located positions
(SURVEY 8f NEXT-1 oracle; definition in DESIGN.md 7c; "paired by plausible
distance").  Plain Python over the oracle's own hits and its full suffix array; shares nothing with
the CUDA path."""
import numpy as np

PAIR_DTYPE = np.dtype([("pos1", "<u4"), ("pos2", "<u4"), ("frag", "<u4"), ("d1", "u1"), ("d2", "u1"), ("strand1", "u1"),
                       ("zero", "u1")])


def placements(SA, hits, max_occ):
    """hits of one read -> list of (pos, strand, d); hits with more than max_occ occurrences are skipped."""
    out, skipped = [], 0
    for h in hits:
        k, l = int(h["k"]), int(h["l"])
        if l - k + 1 > max_occ:
            skipped += 1
            continue
        for j in range(k, l + 1):
            out.append((int(SA[j]), int(h["strand"]), int(h["d"])))
    return out, skipped


def pair_reads(SA, off, hits, lens, min_frag, max_frag, max_occ):
    """CSR of an aligned batch (reads 2i, 2i+1 = ends of pair i) -> (pair_offsets, pairs, skipped)."""
    n_pairs = (off.size - 1) // 2
    recs, counts, skipped = [], [], 0
    for i in range(n_pairs):
        A, s1 = placements(SA, hits[int(off[2 * i]):int(off[2 * i + 1])], max_occ)
        B, s2 = placements(SA, hits[int(off[2 * i + 1]):int(off[2 * i + 2])], max_occ)
        skipped += s1 + s2
        la, lb = int(lens[2 * i]), int(lens[2 * i + 1])
        best = {}
        for (pa, sa, da) in A:
            for (pb, sb, db) in B:
                if sa == sb:
                    continue
                pf, pr, lr = (pa, pb, lb) if sa == 0 else (pb, pa, la)
                if pr < pf:
                    continue
                frag = pr + lr - pf
                if not (min_frag <= frag <= max_frag):
                    continue
                key = (pa, pb, sa)
                val = (da + db, da, db, frag)
                if key not in best or val < best[key]:
                    best[key] = val
        for key in sorted(best):
            dsum, da, db, frag = best[key]
            recs.append((key[0], key[1], frag, da, db, key[2], 0))
        counts.append(len(best))
    po = np.concatenate([[0], np.cumsum(counts)]).astype(np.uint64)
    return po, np.asarray(recs, dtype=PAIR_DTYPE) if recs else np.zeros(0, PAIR_DTYPE), skipped
