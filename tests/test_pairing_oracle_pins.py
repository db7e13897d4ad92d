"""Pins for the pairing oracle (oracle/pairing.py) against hand-worked cases: the definition of
DESIGN.md 7c written out by hand (positions, orientation, fragment length, dedup, max_occ)."""
import numpy as np

from oracle import HIT_DTYPE
from oracle.pairing import pair_reads, placements


def hits(*recs):
    return np.asarray([(k, l, d, s, 0) for (k, l, d, s) in recs], dtype=HIT_DTYPE)


def test_hand_worked_pairs():
    # suffix array rows -> positions chosen by hand: row j sits at position SA[j]
    SA = np.asarray([0, 100, 350, 5000, 100, 40, 900, 650], np.uint32)
    # pair 0: end 1 forward at 100 (row 1, d=0) and AGAIN at 100 via row 4 with d=2 (another interval
    #         holding the same position); end 2 reverse at 350 (row 2, d=1) and at 5000 (row 3, d=0)
    # pair 1: end 1 reverse at 650 (row 7), end 2 forward at 40 (row 5) and forward at 900 (row 6)
    # pair 2: both ends on the same strand -> nothing
    h = hits((1, 1, 0, 0), (4, 4, 2, 0), (2, 3, 1, 1),          # read 0 (two hits), read 1 (one hit, rows 2..3)
             (7, 7, 3, 1), (5, 6, 0, 0),                        # read 2, read 3 (rows 5..6)
             (1, 1, 0, 0), (5, 5, 0, 0))                        # read 4, read 5: both strand 0
    off = np.asarray([0, 2, 3, 4, 5, 6, 7], np.uint64)
    lens = np.asarray([50, 50, 60, 60, 50, 50], np.uint16)
    po, pairs, skipped = pair_reads(SA, off, h, lens, 200, 700, max_occ=8)
    assert po.tolist() == [0, 1, 2, 2] and skipped == 0
    # pair 0: forward end at 100, reverse end at 350, fragment = 350 + 50 - 100 = 300; 5000 is too far;
    #         the two placements at position 100 collapse to the smaller d1
    assert pairs[0].tolist() == (100, 350, 300, 0, 1, 0, 0)
    # pair 1: end 1 is the reverse one (strand1 = 1) at 650, len 60; forward end 2 at 40: 650 + 60 - 40 = 670 ok;
    #         forward end at 900 lies downstream of the reverse end -> not proper
    assert pairs[1].tolist() == (650, 40, 670, 3, 0, 1, 0)
    # window excludes everything
    po2, pairs2, _ = pair_reads(SA, off, h, lens, 301, 669, max_occ=8)
    assert po2.tolist() == [0, 0, 0, 0] and pairs2.size == 0
    # max_occ = 1 skips the 2-row hit of read 1 and of read 3
    po3, pairs3, sk3 = pair_reads(SA, off, h, lens, 200, 700, max_occ=1)
    assert po3.tolist() == [0, 0, 0, 0] and sk3 == 2


def test_placements_expand_rows():
    SA = np.asarray([7, 3, 9, 1], np.uint32)
    pl, sk = placements(SA, hits((1, 3, 2, 1), (0, 3, 0, 0)), max_occ=3)
    assert pl == [(3, 1, 2), (9, 1, 2), (1, 1, 2)] and sk == 1
