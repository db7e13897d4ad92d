"""GPU parity of the best-stratum mode (bc_align_batch_best).  Expected value = the
oracle's EXHAUSTIVE result filtered per read to d <= min(d_min + plus, z) -- the contract's own
definition, computed here in numpy from the oracle output (no GPU value involved)."""
import numpy as np
import pytest

import synthdata as sd
import paper_1505_07855_b200 as bc
from tests.test_gpu_parity import pair_for

pytestmark = pytest.mark.gpu


def best_filter(off, hits, z, plus):
    """exhaustive CSR -> best-stratum CSR (per read: keep d <= min(d_min + plus, z))."""
    n = off.size - 1
    keep = np.zeros(hits.size, bool)
    cnt = np.zeros(n, np.uint64)
    for r in range(n):
        a, b = int(off[r]), int(off[r + 1])
        if b > a:
            d = hits["d"][a:b].astype(np.int64)
            lim = min(int(d.min()) + plus, z)
            keep[a:b] = d <= lim
            cnt[r] = int(keep[a:b].sum())
    off2 = np.concatenate([[0], np.cumsum(cnt)]).astype(np.uint64)
    return off2, hits[keep]


def run_best(ix, codes, opts, plus):
    b2, nm, off, ln = sd.pack_reads(codes)
    d = bc.HostReads(b2, nm, off, ln).to_device()
    res, ws = bc.bc_align_batch_best(ix, d, opts, plus)
    o, h = res.to_numpy()
    return o, h, bc.bc_last_stats(ix)


@pytest.mark.parametrize("name,n,n_reads", [("2", 2_000_000, 3000), ("3", 3_000_000, 3000), ("1", 1_000_000, 5000),
                                             ("5a", 1_000_000, 400)])   # few heavy reads: last-round states change warps
@pytest.mark.parametrize("plus", [0, 1])
def test_best_stratum_equals_filtered_exhaustive(name, n, n_reads, plus):
    cfg, p = pair_for(name, n)
    reads = sd.make_reads(cfg.scaled(n_reads=n_reads), p.T, 0, n_reads)
    opts = cfg.opts.astuple()
    off_o, hits_o = p.oracle.align(reads.codes, opts)
    want_off, want_hits = best_filter(off_o, hits_o, opts[0], plus)
    off_g, hits_g, st = run_best(p.ix, reads.codes, opts, plus)
    assert np.array_equal(off_g, want_off)
    assert hits_g.tobytes() == want_hits.tobytes()
    # the point of the mode: far fewer nodes than the exhaustive search of the same reads
    b2, nm, off, ln = sd.pack_reads(reads.codes)
    bc.bc_align_batch_host(p.ix, bc.HostReads(b2, nm, off, ln), opts)
    full_nodes = bc.bc_last_stats(p.ix)["nodes"]
    assert st["nodes"] < full_nodes


def test_best_stratum_edge_cases():
    cfg, p = pair_for("2", 2_000_000)
    opts = cfg.opts.astuple()
    # plus >= z degenerates to the exhaustive result
    reads = sd.make_reads(cfg.scaled(n_reads=500), p.T, 0, 500)
    off_o, hits_o = p.oracle.align(reads.codes, opts)
    off_g, hits_g, _ = run_best(p.ix, reads.codes, opts, 5)
    assert np.array_equal(off_g, off_o) and hits_g.tobytes() == hits_o.tobytes()
    # z = 0: one pass, exact matches only
    z0 = (0, 0, 0, 0, 0, 5)
    off_o, hits_o = p.oracle.align(reads.codes, z0)
    off_g, hits_g, st = run_best(p.ix, reads.codes, z0, 1)
    assert np.array_equal(off_g, off_o) and hits_g.tobytes() == hits_o.tobytes()
    # reads that match nowhere stay empty and survive every pass
    rng = np.random.default_rng(1)
    junk = rng.integers(0, 4, size=(64, 51)).astype(np.uint8)
    off_o, hits_o = p.oracle.align(junk, opts)
    off_g, hits_g, st = run_best(p.ix, junk, opts, 1)
    assert np.array_equal(off_g, off_o) and hits_g.tobytes() == hits_o.tobytes()
    # invalid stratum
    b2, nm, off, ln = sd.pack_reads(junk)
    d = bc.HostReads(b2, nm, off, ln).to_device()
    ws = bc.BestWorkspace(p.ix, 64, 51, opts)
    assert bc.bc_align_batch_best_raw(p.ix, d, opts, -1, ws) == bc.BC_E_INVAL
    # a hits buffer that is too small is reported, never truncated
    reads = sd.make_reads(cfg.scaled(n_reads=2000), p.T, 0, 2000)
    b2, nm, off, ln = sd.pack_reads(reads.codes)
    d = bc.HostReads(b2, nm, off, ln).to_device()
    ws = bc.BestWorkspace(p.ix, 2000, 51, opts, hits_capacity=100)
    assert bc.bc_align_batch_best_raw(p.ix, d, opts, 1, ws) == bc.BC_E_OVERFLOW


def test_best_stratum_with_a_deep_budget():
    """z >= 9 (the round-1 workspace sizing broke there) and z > 7 (thresholds read from memory, not
    registers): a small batch, plus 0 / 1 / 2, against the filtered oracle result."""
    cfg = sd.CONFIGS["1"].scaled(n=5_000)
    from tests.test_gpu_parity import Pair
    T = sd.make_genome(cfg)
    p = Pair(T)
    rng = np.random.default_rng(21)
    codes = np.stack([T[int(s0):int(s0) + 26] for s0 in rng.integers(0, T.size - 26, size=64)]).astype(np.uint8)
    for r in codes[:48]:                                # 0..6 substitutions: d_min varies from read to read
        for _ in range(int(rng.integers(0, 7))):
            q = int(rng.integers(0, 26))
            r[q] = (r[q] + 1 + int(rng.integers(0, 3))) & 3
    opts = (9, 1, 1, 0, 0, 5)
    off_o, hits_o = p.oracle.align(codes, opts)
    for plus in (0, 1, 2):
        want_off, want_hits = best_filter(off_o, hits_o, opts[0], plus)
        off_g, hits_g, st = run_best(p.ix, codes, opts, plus)
        assert np.array_equal(off_g, want_off), plus
        assert hits_g.tobytes() == want_hits.tobytes(), plus
    assert len(set(np.diff(off_o.astype(np.int64)).tolist())) > 1


def test_best_stratum_and_pairing_with_ragged_lengths_and_N():
    """reads of different lengths (some with N) through the sub-batch gather of the best-stratum
    mode, then through the pairing step (which uses each read's own length)."""
    from oracle.pairing import pair_reads
    cfg, p = pair_for("3", 3_000_000)
    reads = sd.make_reads(cfg.scaled(n_reads=800), p.T, 0, 800)
    rng = np.random.default_rng(8)
    rl = [r[: int(rng.integers(40, reads.m + 1))].copy() for r in reads.codes]
    opts = (3, 1, 2, 24, 1, 5)
    b2, nm, off, ln = sd.pack_ragged(rl)
    d = bc.HostReads(b2, nm, off, ln).to_device()
    res, _ = bc.bc_align_batch_best(p.ix, d, opts, 1)
    off_g, hits_g = res.to_numpy()
    off_o, hits_o = p.oracle.align(rl, opts)
    want_off, want_hits = best_filter(off_o, hits_o, opts[0], 1)
    assert np.array_equal(off_g, want_off) and hits_g.tobytes() == want_hits.tobytes()
    po_g, pairs_g, info = bc.bc_pair_batch(p.ix, res, d, 150, 450, 16)
    po_o, pairs_o, sk = pair_reads(p.oracle.index(0)[0], want_off, want_hits, ln, 150, 450, 16)
    assert np.array_equal(po_g, po_o) and pairs_g.tobytes() == pairs_o.tobytes() and info["skipped_hits"] == sk
