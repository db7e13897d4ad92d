"""GPU parity of bc_pair_batch against the brute-force pairing oracle
(oracle/pairing.py over the oracle's own hits and suffix array)."""
import numpy as np
import pytest

import synthdata as sd
import paper_1505_07855_b200 as bc
from oracle.pairing import pair_reads
from tests.test_gpu_parity import pair_for

pytestmark = pytest.mark.gpu


def run(name, n, n_reads, max_occ, best=None, window=None):
    cfg, p = pair_for(name, n)
    cfg = cfg.scaled(n_reads=n_reads)
    reads = sd.make_reads(cfg, p.T, 0, n_reads)
    opts = cfg.opts.astuple()
    lo, hi = window or (int(cfg.frag_mu - 4 * cfg.frag_sd), int(cfg.frag_mu + 4 * cfg.frag_sd))
    b2, nm, off, ln = sd.pack_reads(reads.codes)
    d = bc.HostReads(b2, nm, off, ln).to_device()
    if best is None:
        res, _ = bc.bc_align_batch(p.ix, d, opts)
    else:
        res, _ = bc.bc_align_batch_best(p.ix, d, opts, best)
    po_g, pairs_g, info = bc.bc_pair_batch(p.ix, res, d, lo, hi, max_occ)
    off_h, hits_h = res.to_numpy()
    SA = p.oracle.index(0)[0]
    # the aligned CSR itself is already proven identical to the oracle's elsewhere; pair the ORACLE's hits
    off_o, hits_o = p.oracle.align(reads.codes, opts)
    if best is not None:
        from tests.test_gpu_best import best_filter
        off_o, hits_o = best_filter(off_o, hits_o, opts[0], best)
    po_o, pairs_o, skipped = pair_reads(SA, off_o, hits_o, ln, lo, hi, max_occ)
    assert np.array_equal(po_g, po_o)
    assert pairs_g.tobytes() == pairs_o.tobytes()
    assert info["skipped_hits"] == skipped and info["pairs"] == pairs_o.size
    return reads, po_g, pairs_g, cfg


def test_pairing_config3_recipe():
    reads, po, pairs, cfg = run("3", 3_000_000, 2000, 32)
    n_pairs = reads.n_reads // 2
    paired = np.diff(po.astype(np.int64)) > 0
    assert paired.mean() > 0.7                           # most synthetic fragments pair up
    # a uniquely paired fragment sits where the generator drew it from
    uniq = np.nonzero(np.diff(po.astype(np.int64)) == 1)[0]
    rec = pairs[po[uniq].astype(np.int64)]
    first_fwd = reads.strand[2 * uniq] == 0
    exp1 = np.where(first_fwd, reads.anchor[2 * uniq], reads.anchor[2 * uniq] - cfg.m)
    assert (np.abs(rec["pos1"].astype(np.int64) - exp1) <= 3).mean() > 0.95


def test_pairing_config4_recipe_best_stratum():
    run("4", 3_000_000, 1200, 16, best=1)


def test_pairing_repeats_small_max_occ_and_tight_window():
    run("3", 3_000_000, 1000, 2, window=(290, 310))
    run("3", 3_000_000, 600, 1000, window=(1, 100000))     # wide window, every repeat copy: many candidates per pair


def test_pairing_edge_cases():
    cfg, p = pair_for("3", 3_000_000)
    reads = sd.make_reads(cfg.scaled(n_reads=64), p.T, 0, 64)
    b2, nm, off, ln = sd.pack_reads(reads.codes)
    d = bc.HostReads(b2, nm, off, ln).to_device()
    res, _ = bc.bc_align_batch(p.ix, d, cfg.opts.astuple())
    with pytest.raises(bc.BcError) as e:                 # min_frag > max_frag
        bc.bc_pair_batch(p.ix, res, d, 500, 100, 8)
    assert e.value.status == bc.BC_E_INVAL
    with pytest.raises(bc.BcError) as e:                 # max_occ = 0
        bc.bc_pair_batch(p.ix, res, d, 100, 500, 0)
    assert e.value.status == bc.BC_E_INVAL
    # junk reads: no hits, no pairs
    rng = np.random.default_rng(3)
    junk = rng.integers(0, 4, size=(32, 76)).astype(np.uint8)
    b2, nm, off, ln = sd.pack_reads(junk)
    dj = bc.HostReads(b2, nm, off, ln).to_device()
    rj, _ = bc.bc_align_batch(p.ix, dj, (1, 0, 0, 0, 0, 5))
    po, pairs, info = bc.bc_pair_batch(p.ix, rj, dj, 100, 500, 8)
    assert po.tolist() == [0] * 17 and pairs.size == 0 and info["placements"] == 0
