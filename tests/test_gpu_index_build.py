"""GPU index construction (bc_index_build_gpu) against the oracle's naive suffix
sort, element by element: BWT, Occ checkpoints, C, primary, SA sample of both directions."""
import numpy as np
import pytest

import synthdata as sd
import paper_1505_07855_b200 as bc
from oracle import Oracle
from tests.test_host_logic import unpack_bwt

pytestmark = pytest.mark.gpu


def check(T, occ_interval=128, sa_interval=32):
    n = T.size
    h = bc.bc_index_build_gpu(T, occ_interval, sa_interval)
    o = Oracle(T)
    for which in (0, 1):
        SA, B, Cc, primary = o.index(which)
        bwt2, occ, Ch, prim_h, oi = h.arrays(which)
        assert prim_h == primary and Ch == Cc.tolist() and oi == occ_interval
        want = B[B != 4]
        assert np.array_equal(unpack_bwt(bwt2, n), want)
        assert not (bwt2[-1] >> np.uint64(2 * (n % 32))) if n % 32 else True      # padding bits are zero
        for c in range(4):
            pref = np.concatenate([[0], np.cumsum(want == c)])
            assert np.array_equal(occ[:, c], pref[np.arange(occ.shape[0]) * occ_interval])
        if which == 0:
            sa, si = h.sa_samples()
            assert si == sa_interval and np.array_equal(sa, SA[::sa_interval])
    return h


@pytest.mark.parametrize("n,oi,si", [(1, 32, 1), (5, 32, 4), (63, 32, 8), (64, 64, 32), (65, 128, 32), (4096, 128, 32),
                                     (100_003, 128, 7)])
def test_gpu_build_matches_naive_suffix_sort(n, oi, si):
    T = (sd.hash_u64(91, 1, np.arange(n, dtype=np.uint64)) >> np.uint64(62)).astype(np.uint8)
    check(T, oi, si)


def test_gpu_build_long_runs_and_repeats():
    # LCPs far beyond the 21-symbol initial key: several doubling rounds
    T = np.concatenate([np.zeros(3000, np.uint8), np.tile(np.asarray([0, 1, 2, 3, 3, 1], np.uint8), 700),
                        np.full(1000, 3, np.uint8), np.zeros(500, np.uint8)])
    check(T)
    check(sd.make_genome(sd.CONFIGS["2"].scaled(n=1_000_000)))


def test_gpu_built_index_is_identical_to_the_host_built_one_and_aligns():
    cfg = sd.CONFIGS["3"].scaled(n=2_000_000, n_reads=1000)
    T = sd.make_genome(cfg)
    hg, hh = bc.bc_index_build_gpu(T), bc.bc_index_build_host(T, 128, 32)
    for which in (0, 1):
        a, b = hg.arrays(which), hh.arrays(which)
        assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1]) and a[2:] == b[2:]
    assert np.array_equal(hg.sa_samples()[0], hh.sa_samples()[0])
    ix = bc.bc_index_upload(hg)
    reads = sd.make_reads(cfg, T, 0, 1000)
    b2, nm, off, ln = sd.pack_reads(reads.codes)
    off_g, hits_g, _ = bc.bc_align_batch_host(ix, bc.HostReads(b2, nm, off, ln), cfg.opts.astuple())
    off_o, hits_o = Oracle(T).align(reads.codes, cfg.opts.astuple())
    assert np.array_equal(off_g, off_o) and hits_g.tobytes() == hits_o.tobytes()
    with pytest.raises(bc.BcError):
        bc.bc_index_build_gpu(np.asarray([0, 1, 5], np.uint8))
