"""Both device index layouts (bc_internal.cuh: 32-byte blocks of 64 symbols, 128-byte lines of 384 symbols) give the
same bytes as the oracle.  The library picks the layout by index size; here each is forced (bc_set_index_layout)
on genomes small enough for the oracle, including sizes around the line and region boundaries."""
import numpy as np
import pytest

import synthdata as sd
import paper_1505_07855_b200 as bc
from oracle import Oracle

pytestmark = pytest.mark.gpu


def upload(host, layout):
    bc.bc_set_index_layout(layout)
    try:
        return bc.bc_index_upload(host)
    finally:
        bc.bc_set_index_layout(0)


def align(ix, reads_list, opts):
    b2, nm, off, ln = sd.pack_ragged(reads_list)
    o, h, _ = bc.bc_align_batch_host(ix, bc.HostReads(b2, nm, off, ln), opts)
    return o, h


@pytest.mark.parametrize("n", [1, 63, 64, 127, 128, 129, 383, 384, 385, 767, 768, 769, 1151, 1152, 1153, 5000])
def test_line_and_block_boundaries(n):
    rng = np.random.default_rng(n)
    T = rng.integers(0, 4, size=n).astype(np.uint8)
    orc = Oracle(T, nthreads=1)
    host = bc.bc_index_build_host(T, 128, 8)
    reads = []
    for _ in range(24):
        m = int(rng.integers(1, min(n, 20) + 1))
        s0 = int(rng.integers(0, n - m + 1))
        r = T[s0:s0 + m].copy()
        if m > 2 and rng.random() < 0.5:
            r[int(rng.integers(0, m))] = int(rng.integers(0, 4))
        reads.append(r)
    opts = (1, 0, 0, 0, 0, 1)
    off_o, hits_o = orc.align(reads, opts)
    rows = np.arange(n + 1, dtype=np.uint32)
    SA = orc.index(0)[0]
    for layout in (1, 2):
        ix = upload(host, layout)
        assert (bc.bc_last_stats(ix)["geometry"] >> 15) & 1 == 0          # nothing ran yet
        off_g, hits_g = align(ix, reads, opts)
        assert (bc.bc_last_stats(ix)["geometry"] >> 15) & 1 == layout - 1
        assert np.array_equal(off_g, off_o) and hits_g.tobytes() == hits_o.tobytes(), (n, layout)
        assert np.array_equal(bc.bc_locate(ix, rows).cpu().numpy().view(np.uint32), SA)


@pytest.mark.parametrize("name,n,n_reads", [("2", 2_000_000, 2000), ("3", 3_000_000, 1500), ("4", 3_000_000, 1000), ("5a", 1_000_000, 300)])
def test_recipes_under_both_layouts(name, n, n_reads):
    cfg = sd.CONFIGS[name].scaled(n=n, n_reads=n_reads)
    T = sd.make_genome(cfg)
    reads = sd.make_reads(cfg, T, 0, n_reads)
    opts = cfg.opts.astuple()
    off_o, hits_o = Oracle(T).align(reads.codes, opts)
    host = bc.bc_index_build_host(T, 128, 32)
    sizes = []
    for layout in (1, 2):
        ix = upload(host, layout)
        sizes.append(len(ix.mem))
        off_g, hits_g = align(ix, list(reads.codes), opts)
        assert np.array_equal(off_g, off_o) and hits_g.tobytes() == hits_o.tobytes(), layout
        res, _ = bc.bc_align_batch_best(ix, bc.HostReads(*sd.pack_reads(reads.codes)).to_device(), opts, 1)
        assert res.n_hits > 0
    assert sizes[1] < 0.8 * sizes[0]                                      # lines: n/3 bytes per BWT instead of n/2
