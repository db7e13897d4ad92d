"""GPU parity at index sizes the other tests do not reach ("GPU tests that reach the full-size
paths"): (a) an index above the 64 MB mark at which the library changes its shared-memory split, (b) an index
well beyond the 126 MB L2, where rank queries really go to HBM.  Same bar as everywhere: byte-identical to
the oracle through the C-ABI.  The oracle's own index comes from its literal suffix sort in (a) and from the
bucketed sort SURVEY C8 allows in (b) (pinned against the literal one in tests/test_oracle_pins2.py)."""
import numpy as np
import pytest

import synthdata as sd
import paper_1505_07855_b200 as bc
from oracle import Oracle

pytestmark = pytest.mark.gpu


def _check(cfg, T, host, oracle, n_reads, spread):
    ix = bc.bc_index_upload(host)
    # reads spread over the config's whole read set, not its first n_reads
    first = np.arange(n_reads, dtype=np.int64) * spread
    codes = np.concatenate([sd.make_reads(cfg, T, int(f) & ~1, 2).codes for f in first[::2]])[:n_reads]
    opts = cfg.opts.astuple()
    b2, nm, off, ln = sd.pack_reads(codes)
    off_g, hits_g, _ = bc.bc_align_batch_host(ix, bc.HostReads(b2, nm if (codes == 4).any() else None, off, ln), opts)
    st = bc.bc_last_stats(ix)
    off_o, hits_o = oracle.align(codes, opts)
    assert np.array_equal(off_g, off_o)
    assert hits_g.tobytes() == hits_o.tobytes()
    assert hits_g.size >= 0.5 * n_reads and st["nodes"] > 1000 * n_reads
    rows = hits_g["k"][:: max(1, hits_g.size // 300)].copy()
    assert np.array_equal(bc.bc_locate(ix, rows).cpu().numpy().view(np.uint32), oracle.locate(rows))
    return ix, st


def test_index_above_64MB_config3_recipe():
    cfg = sd.CONFIGS["3"].scaled(n=60_000_000)
    T = sd.make_genome(cfg)
    host = bc.bc_index_build_host(T, 128, 32)
    assert bc.bc_index_device_bytes(host) > (64 << 20)
    _check(cfg, T, host, Oracle(T, sort="literal"), 1200, 3001)


def test_index_beyond_L2_config4_options():
    cfg = sd.CONFIGS["4"].scaled(n=200_000_000)
    T = sd.make_genome(cfg)
    host = bc.bc_index_build_gpu(T, 128, 32)
    assert bc.bc_index_device_bytes(host) > (200 << 20)
    ix, st = _check(cfg, T, host, Oracle(T, sort="bucketed"), 600, 12007)
    assert st["chain_nodes"] > st["branch_nodes"]            # seed-spent states run as exact-match chains
