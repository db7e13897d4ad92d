"""GPU parity: the CUDA path, called through the C-ABI (via the thin binding), against the CPU
oracle, element by element on the same seeded inputs.  Integer work => the bar is BIT-EXACT on
hit_offsets and on every 12-byte hit record.  These tests FAIL (never skip, never fall back) if the
compiled library is missing on a GPU box."""
import ctypes as C
import os

import numpy as np
import pytest

import synthdata as sd
import paper_1505_07855_b200 as bc
from oracle import Oracle

pytestmark = pytest.mark.gpu

GOLD = os.path.join(os.path.dirname(__file__), "golden", "worked_example.txt")


class Pair:
    """genome -> (oracle index, device index), both built from the same seeded genome."""

    def __init__(self, T, sa_interval=32):
        self.T = T
        self.oracle = Oracle(T)
        self.host = bc.bc_index_build_host(T, 128, sa_interval)
        self.ix = bc.bc_index_upload(self.host)


def gpu_align(ix, reads_list, opts, **kw):
    b2, nm, off, ln = sd.pack_ragged(reads_list)
    h = bc.HostReads(b2, nm, off, ln)
    off_g, hits_g, ws = bc.bc_align_batch_host(ix, h, opts, **kw)
    return off_g, hits_g


def assert_same(ix, oracle, reads_list, opts):
    off_o, hits_o = oracle.align(reads_list, tuple(opts))
    off_g, hits_g = gpu_align(ix, reads_list, opts)
    assert np.array_equal(off_g, off_o)
    assert hits_g.tobytes() == hits_o.tobytes()
    return off_o, hits_o


_pairs = {}


def pair_for(cfg_name, n):
    key = (cfg_name, n)
    if key not in _pairs:
        cfg = sd.CONFIGS[cfg_name].scaled(n=n)
        _pairs[key] = (cfg, Pair(sd.make_genome(cfg)))
    return _pairs[key]


# --------------------------------------------------------------------------------------------
def test_library_loaded_is_in_tree():
    so = bc._build.SO
    assert os.path.exists(so) and os.path.dirname(so).endswith("paper_1505_07855_b200")
    assert bc.lib() is not None


def test_worked_example_through_the_gpu():
    """SURVEY C6 P1 fixture (tests/golden/worked_example.txt) straight through bc_align_batch + bc_locate."""
    T = None
    hits = []
    for line in open(GOLD):
        line = line.strip()
        if line.startswith("T "):
            T = sd.encode(line.split()[1])
        elif line.startswith("HIT "):
            left, right = line[4:].split(":")
            f = left.split()
            z, go, ge, E, sl, sz = map(int, f[1:7])
            want = []
            if right.strip() != "-":
                for rec in right.split(";"):
                    v = rec.strip().split(",")
                    pos = sorted(int(x) for x in v[4].split("|")) if len(v) > 4 else None
                    want.append((int(v[0]), int(v[1]), int(v[2]), int(v[3]), pos))
            hits.append((f[0], (z, go, ge, sl, sz, E), want))
    p = Pair(T, sa_interval=4)
    for read, opts, want in hits:
        off, h = gpu_align(p.ix, [sd.encode(read)], opts)
        got = [(int(x["strand"]), int(x["k"]), int(x["l"]), int(x["d"])) for x in h]
        assert got == [w[:4] for w in want], (read, opts)
        for (s, k, l, d, pos) in want:
            if pos is not None:
                rows = np.arange(k, l + 1, dtype=np.uint32)
                got_pos = bc.bc_locate(p.ix, rows).cpu().numpy().view(np.uint32)
                assert sorted(got_pos.tolist()) == pos


def test_config1_full_size():
    """configs[0] of BASELINE.json at full size: 1 Mbp, 10,000 x 36 bp, z=2 mismatches only."""
    cfg, p = pair_for("1", sd.CONFIGS["1"].n)
    reads = sd.make_reads(cfg, p.T)
    off, hits = assert_same(p.ix, p.oracle, list(reads.codes), cfg.opts.astuple())
    # sanity statistic (most reads match uniquely)
    assert int(off[-1]) >= 0.9 * reads.n_reads


def test_config2_full_size_in_the_bench_configuration():
    """configs[1] of BASELINE.json at FULL size, launched as bench.py launches it (one batch of
    200,000 reads, default geometry): reads sampled across the whole batch are compared with the
    oracle one by one, and properties that hold at any size are checked on the full output."""
    cfg, p = pair_for("2", sd.CONFIGS["2"].n)
    reads = sd.make_reads(cfg, p.T)
    opts = cfg.opts.astuple()
    b2, nm, off, ln = sd.pack_reads(reads.codes)
    off_g, hits_g, _ = bc.bc_align_batch_host(p.ix, bc.HostReads(b2, None, off, ln), opts)
    st = bc.bc_last_stats(p.ix)
    assert off_g.size == reads.n_reads + 1 and int(off_g[-1]) == hits_g.size
    assert np.all(np.diff(off_g.astype(np.int64)) >= 0)
    assert np.all(hits_g["k"] <= hits_g["l"]) and np.all(hits_g["l"] <= cfg.n) and np.all(hits_g["d"] <= opts[0])
    assert np.all(hits_g["zero"] == 0) and np.all(hits_g["strand"] <= 1)
    # sorted by (strand, k, l) and unique inside every read
    rid = np.repeat(np.arange(reads.n_reads), np.diff(off_g.astype(np.int64)))
    same_read = rid[1:] == rid[:-1]
    s0, s1 = hits_g["strand"][:-1], hits_g["strand"][1:]
    k0, k1 = hits_g["k"][:-1], hits_g["k"][1:]
    l0, l1 = hits_g["l"][:-1], hits_g["l"][1:]
    increasing = (s1 > s0) | ((s1 == s0) & ((k1 > k0) | ((k1 == k0) & (l1 > l0))))
    assert np.all(increasing[same_read])                              # strictly by (strand, k, l): sorted and deduplicated
    assert st["nodes"] > 0 and st["lookups"] == 2 * st["nodes"] and st["lines"] >= st["nodes"]
    # sampled reads, one by one
    rng = np.random.default_rng(2)
    pick = np.sort(rng.choice(reads.n_reads, size=3000, replace=False))
    off_o, hits_o = p.oracle.align(reads.codes[pick], opts)
    for j, r in enumerate(pick.tolist()):
        g = hits_g[int(off_g[r]):int(off_g[r + 1])]
        o = hits_o[int(off_o[j]):int(off_o[j + 1])]
        assert g.tobytes() == o.tobytes(), r
    # located positions of unique hits point back at where the read was drawn from (no indel drift > 3)
    uniq = np.nonzero(np.diff(off_g.astype(np.int64))[pick] == 1)[0][:500]
    rows = np.asarray([hits_g[int(off_g[pick[u]])]["k"] for u in uniq], np.uint32)
    pos = bc.bc_locate(p.ix, rows).cpu().numpy().view(np.uint32).astype(np.int64)
    strand = np.asarray([hits_g[int(off_g[pick[u]])]["strand"] for u in uniq])
    exp = np.where(reads.strand[pick[uniq]] == 0, reads.anchor[pick[uniq]], reads.anchor[pick[uniq]] - cfg.m)
    ok = (np.abs(pos - exp) <= 3) & (strand == reads.strand[pick[uniq]])
    assert ok.mean() > 0.95


@pytest.mark.parametrize("name,n,n_reads", [("2", 2_000_000, 1500), ("3", 3_000_000, 1500), ("4", 3_000_000, 1000),
                                             ("5a", 1_000_000, 300), ("5b", 3_000_000, 1000)])
def test_config_recipes_scaled(name, n, n_reads):
    """Every config's recipe (repeats, error profile, paired ends, N, seed, gaps) at a genome size
    the oracle finishes in seconds; spans many warps' worth of queries and a ragged tail."""
    cfg, p = pair_for(name, n)
    cfg = cfg.scaled(n_reads=n_reads)
    reads = sd.make_reads(cfg, p.T, 0, n_reads)
    assert_same(p.ix, p.oracle, list(reads.codes), cfg.opts.astuple())


def test_ragged_lengths_and_N():
    cfg, p = pair_for("3", 3_000_000)
    reads = sd.make_reads(cfg.scaled(n_reads=600), p.T, 0, 600)
    rng = np.random.default_rng(5)
    rl = []
    for i, r in enumerate(reads.codes):
        m = int(rng.integers(1, reads.m + 1))
        r = r[:m].copy()
        if i % 7 == 0:
            r[rng.integers(0, m)] = 4
        rl.append(r)
    rl.append(np.full(40, 4, np.uint8))                 # all N: no hits
    rl.append(np.asarray([2], np.uint8))                # length 1
    for opts in [(2, 1, 2, 0, 0, 3), (3, 1, 2, 20, 1, 5), (1, 0, 0, 0, 0, 0), (2, 2, 2, 0, 0, 0)]:
        # E = 0 with a length-1 read makes "everything" align; keep those reads longer
        rr = rl if opts[5] > 0 else [r for r in rl if len(r) >= 12]
        assert_same(p.ix, p.oracle, rr, opts)


def test_max_read_length_and_exact():
    cfg, p = pair_for("2", 2_000_000)
    rng = np.random.default_rng(9)
    rl = []
    for _ in range(64):
        s = int(rng.integers(0, p.T.size - 256))
        r = p.T[s:s + 256].copy()
        for q in rng.integers(0, 256, size=2):
            r[q] = (r[q] + 1) & 3
        rl.append(r)
    assert_same(p.ix, p.oracle, rl, (3, 1, 2, 32, 1, 5))
    off, hits = assert_same(p.ix, p.oracle, [p.T[1000:1256].copy()], (0, 0, 0, 0, 0, 5))
    assert int(off[-1]) == 1 and int(hits[0]["d"]) == 0 and int(hits[0]["strand"]) == 0
    assert bc.bc_locate(p.ix, np.asarray([hits[0]["k"]], np.uint32)).cpu().numpy().view(np.uint32)[0] == 1000


def test_empty_batch_and_invalid_arguments():
    cfg, p = pair_for("1", sd.CONFIGS["1"].n)
    off, hits = gpu_align(p.ix, [], (2, 0, 0, 0, 0, 5))
    assert off.tolist() == [0] and hits.size == 0
    reads = [p.T[10:46].copy()]
    with pytest.raises(bc.BcError) as e:
        gpu_align(p.ix, reads, (256, 0, 0, 0, 0, 5))
    assert e.value.status == bc.BC_E_INVAL
    with pytest.raises(bc.BcError) as e:
        gpu_align(p.ix, reads, (2, -1, 0, 0, 0, 5))
    assert e.value.status == bc.BC_E_INVAL
    # a read longer than the declared max_len is an error, not a truncation
    b2, nm, o, ln = sd.pack_ragged(reads)
    h = bc.HostReads(b2, nm, o, ln)
    d = h.to_device()
    d.max_len = 20
    ws = bc.Workspace(p.ix, 1, 20, (2, 0, 0, 0, 0, 5))
    assert bc.bc_align_batch_raw(p.ix, d, (2, 0, 0, 0, 0, 5), ws) == bc.BC_E_INVAL


def test_overflow_is_reported_never_truncated():
    """Repeat-rich genome, loose budget: many hits.  Too-small arena / hits buffer => BC_E_OVERFLOW
    with the needed sizes; growing to them gives the oracle's answer."""
    cfg, p = pair_for("2", 2_000_000)
    reads = list(sd.make_reads(cfg.scaled(n_reads=400), p.T, 0, 400).codes)
    opts = cfg.opts.astuple()
    off_o, hits_o = p.oracle.align(reads, opts)
    b2, nm, o, ln = sd.pack_ragged(reads)
    d = bc.HostReads(b2, nm, o, ln).to_device()
    ws = bc.Workspace(p.ix, len(reads), 51, opts, raw_hits_per_read=1, hits_capacity=8)
    rc = bc.bc_align_batch_raw(p.ix, d, opts, ws)
    assert rc == bc.BC_E_OVERFLOW
    need = ws.needed.cpu().numpy().view(np.uint64)
    assert int(need[1]) >= hits_o.size
    ws2 = bc.Workspace(p.ix, len(reads), 51, opts, raw_hits_per_read=int(need[1]) // len(reads) + 1, hits_capacity=8)
    rc = bc.bc_align_batch_raw(p.ix, d, opts, ws2)
    assert rc == bc.BC_E_OVERFLOW
    need = ws2.needed.cpu().numpy().view(np.uint64)
    assert int(need[0]) == hits_o.size
    res, _ = bc.bc_align_batch(p.ix, d, opts, ws2)     # grows and repeats
    off_g, hits_g = res.to_numpy()
    assert np.array_equal(off_g, off_o) and hits_g.tobytes() == hits_o.tobytes()


def test_locate_equals_suffix_array():
    cfg, p = pair_for("2", 2_000_000)
    SA = p.oracle.index(0)[0]
    rng = np.random.default_rng(3)
    rows = np.concatenate([rng.integers(0, p.T.size + 1, size=20000), [0, p.T.size, p.oracle.index(0)[3]]]).astype(np.uint32)
    pos = bc.bc_locate(p.ix, rows).cpu().numpy().view(np.uint32)
    assert np.array_equal(pos, SA[rows])


def test_result_independent_of_kernel_geometry():
    """Deterministic output whatever the scheduling: different CTA/warp geometry => identical bytes."""
    cfg, p = pair_for("2", 2_000_000)
    reads = list(sd.make_reads(cfg.scaled(n_reads=3000), p.T, 0, 3000).codes)
    opts = cfg.opts.astuple()
    outs = []
    for geo in [(0, 0), (1, 4), (2, 8), (5, 1)]:
        bc.bc_set_geometry(p.ix, *geo)
        off, hits = gpu_align(p.ix, reads, opts)
        outs.append((off.tobytes(), hits.tobytes()))
    bc.bc_set_geometry(p.ix, 0, 0)
    assert all(o == outs[0] for o in outs)
    st = bc.bc_last_stats(p.ix)
    assert st["nodes"] > 0 and st["lookups"] == 2 * st["nodes"]


def test_states_move_between_warps_and_results_do_not():
    """A4: a small batch of heavy trees (config 5a's options: 36 bp, z=4, no seed) leaves most warps without
    queries; busy warps give the bottom of their ring away, pollers take it.  The CSR must be byte-identical
    with the exchange on (blocks did move), off, and to the oracle."""
    cfg, p = pair_for("5a", 1_000_000)
    reads = sd.make_reads(cfg.scaled(n_reads=400), p.T, 0, 400)
    opts = cfg.opts.astuple()
    rl = list(reads.codes)
    outs, steals = [], []
    try:
        for geo, pol in [((0, 0), 0), ((0, 0), 256), ((2, 8), 0), ((5, 2), 0)]:
            bc.bc_set_geometry(p.ix, *geo)
            bc.bc_set_tuning(p.ix, 0, 0, pol)
            off, hits = gpu_align(p.ix, rl, opts)
            outs.append((off.tobytes(), hits.tobytes()))
            steals.append(bc.bc_last_stats(p.ix)["passes_or_steals"])
    finally:
        bc.bc_set_geometry(p.ix, 0, 0)
        bc.bc_set_tuning(p.ix, 0, 0, 0)
    assert all(o == outs[0] for o in outs)
    assert steals[0] > 0 and steals[1] == 0 and steals[2] > 0
    off_o, hits_o = p.oracle.align(reads.codes, opts)
    assert outs[0] == (off_o.tobytes(), hits_o.tobytes())


def test_status_codes_for_small_buffers_and_deep_budgets():
    cfg, p = pair_for("1", sd.CONFIGS["1"].n)
    reads = [p.T[10:46].copy()]
    b2, nm, o, ln = sd.pack_ragged(reads)
    d = bc.HostReads(b2, nm, o, ln).to_device()
    opts = (2, 0, 0, 0, 0, 5)
    ws = bc.Workspace(p.ix, 1, 36, opts)
    ws.ws_bytes = 4096                                   # claim a workspace far smaller than *_bytes said
    assert bc.bc_align_batch_raw(p.ix, d, opts, ws) == bc.BC_E_NOMEM
    # a geometry whose pools do not fit the shared memory is refused, not mis-computed
    bc.bc_set_tuning(p.ix, 0, 16)                            # 16 KB / 8 warps: fewer than 224 entries per warp
    try:
        with pytest.raises(bc.BcError) as e:
            bc.Workspace(p.ix, 1, 36, opts)
        assert e.value.status == bc.BC_E_UNSUPPORTED
    finally:
        bc.bc_set_tuning(p.ix, 0, 0)
    # locate: out-of-range rows give the sentinel, not a wild read
    pos = bc.bc_locate(p.ix, np.asarray([p.T.size + 5], np.uint32)).cpu().numpy().view(np.uint32)
    assert pos[0] == 0xFFFFFFFF
    assert bc.bc_measure_random_sectors(1 << 24, 64) > 1e9


def test_deep_budgets_use_the_generic_query_record():
    """z > 7 or seed_z > 3: thresholds are read from memory instead of registers (bc_ws.cuh); z far beyond the
    read length is legal and means "every substring of that length"."""
    cfg = sd.CONFIGS["1"].scaled(n=3000)
    T = sd.make_genome(cfg)
    p = Pair(T)
    rng = np.random.default_rng(12)
    rl = [T[int(s0):int(s0) + 14].copy() for s0 in rng.integers(0, T.size - 14, size=24)]
    for r in rl[:8]:
        r[int(rng.integers(0, 14))] = (r[3] + 1) & 3
    assert_same(p.ix, p.oracle, rl, (9, 1, 2, 10, 4, 2))
    assert_same(p.ix, p.oracle, rl[:6], (40, 0, 0, 0, 0, 5))
    assert_same(p.ix, p.oracle, rl[:6], (12, 2, 3, 0, 0, 0))


def test_spill_area_exhaustion_is_reported_and_recovered():
    """The per-warp spill area of pending branch states is finite: when it runs full the call says so
    (BC_E_NOMEM, never a truncated result) and the binding repeats it with a larger area."""
    cfg, p = pair_for("5a", 1_000_000)
    reads = sd.make_reads(cfg.scaled(n_reads=2000), p.T, 0, 2000)
    opts = cfg.opts.astuple()
    b2, nm, off, ln = sd.pack_reads(reads.codes)
    d = bc.HostReads(b2, None, off, ln).to_device()
    try:
        bc.bc_set_tuning(p.ix, 1, 0)                         # one block of 32 states per warp
        ws = bc.Workspace(p.ix, 2000, 36, opts, 64)
        assert bc.bc_align_batch_raw(p.ix, d, opts, ws) == bc.BC_E_NOMEM
        res, _ = bc.bc_align_batch(p.ix, d, opts, ws)        # grows the area and repeats
        assert p.ix.spill_blocks > 1
        off_g, hits_g = res.to_numpy()
    finally:
        bc.bc_set_tuning(p.ix, 0, 0)
    off_o, hits_o = p.oracle.align(reads.codes, opts)
    assert np.array_equal(off_g, off_o) and hits_g.tobytes() == hits_o.tobytes()
    st = bc.bc_last_stats(p.ix)
    assert st["cancelled"] > 0 and st["spill_blocks"] > 0    # un-pop and spill both fired on this workload


def test_moderately_deep_budget():
    """z = 8 with a seed on short reads: results still match the oracle."""
    cfg, p = pair_for("1", sd.CONFIGS["1"].n)
    rng = np.random.default_rng(4)
    rl = []
    for _ in range(40):
        s0 = int(rng.integers(0, p.T.size - 20))
        rl.append(p.T[s0:s0 + 16].copy())
    assert_same(p.ix, p.oracle, rl, (8, 0, 0, 12, 1, 5))
    rl24 = [p.T[i * 1000:i * 1000 + 24].copy() for i in range(1, 9)]
    assert_same(p.ix, p.oracle, rl24, (5, 1, 2, 0, 0, 3))


def test_autotune_keeps_parity_as_a_hard_constraint():
    from paper_1505_07855_b200.autotune import autotune_geometry, autotune, GENES
    cfg, p = pair_for("2", 2_000_000)
    reads = sd.make_reads(cfg.scaled(n_reads=4000), p.T, 0, 4000)
    opts = cfg.opts.astuple()
    b2, nm, off, ln = sd.pack_reads(reads.codes)
    d = bc.HostReads(b2, nm, off, ln).to_device()
    best, table = autotune_geometry(p.ix, d, opts, candidates=((0, 0), (2, 8), (4, 6), (6, 4)), repeats=1)
    assert all(r["identical"] for r in table if r["status"] == "ok") and best["geometry"] in [r["geometry"] for r in table]
    off_g, hits_g = gpu_align(p.ix, list(reads.codes), opts)          # runs with the winner left set
    off_o, hits_o = p.oracle.align(reads.codes, opts)
    bc.bc_set_geometry(p.ix, 0, 0)
    assert np.array_equal(off_g, off_o) and hits_g.tobytes() == hits_o.tobytes()
    # the evolutionary search over the run-time genes (build-time genes need the compiler; see profiles/r02_autotune_*)
    runtime = {k: v for k, v in GENES.items() if k != "min_ctas"}
    runtime["min_ctas"] = (GENES["min_ctas"][0],)
    best, table = autotune(p.host, bc.HostReads(b2, nm, off, ln), opts, budget=6, repeats=1, genes=runtime)
    ok = [r for r in table if r["status"] == "ok"]
    assert len(table) == 6 and ok and all(r["identical"] for r in ok) and best["search_ms"] <= table[0]["search_ms"]
