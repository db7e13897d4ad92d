"""N>1 host logic on CPU (gloo, world_size 2): read sharding covers the batch exactly once, the
max-over-ranks reduction and the CSR concatenation in rank order.  The per-rank 'aligner' here is
the oracle (tests may call it): the point is the plumbing, which has no GPU in it."""
import os
import socket

import numpy as np
import torch.multiprocessing as mp

import synthdata as sd
from paper_1505_07855_b200 import dist as bdist


def test_shard_range_partitions():
    for n in (0, 1, 7, 200_000, 200_001):
        for w in (1, 2, 3, 8):
            parts = [bdist.shard_range(n, r, w) for r in range(w)]
            assert parts[0][0] == 0 and sum(c for _, c in parts) == n
            for (f0, c0), (f1, _) in zip(parts, parts[1:]):
                assert f0 + c0 == f1
            assert max(c for _, c in parts) - min(c for _, c in parts) <= 1


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, q):
    os.environ.update(RANK=str(rank), WORLD_SIZE=str(world), LOCAL_RANK=str(rank), MASTER_ADDR="127.0.0.1",
                      MASTER_PORT=str(port))
    from oracle import Oracle
    r, w, _ = bdist.init_from_env("gloo")
    assert (r, w) == (rank, world) and bdist.active()
    cfg = sd.CONFIGS["1"].scaled(n=50_000, n_reads=101)
    T = sd.make_genome(cfg)
    first, count = bdist.shard_range(cfg.n_reads, r, w)
    reads = sd.make_reads(cfg, T, first, count)
    off, hits = Oracle(T, nthreads=1).align(reads.codes, cfg.opts.astuple())
    bdist.barrier()
    mx = bdist.max_over_ranks(10.0 + rank)
    g = bdist.gather_csr(off, hits)
    if rank == 0:
        q.put((mx, g[0], g[1]))
    bdist.finish()


def test_two_rank_sharding_matches_single_rank():
    from oracle import Oracle
    ctx = mp.get_context("spawn")
    q = ctx.SimpleQueue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    mx, off, hits = q.get()
    for p in procs:
        p.join(60)
        assert p.exitcode == 0
    assert mx == 11.0
    cfg = sd.CONFIGS["1"].scaled(n=50_000, n_reads=101)
    T = sd.make_genome(cfg)
    off1, hits1 = Oracle(T, nthreads=2).align(sd.make_reads(cfg, T).codes, cfg.opts.astuple())
    assert np.array_equal(off, off1) and hits.tobytes() == hits1.tobytes()


def _bcast_worker(rank, world, port, q):
    os.environ.update(RANK=str(rank), WORLD_SIZE=str(world), LOCAL_RANK=str(rank), MASTER_ADDR="127.0.0.1",
                      MASTER_PORT=str(port))
    import paper_1505_07855_b200 as bc
    bdist.init_from_env("gloo")
    cfg = sd.CONFIGS["2"].scaled(n=30_000)
    host = genome = None
    if rank == 0:                                    # the index is built once, on rank 0 only
        genome = sd.make_genome(cfg)
        host = bc.bc_index_build_host(genome, 128, 32, 2)
    genome = bdist.broadcast_array(genome)
    host = bdist.broadcast_host_index(host)
    a = host.to_arrays()
    q.put((rank, genome.tobytes(), {k: np.asarray(v).tobytes() for k, v in a.items()}))
    bdist.barrier()
    bdist.finish()


def test_index_built_once_and_broadcast():
    """rank 0 builds the index; the other rank receives the genome and every transport array bit for bit."""
    ctx = mp.get_context("spawn")
    q = ctx.SimpleQueue()
    port = _free_port()
    procs = [ctx.Process(target=_bcast_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = dict()
    for _ in range(2):
        r, g, arrs = q.get()
        got[r] = (g, arrs)
    for p in procs:
        p.join(60)
        assert p.exitcode == 0
    assert got[0][0] == got[1][0] and len(got[0][0]) == 30_000
    assert got[0][1].keys() == got[1][1].keys() and len(got[0][1]) == 13
    for k in got[0][1]:
        assert got[0][1][k] == got[1][1][k], k
