#!/usr/bin/env python
"""bench.py -- reads aligned/s of the inexact backward search on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 4] [--impl reference]

One "step" = one pass of the whole hot path (bc_align_batch: query records with D[] bounds, persistent
inexact search, hit emission, per-read sort + dedup -> CSR) over one batch of synthetic reads.
Workload at N=1 (the headline): BASELINE.json configs[3] -- the largest configuration on which the oracle
can stand beside the kernel inside one run, and an index (1.5 GB) far beyond the 126 MB L2, the regime the
metric names ("Occ lookups/s vs HBM random-sector roofline"): 1 Gbp repeat-rich genome, one batch of
1,000,000 x 100 bp reads of its 8 M, z=5, seed 32/2, 1 gap open, 10 extensions; index built by
bc_index_build_gpu (untimed).  The same JSON line carries sub-records (`sub`) for config 2 (16 Mbp, index
L2-resident) and config 5b at its full 3.1 Gbp (no oracle beside that one unless --sub-oracle: its index alone
takes 7 minutes of host time; the full-size oracle comparison is profiles/r02_bench_config5b_full.json).  N>1: the index is built once on rank 0
and broadcast, every rank aligns its own batch of the same recipe (read indices rank*B .. (rank+1)*B), no
data-path collective (weak scaling).  Prints ONE JSON line on rank 0.
"""
from __future__ import annotations

import argparse
import hashlib
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import synthdata as sd  # noqa: E402

METRIC = "reads aligned/sec on 1 B200; Occ lookups/s vs HBM random-sector roofline"
UNIT = "reads/s"
KERNELS_PER_STEP = 12      # prepare, search, 2 x (3 scan kernels), scatter, sort_small, sort_big, write_hits
L2_BYTES = 126 << 20
DEFAULT_BATCH = {"4": 1_000_000, "5a": 100_000, "5b": 1_000_000}   # reads per step when the config's set is streamed

DESC = {
    "1": "config 1: 1 Mbp uniform genome, 10k x 36 bp, z=2 mismatches only",
    "2": "config 2: 16 Mbp genome (20% repeats), 200k x 51 bp reads, z=3, max_gap_open=1, max_gap_ext=3, E=5",
    "3": "config 3: 100 Mbp repeat-rich genome, 4M x 76 bp (2M pairs), z=4, seed 32/2, go=1, ge=6",
    "4": "config 4: 1 Gbp genome (45% repeats, 1000 families), one batch of 1M x 100 bp of the 8M paired-end reads, "
         "z=5, seed 32/2, max_gap_open=1, max_gap_ext=10, E=5",
    "5a": "config 5 (36 bp half): 3.1 Gbp genome, 2x36 bp paired-end reads in batches, z=4, no seed, go=1, ge=10",
    "5b": "config 5 (108 bp half): 3.1 Gbp genome, 2x108 bp paired-end reads in batches of 1M, z=6, seed 32/2, go=1, ge=10",
}


class ClockSampler:
    """nvidia-smi clocks/throttle reasons sampled every 200 ms while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.rows, self.proc, self.th = [], None, None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            if len(r) < 6:
                continue
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
            except ValueError:
                continue
            for nm, v in zip(names, r[2:6]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def spread_sample(n_total: int, n_pick: int) -> np.ndarray:
    """n_pick distinct read indices spread over [0, n_total) by a multiplicative hash (never "the first N")."""
    n_pick = min(n_pick, n_total)
    idx = (np.arange(4 * n_pick + 16, dtype=np.uint64) * np.uint64(2654435761)) % np.uint64(max(1, n_total))
    _, first = np.unique(idx, return_index=True)
    return np.sort(idx[np.sort(first)][:n_pick].astype(np.int64))


def workload(name: str, args):
    cfg = sd.CONFIGS[name]
    desc = DESC.get(name, "config " + name)
    if args.genome_bp:
        cfg = cfg.scaled(n=args.genome_bp)
        desc += f" [genome scaled to {args.genome_bp} bp]"
    B = args.reads if args.reads is not None else DEFAULT_BATCH.get(name, cfg.n_reads)
    return cfg, desc, B


# ------------------------------------------------------------------------------------------------
# reference arm / cpu baseline: the oracle as it stands, on the host cores
# ------------------------------------------------------------------------------------------------
def oracle_rate_probe(orc, codes: np.ndarray, opts, cap: int, target_s: float):
    """How many reads the oracle does in ~target_s seconds (probe with 256 reads spread over the batch)."""
    cores = os.cpu_count() or 1
    pick = spread_sample(codes.shape[0], min(256, cap))
    t0 = time.time()
    orc.align(codes[pick], opts, nthreads=cores)
    dt = max(time.time() - t0, 1e-3)
    return int(max(pick.size, min(cap, pick.size * target_s / dt)))


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    from oracle import Oracle                          # the reference arm IS the oracle
    cfg, desc, B = workload(args.config, args)
    genome = sd.make_genome(cfg)
    cores = os.cpu_count() or 1
    t0 = time.time()
    orc = Oracle(genome, nthreads=cores)
    t_build = time.time() - t0
    opts = cfg.opts.astuple()
    reads = sd.make_reads(cfg, genome, 0, B)
    per_step_s = max(2.0, min(20.0, 150.0 / max(1, args.steps + args.warmup)))
    sample = oracle_rate_probe(orc, reads.codes, opts, B, per_step_s)
    pick = spread_sample(B, sample)
    codes = reads.codes[pick]
    times = []
    for s in range(args.warmup + args.steps):
        t0 = time.time()
        orc.align(codes, opts, nthreads=cores)
        dt = time.time() - t0
        if s >= args.warmup:
            times.append(dt)
    tot = sum(times)
    value = pick.size * len(times) / tot
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * tot / len(times), "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "u32", "data": "synthetic",
        "config": {"workload": desc, "reads_per_step": int(pick.size), "genome_bp": cfg.n,
                   "index_build_s": t_build,
                   "note": "the CPU oracle as it stands (naive suffix sort, bucketed beyond 150 M suffixes as SURVEY C8 "
                           "allows; recursive search); each step = a bounded sample of the workload's batch, spread over it"},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle",
                         "sample": f"{pick.size} reads spread over the workload's batch of {B}, per step"},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }
    print(json.dumps(line), flush=True)
    return 0


# ------------------------------------------------------------------------------------------------
# our arm
# ------------------------------------------------------------------------------------------------
def csr_digest(off: np.ndarray, hits: np.ndarray) -> str:
    return hashlib.sha256(off.tobytes() + hits.tobytes()).hexdigest()


def traffic_for(name: str, reads: int):
    """DRAM bytes per launch of the search kernel from the committed ncu capture of this workload (HEAD kernel)."""
    tp = os.path.join(ROOT, "profiles", "traffic.json")
    try:
        t = json.load(open(tp)).get(name)
        if t and int(t.get("reads", -1)) == reads:
            return t
    except Exception:
        pass
    return None


def measure(name: str, args, dev, rank: int, world: int, steps: int, warmup: int, main: bool):
    """Build the workload `name` on this rank, time it, check it; returns (record dict, context)."""
    import torch
    import paper_1505_07855_b200 as bc
    from paper_1505_07855_b200 import dist as bdist

    cfg, desc, B = workload(name, args)
    # ---- genome + index (untimed): built once on rank 0, shipped to the other ranks ----
    gpath = ipath = None
    if args.index_cache:
        os.makedirs(args.index_cache, exist_ok=True)
        key = f"seed{cfg.seed:x}_n{cfg.n}"
        gpath, ipath = os.path.join(args.index_cache, key + "_genome.npy"), os.path.join(args.index_cache, key + "_index.npz")
    index_build = {"where": "disk cache", "seconds": 0.0}
    genome = host = None
    if rank == 0:
        if gpath and os.path.exists(gpath):
            genome = np.load(gpath)
        else:
            genome = sd.make_genome(cfg)
            if gpath:
                np.save(gpath, genome)
        if ipath and os.path.exists(ipath):
            host = bc.HostIndex.load(ipath)
        else:
            t_b = time.time()
            host = bc.bc_index_build_host(genome, 128, 32) if args.host_index_build else bc.bc_index_build_gpu(genome, 128, 32, dev)
            index_build = {"where": f"host, {os.cpu_count()} threads" if args.host_index_build else "gpu (bc_index_build_gpu)",
                           "seconds": time.time() - t_b,
                           "note": "untimed step before the path; both builders give identical arrays"}
            if ipath:
                host.save(ipath)
            torch.cuda.empty_cache()
    if world > 1:
        genome = bdist.broadcast_array(genome, dev)
        host = bdist.broadcast_host_index(host, dev)
        index_build["shipped"] = "built on rank 0, transport arrays broadcast to the other ranks"
    ix = bc.bc_index_upload(host, dev)
    if args.ctas or args.warps:
        bc.bc_set_geometry(ix, args.ctas, args.warps)
    if args.pool_kb or args.ld_policy:
        bc.bc_set_tuning(ix, 0, args.pool_kb, args.ld_policy)
    first, count = bdist.shard_range(B * world, rank, world)      # weak scaling: B reads per rank
    reads = sd.make_reads(cfg, genome, first, count)
    opts = cfg.opts.astuple()
    b2, nm, off, ln = sd.pack_reads(reads.codes)
    if not (reads.codes == 4).any():
        nm = None
    hreads = bc.HostReads(b2, nm, off, ln)
    dreads = hreads.to_device(dev)
    stream = torch.cuda.current_stream()
    best = args.best is not None and main
    if best:                                                     # best-stratum mode, not the BASELINE metric's mode
        res, ws = bc.bc_align_batch_best(ix, dreads, opts, args.best)
    else:
        res, ws = bc.bc_align_batch(ix, dreads, opts)            # sizes the caller-owned buffers (grows once if needed)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)  # > 126 MB L2

    def one_step():
        rc = (bc.bc_align_batch_best_raw(ix, dreads, opts, args.best, ws, stream) if best
              else bc.bc_align_batch_raw(ix, dreads, opts, ws, stream))
        if rc != bc.BC_OK:
            raise bc.BcError(rc, "bc_align_batch")

    for _ in range(warmup):
        flush.fill_(1)
        one_step()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    sampler = ClockSampler(dev.index) if (rank == 0 and main) else None
    bdist.barrier(); torch.cuda.synchronize()
    search_ns, stats = [], None
    for a, b in ev:
        flush.fill_(1)                                            # L2 flush between timed steps (untimed)
        a.record(stream)
        one_step()
        b.record(stream)
        stats = bc.bc_last_stats(ix)
        search_ns.append(stats["search_ns"])
    torch.cuda.synchronize(); bdist.barrier()
    step_ms = [a.elapsed_time(b) for a, b in ev]
    clocks = sampler.stop() if sampler else None
    t_ms = bdist.max_over_ranks(sum(step_ms), dev)
    n_hits = int(ws.needed.cpu().numpy().view(np.uint64)[0])

    # ---- e2e: host buffers in, host CSR out, copies inside the timed region ----
    e2e_times = []
    off_h = hits_h = None
    for s in range((warmup + steps) if main else 2):
        flush.fill_(1)
        torch.cuda.synchronize(); bdist.barrier()
        t0 = time.perf_counter()
        if best:
            r2, ws = bc.bc_align_batch_best(ix, hreads.to_device(dev), opts, args.best, ws)
            off_h, hits_h = r2.to_numpy()
        else:
            off_h, hits_h, ws = bc.bc_align_batch_host(ix, hreads, opts, ws)
        torch.cuda.synchronize()
        dt = time.perf_counter() - t0
        if s >= (warmup if main else 1):
            e2e_times.append(dt)
    e2e_s = bdist.max_over_ranks(sum(e2e_times), dev)
    h2d = hreads.nbytes
    d2h = int(off_h.nbytes + hits_h.nbytes + 16)
    ctx = dict(cfg=cfg, genome=genome, host=host, ix=ix, reads=reads, hreads=hreads, dreads=dreads, opts=opts, ws=ws,
               off_h=off_h, hits_h=hits_h, first=first, count=count, one_step=one_step, ln=ln, n_hits=n_hits, best=best)
    if rank != 0:
        return None, ctx

    peak, peak_src = measured_peaks()
    k_s = float(np.mean(search_ns)) * 1e-9
    alg_bytes = stats["lines"] * 32           # algorithmic bytes: one 32-byte index block per rank query (+1 when the pair straddles two)
    achieved = alg_bytes / k_s / 1e9 if k_s > 0 else 0.0
    index_bytes = bc.bc_index_device_bytes(host)
    hbm_regime = index_bytes > 2 * L2_BYTES
    tr = traffic_for(name, count) if not best else None
    roof = {"bound": "hbm" if hbm_regime else "l2", "kernel": "bc_search_kernel", "achieved": achieved, "peak": peak, "unit": "GB/s",
            "frac": achieved / peak, "traffic": tr["dram_bytes"] if tr else None,
            "traffic_over_algorithmic": (tr["dram_bytes"] / alg_bytes) if tr else None,
            "traffic_source": tr["source"] if tr else None, "peak_source": peak_src,
            "algorithmic_bytes_per_launch": alg_bytes,
            "kernel_ms": k_s * 1e3, "kernel_ms_best": min(search_ns) * 1e-6, "kernel_share_of_step": k_s * 1e3 / (sum(step_ms) / steps),
            "nodes_per_launch": stats["nodes"], "nodes_per_s": stats["nodes"] / k_s if k_s else 0.0,
            "occ_lookups_per_s": stats["lookups"] / k_s if k_s else 0.0, "sectors_per_launch": stats["lines"],
            "sectors_per_s": stats["lines"] / k_s if k_s else 0.0,
            "branch_nodes": stats["branch_nodes"], "run_nodes": stats["chain_nodes"],
            "lanes_per_branch_step": stats["branch_nodes"] / max(1, stats["branch_steps"]),
            "lanes_per_run_step": stats["chain_nodes"] / max(1, stats["chain_steps"]),
            "pool_max": stats["pool_max"], "cancelled": stats["cancelled"], "spill_blocks": stats["spill_blocks"],
            "spill_max": stats["spill_max"],
            "geometry": {"ctas_per_sm": stats["geometry"] >> 32, "warps_per_cta": (stats["geometry"] >> 16) & 0xFFFF,
                         "pool_entries_per_warp": stats["geometry"] & 0xFFFF},
            "note": ("algorithmic bytes = 32 B x index blocks the search must read (1 or 2 per node, counted by the kernel) / "
                     "search-kernel time from CUDA events on its stream; peak = measured streaming HBM bandwidth.  ") +
                    ("The index is far beyond L2: rank queries go to HBM.  With default cache policies every missing 32-byte "
                     "block costs a whole 128-byte line; the kernel's loads carry the 64-byte L2 prefetch-size hint, which halves "
                     "that (profiles/r02_random_access_ncu.md).  What binds is the RATE of random DRAM accesses, not their bytes: "
                     "see dram_accesses and random_access_probe." if hbm_regime else
                     "This workload's index is L2-resident (DRAM traffic ~0): HBM does not bind it, instruction issue and L2 "
                     "latency do; frac is reported against the HBM peak only for comparability.")}
    if tr:
        acc = tr["dram_bytes"] / 64.0
        roof["dram_accesses"] = {"access_bytes": 64, "per_launch": acc, "per_s": acc / k_s,
                                 "dram_bytes_per_s": tr["dram_bytes"] / k_s, "frac_of_hbm_peak_at_the_pins": tr["dram_bytes"] / k_s / 1e9 / peak}
    rec = {
        "value": count * world * steps / (t_ms * 1e-3), "unit": UNIT, "ms_per_step": t_ms / steps,
        "ms_per_step_best": min(step_ms), "ms_per_step_median": float(np.median(step_ms)),
        "config": {"workload": desc, "reads_per_step_per_gpu": count, "read_len": cfg.m, "genome_bp": cfg.n,
                   "opts": dict(zip(("z", "max_gap_open", "max_gap_ext", "seed_len", "seed_z", "indel_end_skip"), opts)),
                   "index_bytes": index_bytes, "l2": "flushed between steps (256 MiB fill, untimed)",
                   "parallelism": f"dp{world} (index replicated, reads sharded, no collective)",
                   "hits_per_step": n_hits, "index_build": index_build,
                   "mode": ("best-stratum +%d (bc_align_batch_best, budgets 0..%d in one launch)" % (args.best, max(0, stats.get("passes_or_steals", 1) - 1))) if best else "exhaustive (bc_align_batch)"},
        "e2e": {"value": count * world * len(e2e_times) / e2e_s, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h},
        "gpu_launches": KERNELS_PER_STEP * steps,         # both modes: one launch of the hot path per step
        "clocks": clocks, "roofline": roof,
    }
    ctx["stats"] = stats
    ctx["k_s"] = k_s
    return rec, ctx


def checks(rec: dict, ctx: dict, args, dev, with_oracle: bool, sample_target: int):
    """Parity and properties on rank 0 (outside the timed region): oracle on a spread sample, the same CSR under a
    second kernel geometry (SHA-256 over all reads), anchors of uniquely-hit reads."""
    import torch
    import paper_1505_07855_b200 as bc
    cfg, ix, reads, opts, ws = ctx["cfg"], ctx["ix"], ctx["reads"], ctx["opts"], ctx["ws"]
    off_h, hits_h, count, best = ctx["off_h"], ctx["hits_h"], ctx["count"], ctx["best"]
    # ---- a property that holds at any size: unique hits locate to where the generator drew the read ----
    one_hit = np.nonzero(np.diff(off_h.astype(np.int64)) == 1)[0]
    if one_hit.size:
        pick = one_hit[:: max(1, one_hit.size // 20000)]
        hsel = hits_h[off_h[pick].astype(np.int64)]
        posu = bc.bc_locate(ix, np.ascontiguousarray(hsel["k"])).cpu().numpy().view(np.uint32).astype(np.int64)
        exp = np.where(reads.strand[pick] == 0, reads.anchor[pick], reads.anchor[pick] - cfg.m)
        okk = (np.abs(posu - exp) <= 3) & (hsel["strand"] == reads.strand[pick])
        rec["anchor_check"] = {"reads_with_one_hit": int(one_hit.size), "checked": int(pick.size),
                               "located_at_generator_anchor_frac": float(okk.mean())}
    parity = {}
    # ---- the whole CSR must not depend on the kernel geometry (SURVEY 8d "Timing") ----
    if not args.no_geometry_check and not best:
        d0 = csr_digest(off_h, hits_h)
        bc.bc_set_geometry(ix, 2, 8)
        try:
            off2, hits2, ws2 = bc.bc_align_batch_host(ix, ctx["hreads"], opts)
            d1 = csr_digest(off2, hits2)
            del ws2
        finally:
            bc.bc_set_geometry(ix, args.ctas, args.warps)
        parity.update({"csr_sha256": d0, "geometry_hash_equal": d0 == d1,
                       "geometries": "library default vs (2 CTAs/SM, 8 warps), all %d reads of the batch" % count})
        torch.cuda.empty_cache()
    # ---- cpu baseline: the oracle on a bounded sample spread over the same batch, + parity on that sample ----
    if with_oracle:
        from oracle import Oracle
        cores = os.cpu_count() or 1
        t0 = time.time()
        orc = Oracle(ctx["genome"], nthreads=cores)
        t_build = time.time() - t0
        n = oracle_rate_probe(orc, reads.codes, opts, count, args.oracle_seconds)
        if sample_target:                                         # >= 50 k reads when that stays within ~30 s (always with --full-sample)
            n = max(n, sample_target if args.full_sample else min(sample_target, int(n * 30.0 / args.oracle_seconds)))
        n = min(n, count)
        pick = spread_sample(count, n)
        t0 = time.time()
        off_o, hits_o = orc.align(reads.codes[pick], opts, nthreads=cores)
        dt = time.time() - t0
        rec["cpu_baseline"] = {"value": pick.size / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
                               "sample": f"{pick.size} reads spread over the same batch of {count} (multiplicative hash), {dt:.1f} s; "
                                         f"oracle index built in {t_build:.0f} s (untimed)"}
        if best:                                                  # the contract: exhaustive result filtered to d <= min(d_min + plus, z)
            keep = np.zeros(hits_o.size, bool)
            cnts = np.zeros(pick.size, np.uint64)
            for r in range(pick.size):
                a, b = int(off_o[r]), int(off_o[r + 1])
                if b > a:
                    dd = hits_o["d"][a:b].astype(np.int64)
                    keep[a:b] = dd <= min(int(dd.min()) + args.best, opts[0])
                    cnts[r] = int(keep[a:b].sum())
            off_o, hits_o = np.concatenate([[0], np.cumsum(cnts)]).astype(np.uint64), hits_o[keep]
        lo, hi = off_h[pick].astype(np.int64), off_h[pick + 1].astype(np.int64)
        same = bool(np.array_equal(hi - lo, np.diff(off_o.astype(np.int64))))
        if same:
            sel = np.concatenate([np.arange(a, b) for a, b in zip(lo, hi)]) if pick.size else np.zeros(0, np.int64)
            same = hits_h[sel].tobytes() == hits_o.tobytes()
        parity.update({"reads_checked": int(pick.size), "identical_to_oracle": same,
                       "sample": "spread over the batch by a multiplicative hash of the read index"})
        ctx["oracle"], ctx["oracle_pick"], ctx["off_o"], ctx["hits_o"] = orc, pick, off_o, hits_o
    if parity:
        rec["parity"] = parity


def run_ours(args):
    import torch
    import paper_1505_07855_b200 as bc
    from paper_1505_07855_b200 import dist as bdist

    rank, world, local = bdist.init_from_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback")
    dev = torch.device("cuda", local % torch.cuda.device_count())   # (modulo only matters for the one-GPU plumbing test)
    torch.cuda.set_device(dev)

    rec, ctx = measure(args.config, args, dev, rank, world, args.steps, args.warmup, True)
    if rank != 0:
        bdist.finish()
        return 0
    out = {"metric": METRIC, "value": rec["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
           "ms_per_step": rec["ms_per_step"], "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
           "dtype": "u32", "data": "synthetic"}
    out.update({k: v for k, v in rec.items() if k not in ("value", "unit", "ms_per_step")})
    cfg, ix, stats, k_s = ctx["cfg"], ctx["ix"], ctx["stats"], ctx["k_s"]

    # ---- measured random-access rates (the metric's own denominator), outside the timed region ----
    if not args.no_probe:
        idx_bytes = int(out["config"]["index_bytes"])
        rs_res = bc.bc_measure_random_sectors(min(idx_bytes, 8 << 30), 512, dev, ld_policy=1)
        rs_hbm = bc.bc_measure_random_sectors(8 << 30, 256, dev, ld_policy=1)
        rs_hbm0 = bc.bc_measure_random_sectors(8 << 30, 256, dev, ld_policy=0)
        sect_s = stats["lines"] / k_s if k_s else 0.0
        probe = {
            "unit": "G loads/s (one 32-byte block each)", "search_kernel_blocks": sect_s / 1e9,
            "probe_index_sized_table": rs_res / 1e9, "probe_8GiB_table_hbm": rs_hbm / 1e9,
            "probe_8GiB_table_hbm_default_cache_policy": rs_hbm0 / 1e9,
            "how": "bc_measure_random_sectors2: 64 warps/SM, 4 independent 256-bit loads in flight per thread, uniformly random "
                   "32-byte blocks, the search kernel's load policy (no L1 allocation, 64-byte L2 prefetch size).  ncu on the "
                   "8 GiB table: 1.99 DRAM sectors per load with that policy, 3.96 with the default one, the SAME loads/s "
                   "(profiles/r02_random_access_ncu.md): on B200 random HBM access is bound by the access RATE (~44 G/s), not "
                   "by bytes.  The kernel's block rate exceeds the probe's because part of its blocks are L1/L2 hits (top of "
                   "the search trees) and both ends of a narrow interval share an access."}
        da = out["roofline"].get("dram_accesses")
        if da:
            probe["search_kernel_dram_accesses"] = da["per_s"] / 1e9
            probe["frac_of_random_access_rate"] = da["per_s"] / rs_hbm
        out["random_access_probe"] = probe
    # ---- optional: K batches streamed end to end, H2D of batch b+1 overlapped with the search of batch b ----
    if args.batches > 1:
        genome, first, count, opts, ws, best = ctx["genome"], ctx["first"], ctx["count"], ctx["opts"], ctx["ws"], ctx["best"]
        copy_stream = torch.cuda.Stream(device=dev)
        hb = []
        for b in range(args.batches):                             # host side, untimed: generate and pin every batch
            rb = sd.make_reads(cfg, genome, first + b * count, count)
            pb = sd.pack_reads(rb.codes)
            hb.append(bc.HostReads(pb[0], pb[1] if (rb.codes == 4).any() else None, pb[2], pb[3]))
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        with torch.cuda.stream(copy_stream):
            nxt = hb[0].to_device(dev)
        total_hits = 0
        sha = hashlib.sha256()
        for b in range(args.batches):
            copy_stream.synchronize()                             # batch b is on the device
            cur = nxt
            if b + 1 < args.batches:
                with torch.cuda.stream(copy_stream):              # next batch's H2D runs under this batch's kernels
                    nxt = hb[b + 1].to_device(dev)
            if best:
                rb_, ws = bc.bc_align_batch_best(ix, cur, opts, args.best, ws)
            else:
                rb_, ws = bc.bc_align_batch(ix, cur, opts, ws)
            o_, h_ = rb_.to_numpy()                               # CSR back to the host (the call has synchronised)
            total_hits += int(h_.size)
            sha.update(o_.tobytes()); sha.update(h_.tobytes())
        torch.cuda.synchronize()
        dts = time.perf_counter() - t0
        ctx["ws"] = ws
        out["stream"] = {"batches": args.batches, "reads": args.batches * count, "seconds": dts,
                         "value": args.batches * count / dts, "unit": UNIT, "hits": total_hits,
                         "h2d_bytes": sum(h.nbytes for h in hb), "csr_sha256_all_batches": sha.hexdigest(),
                         "note": "pinned host batches -> device on a second stream, overlapped with the previous batch's "
                                 "search; results copied back per batch; wall clock over all batches"}
    # ---- optional: the step after the path -- pairing the ends, timed end to end ----
    pair_res = None
    if args.pair and cfg.paired:
        lo, hi = int(cfg.frag_mu - 4 * cfg.frag_sd), int(cfg.frag_mu + 4 * cfg.frag_sd)
        ws, count = ctx["ws"], ctx["count"]
        ctx["one_step"]()                                         # the device result of the last mode run
        resd = bc.AlignResult(ws.hit_offsets, ws.hits, ctx["n_hits"], 0)
        pair_res = bc.bc_pair_batch(ix, resd, ctx["dreads"], lo, hi, 32)   # sizes the buffers
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        for _ in range(args.steps):
            pair_res = bc.bc_pair_batch(ix, resd, ctx["dreads"], lo, hi, 32)
        torch.cuda.synchronize()
        dtp = (time.perf_counter() - t0) / args.steps
        out["pairing"] = {"pairs_of_reads_per_s": (count // 2) / dtp, "ms_per_batch": dtp * 1e3, "window": [lo, hi],
                          "max_occ": 32, **pair_res[2],
                          "fragments_paired_frac": float((np.diff(pair_res[0].astype(np.int64)) > 0).mean()),
                          "note": "bc_pair_batch on the device CSR of the step above; wall clock incl. buffer allocation "
                                  "and the copy of the pairs to the host"}
    checks(out, ctx, args, dev, with_oracle=not args.no_cpu and world == 1, sample_target=50_000)
    if pair_res is not None and "oracle" in ctx and not ctx["best"]:
        # brute-force pairing of the oracle's own located hits needs whole pairs: the first reads of the batch
        from oracle.pairing import pair_reads
        ns = min(2000, ctx["count"]) & ~1
        off_o, hits_o = ctx["oracle"].align(ctx["reads"].codes[:ns], ctx["opts"])
        SA = ctx["oracle"].index(0)[0]
        po_o, pairs_o, _ = pair_reads(SA, off_o, hits_o, ctx["ln"][:ns], lo, hi, 32)
        out["pairing"]["parity"] = {"pairs_of_reads_checked": ns // 2, "identical_to_oracle": bool(
            np.array_equal(pair_res[0][: ns // 2 + 1], po_o) and pair_res[1][: int(po_o[-1])].tobytes() == pairs_o.tobytes())}
    # ---- sub-records: the other regimes, same checks, fewer steps; never the headline ----
    subs = [s for s in (args.sub.split(",") if args.sub else []) if s and s != args.config]
    if subs and world == 1:
        out["sub"] = {}
        for k in list(ctx):                                       # free the headline workload's device memory first
            ctx[k] = None
        del ix
        torch.cuda.empty_cache()
        sub_args = argparse.Namespace(**vars(args))
        sub_args.reads = sub_args.genome_bp = None
        sub_args.best = None
        sub_args.batches, sub_args.pair = 1, False
        for name in subs:
            c2 = {}
            try:                                                  # a sub-record must never cost the headline its line
                r2, c2 = measure(name, sub_args, dev, 0, 1, max(3, min(args.steps, 5)), 3, False)
                small = sd.CONFIGS[name].n <= 200_000_000         # the oracle's index builds in seconds to a minute
                checks(r2, c2, sub_args, dev, with_oracle=(not args.no_cpu) and (small or args.sub_oracle), sample_target=50_000)
                out["sub"]["config " + name] = r2
            except Exception as e:                                # noqa: BLE001
                out["sub"]["config " + name] = {"error": f"{type(e).__name__}: {e}"}
            for k in list(c2):
                c2[k] = None
            del c2
            torch.cuda.empty_cache()
    print(json.dumps(out), flush=True)
    bdist.finish()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=8)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="4", choices=sorted(sd.CONFIGS))
    ap.add_argument("--sub", default="2,5b", help="comma-separated configs measured as sub-records of the same line (N=1 only)")
    ap.add_argument("--sub-oracle", action="store_true", help="run the oracle beside the large sub-records too (3.1 Gbp: ~10 min)")
    ap.add_argument("--reads", type=int, default=None, help="reads per step per GPU (default: the config's batch)")
    ap.add_argument("--genome-bp", type=int, default=None,
                    help="same recipe on a smaller genome (exploration only; the default is the config's own size)")
    ap.add_argument("--index-cache", default=None, metavar="DIR", help="cache genome and host index here (untimed)")
    ap.add_argument("--host-index-build", action="store_true", help="build the index on the host instead of bc_index_build_gpu")
    ap.add_argument("--gpu-index-build", action="store_true", help="(default; kept for older command lines)")
    ap.add_argument("--ctas", type=int, default=0)
    ap.add_argument("--warps", type=int, default=0)
    ap.add_argument("--pool-kb", type=int, default=0)
    ap.add_argument("--ld-policy", type=int, default=0)
    ap.add_argument("--best", type=int, default=None, metavar="PLUS",
                    help="best-stratum mode: keep hits with d <= min(d_min + PLUS, z) (bc_align_batch_best)")
    ap.add_argument("--batches", type=int, default=1, help="also stream this many batches end to end (config 5: 1M-read batches)")
    ap.add_argument("--pair", action="store_true", help="also time bc_pair_batch on the result (paired configs)")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline / oracle parity leg (profiling runs)")
    ap.add_argument("--no-probe", action="store_true", help="skip the random-access microbenchmark")
    ap.add_argument("--no-geometry-check", action="store_true", help="skip the second-geometry CSR hash")
    ap.add_argument("--oracle-seconds", type=float, default=12.0, help="CPU seconds the cpu_baseline sample aims at")
    ap.add_argument("--full-sample", action="store_true",
                    help="oracle parity on at least 50,000 reads even when that takes longer than --oracle-seconds")
    args = ap.parse_args()
    return run_reference(args) if args.impl == "reference" else run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
