#!/usr/bin/env python
"""bench.py -- reads aligned/s of the inexact backward search on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 2] [--impl reference]

One "step" = one pass of the whole hot path (bc_align_batch: D[] bounds, persistent inexact search,
hit emission, per-read sort + dedup -> CSR) over one batch of synthetic reads.  Workload at N=1:
configs[1] of BASELINE.json (16 Mbp repeat-rich genome, 200,000 x 51 bp reads, z=3, 1 gap open,
3 extensions).  N>1: the index is replicated, every rank aligns its own batch of the same recipe
(read indices rank*B .. (rank+1)*B), no data-path collective (weak scaling).
Prints ONE JSON line on rank 0.
"""
from __future__ import annotations

import argparse
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


def workload(name: str):
    cfg = sd.CONFIGS[name]
    desc = {
        "1": "config 1: 1 Mbp uniform genome, 10k x 36 bp, z=2 mismatches only",
        "2": "config 2: 16 Mbp genome (20% repeats), 200k x 51 bp reads, z=3, max_gap_open=1, max_gap_ext=3, E=5",
        "3": "config 3: 100 Mbp repeat-rich genome, 4M x 76 bp (2M pairs), z=4, seed 32/2, go=1, ge=6",
    }.get(name, "config " + name)
    return cfg, desc


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


# ------------------------------------------------------------------------------------------------
# reference arm / cpu baseline: the oracle as it stands, on the host cores
# ------------------------------------------------------------------------------------------------
def calibrate_sample(cfg, genome, target_s: float, cap: int):
    """Pick how many reads the oracle can do in ~target_s seconds (probe with 256 reads)."""
    from oracle import Oracle
    cores = os.cpu_count() or 1
    probe = min(256, cap)
    orc = Oracle(genome, nthreads=cores)
    reads = sd.make_reads(cfg, genome, 0, probe)
    t0 = time.time()
    orc.align(reads.codes, cfg.opts.astuple(), nthreads=cores)
    dt = max(time.time() - t0, 1e-3)
    return orc, int(max(probe, min(cap, probe * target_s / dt)))


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    cfg, desc = workload(args.config)
    genome = sd.make_genome(cfg)
    from oracle import Oracle  # noqa: F401  (the reference arm IS the oracle)
    cores = os.cpu_count() or 1
    per_step_s = max(2.0, min(20.0, 150.0 / max(1, args.steps + args.warmup)))
    orc, sample = calibrate_sample(cfg, genome, per_step_s, cfg.n_reads)
    opts = cfg.opts.astuple()
    times = []
    for s in range(args.warmup + args.steps):
        reads = sd.make_reads(cfg, genome, 0, sample)
        t0 = time.time()
        orc.align(reads.codes, opts, nthreads=cores)
        dt = time.time() - t0
        if s >= args.warmup:
            times.append(dt)
    tot = sum(times)
    value = sample * len(times) / tot
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * tot / len(times), "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "u32", "data": "synthetic",
        "config": {"workload": desc, "reads_per_step": sample,
                   "note": "the CPU oracle as it stands (naive suffix sort + recursive search), bounded sample per step"},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle",
                         "sample": f"first {sample} reads of the workload per step"},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }
    print(json.dumps(line), flush=True)
    return 0


# ------------------------------------------------------------------------------------------------
# our arm
# ------------------------------------------------------------------------------------------------
def run_ours(args):
    import torch
    import paper_1505_07855_b200 as bc
    from paper_1505_07855_b200 import dist as bdist

    rank, world, local = bdist.init_from_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback")
    dev = torch.device("cuda", local % torch.cuda.device_count())   # (modulo only matters for the one-GPU plumbing test)
    torch.cuda.set_device(dev)

    cfg, desc = workload(args.config)
    if args.genome_bp:
        cfg = cfg.scaled(n=args.genome_bp)
        desc += f" [genome scaled to {args.genome_bp} bp]"
    B = cfg.n_reads if args.reads is None else args.reads
    # genome + host index, optionally cached on disk (config 5: "index built once on the host and cached; not timed")
    gpath = ipath = None
    if args.index_cache:
        os.makedirs(args.index_cache, exist_ok=True)
        key = f"seed{cfg.seed:x}_n{cfg.n}"
        gpath, ipath = os.path.join(args.index_cache, key + "_genome.npy"), os.path.join(args.index_cache, key + "_index.npz")
    if gpath and os.path.exists(gpath):
        genome = np.load(gpath)
    else:
        genome = sd.make_genome(cfg)
        if gpath and rank == 0:
            np.save(gpath, genome)
    first, count = bdist.shard_range(B * world, rank, world)      # weak scaling: B reads per rank
    reads = sd.make_reads(cfg, genome, first, count)
    opts = cfg.opts.astuple()
    index_build = {"where": "disk cache", "seconds": 0.0}
    if ipath and os.path.exists(ipath):
        host = bc.HostIndex.load(ipath)
    else:
        t_b = time.time()
        host = bc.bc_index_build_gpu(genome, 128, 32, dev) if args.gpu_index_build else bc.bc_index_build_host(genome, 128, 32)
        index_build = {"where": "gpu (bc_index_build_gpu)" if args.gpu_index_build else f"host, {os.cpu_count()} threads",
                       "seconds": time.time() - t_b, "note": "untimed step before the path; both builders give identical arrays"}
        if ipath and rank == 0:
            host.save(ipath)
    ix = bc.bc_index_upload(host, dev)
    if args.ctas or args.warps:
        bc.bc_set_geometry(ix, args.ctas, args.warps)
    b2, nm, off, ln = sd.pack_reads(reads.codes)
    if not (reads.codes == 4).any():
        nm = None
    hreads = bc.HostReads(b2, nm, off, ln)
    dreads = hreads.to_device(dev)
    stream = torch.cuda.current_stream()
    best = args.best is not None
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

    for _ in range(args.warmup):
        flush.fill_(1)
        one_step()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    sampler = ClockSampler(dev.index) if rank == 0 else None
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
    t_ms = sum(a.elapsed_time(b) for a, b in ev)
    clocks = sampler.stop() if sampler else None
    t_ms = bdist.max_over_ranks(t_ms, dev)
    n_hits = int(ws.needed.cpu().numpy().view(np.uint64)[0])

    # ---- e2e: host buffers in, host CSR out, copies inside the timed region ----
    e2e_times = []
    for s in range(args.warmup + args.steps):
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
        if s >= args.warmup:
            e2e_times.append(dt)
    e2e_s = bdist.max_over_ranks(sum(e2e_times), dev)
    h2d = hreads.nbytes
    d2h = int(off_h.nbytes + hits_h.nbytes + 16)

    if rank != 0:
        bdist.finish()
        return 0

    value = count * world * args.steps / (t_ms * 1e-3)
    peak, peak_src = measured_peaks()
    k_s = float(np.mean(search_ns)) * 1e-9
    line_bytes = stats["lines"] * 32          # algorithmic bytes: one 32-byte index sector per rank query (+1 when the pair straddles)
    achieved = line_bytes / k_s / 1e9 if k_s > 0 else 0.0
    traffic = None
    tp = os.path.join(ROOT, "profiles", "traffic.json")
    if os.path.exists(tp):
        try:
            traffic = json.load(open(tp)).get(args.config)
        except Exception:
            traffic = None
    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": t_ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "u32", "data": "synthetic",
        "config": {"workload": desc, "reads_per_step_per_gpu": count, "read_len": cfg.m, "genome_bp": cfg.n,
                   "opts": dict(zip(("z", "max_gap_open", "max_gap_ext", "seed_len", "seed_z", "indel_end_skip"), opts)),
                   "index_bytes": bc.bc_index_device_bytes(host), "l2": "flushed between steps (256 MiB fill, untimed)",
                   "parallelism": f"dp{world} (index replicated, reads sharded, no collective)",
                   "hits_per_step": n_hits, "index_build": index_build,
                   "mode": ("best-stratum +%d (bc_align_batch_best, %d passes)" % (args.best, stats.get("passes", 0))) if best else "exhaustive (bc_align_batch)"},
        "e2e": {"value": count * world * args.steps / e2e_s, "unit": UNIT, "h2d_bytes_per_step": h2d,
                "d2h_bytes_per_step": d2h},
        "gpu_launches": (args.steps * (stats.get("passes", 0) * (KERNELS_PER_STEP + 9) + 5)) if best
                        else KERNELS_PER_STEP * args.steps,   # best mode: per pass + gather, classify, 2 scans, commit; + init, scan, write
        "clocks": clocks,
        "roofline": {"bound": "hbm", "kernel": "bc_search_kernel", "achieved": achieved, "peak": peak, "unit": "GB/s",
                     "frac": achieved / peak, "traffic": traffic, "peak_source": peak_src,
                     "kernel_ms": k_s * 1e3, "kernel_share_of_step": k_s * 1e3 / (t_ms / args.steps),
                     "nodes_per_launch": stats["nodes"], "occ_lookups_per_s": stats["lookups"] / k_s if k_s else 0.0,
                     "lines_per_launch": stats["lines"],
                     "branch_nodes": stats["branch_nodes"], "chain_nodes": stats["chain_nodes"],
                     "lanes_per_branch_step": stats["branch_nodes"] / max(1, stats["branch_steps"]),
                     "lanes_per_chain_step": stats["chain_nodes"] / max(1, stats["chain_steps"]),
                     "pool_max": stats["pool_max"], "cancelled": stats["cancelled"], "spill_blocks": stats["spill_blocks"], "geometry": {"ctas_per_sm": stats["geometry"] >> 32,
                                                                 "warps_per_cta": (stats["geometry"] >> 16) & 0xFFFF,
                                                                 "pool_entries_per_warp": stats["geometry"] & 0xFFFF},
                     "sectors_per_s": stats["lines"] / k_s if k_s else 0.0,
                     "note": "algorithmic bytes = 32 B x index sectors the search must read (1 or 2 per node, "
                             "counted by the kernel) / search-kernel time from CUDA events on its stream; peak = "
                             "measured streaming HBM bandwidth.  This workload's 16 MB index is L2-resident, so HBM "
                             "does not bind it: see random_sector (measured) and DESIGN.md 'Rooflines'"},
    }
    # ---- measured random-sector rates (the metric's own denominator), outside the timed region ----
    if not args.no_probe:
        idx_bytes = 2 * (cfg.n // 64 + 1) * 32
        rs_res = bc.bc_measure_random_sectors(idx_bytes, 512, dev)
        rs_hbm = bc.bc_measure_random_sectors(8 << 30, 256, dev)
        sect_s = stats["lines"] / k_s if k_s else 0.0
        out["random_sector"] = {"unit": "G sectors/s (32 B)", "search_kernel": sect_s / 1e9,
                                "peak_index_sized_table": rs_res / 1e9, "peak_8GiB_table_hbm": rs_hbm / 1e9,
                                "frac_of_index_sized_peak": sect_s / rs_res, "frac_of_hbm_random_peak": sect_s / rs_hbm,
                                "how": "bc_measure_random_sectors: 64 warps/SM, 4 independent 256-bit loads in flight per thread"}
    # ---- optional: K batches streamed end to end, H2D of batch b+1 overlapped with the search of batch b ----
    if args.batches > 1:
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
        outs, total_hits = [], 0
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
        torch.cuda.synchronize()
        dts = time.perf_counter() - t0
        out["stream"] = {"batches": args.batches, "reads": args.batches * count, "seconds": dts,
                         "value": args.batches * count / dts, "unit": UNIT, "hits": total_hits,
                         "h2d_bytes": sum(h.nbytes for h in hb),
                         "note": "pinned host batches -> device on a second stream, overlapped with the previous batch's "
                                 "search; results copied back per batch; wall clock over all batches"}
    # ---- a property that holds at any size: unique hits locate to where the generator drew the read ----
    one_hit = np.nonzero(np.diff(off_h.astype(np.int64)) == 1)[0]
    if one_hit.size:
        pick = one_hit[:: max(1, one_hit.size // 20000)]
        hsel = hits_h[off_h[pick].astype(np.int64)]
        posu = bc.bc_locate(ix, np.ascontiguousarray(hsel["k"])).cpu().numpy().view(np.uint32).astype(np.int64)
        exp = np.where(reads.strand[pick] == 0, reads.anchor[pick], reads.anchor[pick] - cfg.m)
        okk = (np.abs(posu - exp) <= 3) & (hsel["strand"] == reads.strand[pick])
        out["anchor_check"] = {"reads_with_one_hit": int(one_hit.size), "checked": int(pick.size),
                               "located_at_generator_anchor_frac": float(okk.mean())}
    # ---- optional: the step after the path -- pairing the ends, timed end to end ----
    pair_res = None
    if args.pair and cfg.paired:
        lo, hi = int(cfg.frag_mu - 4 * cfg.frag_sd), int(cfg.frag_mu + 4 * cfg.frag_sd)
        resd = bc.AlignResult(ws.hit_offsets, ws.hits, n_hits, 0)
        one_step()                                                # the device result of the last mode run
        pair_res = bc.bc_pair_batch(ix, resd, dreads, lo, hi, 32)   # sizes the buffers
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        for _ in range(args.steps):
            pair_res = bc.bc_pair_batch(ix, resd, dreads, lo, hi, 32)
        torch.cuda.synchronize()
        dtp = (time.perf_counter() - t0) / args.steps
        out["pairing"] = {"pairs_of_reads_per_s": (count // 2) / dtp, "ms_per_batch": dtp * 1e3, "window": [lo, hi],
                          "max_occ": 32, **pair_res[2],
                          "fragments_paired_frac": float((np.diff(pair_res[0].astype(np.int64)) > 0).mean()),
                          "note": "bc_pair_batch on the device CSR of the step above; wall clock incl. buffer allocation "
                                  "and the copy of the pairs to the host"}
    # ---- cpu baseline: the oracle on a bounded sample of the same batch, + parity on that sample ----
    if not args.no_cpu:
        orc, sample = calibrate_sample(cfg, genome, 12.0, count)
        sreads = sd.make_reads(cfg, genome, first, sample)
        cores = os.cpu_count() or 1
        t0 = time.time()
        off_o, hits_o = orc.align(sreads.codes, opts, nthreads=cores)
        dt = time.time() - t0
        out["cpu_baseline"] = {"value": sample / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
                               "sample": f"first {sample} reads of the same batch, {dt:.1f} s"}
        if best:                                                  # the contract: exhaustive result filtered to d <= min(d_min + plus, z)
            keep = np.zeros(hits_o.size, bool)
            cnts = np.zeros(sample, np.uint64)
            for r in range(sample):
                a, b = int(off_o[r]), int(off_o[r + 1])
                if b > a:
                    dd = hits_o["d"][a:b].astype(np.int64)
                    keep[a:b] = dd <= min(int(dd.min()) + args.best, opts[0])
                    cnts[r] = int(keep[a:b].sum())
            off_o, hits_o = np.concatenate([[0], np.cumsum(cnts)]).astype(np.uint64), hits_o[keep]
        same = bool(np.array_equal(off_h[: sample + 1], off_o) and
                    hits_h[: int(off_o[-1])].tobytes() == hits_o.tobytes())
        out["parity"] = {"reads_checked": sample, "identical_to_oracle": same}
        if pair_res is not None:                                  # brute-force pairing of the oracle's own located hits
            from oracle.pairing import pair_reads
            ns = sample & ~1
            SA = orc.index(0)[0]
            po_o, pairs_o, _ = pair_reads(SA, off_o[: ns + 1], hits_o, ln[:ns], lo, hi, 32)
            po_g, pairs_g = pair_res[0], pair_res[1]
            out["pairing"]["parity"] = {"pairs_of_reads_checked": ns // 2, "identical_to_oracle": bool(
                np.array_equal(po_g[: ns // 2 + 1], po_o) and pairs_g[: int(po_o[-1])].tobytes() == pairs_o.tobytes())}
    print(json.dumps(out), flush=True)
    bdist.finish()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="2", choices=sorted(sd.CONFIGS))
    ap.add_argument("--reads", type=int, default=None, help="reads per step per GPU (default: the config's)")
    ap.add_argument("--genome-bp", type=int, default=None,
                    help="same recipe on a smaller genome (exploration only; the default is the config's own size)")
    ap.add_argument("--index-cache", default=None, metavar="DIR", help="cache genome and host index here (untimed)")
    ap.add_argument("--gpu-index-build", action="store_true", help="build the index with bc_index_build_gpu instead of on the host")
    ap.add_argument("--ctas", type=int, default=0)
    ap.add_argument("--warps", type=int, default=0)
    ap.add_argument("--best", type=int, default=None, metavar="PLUS",
                    help="best-stratum mode: keep hits with d <= min(d_min + PLUS, z) (bc_align_batch_best)")
    ap.add_argument("--batches", type=int, default=1, help="also stream this many batches end to end (config 5: 1M-read batches)")
    ap.add_argument("--pair", action="store_true", help="also time bc_pair_batch on the result (paired configs)")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg (profiling runs)")
    ap.add_argument("--no-probe", action="store_true", help="skip the random-sector microbenchmark")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "ours" and not args.no_cpu:
        pass                                                     # the driver's contract asks W >= 3; honoured by default
    return run_reference(args) if args.impl == "reference" else run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
