"""Autotuning in the spirit of the paper's genetic improvement (the GI
version owes its speed-up to evolved source edits AND tuned parameters).  The GI framework and the original
source are not available; what is kept is the method: variants of the kernel are generated, each is RUN, its
output must be byte-identical to the reference output (a variant that changes one byte is rejected, however
fast), and the fastest survivor becomes the default.

A variant is a point in the space below.  `min_ctas` is a BUILD-time gene (launch bounds, hence the register
budget ptxas works with): every value is compiled as its own shared library (`_build.build_variant`) and loaded
in turn; the others are run-time genes of the C ABI (`bc_set_geometry`, `bc_set_tuning`).  The search is a small
(1 + lambda) evolution: start from the library defaults, mutate one or two genes of the best individual, keep
improvements; every evaluated point is recorded, so a full grid is just a large budget.

The committed tables (profiles/r02_autotune_*.json) came from `python -m paper_1505_07855_b200.autotune`; the
rule in csrc/bc_align.cu (`choose_geometry`) and the cache policy by index size are their result.
"""
from __future__ import annotations

import hashlib
import json
import random
import sys

import paper_1505_07855_b200 as bc
from . import _build

GENES = {                                   # value 0 = "library default" for the run-time genes
    "min_ctas": (4, 3, 5),                  # BUILD-time: __launch_bounds__(224, min_ctas) of the default flavour
    "ctas": (0, 2, 3, 4, 5, 6),             # CTAs per SM launched
    "warps": (0, 4, 6, 7, 8),               # warps per CTA (8: the 256-thread flavour, 3 CTAs per SM)
    "pool_kb": (0, 128, 144, 160, 176, 192, 208),   # shared memory per SM given to the state pools
    "ld_policy": (0, 1, 2),                 # cache policy of the index loads (bc_set_tuning)
    "layout": (0, 1, 2),                    # device index layout (bc_set_index_layout; needs a re-upload)
}
DEFAULT = {k: v[0] for k, v in GENES.items()}


def _digest(res) -> str:
    off, hits = res.to_numpy()
    return hashlib.sha256(off.tobytes() + hits.tobytes()).hexdigest()


class Evaluator:
    """Runs one variant on one workload: (search-kernel ms, digest of the whole CSR)."""

    def __init__(self, host: "bc.HostIndex", hreads: "bc.HostReads", opts, device="cuda:0", repeats: int = 2, best_plus=None):
        self.arrays = {k: v.copy() for k, v in host.to_arrays().items()}     # survives library switches
        self.hreads, self.opts, self.device, self.repeats, self.best_plus = hreads, opts, device, repeats, best_plus
        self._lib_for, self._ix = None, None

    def _index(self, min_ctas: int, layout: int):
        if self._lib_for != (min_ctas, layout):
            if self._ix is not None:
                self._ix.free()
            so = None if min_ctas == DEFAULT["min_ctas"] else _build.build_variant({"BC_SEARCH_MIN_CTAS": min_ctas})
            bc.use_library(so)
            bc.bc_set_index_layout(layout)
            try:
                self._ix = bc.bc_index_upload(bc.HostIndex.from_arrays(self.arrays), self.device)
            finally:
                bc.bc_set_index_layout(0)
            self._lib_for = (min_ctas, layout)
        return self._ix

    def __call__(self, g: dict):
        ix = self._index(g["min_ctas"], g.get("layout", 0))
        bc.bc_set_geometry(ix, g["ctas"], g["warps"])
        bc.bc_set_tuning(ix, 0, g["pool_kb"], g["ld_policy"])
        d = self.hreads.to_device(self.device)
        times = []
        for _ in range(max(1, self.repeats)):
            if self.best_plus is None:
                res, _ws = bc.bc_align_batch(ix, d, self.opts)
            else:
                res, _ws = bc.bc_align_batch_best(ix, d, self.opts, self.best_plus)
            times.append(bc.bc_last_stats(ix)["search_ns"] / 1e6)
        return min(times), _digest(res)

    def close(self):
        if self._ix is not None:
            self._ix.free()
            self._ix = None
        bc.use_library(None)


def evolve(evaluate, budget: int = 40, seed: int = 0, lam: int = 4, genes: dict = GENES):
    """(1 + lambda) evolution with parity as a hard constraint.  Returns (best_row, table)."""
    rng = random.Random(seed)
    table, seen = [], {}

    def run(g):
        key = tuple(sorted(g.items()))
        if key in seen:
            return seen[key]
        row = {"genes": dict(g), "search_ms": None, "identical": None, "status": "ok"}
        try:
            ms, dig = evaluate(g)
            row["search_ms"], row["digest"] = ms, dig
        except bc.BcError as e:                  # e.g. pools that do not fit this geometry
            row["status"] = str(e)
        table.append(row)
        seen[key] = row
        return row

    ref = run(dict(DEFAULT))
    if ref["status"] != "ok":
        raise RuntimeError("autotune: the default variant did not run: " + ref["status"])
    ref["identical"] = True
    best = ref
    while len(table) < budget:
        kids = []
        for _ in range(lam):
            g = dict(best["genes"])
            for name in rng.sample(sorted(genes), rng.choice((1, 1, 2))):
                g[name] = rng.choice(genes[name])
            kids.append(run(g))
            if len(table) >= budget:
                break
        for row in kids:
            if row["status"] != "ok":
                continue
            row["identical"] = row["digest"] == ref["digest"]
            if row["identical"] and row["search_ms"] < best["search_ms"]:
                best = row
    for row in table:
        row.pop("digest", None)
    return best, table


def autotune(host, hreads, opts, device="cuda:0", budget: int = 40, seed: int = 0, repeats: int = 2, best_plus=None,
             genes: dict = GENES):
    """`genes` may restrict the space, e.g. to the run-time genes (no compiler needed)."""
    ev = Evaluator(host, hreads, opts, device, repeats, best_plus)
    try:
        return evolve(ev, budget, seed, genes=genes)
    finally:
        ev.close()


def autotune_geometry(ix, reads, opts, candidates=((0, 0), (2, 8), (3, 8), (4, 8), (4, 6), (5, 6), (6, 4)), repeats: int = 2):
    """Round-1 entry point, kept: grid over (CTAs per SM, warps per CTA) on an uploaded index; leaves the winner set."""
    table, ref, best = [], None, None
    for geo in candidates:
        row = {"geometry": tuple(geo), "search_ms": None, "identical": None, "status": "ok"}
        try:
            bc.bc_set_geometry(ix, *geo)
            times = []
            for _ in range(max(1, repeats)):
                res, _ws = bc.bc_align_batch(ix, reads, opts)
                times.append(bc.bc_last_stats(ix)["search_ns"] / 1e6)
            dig = _digest(res)
            ref = ref or dig
            row["search_ms"], row["identical"] = min(times), dig == ref
            if row["identical"] and (best is None or row["search_ms"] < best["search_ms"]):
                best = row
        except bc.BcError as e:
            row["status"] = str(e)
        table.append(row)
    if best is None:
        bc.bc_set_geometry(ix, 0, 0)
        raise RuntimeError("autotune: no candidate geometry ran")
    bc.bc_set_geometry(ix, *best["geometry"])
    return best, table


def main(argv=None):
    """python -m paper_1505_07855_b200.autotune CONFIG [READS] [BUDGET] [GENOME_BP]  -> one JSON document on stdout."""
    import numpy as np
    import synthdata as sd
    argv = list(sys.argv[1:] if argv is None else argv)
    name = argv[0] if argv else "2"
    cfg = sd.CONFIGS[name]
    n_reads = int(argv[1]) if len(argv) > 1 else min(cfg.n_reads, 200_000)
    budget = int(argv[2]) if len(argv) > 2 else 40
    if len(argv) > 3:
        cfg = cfg.scaled(n=int(argv[3]))
    genome = sd.make_genome(cfg)
    host = bc.bc_index_build_gpu(genome, 128, 32)
    reads = sd.make_reads(cfg, genome, 0, n_reads)
    b2, nm, off, ln = sd.pack_reads(reads.codes)
    hreads = bc.HostReads(b2, nm if (reads.codes == 4).any() else None, off, ln)
    best, table = autotune(host, hreads, cfg.opts.astuple(), budget=budget)
    ok = [r for r in table if r["status"] == "ok"]
    print(json.dumps({"workload": f"config {name}, genome {cfg.n} bp, {n_reads} reads", "evaluated": len(table),
                      "rejected_for_parity": sum(1 for r in ok if r["identical"] is False),
                      "default_ms": table[0]["search_ms"], "best": best,
                      "table": sorted(ok, key=lambda r: r["search_ms"]) + [r for r in table if r["status"] != "ok"]}))
    return 0


if __name__ == "__main__":
    sys.exit(main())
