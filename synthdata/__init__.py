"""Seeded synthetic genomes and reads.

This module only *draws inputs*.  It holds none of the aligner's arithmetic (no BWT, no rank,
no search) and is the one module that both the oracle-side tests and the CUDA-side code may
import.  All randomness is a counter-based hash, splitmix64(seed, stream tag, index), so every
value is a pure function of (config, index) and generation is order-free.

Stand-in statement: the paper measures on hg19 + 1000-Genomes ERR001270 (36 bp PE) and GCAT
gcat_set_037 (100 bp PE).  None of these is in the container; the generators
below produce inputs with the same shapes (lengths, pairing, error profile, repeat content).
"""
from __future__ import annotations

import dataclasses
import numpy as np

U64 = np.uint64
_M64 = (1 << 64) - 1

# stream tags
T_BASE, T_CONS, T_FAM, T_GAP, T_SUB, T_SUBB, T_NRUN, T_NBASE = 1, 2, 3, 4, 5, 6, 7, 8
T_RPOS, T_RSTRAND, T_RSUB, T_RSUBB, T_RIND, T_RINDK, T_RINDB, T_RN = 20, 21, 22, 23, 24, 25, 26, 27
T_FRAG1, T_FRAG2, T_FLEN, T_FDIV = 30, 31, 32, 33


def splitmix64(x: np.ndarray) -> np.ndarray:
    """splitmix64 finaliser on a uint64 array (wrap-around arithmetic)."""
    with np.errstate(over="ignore"):
        z = (x + U64(0x9E3779B97F4A7C15)).astype(U64)
        z = (z ^ (z >> U64(30))) * U64(0xBF58476D1CE4E5B9)
        z = (z ^ (z >> U64(27))) * U64(0x94D049BB133111EB)
        return z ^ (z >> U64(31))


def hash_u64(seed: int, tag: int, idx) -> np.ndarray:
    """hash of (seed, tag, idx[...]) -> uint64 array, same shape as idx."""
    idx = np.asarray(idx, dtype=U64)
    key = splitmix64(np.asarray([(seed * 0x100 + tag) & _M64], dtype=U64))[0]
    with np.errstate(over="ignore"):
        return splitmix64(idx ^ key)


def u01(seed: int, tag: int, idx) -> np.ndarray:
    """uniform double in [0,1) from the hash."""
    return (hash_u64(seed, tag, idx) >> U64(11)).astype(np.float64) * (1.0 / (1 << 53))


@dataclasses.dataclass(frozen=True)
class Opts:
    """Search options = bc_opts of include/barracuda_b200.h (same field order)."""
    z: int
    max_gap_open: int
    max_gap_ext: int
    seed_len: int
    seed_z: int
    indel_end_skip: int

    def astuple(self):
        return (self.z, self.max_gap_open, self.max_gap_ext, self.seed_len, self.seed_z,
                self.indel_end_skip)


@dataclasses.dataclass(frozen=True)
class Config:
    """One workload of BASELINE.json `configs` (numbers 1..5; 5 is split into 5a/5b)."""
    name: str
    seed: int
    n: int                       # genome length
    n_fam: int = 0               # repeat families (0 = none)
    fam_len: tuple = (300, 300)  # family consensus length range (uniform, inclusive)
    fam_div: tuple = (0.10, 0.10)  # per-family divergence range (uniform)
    rep_frac: float = 0.0        # fraction of the genome covered by repeat copies
    nrun_frac: float = 0.0       # fraction of the genome inside (re-randomised) N runs
    n_reads: int = 0             # number of reads (ends); paired => even
    m: int = 36
    paired: bool = False
    frag_mu: float = 0.0
    frag_sd: float = 0.0
    p0: float = 0.01             # substitution rate at the 5' end
    p1: float = 0.01             # ... at the 3' end
    indel: float = 0.0           # indel event rate per base (length uniform 1..3)
    read_n: float = 0.0          # per-base probability of an N in a read
    opts: Opts = Opts(2, 0, 0, 0, 0, 5)

    def scaled(self, n: int | None = None, n_reads: int | None = None) -> "Config":
        """Same recipe at a smaller size (used by parity tests; DESIGN.md says which)."""
        return dataclasses.replace(self, n=n or self.n, n_reads=n_reads or self.n_reads)


_R45 = dict(n_fam=1000, fam_len=(100, 6000), fam_div=(0.05, 0.20), rep_frac=0.45)
CONFIGS = {
    "1": Config("1", 0xBC0001, 1_000_000, n_reads=10_000, m=36, p0=0.01, p1=0.01,
                opts=Opts(2, 0, 0, 0, 0, 5)),
    "2": Config("2", 0xBC0002, 16_000_000, n_fam=50, rep_frac=0.20, n_reads=200_000, m=51,
                p0=0.005, p1=0.03, indel=0.0002, opts=Opts(3, 1, 3, 0, 0, 5)),
    "3": Config("3", 0xBC0003, 100_000_000, n_fam=50, rep_frac=0.20, nrun_frac=0.001,
                n_reads=4_000_000, m=76, paired=True, frag_mu=300, frag_sd=30, p0=0.005, p1=0.03,
                indel=0.0002, read_n=0.001, opts=Opts(4, 1, 6, 32, 2, 5)),
    "4": Config("4", 0xBC0004, 1_000_000_000, n_reads=8_000_000, m=100, paired=True, frag_mu=400,
                frag_sd=40, p0=0.005, p1=0.04, indel=0.0005, opts=Opts(5, 1, 10, 32, 2, 5), **_R45),
    # config 5: BASELINE.json gives no gap limits; SURVEY 8d proposes config 4's (1, 10).
    "5a": Config("5a", 0xBC0005, 3_100_000_000, n_reads=20_000_000, m=36, paired=True, frag_mu=350,
                 frag_sd=35, p0=0.005, p1=0.04, indel=0.0005, opts=Opts(4, 1, 10, 0, 0, 5), **_R45),
    "5b": Config("5b", 0xBC0005, 3_100_000_000, n_reads=20_000_000, m=108, paired=True,
                 frag_mu=350, frag_sd=35, p0=0.005, p1=0.04, indel=0.0005,
                 opts=Opts(6, 1, 10, 32, 2, 5), **_R45),
}


# ----------------------------------------------------------------------------------------------
# genome
# ----------------------------------------------------------------------------------------------
def make_genome(cfg: Config, chunk: int = 1 << 24) -> np.ndarray:
    """Genome as uint8 codes A,C,G,T = 0..3 (no N: N runs are re-randomised)."""
    n, seed = cfg.n, cfg.seed
    g = np.empty(n, dtype=np.uint8)
    for s in range(0, n, chunk):
        e = min(n, s + chunk)
        g[s:e] = (hash_u64(seed, T_BASE, np.arange(s, e, dtype=U64)) >> U64(62)).astype(np.uint8)
    if cfg.n_fam > 0 and cfg.rep_frac > 0:
        F = cfg.n_fam
        fid = np.arange(F, dtype=U64)
        lo, hi = cfg.fam_len
        flen = (lo + (hash_u64(seed, T_FLEN, fid) % U64(hi - lo + 1)).astype(np.int64))
        fdiv = cfg.fam_div[0] + (cfg.fam_div[1] - cfg.fam_div[0]) * u01(seed, T_FDIV, fid)
        foff = np.concatenate([[0], np.cumsum(flen)])
        cons = (hash_u64(seed, T_CONS, np.arange(foff[-1], dtype=U64)) >> U64(62)).astype(np.uint8)
        mean_len = float(flen.mean())
        mean_gap = mean_len * (1.0 - cfg.rep_frac) / cfg.rep_frac
        k_max = int(n / (mean_len + mean_gap) * 1.2) + 16
        cid = np.arange(k_max, dtype=U64)
        fam = (hash_u64(seed, T_FAM, cid) % U64(F)).astype(np.int64)
        gap = np.floor(-np.log1p(-u01(seed, T_GAP, cid)) * mean_gap).astype(np.int64)
        clen = flen[fam]
        start = np.cumsum(gap + np.concatenate([[0], clen[:-1]]))
        ok = start + clen <= n
        fam, clen, start = fam[ok], clen[ok], start[ok]
        # process copies in groups to bound temporaries
        grp = max(1, int(chunk // max(1, int(mean_len))))
        for a in range(0, len(fam), grp):
            f, L, st = fam[a:a + grp], clen[a:a + grp], start[a:a + grp]
            tot = int(L.sum())
            if tot == 0:
                continue
            rep_start = np.repeat(st, L)
            within = np.arange(tot, dtype=np.int64) - np.repeat(np.cumsum(L) - L, L)
            pos = rep_start + within
            base = cons[np.repeat(foff[f], L) + within]
            pu = pos.astype(U64)
            sub = u01(seed, T_SUB, pu) < np.repeat(fdiv[f], L)
            delta = (1 + (hash_u64(seed, T_SUBB, pu) % U64(3))).astype(np.uint8)
            g[pos] = np.where(sub, (base + delta) & 3, base)
    if cfg.nrun_frac > 0:
        mean_run = 275.0
        k = int(n * cfg.nrun_frac / mean_run)
        rid = np.arange(k, dtype=U64)
        rlen = 50 + (hash_u64(seed, T_NRUN, rid) % U64(451)).astype(np.int64)
        rst = (u01(seed, T_NRUN, rid + U64(1 << 40)) * (n - 500)).astype(np.int64)
        for s0, L in zip(rst.tolist(), rlen.tolist()):
            p = np.arange(s0, s0 + L, dtype=U64)
            g[s0:s0 + L] = (hash_u64(seed, T_NBASE, p) >> U64(62)).astype(np.uint8)
    return g


# ----------------------------------------------------------------------------------------------
# reads
# ----------------------------------------------------------------------------------------------
@dataclasses.dataclass
class Reads:
    codes: np.ndarray      # (n_reads, m) uint8, 0..3 and 4 = N   (all reads of a batch share m here)
    anchor: np.ndarray     # (n_reads,) int64: genome coordinate of the read's 5' end (see strand)
    strand: np.ndarray     # (n_reads,) uint8: 0 = forward copy of genome[anchor:...], 1 = revcomp of genome[...:anchor]

    @property
    def n_reads(self):
        return self.codes.shape[0]

    @property
    def m(self):
        return self.codes.shape[1]


_SLACK = 12


def make_reads(cfg: Config, genome: np.ndarray, first: int = 0, count: int | None = None) -> Reads:
    """Reads `first .. first+count` of the config's read set (pure function of the index)."""
    n, m, seed = cfg.n, cfg.m, cfg.seed
    count = cfg.n_reads - first if count is None else count
    rid = np.arange(first, first + count, dtype=U64)
    span = m + _SLACK
    if not cfg.paired:
        strand = (hash_u64(seed, T_RSTRAND, rid) & U64(1)).astype(np.uint8)
        lo = (u01(seed, T_RPOS, rid) * (n - span)).astype(np.int64)       # leftmost genome base used
        anchor = np.where(strand == 0, lo, lo + span)
    else:
        pid = rid >> U64(1)
        end2 = (rid & U64(1)).astype(np.uint8)
        u1 = np.maximum(u01(seed, T_FRAG1, pid), 1e-300)
        u2 = u01(seed, T_FRAG2, pid)
        gauss = np.sqrt(-2.0 * np.log(u1)) * np.cos(2.0 * np.pi * u2)
        flen = np.maximum(np.rint(cfg.frag_mu + cfg.frag_sd * gauss).astype(np.int64), span)
        fstart = (u01(seed, T_RPOS, pid) * (n - flen)).astype(np.int64)
        fstrand = (hash_u64(seed, T_RSTRAND, pid) & U64(1)).astype(np.uint8)
        # end 1 = first m bases of the fragment, end 2 = revcomp of its last m bases
        strand = fstrand ^ end2
        anchor = np.where(strand == 0, fstart, fstart + flen)
    # gather source bases, 5'->3' of the read
    j = np.arange(span, dtype=np.int64)[None, :]
    src = np.where(strand[:, None] == 0, anchor[:, None] + j, anchor[:, None] - 1 - j)
    frag = genome[src]
    frag = np.where(strand[:, None] == 0, frag, 3 - frag).astype(np.uint8)
    # substitutions, probability linear along the read
    cell = rid[:, None] * U64(512) + np.arange(span, dtype=U64)[None, :]
    pt = cfg.p0 + (cfg.p1 - cfg.p0) * (np.arange(span) / max(1, m - 1))
    sub = u01(seed, T_RSUB, cell) < pt[None, :]
    delta = (1 + (hash_u64(seed, T_RSUBB, cell) % U64(3))).astype(np.uint8)
    frag = np.where(sub, (frag + delta) & 3, frag).astype(np.uint8)
    out = frag[:, :m].copy()
    if cfg.indel > 0:
        ev = u01(seed, T_RIND, cell[:, :m]) < cfg.indel
        rows = np.nonzero(ev.any(axis=1))[0]
        for r in rows.tolist():
            src_row = frag[r].tolist()
            res, t = [], 0
            while len(res) < m and t < span:
                if t < m and ev[r, t]:
                    ev[r, t] = False                     # one event per source position
                    c = int(cell[r, t])
                    kind = int(hash_u64(seed, T_RINDK, [c])[0])
                    L = 1 + (kind >> 8) % 3
                    if kind & 1:                         # insertion of L hashed bases before base t
                        ins = hash_u64(seed, T_RINDB, np.arange(c * 4, c * 4 + L, dtype=U64)) >> U64(62)
                        res.extend(int(x) for x in ins)
                    else:                                # deletion: skip L source bases
                        t += L
                    continue
                res.append(src_row[t])
                t += 1
            res = (res + [0] * m)[:m]
            out[r] = np.asarray(res, dtype=np.uint8)
    if cfg.read_n > 0:
        isn = u01(seed, T_RN, cell[:, :m]) < cfg.read_n
        out = np.where(isn, 4, out).astype(np.uint8)
    return Reads(out, anchor, strand)


def _pack_stream(flat: np.ndarray):
    """flat codes (0..3, 4 = N) -> (bases2 uint32[], nmask uint32[]) of the bc_reads transport layout."""
    total = flat.size
    isn = flat == 4
    two = np.where(isn, 0, flat).astype(np.uint32)
    pad = (-total) % 16
    two = np.concatenate([two, np.zeros(pad, dtype=np.uint32)]).reshape(-1, 16)
    shifts = (2 * np.arange(16, dtype=np.uint32))[None, :]
    bases2 = np.bitwise_or.reduce(two << shifts, axis=1).astype(np.uint32)
    padn = (-total) % 32
    nb = np.concatenate([isn.astype(np.uint32), np.zeros(padn, dtype=np.uint32)]).reshape(-1, 32)
    nmask = np.bitwise_or.reduce(nb << np.arange(32, dtype=np.uint32)[None, :], axis=1).astype(np.uint32)
    return bases2, nmask


def pack_reads(codes: np.ndarray):
    """Pack (n_reads, m) codes into the bc_reads transport layout.

    Returns (bases2 uint32[], nmask uint32[], off uint64[n_reads], len uint16[n_reads]).
    Base i of the stream sits at bits 2*(i%16) of bases2[i//16]; N -> code 0 and its nmask bit
    (bit i%32 of nmask[i//32]) set.  Reads are concatenated without padding.
    """
    nr, m = codes.shape
    bases2, nmask = _pack_stream(codes.reshape(-1))
    off = (np.arange(nr, dtype=np.uint64) * np.uint64(m))
    ln = np.full(nr, m, dtype=np.uint16)
    return bases2, nmask, off, ln


def pack_ragged(reads: list):
    """Same layout for reads of different lengths (list of uint8 code arrays)."""
    lens = np.asarray([len(r) for r in reads], dtype=np.int64)
    off = np.concatenate([[0], np.cumsum(lens)[:-1]]).astype(np.uint64) if len(reads) else np.zeros(0, np.uint64)
    flat = np.concatenate([np.asarray(r, dtype=np.uint8) for r in reads]) if len(reads) else np.zeros(0, np.uint8)
    b2, nm = _pack_stream(flat) if flat.size else (np.zeros(0, np.uint32), np.zeros(0, np.uint32))
    return b2, nm, off, lens.astype(np.uint16)


_ALPHA = "ACGTN"


def encode(s: str) -> np.ndarray:
    return np.asarray([_ALPHA.index(c) for c in s.upper()], dtype=np.uint8)


def decode(a) -> str:
    return "".join(_ALPHA[int(c)] for c in a)
