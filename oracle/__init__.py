"""ORACLE -- test infrastructure, not product code (see bc_oracle.cpp header).

ctypes loader for oracle/bc_oracle.cpp.  Only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this package.  It imports nothing from
paper_1505_07855_b200 and shares no code with it.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_DIR = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_DIR, "bc_oracle.cpp")
_SO = os.path.join(_DIR, "libbc_oracle.so")

FLAG_PRUNE, FLAG_BAN_ID, FLAG_PLUS_5P_FIRST = 1, 2, 4
DEFAULT_FLAGS = FLAG_PRUNE | FLAG_BAN_ID | FLAG_PLUS_5P_FIRST

HIT_DTYPE = np.dtype([("k", "<u4"), ("l", "<u4"), ("d", "u1"), ("strand", "u1"), ("zero", "<u2")])


def build(force: bool = False) -> str:
    """Compile the oracle with g++ (building the checker is not using it)."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        subprocess.check_call(["g++", "-O2", "-std=c++17", "-shared", "-fPIC", "-pthread", _SRC, "-o", _SO])
    return _SO


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        L.orc_index_build.restype = C.c_void_p
        L.orc_index_build.argtypes = [C.c_void_p, C.c_uint64, C.c_int]
        L.orc_index_build2.restype = C.c_void_p
        L.orc_index_build2.argtypes = [C.c_void_p, C.c_uint64, C.c_int, C.c_int]
        L.orc_index_free.argtypes = [C.c_void_p]
        L.orc_index_get.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_occ.restype = C.c_uint64
        L.orc_occ.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int64]
        L.orc_D.argtypes = [C.c_void_p, C.c_void_p, C.c_int, C.c_void_p]
        L.orc_D_range.argtypes = [C.c_void_p, C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_void_p]
        L.orc_locate.argtypes = [C.c_void_p, C.c_void_p, C.c_uint64, C.c_void_p]
        L.orc_align.restype = C.c_void_p
        L.orc_align.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_uint64, C.c_void_p, C.c_int, C.c_int]
        for f in ("orc_result_total", "orc_result_nodes", "orc_result_lookups"):
            getattr(L, f).restype = C.c_uint64
            getattr(L, f).argtypes = [C.c_void_p]
        L.orc_result_copy.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_result_free.argtypes = [C.c_void_p]
        _lib = L
    return _lib


def _ptr(a):
    return a.ctypes.data_as(C.c_void_p)


class Oracle:
    """Index of one genome (codes 0..3) + the reference search."""

    def __init__(self, genome: np.ndarray, nthreads: int | None = None, sort: str = "auto"):
        """sort: "literal" (one comparison sort of all suffixes), "bucketed" (by the first 12
        bases, then a comparison sort per bucket) or "auto" (literal up to 150 M suffixes)."""
        self.T = np.ascontiguousarray(genome, dtype=np.uint8)
        assert self.T.size == 0 or self.T.max() <= 3
        self.n = int(self.T.size)
        self.nthreads = nthreads or os.cpu_count() or 1
        mode = {"literal": 0, "bucketed": 1, "auto": -1}[sort]
        self._h = lib().orc_index_build2(_ptr(self.T), self.n, self.nthreads, mode)

    def __del__(self):
        if getattr(self, "_h", None):
            lib().orc_index_free(self._h)
            self._h = None

    def index(self, which: int = 0):
        """(SA uint32[n+1], B uint8[n+1] with 4='$', C[5], primary) of the fwd (0) / rev (1) index."""
        SA = np.empty(self.n + 1, np.uint32)
        B = np.empty(self.n + 1, np.uint8)
        Cc = np.empty(5, np.uint64)
        pr = C.c_uint64(0)
        lib().orc_index_get(self._h, which, _ptr(SA), _ptr(B), _ptr(Cc), C.byref(pr))
        return SA, B, Cc, int(pr.value)

    def occ(self, which: int, c: int, j: int) -> int:
        return int(lib().orc_occ(self._h, which, c, j))

    def D(self, Q) -> np.ndarray:
        Q = np.ascontiguousarray(Q, dtype=np.uint8)
        out = np.empty(Q.size, np.int32)
        lib().orc_D(self._h, _ptr(Q), Q.size, _ptr(out))
        return out

    def D_range(self, Q, lo: int, hi: int) -> np.ndarray:
        """Ds: the D loop restricted to Q[lo..hi); entries outside the range are 0."""
        Q = np.ascontiguousarray(Q, dtype=np.uint8)
        out = np.empty(Q.size, np.int32)
        lib().orc_D_range(self._h, _ptr(Q), Q.size, lo, hi, _ptr(out))
        return out

    def locate(self, rows) -> np.ndarray:
        rows = np.ascontiguousarray(rows, dtype=np.uint32)
        out = np.empty(rows.size, np.uint32)
        lib().orc_locate(self._h, _ptr(rows), rows.size, _ptr(out))
        return out

    def align(self, reads, opts, flags: int = DEFAULT_FLAGS, nthreads: int | None = None, stats: dict | None = None):
        """reads: (n_reads, m) uint8 array or list of code arrays; opts: 6-tuple
        (z, max_gap_open, max_gap_ext, seed_len, seed_z, indel_end_skip).
        Returns (hit_offsets uint64[n_reads+1], hits HIT_DTYPE[]): per read R_0 then R_1, each
        sorted by (k,l)."""
        if isinstance(reads, np.ndarray) and reads.ndim == 2:
            nr, m = reads.shape
            flat = np.ascontiguousarray(reads.reshape(-1), dtype=np.uint8)
            off = np.arange(nr, dtype=np.uint64) * np.uint64(m)
            ln = np.full(nr, m, np.uint16)
        else:
            nr = len(reads)
            lens = np.asarray([len(r) for r in reads], dtype=np.int64)
            off = (np.cumsum(lens) - lens).astype(np.uint64)
            ln = lens.astype(np.uint16)
            flat = np.concatenate([np.asarray(r, np.uint8) for r in reads]) if nr else np.zeros(0, np.uint8)
        o = np.asarray(tuple(opts), dtype=np.int32)
        assert o.size == 6
        r = lib().orc_align(self._h, _ptr(flat), _ptr(off), _ptr(ln), nr, _ptr(o), flags, nthreads or self.nthreads)
        try:
            tot = int(lib().orc_result_total(r))
            offs = np.empty(nr + 1, np.uint64)
            hits = np.empty(tot, HIT_DTYPE)
            lib().orc_result_copy(r, _ptr(offs), _ptr(hits))
            if stats is not None:
                stats["nodes"] = int(lib().orc_result_nodes(r))
                stats["lookups"] = int(lib().orc_result_lookups(r))
        finally:
            lib().orc_result_free(r)
        return offs, hits
