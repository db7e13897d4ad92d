"""Thin Python binding of the C-ABI library of include/barracuda_b200.h (same names).

Argument marshalling only: every step of the hot path (D[] bounds, inexact search, hit emission,
sort + dedup, locate) runs in the CUDA kernels of csrc/.  PyTorch provides device memory and
streams, nothing else.  There is no CPU fallback: without the compiled library (and, for the
compute calls, a CUDA device) everything here raises.

Paper passages behind each call are cited in include/barracuda_b200.h; the readings of what the
paper leaves open are in DESIGN.md.
"""
from __future__ import annotations

import ctypes as C
import dataclasses
import os

import numpy as np

from . import _build

BC_OK, BC_E_INVAL, BC_E_NOMEM, BC_E_CUDA, BC_E_OVERFLOW, BC_E_UNSUPPORTED = 0, -1, -2, -3, -4, -5
BC_MAX_READ_LEN = 256

HIT_DTYPE = np.dtype([("k", "<u4"), ("l", "<u4"), ("d", "u1"), ("strand", "u1"), ("zero", "<u2")])


class bc_bwt_host(C.Structure):
    _fields_ = [("n", C.c_uint64), ("primary", C.c_uint64), ("bwt2", C.c_void_p), ("occ_interval", C.c_uint32),
                ("occ", C.c_void_p), ("C", C.c_uint64 * 5)]


class bc_index_host(C.Structure):
    _fields_ = [("fwd", bc_bwt_host), ("rev", bc_bwt_host), ("sa_interval", C.c_uint32), ("sa", C.c_void_p)]


class bc_opts(C.Structure):
    _fields_ = [(f, C.c_int32) for f in ("z", "max_gap_open", "max_gap_ext", "seed_len", "seed_z", "indel_end_skip")]


class bc_reads(C.Structure):
    _fields_ = [("bases2", C.c_void_p), ("nmask", C.c_void_p), ("off", C.c_void_p), ("len", C.c_void_p),
                ("n_reads", C.c_uint32), ("max_len", C.c_uint32)]


class bc_result(C.Structure):
    _fields_ = [("hit_offsets", C.c_void_p), ("hits", C.c_void_p), ("hits_capacity", C.c_uint64),
                ("n_hits_needed", C.c_void_p)]


class bc_pair_opts(C.Structure):
    _fields_ = [("min_frag", C.c_uint32), ("max_frag", C.c_uint32), ("max_occ", C.c_uint32)]


class bc_pair_result(C.Structure):
    _fields_ = [("pair_offsets", C.c_void_p), ("pairs", C.c_void_p), ("pairs_capacity", C.c_uint64),
                ("n_needed", C.c_void_p)]


PAIR_DTYPE = np.dtype([("pos1", "<u4"), ("pos2", "<u4"), ("frag", "<u4"), ("d1", "u1"), ("d2", "u1"), ("strand1", "u1"),
                       ("zero", "u1")])


class BcError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        super().__init__(f"{where}: {strerror(status)} ({status})")


_lib = None
_lib_path = None


def use_library(path: str | None):
    """Load a build-time variant of the library (see _build.build_variant) instead of the default one; None =
    back to the default.  Handles created by one library must not be passed to another: call this first."""
    global _lib, _lib_path
    _lib, _lib_path = None, path


def lib():
    """The loaded C-ABI library.  Built in-tree with nvcc if missing or stale; raises otherwise."""
    global _lib
    if _lib is None:
        so = _lib_path or os.environ.get("BC_LIBRARY") or _build.build()
        if not os.path.exists(so):
            raise ImportError("libbarracuda_b200.so is missing and could not be built; there is no CPU fallback")
        L = C.CDLL(so)
        vp, u32, u64, i32 = C.c_void_p, C.c_uint32, C.c_uint64, C.c_int
        L.bc_index_device_bytes.argtypes = [C.POINTER(bc_index_host), C.POINTER(C.c_size_t)]
        L.bc_index_upload.argtypes = [C.POINTER(bc_index_host), vp, C.c_size_t, vp, C.POINTER(vp)]
        L.bc_index_free.argtypes = [vp]
        L.bc_align_workspace_bytes.argtypes = [vp, u32, u32, C.POINTER(bc_opts), u32, C.POINTER(C.c_size_t)]
        L.bc_align_batch.argtypes = [vp, C.POINTER(bc_reads), C.POINTER(bc_opts), C.POINTER(bc_result), vp, C.c_size_t, vp]
        L.bc_align_best_workspace_bytes.argtypes = [vp, u32, u32, C.POINTER(bc_opts), u32, u64, C.POINTER(C.c_size_t)]
        L.bc_align_batch_best.argtypes = [vp, C.POINTER(bc_reads), C.POINTER(bc_opts), C.c_int32, C.POINTER(bc_result), vp,
                                          C.c_size_t, vp]
        L.bc_pair_workspace_bytes.argtypes = [u32, u64, u64, C.POINTER(C.c_size_t)]
        L.bc_pair_batch.argtypes = [vp, vp, vp, vp, u32, C.POINTER(bc_pair_opts), u64, u64, C.POINTER(bc_pair_result), vp,
                                    C.c_size_t, vp]
        L.bc_locate.argtypes = [vp, vp, u64, vp, vp]
        L.bc_last_stats.argtypes = [vp, C.POINTER(u64 * 16)]
        L.bc_set_geometry.argtypes = [vp, u32, u32]
        L.bc_set_tuning.argtypes = [vp, u32, u32, u32]
        L.bc_set_index_layout.argtypes = [i32]
        L.bc_index_build_host.argtypes = [vp, u64, u32, u32, i32, C.POINTER(C.POINTER(bc_index_host))]
        L.bc_index_host_free.argtypes = [C.POINTER(bc_index_host)]
        L.bc_index_build_gpu_bytes.argtypes = [u64, u32, u32, C.POINTER(C.c_size_t)]
        L.bc_index_build_gpu.argtypes = [vp, u64, u32, u32, vp, C.c_size_t, vp, C.POINTER(C.POINTER(bc_index_host))]
        L.bc_measure_random_sectors.argtypes = [vp, C.c_size_t, u32, vp, vp, C.POINTER(C.c_double)]
        L.bc_measure_random_sectors2.argtypes = [vp, C.c_size_t, u32, i32, vp, vp, C.POINTER(C.c_double)]
        L.bc_exclusive_scan_scratch_bytes.argtypes = [u64]
        L.bc_exclusive_scan_scratch_bytes.restype = C.c_size_t
        L.bc_exclusive_scan_u32.argtypes = [vp, u64, vp, C.c_size_t, vp, vp]
        L.bc_exclusive_scan_u32_static.argtypes = [vp, u64, vp, vp]
        L.bc_scan_static_max_n.argtypes = []
        L.bc_scan_static_max_n.restype = u64
        L.bc_scan_static_setup.argtypes = []
        for f in ("bc_exclusive_scan_u32", "bc_exclusive_scan_u32_static", "bc_scan_static_setup"):
            getattr(L, f).restype = i32
        L.bc_strerror.argtypes = [i32]
        L.bc_strerror.restype = C.c_char_p
        for f in ("bc_index_device_bytes", "bc_index_upload", "bc_index_free", "bc_align_workspace_bytes",
                  "bc_align_batch", "bc_locate", "bc_last_stats", "bc_set_geometry", "bc_set_tuning", "bc_set_index_layout", "bc_index_build_host",
                  "bc_index_host_free", "bc_measure_random_sectors", "bc_measure_random_sectors2", "bc_align_best_workspace_bytes",
                  "bc_align_batch_best", "bc_pair_workspace_bytes", "bc_pair_batch", "bc_index_build_gpu_bytes", "bc_index_build_gpu"):
            getattr(L, f).restype = i32
        _lib = L
    return _lib


def strerror(status: int) -> str:
    return lib().bc_strerror(status).decode()


def _check(status: int, where: str):
    if status != BC_OK:
        raise BcError(status, where)


def _torch():
    import torch
    if not torch.cuda.is_available():
        raise RuntimeError("paper_1505_07855_b200 needs a CUDA device (sm_100a); there is no CPU fallback")
    return torch


def _stream_ptr(torch, stream):
    s = stream if stream is not None else torch.cuda.current_stream()
    return C.c_void_p(s.cuda_stream)


def make_opts(o) -> bc_opts:
    if isinstance(o, bc_opts):
        return o
    t = o.astuple() if hasattr(o, "astuple") else tuple(o)
    return bc_opts(*[int(x) for x in t])


# --------------------------------------------------------------------------------------------
# host index (transport arrays)
# --------------------------------------------------------------------------------------------
class HostIndex:
    """Owner of a bc_index_host built by bc_index_build_host (host memory, library-allocated)."""

    def __init__(self, ptr):
        self._p = ptr

    @property
    def struct(self) -> bc_index_host:
        return self._p.contents

    @property
    def n(self) -> int:
        return int(self.struct.fwd.n)

    def arrays(self, which: int = 0):
        """(bwt2 uint64[], occ uint32[][4], C[5], primary, occ_interval) views of the fwd/rev BWT."""
        b = self.struct.rev if which else self.struct.fwd
        n = int(b.n)
        bwt2 = np.ctypeslib.as_array(C.cast(b.bwt2, C.POINTER(C.c_uint64)), shape=(n // 32 + 1,))
        occ = np.ctypeslib.as_array(C.cast(b.occ, C.POINTER(C.c_uint32)), shape=(n // b.occ_interval + 1, 4))
        return bwt2, occ, [int(x) for x in b.C], int(b.primary), int(b.occ_interval)

    def sa_samples(self):
        s = self.struct
        cnt = self.n // s.sa_interval + 1
        return np.ctypeslib.as_array(C.cast(s.sa, C.POINTER(C.c_uint32)), shape=(cnt,)), int(s.sa_interval)

    def to_arrays(self) -> dict:
        """The transport arrays as a dict of numpy arrays (views; copy before the index is freed)."""
        st = self.struct
        d = {"n": np.uint64(self.n), "sa_interval": np.uint32(st.sa_interval), "sa": self.sa_samples()[0]}
        for name, which in (("fwd", 0), ("rev", 1)):
            bwt2, occ, Cc, primary, oi = self.arrays(which)
            d[name + "_bwt2"], d[name + "_occ"] = bwt2, occ
            d[name + "_C"], d[name + "_primary"], d[name + "_oi"] = np.asarray(Cc, np.uint64), np.uint64(primary), np.uint32(oi)
        return d

    @staticmethod
    def from_arrays(arrs: dict) -> "HostIndex":
        """A bc_index_host over numpy arrays (to_arrays() of another process, or a file); Python owns the memory."""
        keep = {k: np.ascontiguousarray(v) for k, v in arrs.items()}

        def scalar(name):
            return int(keep[name].reshape(-1)[0])
        h = bc_index_host()
        for name, b in (("fwd", h.fwd), ("rev", h.rev)):
            b.n = scalar("n"); b.primary = scalar(name + "_primary"); b.occ_interval = scalar(name + "_oi")
            b.bwt2 = keep[name + "_bwt2"].ctypes.data; b.occ = keep[name + "_occ"].ctypes.data
            for c in range(5):
                b.C[c] = int(keep[name + "_C"].reshape(-1)[c])
        h.sa_interval = scalar("sa_interval"); h.sa = keep["sa"].ctypes.data
        obj = HostIndex(C.pointer(h))
        obj._owned, obj._keep = False, (keep, h)
        return obj

    def save(self, path: str):
        """Cache the transport arrays on disk (config 5: "index built once on the host and cached")."""
        np.savez(path, **self.to_arrays())

    @staticmethod
    def load(path: str) -> "HostIndex":
        z = np.load(path)
        return HostIndex.from_arrays({k: z[k] for k in z.files})

    def free(self):
        if self._p is not None:
            if getattr(self, "_owned", True):
                lib().bc_index_host_free(self._p)
            self._p = None

    def __del__(self):
        try:
            self.free()
        except Exception:
            pass


def bc_index_build_host(text: np.ndarray, occ_interval: int = 128, sa_interval: int = 32,
                        n_threads: int | None = None) -> HostIndex:
    """Suffix-sort T$ and reverse(T)$ on the host (untimed helper)."""
    text = np.ascontiguousarray(text, dtype=np.uint8)
    out = C.POINTER(bc_index_host)()
    rc = lib().bc_index_build_host(text.ctypes.data_as(C.c_void_p), text.size, occ_interval, sa_interval,
                                   n_threads or os.cpu_count() or 1, C.byref(out))
    _check(rc, "bc_index_build_host")
    return HostIndex(out)


# --------------------------------------------------------------------------------------------
# device index
# --------------------------------------------------------------------------------------------
class DeviceIndex:
    """bc_index handle + the torch buffer that backs it."""

    def __init__(self, handle, mem, n, device):
        self._h, self.mem, self.n, self.device = handle, mem, n, device
        self.spill_blocks, self.pool_kb, self.ld_policy = 0, 0, 0

    @property
    def handle(self):
        if self._h is None:
            raise RuntimeError("index was freed")
        return self._h

    def free(self):
        if self._h is not None:
            lib().bc_index_free(self._h)
            self._h = None
            self.mem = None

    def __del__(self):
        try:
            self.free()
        except Exception:
            pass


def bc_index_device_bytes(h: HostIndex) -> int:
    b = C.c_size_t(0)
    _check(lib().bc_index_device_bytes(h._p, C.byref(b)), "bc_index_device_bytes")
    return int(b.value)


def bc_index_upload(h: HostIndex, device="cuda:0", stream=None) -> DeviceIndex:
    """Index wholly resident in GPU memory, re-laid out as 64-byte rank lines."""
    torch = _torch()
    nbytes = bc_index_device_bytes(h)
    dev = torch.device(device)
    with torch.cuda.device(dev):
        mem = torch.empty(nbytes + 256, dtype=torch.uint8, device=dev)
        ptr = (mem.data_ptr() + 255) & ~255
        out = C.c_void_p()
        rc = lib().bc_index_upload(h._p, C.c_void_p(ptr), nbytes, _stream_ptr(torch, stream), C.byref(out))
    _check(rc, "bc_index_upload")
    return DeviceIndex(out, mem, h.n, dev)


def bc_set_geometry(ix: DeviceIndex, ctas_per_sm: int = 0, warps_per_cta: int = 0):
    _check(lib().bc_set_geometry(ix.handle, ctas_per_sm, warps_per_cta), "bc_set_geometry")


def bc_set_index_layout(choice: int = 0):
    """Device layout of indexes uploaded from now on: 0 by size, 1 = 32-byte blocks, 2 = 128-byte lines."""
    _check(lib().bc_set_index_layout(choice), "bc_set_index_layout")


def bc_set_tuning(ix: DeviceIndex, spill_blocks: int = 0, pool_kb: int = 0, ld_policy: int = 0):
    _check(lib().bc_set_tuning(ix.handle, spill_blocks, pool_kb, ld_policy), "bc_set_tuning")
    ix.spill_blocks, ix.pool_kb, ix.ld_policy = spill_blocks, pool_kb, ld_policy


STAT_NAMES = ("nodes", "lookups", "lines", "raw_hits", "d_lookups", "pool_max", "search_ns", "geometry",
              "branch_steps", "branch_nodes", "chain_steps", "chain_nodes", "cancelled", "spill_blocks", "spill_max", "passes_or_steals")


def bc_last_stats(ix: DeviceIndex) -> dict:
    a = (C.c_uint64 * 16)()
    _check(lib().bc_last_stats(ix.handle, C.byref(a)), "bc_last_stats")
    return dict(zip(STAT_NAMES, [int(x) for x in a]))


# --------------------------------------------------------------------------------------------
# reads and results
# --------------------------------------------------------------------------------------------
@dataclasses.dataclass
class DeviceReads:
    """bc_reads with torch-owned device tensors (int-typed views of the unsigned transport arrays)."""
    bases2: object      # int32 tensor  (uint32 words)
    nmask: object       # int32 tensor or None
    off: object         # int64 tensor  (uint64)
    len: object         # int16 tensor  (uint16)
    n_reads: int
    max_len: int

    def struct(self) -> bc_reads:
        return bc_reads(self.bases2.data_ptr() if self.n_reads else None,
                        self.nmask.data_ptr() if (self.nmask is not None and self.n_reads) else None,
                        self.off.data_ptr() if self.n_reads else None,
                        self.len.data_ptr() if self.n_reads else None, self.n_reads, self.max_len)


class HostReads:
    """Packed reads in pinned host memory (the transport layout of bc_reads)."""

    def __init__(self, bases2: np.ndarray, nmask, off: np.ndarray, ln: np.ndarray, pin: bool = True):
        import torch
        self.n_reads = int(ln.size)
        self.max_len = int(ln.max()) if ln.size else 1

        def t(a, dt):
            x = torch.from_numpy(np.ascontiguousarray(a).view(dt))
            return x.pin_memory() if (pin and torch.cuda.is_available() and x.numel()) else x
        self.bases2 = t(bases2.astype(np.uint32, copy=False), np.int32)
        self.nmask = None if nmask is None else t(nmask.astype(np.uint32, copy=False), np.int32)
        self.off = t(off.astype(np.uint64, copy=False), np.int64)
        self.len = t(ln.astype(np.uint16, copy=False), np.int16)

    @property
    def nbytes(self) -> int:
        ts = [self.bases2, self.off, self.len] + ([self.nmask] if self.nmask is not None else [])
        return sum(x.numel() * x.element_size() for x in ts)

    def to_device(self, device="cuda:0") -> DeviceReads:
        _torch()
        nm = None if self.nmask is None else self.nmask.to(device, non_blocking=True)
        return DeviceReads(self.bases2.to(device, non_blocking=True), nm, self.off.to(device, non_blocking=True),
                           self.len.to(device, non_blocking=True), self.n_reads, self.max_len)


@dataclasses.dataclass
class AlignResult:
    hit_offsets: object     # int64 tensor [n_reads+1] (device)
    hits: object            # uint8 tensor [n_hits*12] (device), records of HIT_DTYPE
    n_hits: int
    n_raw: int

    def to_numpy(self):
        """(hit_offsets uint64[n_reads+1], hits HIT_DTYPE[n_hits]) on the host."""
        off = self.hit_offsets.cpu().numpy().view(np.uint64)
        hits = self.hits[: self.n_hits * 12].cpu().numpy().view(HIT_DTYPE)
        return off, hits


class Workspace:
    """Caller-owned device buffers of bc_align_batch, reusable across batches of the same shape."""

    def __init__(self, ix: DeviceIndex, n_reads: int, max_len: int, opts, raw_hits_per_read: int = 16,
                 hits_capacity: int | None = None):
        torch = _torch()
        self.ix, self.n_reads, self.max_len = ix, n_reads, max_len
        self.opts = make_opts(opts)
        b = C.c_size_t(0)
        _check(lib().bc_align_workspace_bytes(ix.handle, n_reads, max_len, C.byref(self.opts), raw_hits_per_read,
                                              C.byref(b)), "bc_align_workspace_bytes")
        self.ws_bytes = int(b.value)
        self.raw_hits_per_read = raw_hits_per_read
        with torch.cuda.device(ix.device):
            self.mem = torch.empty(self.ws_bytes + 256, dtype=torch.uint8, device=ix.device)
            self.hits_capacity = int(hits_capacity if hits_capacity is not None else max(1024, 4 * n_reads))
            self.hit_offsets = torch.empty(n_reads + 1, dtype=torch.int64, device=ix.device)
            self.hits = torch.empty(self.hits_capacity * 12, dtype=torch.uint8, device=ix.device)
            self.needed = torch.zeros(2, dtype=torch.int64, device=ix.device)

    @property
    def ptr(self) -> int:
        return (self.mem.data_ptr() + 255) & ~255


def bc_align_workspace_bytes(ix: DeviceIndex, n_reads: int, max_len: int, opts, raw_hits_per_read: int = 0) -> int:
    b = C.c_size_t(0)
    o = make_opts(opts)
    _check(lib().bc_align_workspace_bytes(ix.handle, n_reads, max_len, C.byref(o), raw_hits_per_read, C.byref(b)),
           "bc_align_workspace_bytes")
    return int(b.value)


def bc_align_batch_raw(ix: DeviceIndex, reads: DeviceReads, opts, ws: Workspace, stream=None) -> int:
    """One call of the C entry point; returns its status code (no retry, no exception)."""
    torch = _torch()
    o = make_opts(opts)
    r = reads.struct()
    res = bc_result(ws.hit_offsets.data_ptr(), ws.hits.data_ptr(), ws.hits_capacity, ws.needed.data_ptr())
    with torch.cuda.device(ix.device):
        return lib().bc_align_batch(ix.handle, C.byref(r), C.byref(o), C.byref(res), C.c_void_p(ws.ptr), ws.ws_bytes,
                                    _stream_ptr(torch, stream))


def bc_align_batch(ix: DeviceIndex, reads: DeviceReads, opts, ws: Workspace | None = None, stream=None,
                   grow: bool = True):
    """The hot path: per read, the deduplicated sorted SA intervals with
    their minimum difference counts.  On BC_E_OVERFLOW the caller-owned buffers are re-allocated at
    the size the library reports and the call is repeated (grow=True), else BcError is raised.
    Returns (AlignResult, Workspace)."""
    if ws is None:
        ws = Workspace(ix, reads.n_reads, max(1, reads.max_len), opts)
    for _ in range(7):
        rc = bc_align_batch_raw(ix, reads, opts, ws, stream)
        if rc == BC_OK:
            need = ws.needed.cpu().numpy().view(np.uint64)
            return AlignResult(ws.hit_offsets, ws.hits, int(need[0]), int(need[1])), ws
        if rc == BC_E_NOMEM and grow and (ix.spill_blocks or 128) < 8192:
            # a warp's spill area of pending branch states ran full: give it more and repeat (never truncated)
            bc_set_tuning(ix, 4 * (ix.spill_blocks or 128), ix.pool_kb, ix.ld_policy)
            ws = Workspace(ix, reads.n_reads, max(1, reads.max_len), opts, ws.raw_hits_per_read, ws.hits_capacity)
            continue
        if rc != BC_E_OVERFLOW or not grow:
            raise BcError(rc, "bc_align_batch")
        need = ws.needed.cpu().numpy().view(np.uint64)
        n_dedup, n_raw = int(need[0]), int(need[1])
        per_read = max(ws.raw_hits_per_read, -(-n_raw // max(1, reads.n_reads)) + 1)
        cap = max(ws.hits_capacity, n_dedup if n_dedup else ws.hits_capacity)
        ws = Workspace(ix, reads.n_reads, max(1, reads.max_len), opts, per_read, cap)
    raise BcError(BC_E_OVERFLOW, "bc_align_batch (after growing)")


def bc_align_batch_host(ix: DeviceIndex, hreads: HostReads, opts, ws: Workspace | None = None, stream=None):
    """End-to-end call with HOST buffers: pinned host reads -> device, bc_align_batch, CSR result
    back to the host.  Returns (hit_offsets uint64[], hits HIT_DTYPE[], Workspace)."""
    torch = _torch()
    with torch.cuda.device(ix.device):
        dreads = hreads.to_device(ix.device)
        res, ws = bc_align_batch(ix, dreads, opts, ws, stream)
        off, hits = res.to_numpy()
    return off, hits, ws


def bc_locate(ix: DeviceIndex, rows, stream=None):
    """SA rows -> text coordinates: pos[i] = SA_fwd[rows[i]]."""
    torch = _torch()
    rows_t = torch.as_tensor(np.ascontiguousarray(rows, dtype=np.uint32).view(np.int32), device=ix.device) \
        if not hasattr(rows, "data_ptr") else rows
    pos = torch.empty_like(rows_t)
    with torch.cuda.device(ix.device):
        rc = lib().bc_locate(ix.handle, C.c_void_p(rows_t.data_ptr()), rows_t.numel(), C.c_void_p(pos.data_ptr()),
                             _stream_ptr(torch, stream))
    _check(rc, "bc_locate")
    return pos


def bc_measure_random_sectors(table_bytes: int, loads_per_thread: int = 256, device="cuda:0", stream=None, ld_policy: int = 0) -> float:
    """Random 32-byte-sector load rate (sectors/s) over a torch-allocated table of `table_bytes`; ld_policy 0 =
    default cache policies, 1 = the search kernel's (no L1 allocation, 64-byte L2 prefetch size)."""
    torch = _torch()
    dev = torch.device(device)
    with torch.cuda.device(dev):
        table = torch.empty(table_bytes // 4, dtype=torch.int32, device=dev)
        table.fill_(0x5A5A5A5A)
        sink = torch.zeros(4, dtype=torch.int32, device=dev)
        out = C.c_double(0.0)
        rc = lib().bc_measure_random_sectors2(C.c_void_p(table.data_ptr()), table.numel() * 4, loads_per_thread, ld_policy,
                                              C.c_void_p(sink.data_ptr()), _stream_ptr(torch, stream), C.byref(out))
    _check(rc, "bc_measure_random_sectors")
    return float(out.value)


def bc_exclusive_scan_u32(counts, scratch=None, stream=None):
    """Exclusive scan of a uint32 device tensor (int32 view) into n+1 uint64 offsets (int64 view); the scratch is a
    caller-owned device tensor (allocated here by torch when None).  Enqueues on the stream; no synchronise."""
    torch = _torch()
    n = counts.numel()
    out = torch.empty(n + 1, dtype=torch.int64, device=counts.device)
    need = int(lib().bc_exclusive_scan_scratch_bytes(n))
    if scratch is None:
        scratch = torch.empty(need, dtype=torch.uint8, device=counts.device)
    with torch.cuda.device(counts.device):
        rc = lib().bc_exclusive_scan_u32(C.c_void_p(counts.data_ptr() if n else None), n, C.c_void_p(scratch.data_ptr()),
                                         scratch.numel() * scratch.element_size(), C.c_void_p(out.data_ptr()),
                                         _stream_ptr(torch, stream))
    _check(rc, "bc_exclusive_scan_u32")
    return out


def bc_scan_static_max_n() -> int:
    return int(lib().bc_scan_static_max_n())


def bc_exclusive_scan_u32_static(counts, out, stream=None):
    """The same scan with NO allocation anywhere: scratch in a static device array of the library (n up to
    bc_scan_static_max_n() = 67,108,864), `out` (int64, n+1) provided by the caller.  Calls that overlap on the GPU
    race on the shared scratch; calls on one stream are safe."""
    torch = _torch()
    n = counts.numel()
    if out.numel() < n + 1:
        raise ValueError("out must hold n + 1 offsets")
    with torch.cuda.device(counts.device):
        rc = lib().bc_exclusive_scan_u32_static(C.c_void_p(counts.data_ptr() if n else None), n, C.c_void_p(out.data_ptr()),
                                                _stream_ptr(torch, stream))
    if rc == BC_E_UNSUPPORTED:
        raise BcError(rc, f"bc_exclusive_scan_u32_static: n = {n} exceeds the static scratch limit {bc_scan_static_max_n()}")
    _check(rc, "bc_exclusive_scan_u32_static")
    return out


class BestWorkspace:
    """Caller-owned device buffers of bc_align_batch_best."""

    def __init__(self, ix: DeviceIndex, n_reads: int, max_len: int, opts, raw_hits_per_read: int = 16,
                 hits_capacity: int | None = None):
        torch = _torch()
        self.ix, self.n_reads, self.max_len = ix, n_reads, max_len
        self.opts = make_opts(opts)
        self.raw_hits_per_read = raw_hits_per_read
        self.hits_capacity = int(hits_capacity if hits_capacity is not None else max(1024, 4 * n_reads))
        b = C.c_size_t(0)
        _check(lib().bc_align_best_workspace_bytes(ix.handle, n_reads, max_len, C.byref(self.opts), raw_hits_per_read,
                                                   self.hits_capacity, C.byref(b)), "bc_align_best_workspace_bytes")
        self.ws_bytes = int(b.value)
        with torch.cuda.device(ix.device):
            self.mem = torch.empty(self.ws_bytes + 256, dtype=torch.uint8, device=ix.device)
            self.hit_offsets = torch.empty(n_reads + 1, dtype=torch.int64, device=ix.device)
            self.hits = torch.empty(self.hits_capacity * 12, dtype=torch.uint8, device=ix.device)
            self.needed = torch.zeros(2, dtype=torch.int64, device=ix.device)

    @property
    def ptr(self) -> int:
        return (self.mem.data_ptr() + 255) & ~255


def bc_align_batch_best_raw(ix: DeviceIndex, reads: DeviceReads, opts, stratum_plus: int, ws: BestWorkspace, stream=None) -> int:
    torch = _torch()
    o = make_opts(opts)
    r = reads.struct()
    res = bc_result(ws.hit_offsets.data_ptr(), ws.hits.data_ptr(), ws.hits_capacity, ws.needed.data_ptr())
    with torch.cuda.device(ix.device):
        return lib().bc_align_batch_best(ix.handle, C.byref(r), C.byref(o), stratum_plus, C.byref(res), C.c_void_p(ws.ptr),
                                         ws.ws_bytes, _stream_ptr(torch, stream))


def bc_align_batch_best(ix: DeviceIndex, reads: DeviceReads, opts, stratum_plus: int = 1, ws: BestWorkspace | None = None,
                        stream=None):
    """Best-stratum mode: per read the hits with d <= min(d_min + stratum_plus, z).  Grows the
    caller-owned buffers and repeats on BC_E_OVERFLOW.  Returns (AlignResult, BestWorkspace)."""
    if ws is None:
        ws = BestWorkspace(ix, reads.n_reads, max(1, reads.max_len), opts)
    for _ in range(8):
        rc = bc_align_batch_best_raw(ix, reads, opts, stratum_plus, ws, stream)
        need = ws.needed.cpu().numpy().view(np.uint64)
        if rc == BC_OK:
            return AlignResult(ws.hit_offsets, ws.hits, int(need[0]), int(need[1])), ws
        if rc == BC_E_NOMEM and (ix.spill_blocks or 128) < 8192:     # spill area exhausted: more of it, repeat
            bc_set_tuning(ix, 4 * (ix.spill_blocks or 128), ix.pool_kb, ix.ld_policy)
            ws = BestWorkspace(ix, reads.n_reads, max(1, reads.max_len), opts, ws.raw_hits_per_read, ws.hits_capacity)
            continue
        if rc != BC_E_OVERFLOW:
            raise BcError(rc, "bc_align_batch_best")
        # need = {hits after dedup (0 when the raw arena overflowed: nothing was sorted), raw hits}: grow what was short
        per_read = max(ws.raw_hits_per_read, -(-int(need[1]) // max(1, reads.n_reads)) + 1)
        if per_read == ws.raw_hits_per_read and int(need[0]) <= ws.hits_capacity:
            per_read *= 2
        cap = max(ws.hits_capacity, int(need[0]) + 1) if int(need[0]) > ws.hits_capacity else ws.hits_capacity
        ws = BestWorkspace(ix, reads.n_reads, max(1, reads.max_len), opts, per_read, cap)
    raise BcError(BC_E_OVERFLOW, "bc_align_batch_best (after growing)")


def bc_pair_batch(ix: DeviceIndex, result: AlignResult, reads: DeviceReads, min_frag: int, max_frag: int, max_occ: int = 32,
                  stream=None):
    """Pair the two ends of every fragment (reads 2i, 2i+1) by plausible distance.
    Returns (pair_offsets uint64[n_pairs+1], pairs PAIR_DTYPE[], needed dict) on the host; buffers are
    grown and the call repeated on BC_E_OVERFLOW."""
    torch = _torch()
    n_reads = reads.n_reads
    o = bc_pair_opts(min_frag, max_frag, max_occ)
    max_place, max_raw, cap = max(1024, 4 * n_reads), max(1024, 2 * n_reads), max(1024, n_reads)
    for _ in range(4):
        b = C.c_size_t(0)
        _check(lib().bc_pair_workspace_bytes(n_reads, max_place, max_raw, C.byref(b)), "bc_pair_workspace_bytes")
        with torch.cuda.device(ix.device):
            mem = torch.empty(int(b.value) + 256, dtype=torch.uint8, device=ix.device)
            poff = torch.empty(n_reads // 2 + 1, dtype=torch.int64, device=ix.device)
            pairs = torch.empty(cap * 16, dtype=torch.uint8, device=ix.device)
            need = torch.zeros(4, dtype=torch.int64, device=ix.device)
            res = bc_pair_result(poff.data_ptr(), pairs.data_ptr(), cap, need.data_ptr())
            rc = lib().bc_pair_batch(ix.handle, C.c_void_p(result.hit_offsets.data_ptr()), C.c_void_p(result.hits.data_ptr()),
                                     C.c_void_p(reads.len.data_ptr()), n_reads, C.byref(o), max_place, max_raw, C.byref(res),
                                     C.c_void_p((mem.data_ptr() + 255) & ~255), int(b.value), _stream_ptr(torch, stream))
        nd = need.cpu().numpy().view(np.uint64)
        info = {"pairs": int(nd[0]), "raw_pairs": int(nd[1]), "placements": int(nd[2]), "skipped_hits": int(nd[3])}
        if rc == BC_OK:
            return poff.cpu().numpy().view(np.uint64), pairs[: info["pairs"] * 16].cpu().numpy().view(PAIR_DTYPE), info
        if rc != BC_E_OVERFLOW:
            raise BcError(rc, "bc_pair_batch")
        max_place = max(max_place, info["placements"] + 1)
        max_raw = max(max_raw, info["raw_pairs"] + 1)
        cap = max(cap, info["pairs"] + 1, info["raw_pairs"] + 1)
    raise BcError(BC_E_OVERFLOW, "bc_pair_batch (after growing)")


def bc_index_build_gpu(text: np.ndarray, occ_interval: int = 128, sa_interval: int = 32, device="cuda:0",
                       stream=None) -> HostIndex:
    """Index construction on the GPU (prefix doubling); same transport arrays as bc_index_build_host."""
    torch = _torch()
    text = np.ascontiguousarray(text, dtype=np.uint8)
    b = C.c_size_t(0)
    _check(lib().bc_index_build_gpu_bytes(text.size, occ_interval, sa_interval, C.byref(b)), "bc_index_build_gpu_bytes")
    dev = torch.device(device)
    out = C.POINTER(bc_index_host)()
    with torch.cuda.device(dev):
        mem = torch.empty(int(b.value) + 256, dtype=torch.uint8, device=dev)
        rc = lib().bc_index_build_gpu(text.ctypes.data_as(C.c_void_p), text.size, occ_interval, sa_interval,
                                      C.c_void_p((mem.data_ptr() + 255) & ~255), int(b.value), _stream_ptr(torch, stream),
                                      C.byref(out))
    _check(rc, "bc_index_build_gpu")
    return HostIndex(out)
