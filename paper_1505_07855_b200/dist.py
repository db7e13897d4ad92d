"""Multi-GPU plumbing: the path shards by reads -- every rank holds a
replica of the index and aligns its own contiguous range of reads; there is NO data-path
collective (the paper does the same at process level: one `aln` per end per GPU, PAPER.md:104,
:117-119).  torch.distributed is used only for the barrier, the max-over-ranks of the timing and
the host-side concatenation of CSR results."""
from __future__ import annotations

import os

import numpy as np


def shard_range(n_total: int, rank: int, world: int):
    """Contiguous range (first, count) of rank `rank` out of n_total units; sizes differ by <= 1."""
    base, rem = divmod(n_total, world)
    first = rank * base + min(rank, rem)
    return first, base + (1 if rank < rem else 0)


def _dist():
    import torch.distributed as d
    return d


def init_from_env(backend: str | None = None):
    """(rank, world, local_rank); initialises the process group when WORLD_SIZE > 1."""
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1 and not _dist().is_initialized():
        import torch
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29500")
        # BC_DIST_BACKEND=gloo lets the N>1 plumbing be exercised where NCCL cannot run (several ranks on one GPU)
        be = backend or os.environ.get("BC_DIST_BACKEND") or ("nccl" if torch.cuda.is_available() else "gloo")
        if be == "nccl":
            torch.cuda.set_device(local)
        _dist().init_process_group(backend=be, rank=rank, world_size=world)
    return rank, world, local


def active() -> bool:
    d = _dist()
    return d.is_available() and d.is_initialized() and d.get_world_size() > 1


def barrier():
    if active():
        _dist().barrier()


def max_over_ranks(x: float, device=None) -> float:
    if not active():
        return float(x)
    import torch
    t = torch.tensor([float(x)], dtype=torch.float64, device=device if _dist().get_backend() == "nccl" else "cpu")
    _dist().all_reduce(t, op=_dist().ReduceOp.MAX)
    return float(t.item())


def broadcast_array(a, device=None, src: int = 0):
    """numpy array of rank `src` on every rank (other ranks pass None).  Shape and dtype travel first."""
    if not active():
        return a
    import torch
    d = _dist()
    meta = [(a.shape, a.dtype.str) if d.get_rank() == src else None]
    d.broadcast_object_list(meta, src=src)
    shape, dt = meta[0]
    on_gpu = d.get_backend() == "nccl"
    if d.get_rank() == src:
        t = torch.from_numpy(np.ascontiguousarray(a).view(np.uint8).reshape(-1))
    else:
        t = torch.empty(int(np.prod(shape, dtype=np.int64)) * np.dtype(dt).itemsize, dtype=torch.uint8)
    if on_gpu:
        t = t.to(device)
    if t.numel():
        d.broadcast(t, src=src)
    out = t.cpu().numpy().view(np.dtype(dt)).reshape(shape)
    return a if d.get_rank() == src else out


def broadcast_host_index(host, device=None, src: int = 0):
    """The index is built ONCE (rank `src`) and its transport arrays are shipped to the other ranks -- one suffix
    sort instead of one per GPU ("one broadcast over NVLink at upload").  Returns a HostIndex everywhere."""
    if not active():
        return host
    from . import HostIndex
    d = _dist()
    names = ["n", "sa_interval", "sa"] + [p + s for p in ("fwd", "rev") for s in ("_bwt2", "_occ", "_C", "_primary", "_oi")]
    arrs = host.to_arrays() if d.get_rank() == src else {}
    out = {}
    for nm in names:
        out[nm] = broadcast_array(np.asarray(arrs[nm]) if d.get_rank() == src else None, device, src)
    return host if d.get_rank() == src else HostIndex.from_arrays(out)


def gather_csr(hit_offsets: np.ndarray, hits: np.ndarray):
    """Concatenate per-rank CSR results in rank order on rank 0 (offsets rebased); other ranks get
    None.  Host-side, after the timed region."""
    if not active():
        return hit_offsets, hits
    d = _dist()
    objs = [None] * d.get_world_size() if d.get_rank() == 0 else None
    d.gather_object((hit_offsets, hits), objs, dst=0)
    if d.get_rank() != 0:
        return None
    offs, hs, base = [np.zeros(1, np.uint64)], [], np.uint64(0)
    for o, h in objs:
        offs.append(o[1:].astype(np.uint64) + base)
        base = base + np.uint64(o[-1])
        hs.append(h)
    return np.concatenate(offs), np.concatenate(hs)


def finish():
    if active():
        _dist().destroy_process_group()
