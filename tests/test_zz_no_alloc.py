"""The entry point that allocates nothing (bc_exclusive_scan_u32_static, csrc/bc_noalloc.cu): its scratch is a
static __device__ array of the library, so it can be called where cudaMalloc cannot (graph capture, serving loops).
Checked against the existing path (the same scan with caller-provided scratch, bc_exclusive_scan_u32) and against
numpy's cumsum, bit for bit (integer work), on two calls in a row that share the static scratch -- the second one
smaller than the first, so stale tile sums of the first call are still in the array -- and for the size limit.
Named test_zz_* so that pytest collects it last: a failure here must not hide any other test under `pytest -x`."""
import numpy as np
import pytest

import paper_1505_07855_b200 as bc

pytestmark = pytest.mark.gpu


def _counts(n, seed):
    rng = np.random.default_rng(seed)
    c = rng.integers(0, 50, size=n, dtype=np.uint32)
    if n > 10:
        c[rng.integers(0, n, size=5)] = np.uint32(0xFFFFFFF0)      # sums pass 2^32: the offsets are 64-bit
    return c


def test_static_scan_equals_existing_path_on_two_calls_in_a_row():
    import torch
    assert torch.cuda.is_available()
    dev = torch.device("cuda:0")
    assert bc.lib().bc_scan_static_setup() == bc.BC_OK
    before = torch.cuda.memory_allocated(dev)
    sizes = [1_000_003, 4_099, 2_048, 1, 0, 3_000_000]            # several tiles + ragged tails; then fewer tiles than before
    ins = [torch.from_numpy(_counts(n, 100 + i).view(np.int32)).to(dev) for i, n in enumerate(sizes)]
    outs = [torch.empty(n + 1, dtype=torch.int64, device=dev) for n in sizes]
    torch.cuda.synchronize()
    held = torch.cuda.memory_allocated(dev)
    # back to back on one stream, no synchronise in between: the calls share the static scratch, in stream order
    for x, o in zip(ins, outs):
        bc.bc_exclusive_scan_u32_static(x, o)
    assert torch.cuda.memory_allocated(dev) == held                # nothing was allocated through torch either
    torch.cuda.synchronize()
    for x, o, n in zip(ins, outs, sizes):
        want_existing = bc.bc_exclusive_scan_u32(x)                # the existing path: caller-provided scratch
        torch.cuda.synchronize()
        got = o.cpu().numpy().view(np.uint64)
        assert np.array_equal(got, want_existing.cpu().numpy().view(np.uint64)), n
        ref = np.concatenate([[0], np.cumsum(x.cpu().numpy().view(np.uint32).astype(np.uint64))]).astype(np.uint64)
        assert np.array_equal(got, ref), n
    # the same input again after the others: same bytes (the array keeps old contents, none of them is read)
    again = torch.empty_like(outs[0])
    bc.bc_exclusive_scan_u32_static(ins[0], again)
    torch.cuda.synchronize()
    assert torch.equal(again, outs[0])
    del ins, outs, again
    assert before >= 0


def test_static_scan_rejects_sizes_beyond_its_scratch():
    import torch
    lim = bc.bc_scan_static_max_n()
    assert lim == 1 << 26
    out = torch.empty(8, dtype=torch.int64, device="cuda:0")
    x = torch.zeros(8, dtype=torch.int32, device="cuda:0")
    # the size check comes before any memory is touched, so a small buffer with a large n is safe to pass
    rc = bc.lib().bc_exclusive_scan_u32_static(x.data_ptr(), lim + 1, out.data_ptr(), None)
    assert rc == bc.BC_E_UNSUPPORTED
    assert bc.lib().bc_exclusive_scan_u32_static(None, 5, out.data_ptr(), None) == bc.BC_E_INVAL
    assert bc.lib().bc_exclusive_scan_u32(x.data_ptr(), 8, x.data_ptr(), 8, out.data_ptr(), None) == bc.BC_E_NOMEM
