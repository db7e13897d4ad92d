"""CPU-only checks of the product's host logic: the C-ABI library loads and exports every symbol
the header declares, argument validation returns status codes (no compute calls), and the host
index builder (bucketed suffix sort -> transport arrays) agrees with the oracle's naive suffix sort
and with first principles (BWT inversion, Occ totals)."""
import ctypes as C
import os
import re

import numpy as np
import pytest

import synthdata as sd
import paper_1505_07855_b200 as bc
from oracle import Oracle

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_functions():
    src = open(os.path.join(ROOT, "include", "barracuda_b200.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(bc_[a-z_0-9]+)\s*\(", src)))


def test_library_exports_every_declared_symbol():
    L = bc.lib()
    names = declared_functions()
    assert {"bc_index_upload", "bc_align_batch", "bc_locate", "bc_index_device_bytes", "bc_align_workspace_bytes",
            "bc_index_free", "bc_strerror"} <= set(names)
    for f in names:
        assert hasattr(L, f), f


def test_strerror_and_invalid_arguments():
    L = bc.lib()
    assert bc.strerror(0) == "ok"
    assert "small" in bc.strerror(bc.BC_E_OVERFLOW)
    b = C.c_size_t(0)
    assert L.bc_index_device_bytes(None, C.byref(b)) == bc.BC_E_INVAL
    assert L.bc_index_free(None) == bc.BC_E_INVAL
    assert L.bc_locate(None, None, 0, None, None) == bc.BC_E_INVAL
    out = C.POINTER(bc.bc_index_host)()
    bad = np.asarray([0, 1, 2, 7], np.uint8)
    assert L.bc_index_build_host(bad.ctypes.data_as(C.c_void_p), 4, 128, 32, 1, C.byref(out)) == bc.BC_E_INVAL
    ok = np.asarray([0, 1, 2, 3], np.uint8)
    assert L.bc_index_build_host(ok.ctypes.data_as(C.c_void_p), 4, 100, 32, 1, C.byref(out)) == bc.BC_E_INVAL
    assert L.bc_index_build_host(ok.ctypes.data_as(C.c_void_p), 4, 128, 0, 1, C.byref(out)) == bc.BC_E_INVAL


def test_compute_entry_points_reject_bad_arguments_without_a_gpu():
    L = bc.lib()
    b = C.c_size_t(0)
    o = bc.make_opts((2, 0, 0, 0, 0, 5))
    assert L.bc_align_workspace_bytes(None, 10, 36, C.byref(o), 0, C.byref(b)) == bc.BC_E_INVAL
    assert L.bc_align_batch(None, None, None, None, None, 0, None) == bc.BC_E_INVAL
    out = C.c_double(0)
    assert L.bc_measure_random_sectors(None, 1 << 20, 64, None, None, C.byref(out)) == bc.BC_E_INVAL
    assert L.bc_last_stats(None, None) == bc.BC_E_INVAL
    assert L.bc_set_geometry(None, 1, 1) == bc.BC_E_INVAL
    assert L.bc_index_host_free(None) == bc.BC_E_INVAL


def unpack_bwt(bwt2, n):
    w = np.repeat(bwt2, 32)[:n]
    sh = (2 * (np.arange(n, dtype=np.uint64) % np.uint64(32))).astype(np.uint64)
    return ((w >> sh) & np.uint64(3)).astype(np.uint8)


def check_against_oracle(T, occ_interval, sa_interval):
    n = T.size
    h = bc.bc_index_build_host(T, occ_interval, sa_interval, 4)
    o = Oracle(T, nthreads=4)
    assert bc.bc_index_device_bytes(h) > 2 * (n // 128 + 1) * 64
    for which in (0, 1):
        SA, B, Cc, primary = o.index(which)
        bwt2, occ, Ch, prim_h, oi = h.arrays(which)
        assert prim_h == primary and Ch == Cc.tolist() and oi == occ_interval
        got = unpack_bwt(bwt2, n)
        want = B[B != 4]
        assert np.array_equal(got, want)
        # Occ checkpoints = prefix counts of the '$'-less string
        for c in range(4):
            pref = np.concatenate([[0], np.cumsum(want == c)])
            idx = np.arange(occ.shape[0]) * occ_interval
            assert np.array_equal(occ[:, c], pref[idx])
        if which == 0:
            sa, si = h.sa_samples()
            assert si == sa_interval and np.array_equal(sa, SA[::sa_interval])
    h.free()


@pytest.mark.parametrize("n,occ_interval,sa_interval", [(1, 32, 1), (5, 32, 4), (127, 64, 32), (128, 128, 32), (191, 64, 32), (192, 128, 32),
                                                         (193, 128, 7), (4096, 128, 32), (50_000, 128, 32)])
def test_host_index_matches_naive_suffix_sort(n, occ_interval, sa_interval):
    T = (sd.hash_u64(77, 1, np.arange(n, dtype=np.uint64)) >> np.uint64(62)).astype(np.uint8)
    check_against_oracle(T, occ_interval, sa_interval)


def test_host_index_on_repeats_and_runs():
    # long runs and tandem repeats stress the comparator past the 12-base bucket key
    T = np.concatenate([np.zeros(3000, np.uint8), np.tile(np.asarray([0, 1, 2, 3, 3, 1], np.uint8), 700),
                        np.full(1000, 3, np.uint8), np.zeros(500, np.uint8)])
    check_against_oracle(T, 128, 32)
    cfg = sd.CONFIGS["2"].scaled(n=300_000)
    check_against_oracle(sd.make_genome(cfg), 128, 32)


def test_host_index_bwt_inversion_reproduces_text():
    """LF-walk from `primary` over the transport arrays reproduces T -- first
    principles, no oracle involved."""
    cfg = sd.CONFIGS["1"].scaled(n=20_000)
    T = sd.make_genome(cfg)
    n = T.size
    h = bc.bc_index_build_host(T, 128, 32, 2)
    bwt2, occ, Cc, primary, _ = h.arrays(0)
    Bs = unpack_bwt(bwt2, n)
    pref = np.zeros((4, n + 1), np.int64)
    for c in range(4):
        pref[c, 1:] = np.cumsum(Bs == c)
    out = np.empty(n, np.uint8)
    j = primary                                  # row with SA = 0: B = '$'; walk from the row of suffix 0 ... backwards
    # start from row 0 (suffix '$', SA = n): B[0] = T[n-1]
    j = 0
    for i in range(n - 1, -1, -1):
        p = j - (1 if j > primary else 0)
        c = int(Bs[p])
        out[i] = c
        j = Cc[c] + int(pref[c, p]) + 1          # C[c] + O(c, j) with O inclusive of row j
    assert j == primary
    assert np.array_equal(out, T)
    assert Cc[4] == n and sum(int(pref[c, n]) for c in range(4)) == n
    h.free()
