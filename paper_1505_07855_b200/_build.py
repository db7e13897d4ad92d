"""In-tree build of the C-ABI library (nvcc, sm_100a only).  No JIT cache: the .so sits next to
this file so that it travels with the repo snapshot to the GPU box."""
from __future__ import annotations

import os
import shutil
import subprocess

_DIR = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_DIR, "csrc")
SO = os.path.join(_DIR, "libbarracuda_b200.so")
SOURCES = ["bc_index.cu", "bc_search.cu", "bc_post.cu", "bc_align.cu", "bc_best.cu", "bc_pair.cu", "bc_build_gpu.cu", "bc_roofline.cu", "bc_noalloc.cu", "bc_index_build.cpp"]
HEADERS = ["bc_internal.cuh", "bc_ws.cuh", "bc_host_index.h", os.path.join("..", "..", "include", "barracuda_b200.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC,-pthread,-O3", "-shared"]


def _nvcc() -> str:
    for c in (shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if c and os.path.exists(c):
            return c
    raise RuntimeError("nvcc not found: cannot build libbarracuda_b200.so")


def stale() -> bool:
    if not os.path.exists(SO):
        return True
    t = os.path.getmtime(SO)
    deps = [os.path.join(CSRC, s) for s in SOURCES + HEADERS]
    return any(os.path.getmtime(d) > t for d in deps)


def build_variant(defines: dict, force: bool = False) -> str:
    """A build-time VARIANT of the library (autotuner): the same sources compiled with
    -DNAME=VALUE for every item of `defines`, as paper_1505_07855_b200/variants/libbarracuda_b200_<tag>.so."""
    tag = "_".join(f"{k.lower().replace('bc_', '')}{v}" for k, v in sorted(defines.items())) or "default"
    out_dir = os.path.join(_DIR, "variants")
    os.makedirs(out_dir, exist_ok=True)
    so = os.path.join(out_dir, f"libbarracuda_b200_{tag}.so")
    deps = [os.path.join(CSRC, s) for s in SOURCES + HEADERS]
    if not force and os.path.exists(so) and all(os.path.getmtime(d) <= os.path.getmtime(so) for d in deps):
        return so
    cmd = [_nvcc()] + NVCC_FLAGS + [f"-D{k}={v}" for k, v in sorted(defines.items())] + ["-o", so] + \
          [os.path.join(CSRC, s) for s in SOURCES]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("nvcc failed:\n" + r.stdout + r.stderr)
    return so


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile every CUDA source of the library for sm_100a into one shared object."""
    if not force and not stale():
        return SO
    cmd = [_nvcc()] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-o", SO] + \
          [os.path.join(CSRC, s) for s in SOURCES]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("nvcc failed:\n" + r.stdout + r.stderr)
    if verbose:
        print(r.stderr)
    return SO


if __name__ == "__main__":
    print(build(force=True, verbose=True))
