"""Build libmhd.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_0908_4362_b200.build [--force] [--verbose] [--jitter]

The shared library is git-ignored but travels to the GPU box with the repo snapshot.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libmhd.so")
# the same sources with -DMHD_JITTER (csrc/mhd_async.cuh): random sleeps around every mbarrier operation, for
# tests/test_gpu_jitter.py (compute-sanitizer is closed on this pool); never loaded by the product path
LIB_JITTER = os.path.join(HERE, "libmhd_jitter.so")
SOURCES = ["mhd_api.cu", "mhd_noalloc.cu"]
NVCC_FLAGS = [
    "-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
    "-shared", "-Xcompiler", "-fPIC", "--cudart=static",
]


def _newest_source_mtime() -> float:
    m = 0.0
    for root in (CSRC, os.path.join(os.path.dirname(HERE), "include")):
        for fn in os.listdir(root):
            m = max(m, os.path.getmtime(os.path.join(root, fn)))
    return m


def _compile(lib: str, extra, verbose: bool) -> None:
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    cmd = [nvcc] + NVCC_FLAGS + list(extra) + os.environ.get("MHD_NVCC_EXTRA", "").split() + (["-Xptxas", "-v"] if verbose else []) + ["-o", lib] + [os.path.join(CSRC, s) for s in SOURCES]
    res = subprocess.run(cmd, capture_output=True, text=True)
    if verbose or res.returncode != 0:
        sys.stderr.write(res.stdout + res.stderr)
    if res.returncode != 0:
        raise RuntimeError(f"nvcc failed building {os.path.basename(lib)}")


def _stale(lib: str, force: bool) -> bool:
    return force or not os.path.exists(lib) or os.path.getmtime(lib) < _newest_source_mtime()


def build(force: bool = False, verbose: bool = False) -> str:
    """The product library only.  (The jitter build is test infrastructure: build_jitter(), called by the test that
    loads it, so that importing the package never waits for, or fails on, a second nvcc run.)"""
    if _stale(LIB, force):
        _compile(LIB, [], verbose)
    return LIB


def build_jitter(force: bool = False, verbose: bool = False) -> str:
    """libmhd_jitter.so for tests/test_gpu_jitter.py; never loaded by the product path."""
    if _stale(LIB_JITTER, force):
        _compile(LIB_JITTER, ["-DMHD_JITTER"], verbose)
    return LIB_JITTER


if __name__ == "__main__":
    if "--jitter" in sys.argv:
        print(build_jitter(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
    else:
        print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
