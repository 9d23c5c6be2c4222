"""Build libmhd.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_0908_4362_b200.build [--force] [--verbose]

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


def build(force: bool = False, verbose: bool = False) -> str:
    newest = _newest_source_mtime()
    jobs = [(lib, extra) for lib, extra in ((LIB, []), (LIB_JITTER, ["-DMHD_JITTER"]))
            if force or not os.path.exists(lib) or os.path.getmtime(lib) < newest]
    if len(jobs) == 2 and not verbose:             # both stale: compile them side by side
        import concurrent.futures
        with concurrent.futures.ThreadPoolExecutor(2) as ex:
            for f in [ex.submit(_compile, lib, extra, False) for lib, extra in jobs]:
                f.result()
    else:
        for lib, extra in jobs:
            _compile(lib, extra, verbose)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
