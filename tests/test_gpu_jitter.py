"""Scrambled warp interleavings must not change a single bit (-m gpu).

The march kernels (mhd_yz2.cuh, mhd_bring.cuh, mhd_lrev.cuh) have no block barrier: warps drift, an elected lane refills
shared-memory ring stages behind full/empty mbarriers, and the fused sweeps chain warp groups through further rings --
the neighbour hazard the paper splits its kernels for.  compute-sanitizer is closed on this pool (it has
left GPUs needing a reset), so the guard is a second build of the same sources, libmhd_jitter.so (-DMHD_JITTER), in which
about one mbarrier operation in sixteen is preceded by a 0.2-2.2 us sleep that depends on the clock and on the warp: a
hand-over that only holds for the interleavings the hardware usually produces then reads a stage too early or too late
and gives other bits, or deadlocks.  The child process runs tests/jitter_worker.py with that library, twice (the sleeps
differ from run to run); this process runs the same cases with the product library; all three must agree bit for bit."""
import os
import subprocess
import sys

import numpy as np
import pytest

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_jittered_build_gives_identical_bits(tmp_path):
    from paper_0908_4362_b200 import build as bld
    bld.build()
    bld.build_jitter()         # nvcc runs on the GPU box only if the library did not travel with the snapshot
    assert os.path.exists(bld.LIB_JITTER)
    from tests import jitter_worker
    ref = jitter_worker.run_all()
    for rep in range(2):
        out = tmp_path / f"jitter{rep}.npz"
        env = dict(os.environ, MHD_LIB=bld.LIB_JITTER)
        res = subprocess.run([sys.executable, os.path.join(ROOT, "tests", "jitter_worker.py"), str(out)], env=env, cwd=ROOT,
                             capture_output=True, text=True, timeout=900)       # a deadlock shows up as the timeout
        assert res.returncode == 0, res.stderr[-2000:]
        got = np.load(out)
        assert sorted(got.files) == sorted(ref)
        for k in ref:
            assert np.array_equal(got[k], ref[k]), (rep, k)
