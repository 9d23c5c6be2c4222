"""Small cases that drive every kernel family of the hot path once (-m gpu), sized so that the whole file also runs
under compute-sanitizer in a few minutes:

    compute-sanitizer --tool memcheck  python -m pytest tests/test_gpu_sanitizer_cases.py -m gpu -q
    compute-sanitizer --tool racecheck python -m pytest tests/test_gpu_sanitizer_cases.py -m gpu -q

(one tool per run; summaries under profiles/).  The march kernels have no block barrier in the march: warps drift and
an elected lane refills shared-memory ring stages behind full/empty mbarriers, which is exactly the neighbour hazard
the paper splits its kernels for.  Every case is also checked against the oracle, so the file is an
ordinary parity test when run without the sanitizer."""
import numpy as np
import pytest

import oracle
from tests.parity_utils import max_rel, random_state, worst

pytestmark = pytest.mark.gpu

# (nx, ny, nz), bc: ring marches with 256- and 128-wide tiles, packed x kernels, fused reverse L_x, generic fallbacks
# (outflow along x, ragged extents), extent-1 axes, several march segments
CASES = [((256, 12, 16), 0), ((128, 16, 12), 1), ((512, 8, 9), 0), ((40, 24, 20), 1), ((64, 32, 1), 0), ((48, 1, 1), 1)]


@pytest.mark.parametrize("prec", ["f32", "f64"])
@pytest.mark.parametrize("shape,bc", CASES)
def test_all_kernel_families_small(shape, bc, prec):
    from paper_0908_4362_b200 import binding as B
    nx, ny, nz = shape
    dtp = np.float32 if prec == "f32" else np.float64
    f = [np.ascontiguousarray(a, dtype=dtp) for a in random_state(nx, ny, nz, seed=1)]
    ref = [np.array(a, dtype=np.float64) for a in f]
    s = B.Solver(nx, ny, nz, 1.4, prec, bc)
    s.set_option("graph", 0)
    s.set_state(f)
    for k in range(3):                                  # all three rotations
        dt, _ = s.cfl_dt(0.8)
        cur = [np.array(a, dtype=np.float64) for a in s.get_state()]
        oracle.step_fixed(cur, 1.4, bc, k, dt)
        s.step_fixed(1, dt)
        assert worst(max_rel(s.get_state(), cur)) <= (1e-12 if prec == "f64" else 1e-5), (shape, bc, prec, k)
    s.step(2, 0.8)                                      # fused c_max reduction + dt on the device
    n, t = s.run_until(s.time() + 0.3, 0.8)             # device-side stop test and clipping
    assert n >= 1
    s.set_option("graph", 1)                            # whole steps as a replayed CUDA graph
    s.step(2, 0.8)
    s.diagnostics()
    s.close()
