"""GPU parity of the fused sweeps along y and z (mhd_lrev.cuh; -m gpu): the reverse L_d as one kernel (B pair, then fluid,
PAPER.md:317) and the middle pair of a step (forward L_d then reverse L_d, eqs (23)-(25) PAPER.md:164-170) with its two B
pairs and the fluid update chained through shared memory.  Every case is compared element by
element with the oracle's operator sequence, and with the unfused kernels to a few ulp (same arithmetic templates, other
plumbing: nvcc contracts a*b+c into FMAs kernel by kernel, so the last bit may differ)."""
import numpy as np
import pytest

import oracle
from paper_0908_4362_b200 import inputs
from tests.parity_utils import max_rel, random_state, worst

pytestmark = pytest.mark.gpu
ULPS = {"f64": 2e-15, "f32": 1e-6}          # fused against unfused kernels, relative to the largest value of the field group
P, O = inputs.PERIODIC, inputs.OUTFLOW

# nx a multiple of the tile (128 fp32 / 64 fp64), several tiles, rows and march segments, ragged extents along the march
SHAPES = [(128, 36, 40), (256, 48, 33), (384, 32, 70), (128, 1, 64), (128, 64, 1), (64, 40, 32), (192, 33, 47)]


@pytest.fixture(scope="module")
def B():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_0908_4362_b200 import binding
    return binding


def _solver(B, f, gamma, bc, prec, **opts):
    nz, ny, nx = f[0].shape
    s = B.Solver(nx, ny, nz, gamma, prec, bc)
    for k, v in opts.items():
        s.set_option(k, v)
    s.set_state([np.ascontiguousarray(a, dtype=np.float32 if prec == "f32" else np.float64) for a in f])
    return s


def _ref(f, prec):
    dt = np.float32 if prec == "f32" else np.float64
    return [np.array(np.asarray(a, dtype=dt), dtype=np.float64) for a in f]


@pytest.mark.parametrize("seg", [-1, 16, 24])
@pytest.mark.parametrize("shape", SHAPES)
@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_fused_operators_match_oracle_and_unfused_kernels(B, shape, prec, seg):
    nx, ny, nz = shape
    if seg != -1 and shape not in SHAPES[:3]:
        pytest.skip("segment sweep on the first three shapes only")
    f0 = random_state(nx, ny, nz, seed=nx + 3 * ny + 5 * nz)
    gamma, dt = 5.0 / 3.0, 0.21
    tol = 1e-12 if prec == "f64" else 1e-5
    for d in (1, 2):
        for op in (B.MHD_OP_SWEEP_REVERSE, B.MHD_OP_MIDDLE_PAIR):
            ref = _ref(f0, prec)
            if op == B.MHD_OP_MIDDLE_PAIR:
                oracle.sweep(ref, gamma, P, d, False, dt)
            oracle.sweep(ref, gamma, P, d, True, dt)
            outs = []
            for fuse in (0, 1, 2):
                s = _solver(B, f0, gamma, P, prec, fuse=fuse, segment=seg)
                l0 = s.launch_count()
                s.apply(op, d, 0, dt)
                outs.append((s.get_state(), s.launch_count() - l0))
                s.close()
            e = max_rel(outs[1][0], ref)
            assert worst(e) <= tol, (shape, prec, d, op, e)
            for fuse in (1, 2):
                assert worst(max_rel(outs[fuse][0], outs[0][0])) <= ULPS[prec], (shape, prec, d, op, fuse)
            fusable = (ny if d == 1 else nz) >= 32 and nx % (128 if prec == "f32" else 64) == 0
            if fusable:          # the fused path really ran: fewer launches than the unfused sequence (each + 1 for set_dt)
                assert outs[1][1] < outs[0][1], (shape, prec, d, op, outs[0][1], outs[1][1])


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_fused_steps_all_rotations_with_cmax(B, prec):
    """whole steps (all three rotations, fused c_max reduction in the last kernel) with and without the fused sweeps"""
    f0 = random_state(128, 40, 48, seed=17)
    gamma = 1.4
    outs = []
    for fuse in (0, 1, 2):
        s = _solver(B, f0, gamma, P, prec, fuse=fuse, graph=0)
        t = s.step(6, 0.8)
        outs.append((s.get_state(), t, s.launch_count()))
        s.close()
    for other in outs[1:]:
        assert abs(other[1] - outs[0][1]) <= 10 * ULPS[prec] * outs[0][1]
        assert worst(max_rel(other[0], outs[0][0])) <= 20 * ULPS[prec]
    assert outs[1][2] < outs[2][2] < outs[0][2]
    ref = _ref(f0, prec)
    t_ref = oracle.run(ref, gamma, P, 0, 6, 0.8)
    assert abs(t_ref - outs[1][1]) <= (1e-12 if prec == "f64" else 1e-5) * t_ref
    assert worst(max_rel(outs[1][0], ref)) <= (6e-12 if prec == "f64" else 6e-5)


def test_outflow_grids_run_unfused(B):
    """chaining through ghost cells is exact for periodic boundaries only (mhd_lrev.cuh): outflow grids keep the
    unfused kernels, same launch count with fuse = 0 and 1"""
    f0 = random_state(128, 36, 40, seed=2)
    counts = []
    for fuse in (0, 1):
        s = _solver(B, f0, 1.4, O, "f32", fuse=fuse, graph=0)
        s.step_fixed(3, 0.1)
        counts.append(s.launch_count())
        s.close()
    assert counts[0] == counts[1]
