"""GPU twin of test_oracle_pins.py::test_upwind_tie_takes_the_cell_on_the_right  (-m gpu).

Eq (21): at an exact tie v_{i+1/2} = 0 the first-order flux comes from cell i+1.  The worked example there
(16 cells, dyadic data, B_7 = 1399/864 and B_8 = 1193/864 by hand) is run through every kernel that evaluates the switch:
the generic marching kernels (path = 1), the x kernels (B pair alone and the fused reverse L_x), the ring kernels along
y / z (one and two rows per thread), in fp64 and fp32, with the 16 cells placed across a tile / segment seam as well.  The
data are exact in both precisions, so the tie is exact in both, and the two possible outcomes differ by 0.24: the tolerance
only has to cover rounding of the one limiter quotient (fp32: rcp.approx).  The whole field is also compared with the
oracle element by element."""
import numpy as np
import pytest

import oracle
from paper_0908_4362_b200 import inputs
from tests.test_oracle_pins import TIE_B7, TIE_B8, tie_state

pytestmark = pytest.mark.gpu
P = inputs.PERIODIC

# (nx, ny, nz), sweep direction d, where the 16 cells start along d
CASES = [((16, 1, 1), 0, 0), ((1, 16, 1), 1, 0), ((1, 1, 16), 2, 0),            # 1-D pencils
         ((16, 8, 6), 0, 0), ((256, 6, 4), 0, 120), ((512, 4, 2), 0, 249),      # x kernels; 120..135 and 249..264 straddle thread / tile seams
         ((256, 32, 6), 1, 8), ((256, 6, 48), 2, 23), ((128, 40, 4), 1, 11),    # ring kernels along y / z
         ((320, 24, 5), 1, 3), ((64, 24, 24), 2, 5)]


@pytest.fixture(scope="module")
def B():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_0908_4362_b200 import binding
    return binding


@pytest.mark.parametrize("opts", [{}, {"path": 1}, {"brows": 1}, {"segment": 12}], ids=["default", "generic", "brows1", "seg12"])
@pytest.mark.parametrize("prec,tol", [("f64", 1e-14), ("f32", 1e-6)])
@pytest.mark.parametrize("case", CASES, ids=[f"{c[0][0]}x{c[0][1]}x{c[0][2]}-d{c[1]}" for c in CASES])
def test_upwind_tie_on_the_gpu(B, case, prec, tol, opts):
    shape3, d, off = case
    npdt = np.float32 if prec == "f32" else np.float64
    for t in ((d + 1) % 3, (d + 2) % 3):
        for reverse in (0, 1):
            f = tie_state(d, t, shape3, npdt, offset=off)
            ref = [np.array(a, dtype=np.float64) for a in f]
            # the B pair is B_{t1->d} then B_{t2->d} (reverse: t2 first); the component that is zero stays zero
            for tt in ([(d + 1) % 3, (d + 2) % 3] if not reverse else [(d + 2) % 3, (d + 1) % 3]):
                oracle.badvect(ref, 5.0 / 3.0, P, d, tt, 0.5)
            s = B.Solver(*shape3, 5.0 / 3.0, prec, P)
            for k, v in opts.items():
                s.set_option(k, v)
            s.set_state(f)
            s.apply(B.MHD_OP_BPAIR, d, reverse, 0.5)
            got = [np.asarray(a, dtype=np.float64) for a in s.get_state()]
            s.close()
            line = np.moveaxis(got[5 + t], 2 - d, 0).reshape(shape3[d], -1)
            assert np.all(np.abs(line[off + 7] - TIE_B7) <= tol * TIE_B7), (t, reverse, line[off + 7].ravel()[:4], TIE_B7)
            assert np.all(np.abs(line[off + 8] - TIE_B8) <= tol * TIE_B8), (t, reverse, line[off + 8].ravel()[:4], TIE_B8)
            for c in range(8):
                assert np.abs(got[c] - ref[c]).max() <= tol * 2.0, (c, t, reverse)


@pytest.mark.parametrize("prec,tol", [("f64", 1e-12), ("f32", 1e-5)])
def test_upwind_tie_inside_the_fused_reverse_sweep(B, prec, tol):
    """reverse L_x = B pair then fluid_x in ONE kernel (lrev_x2, the default at these sizes in fp32): the same tie, the
    whole operator against the oracle at the plain per-step tolerance"""
    npdt = np.float32 if prec == "f32" else np.float64
    for shape3, off in (((256, 8, 6), 120), ((512, 4, 4), 249)):
        f = tie_state(0, 1, shape3, npdt, offset=off)
        f[4] = f[4] + 2.0                                    # pressure well above zero with |v| = 1, |B| = 1
        ref = [np.array(a, dtype=np.float64) for a in f]
        oracle.sweep(ref, 5.0 / 3.0, P, 0, True, 0.25)
        s = B.Solver(*shape3, 5.0 / 3.0, prec, P)
        s.set_state(f)
        s.apply(B.MHD_OP_SWEEP_REVERSE, 0, 0, 0.25)
        got = [np.asarray(a, dtype=np.float64) for a in s.get_state()]
        s.close()
        for c in range(8):
            scale = max(1.0, float(np.abs(ref[c]).max()))
            assert np.abs(got[c] - ref[c]).max() <= tol * scale, (shape3, c)
