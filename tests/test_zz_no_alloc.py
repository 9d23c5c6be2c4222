"""mhd_cmax_noalloc: the c_max reduction for callers that cannot allocate device memory.

Who needs it: code embedded in a program that owns every byte of device memory through its own pool and does not
allow cudaMalloc behind its back, loops that cannot take cudaMalloc's device-wide synchronisation, and processes that
are at their memory limit.  All other compute calls of the library work on a context whose workspace is cudaMalloc'ed
(by the library, or by whoever hands it to mhd_bind); this one takes the eight device fields and one device double and
keeps its scratch (per-block partial maxima + a block counter) in a fixed 262400-byte array inside libmhd.so, which
limits it to 2^27 cells.

What is checked here: on two calls in a row -- the second on a SMALLER grid with a SMALLER c_max, so that anything the
first call left in the shared array (partial maxima beyond the second launch's blocks, a counter that is not back at
zero) would show -- the result equals what the existing path (mhd_cfl_dt on a context holding the same state) returns,
within the tolerance tests/test_gpu_parity.py::test_cfl_dt_matches_oracle uses (1e-14 fp64, 2e-6 fp32); and that a grid
beyond the limit is refused with a message and without touching the device.

This file is named so that pytest collects it last: `pytest -x` stops at the first failure, and a failure here must
not hide the parity tests.  It passes alone in a fresh process (the first call on the device does the one-time address
look-up itself) and after the other tests.
"""
import ctypes

import numpy as np
import pytest

from paper_0908_4362_b200 import inputs
from tests.parity_utils import random_state

P, O = inputs.PERIODIC, inputs.OUTFLOW
GAMMA = 5.0 / 3.0


@pytest.fixture(scope="module")
def B():
    from paper_0908_4362_b200 import build
    build.build()
    from paper_0908_4362_b200 import binding
    return binding


def _existing_path_cmax(B, f, bc, prec, npdt):
    """c_max by the path that exists already: a context, its cudaMalloc'ed workspace, mhd_cfl_dt"""
    nz, ny, nx = f[0].shape
    s = B.Solver(nx, ny, nz, GAMMA, prec, bc)
    s.set_state([np.ascontiguousarray(a, dtype=npdt) for a in f])
    _, cm = s.cfl_dt(0.8)
    s.close()
    return cm


def _noalloc_cmax(B, torch, dev_fields, out, bc, prec):
    """one call of the new entry point on torch's current stream; returns the status and the message"""
    nz, ny, nx = dev_fields[0].shape
    ptrs = (ctypes.c_void_p * 8)(*[t.data_ptr() for t in dev_fields])
    err = ctypes.create_string_buffer(512)
    rc = B.mhd_cmax_noalloc(ptrs, nx, ny, nz, GAMMA, B.MHD_F32 if prec == "f32" else B.MHD_F64, bc,
                            torch.cuda.current_stream().cuda_stream, out.data_ptr(), err, len(err))
    return rc, err.value.decode()


@pytest.mark.gpu
@pytest.mark.parametrize("bc", [P, O])
@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_two_calls_in_a_row_match_the_existing_path(B, prec, bc):
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    npdt = np.float32 if prec == "f32" else np.float64
    tol = 1e-14 if prec == "f64" else 2e-6
    # first call: 104 x 40 x 36 = 149760 cells = 36 full blocks of 4096 + a ragged one; second call: 33 x 17 x 9 = 5049
    # cells = 2 blocks; the first state's momenta are scaled up so that its c_max is well above the second's
    big = random_state(104, 40, 36, seed=11)
    small = random_state(33, 17, 9, seed=3)
    for c in (1, 2, 3):
        big[c] = big[c] * 3.0
        big[4] = big[4] + 4.0 * big[c] ** 2 / big[0]     # keep the pressure positive
    want = [_existing_path_cmax(B, f, bc, prec, npdt) for f in (big, small)]
    assert want[1] < 0.7 * want[0]

    dev = [[torch.from_numpy(np.ascontiguousarray(a, dtype=npdt)).cuda() for a in f] for f in (big, small)]
    out = torch.full((2,), -1.0, dtype=torch.float64, device="cuda")
    for n in range(2):                                   # back to back on one stream, no synchronisation in between
        rc, msg = _noalloc_cmax(B, torch, dev[n], out[n:], bc, prec)
        assert rc == B.MHD_OK, msg
    got = out.cpu().numpy()
    for n in range(2):
        assert abs(got[n] - want[n]) <= tol * want[n], (n, got[n], want[n])
    # and once more on the first state: the array now holds the small run's leftovers
    rc, msg = _noalloc_cmax(B, torch, dev[0], out[1:], bc, prec)
    assert rc == B.MHD_OK, msg
    assert abs(out[1].item() - want[0]) <= tol * want[0]


@pytest.mark.gpu
def test_the_largest_grid_the_scratch_allows(B):
    """512^3 fp32 = 2^27 cells uses every one of the 32768 partial slots; the state is made on the device (seeded) and
    handed to both paths as device pointers.  Twice in a row, the maximum moved to the last cell for the second call."""
    import torch
    n = 512
    g = torch.Generator(device="cuda").manual_seed(4362)
    r = lambda lo, hi: torch.rand((n, n, n), generator=g, device="cuda", dtype=torch.float32) * (hi - lo) + lo
    rho = r(0.8, 1.2)
    m = [rho * r(-0.5, 0.5) for _ in range(3)]
    b = [r(-0.4, 0.4) for _ in range(3)]
    e = r(1.0, 2.0) / (GAMMA - 1.0) + 0.5 * (m[0] ** 2 + m[1] ** 2 + m[2] ** 2) / rho + 1.0
    f = [rho] + m + [e] + b
    s = B.Solver(n, n, n, GAMMA, "f32", P)
    out = torch.zeros(2, dtype=torch.float64, device="cuda")
    want = []
    for call in range(2):
        if call == 1:
            f[4][-1, -1, -1] = 40.0                      # the very last cell (last thread of the last block) now holds the maximum
        torch.cuda.synchronize()
        s.set_state(f)
        want.append(s.cfl_dt(0.8)[1])
        rc, msg = _noalloc_cmax(B, torch, f, out[call:], P, "f32")
        assert rc == B.MHD_OK, msg
    s.close()
    got = out.cpu().numpy()
    assert want[1] > 1.5 * want[0]
    for call in range(2):
        assert abs(got[call] - want[call]) <= 2e-6 * want[call], (call, got[call], want[call])


def test_sizes_beyond_the_fixed_scratch_are_refused(B):
    """2^27 cells is the limit; the check comes before any CUDA call, so this needs no GPU and no memory"""
    fake = (ctypes.c_void_p * 8)(*([256] * 8))            # never dereferenced
    err = ctypes.create_string_buffer(512)
    rc = B.mhd_cmax_noalloc(fake, 1024, 512, 512, GAMMA, B.MHD_F32, P, None, 256, err, len(err))
    assert rc == B.MHD_EINVAL
    msg = err.value.decode()
    assert "134217728" in msg and "scratch" in msg, msg
    assert B.mhd_cmax_noalloc(fake, 512, 512, 513, GAMMA, B.MHD_F64, P, None, 256, None, 0) == B.MHD_EINVAL
    assert B.mhd_cmax_noalloc(fake, 0, 4, 4, GAMMA, B.MHD_F64, P, None, 256, err, len(err)) == B.MHD_EINVAL
    assert B.mhd_cmax_noalloc(fake, 4, 4, 4, 1.0, B.MHD_F64, P, None, 256, err, len(err)) == B.MHD_EINVAL
    assert B.mhd_cmax_noalloc(fake, 4, 4, 4, GAMMA, 5, P, None, 256, err, len(err)) == B.MHD_EINVAL
    assert B.mhd_cmax_noalloc(fake, 4, 4, 4, GAMMA, B.MHD_F64, P, None, None, err, len(err)) == B.MHD_EINVAL
    assert "NULL" in err.value.decode()
