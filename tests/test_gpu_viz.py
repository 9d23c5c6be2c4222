"""GPU parity of the headless visualisation stage (section 8): the CUDA kernels
behind mhd_viz_* against oracle/viz.py, byte for byte / bit for bit (-m gpu).  include/mhd.h fixes the arithmetic."""
import numpy as np
import pytest

from oracle import viz
from paper_0908_4362_b200 import inputs
from tests.parity_utils import random_state

pytestmark = pytest.mark.gpu
P, O = inputs.PERIODIC, inputs.OUTFLOW


@pytest.fixture(scope="module")
def env():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_0908_4362_b200 import binding
    return binding, torch


def _lut(seed):
    rng = np.random.default_rng(seed)
    lut = rng.integers(0, 256, size=(256, 4), dtype=np.uint8)
    lut[:, 3] = np.clip(rng.integers(0, 90, size=256), 0, 255)        # mostly translucent
    lut[::37, 3] = 255                                                  # a few opaque entries: early termination
    return lut


@pytest.mark.parametrize("shape", [(40, 24, 20), (37, 5, 3), (512, 1, 1), (64, 33, 1), (16, 16, 70)])
@pytest.mark.parametrize("prec", ["f32", "f64"])
@pytest.mark.parametrize("bc", [P, O])
def test_viz_matches_oracle_exactly(env, shape, prec, bc):
    B, torch = env
    nx, ny, nz = shape
    gamma = 5.0 / 3.0
    dtp = np.float32 if prec == "f32" else np.float64
    f = [np.ascontiguousarray(a, dtype=dtp) for a in random_state(nx, ny, nz, seed=nx + 3 * ny + nz)]
    s = B.Solver(nx, ny, nz, gamma, prec, bc)
    s.set_state(f)
    lut = _lut(nx)
    lut_d = torch.from_numpy(lut).cuda()
    for field in (0, 4, 6, B.MHD_VIZ_PRESSURE):
        lo, hi = s.viz_range(field)
        assert (lo, hi) == viz.value_range(f, field, gamma, bc)
        j, k = ny // 2, nz - 1
        xy = torch.empty((nx, 2), dtype=torch.float32, device="cuda")
        s.viz_curve(field, j, k, lo, hi, xy)
        rgba = torch.empty((ny, nx, 4), dtype=torch.uint8, device="cuda")
        s.viz_slice(field, k, lo, hi, lut_d, rgba)
        vol = torch.empty((ny, nx, 4), dtype=torch.uint8, device="cuda")
        s.viz_volume(field, lo + 0.1 * (hi - lo), hi - 0.2 * (hi - lo), lut_d, 0.35, vol)     # clamps on both sides
        torch.cuda.synchronize()
        want_xy = viz.curve(f, field, gamma, bc, j, k, lo, hi)
        assert np.array_equal(xy.cpu().numpy().view(np.uint32), want_xy.view(np.uint32))          # bit for bit
        assert np.array_equal(rgba.cpu().numpy(), viz.slice_rgba(f, field, gamma, bc, k, lo, hi, lut))
        assert np.array_equal(vol.cpu().numpy(),
                              viz.volume_rgba(f, field, gamma, bc, lo + 0.1 * (hi - lo), hi - 0.2 * (hi - lo), lut, 0.35))
    s.close()


def test_viz_follows_the_state_and_edge_cases(env):
    B, torch = env
    f, meta = inputs.orszag_tang(64)
    s = B.Solver(64, 64, 1, meta["gamma"], "f32", meta["bc"])
    st = [np.ascontiguousarray(a, dtype=np.float32) for a in f]
    s.set_state(st)
    lut = _lut(1)
    lut_d = torch.from_numpy(lut).cuda()
    img = torch.empty((64, 64, 4), dtype=torch.uint8, device="cuda")
    s.step(5, 0.8)                                                       # the stage reads the CURRENT state in place
    now = s.get_state()
    lo, hi = s.viz_range(B.MHD_VIZ_PRESSURE)
    s.viz_slice(B.MHD_VIZ_PRESSURE, 0, lo, hi, lut_d, img)
    torch.cuda.synchronize()
    assert np.array_equal(img.cpu().numpy(), viz.slice_rgba(now, viz.PRESSURE, meta["gamma"], meta["bc"], 0, lo, hi, lut))
    # a NaN cell is skipped by the range and drawn with lut[0]
    st[1][0, 3, 5] = np.nan                                                # (the Orszag-Tang density is uniform: use m_x)
    s.set_state(st)
    lo, hi = s.viz_range(1)
    assert np.isfinite(lo) and np.isfinite(hi) and (lo, hi) == viz.value_range(st, 1, meta["gamma"], meta["bc"])
    s.viz_slice(1, 0, lo, hi, lut_d, img)
    torch.cuda.synchronize()
    assert tuple(img.cpu().numpy()[3, 5]) == tuple(lut[0])
    # +-Inf cells are skipped by the range as well (mhd.h: smallest and largest FINITE value)
    st[1][0, 7, 9] = np.inf
    st[1][0, 8, 2] = -np.inf
    s.set_state(st)
    lo2, hi2 = s.viz_range(1)
    assert (lo2, hi2) == (lo, hi) == viz.value_range(st, 1, meta["gamma"], meta["bc"])
    # argument errors
    for bad in (lambda: s.viz_slice(9, 0, 0.0, 1.0, lut_d, img), lambda: s.viz_slice(0, 1, 0.0, 1.0, lut_d, img),
                lambda: s.viz_slice(0, 0, 1.0, 1.0, lut_d, img), lambda: s.viz_volume(0, 0.0, 1.0, lut_d, 0.0, img),
                lambda: s.viz_curve(0, 64, 0, 0.0, 1.0, img)):
        with pytest.raises(B.MHDError):
            bad()
    s.close()
    e = B.Solver(16, 16, 1, 1.4, "f32", 0)
    with pytest.raises(B.MHDError):
        e.viz_range(0)                                                   # no state yet
    e.close()
