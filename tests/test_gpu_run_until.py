"""GPU: the device-resident time loop (mhd_run_until) and whole-step CUDA graph replay  (-m gpu).

SURVEY.md 8(f) rank 2: the flow loop of PAPER.md:233-243 with dt, t and the final-step clipping (reading R14) kept on
the device.  Checked three ways: bit for bit against the per-step host loop through mhd_cfl_dt / mhd_step_fixed
(same kernels, same dt arithmetic), against the oracle driven by the same rule, and graph replay against plain
stream launches.
"""
import numpy as np
import pytest

import oracle
from paper_0908_4362_b200 import inputs
from tests.parity_utils import max_rel, random_state, worst

pytestmark = pytest.mark.gpu

P, O = inputs.PERIODIC, inputs.OUTFLOW


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
    dt = np.float32 if prec == "f32" else np.float64
    s.set_state([np.ascontiguousarray(a, dtype=dt) for a in f])
    return s


def _host_loop(s, t_end, cfl):
    """the rule mhd_run_until implements, driven from the host one step at a time"""
    t, k = 0.0, 0
    while t < t_end:
        dt, _ = s.cfl_dt(cfl)
        rem = 0.5 * (t_end - t)
        if dt >= rem:
            dt, t = rem, t_end
        else:
            t += 2.0 * dt
        s.step_fixed(1, dt)
        k += 1
    return k, t


def _oracle_loop(ref, gamma, bc, t_end, cfl):
    t, k = 0.0, 0
    while t < t_end:
        dt = cfl / oracle.cmax(ref, gamma, bc)
        rem = 0.5 * (t_end - t)
        if dt >= rem:
            dt, t = rem, t_end
        else:
            t += 2.0 * dt
        oracle.step_fixed(ref, gamma, bc, k, dt)
        k += 1
    return k, t


@pytest.mark.parametrize("graph", [0, 1])
def test_config1_brio_wu_run_until(B, graph):
    """BASELINE.json configs[0]: 512x1x1 fp64, outflow, cfl 0.8 to t = 0.1 (51.2 in grid units), last step clipped"""
    f, meta = inputs.brio_wu(512)
    t_end = 0.1 * 512
    a = _solver(B, f, meta["gamma"], meta["bc"], "f64", graph=graph)
    n, t = a.run_until(t_end, 0.8)
    got = a.get_state()
    assert a.step_index == n and a.time() == t_end == t
    a.close()
    b = _solver(B, f, meta["gamma"], meta["bc"], "f64", graph=0)
    k, _ = _host_loop(b, t_end, 0.8)
    want = b.get_state()
    b.close()
    assert n == k and 100 < n < 200
    for x, y in zip(got, want):
        assert np.array_equal(x, y)                      # same kernels, same dt: bit for bit
    ref = [np.array(x, dtype=np.float64) for x in f]
    ko, _ = _oracle_loop(ref, meta["gamma"], meta["bc"], t_end, 0.8)
    assert ko == n
    assert worst(max_rel(got, ref)) <= 1e-10             # accumulated over ~143 steps


@pytest.mark.parametrize("prec", ["f32", "f64"])
def test_run_until_3d_against_oracle_and_host_loop(B, prec):
    f, gamma = random_state(32, 16, 24, seed=11), 5.0 / 3.0
    dtp = np.float32 if prec == "f32" else np.float64
    f = [np.asarray(x, dtype=dtp) for x in f]
    a = _solver(B, f, gamma, P, prec)
    dt0, _ = a.cfl_dt(0.8)
    t_end = 2 * dt0 * 7.3                                 # 8 steps, the last one clipped
    n, t = a.run_until(t_end, 0.8)
    got = a.get_state()
    a.close()
    b = _solver(B, f, gamma, P, prec, graph=0)
    k, _ = _host_loop(b, t_end, 0.8)
    want = b.get_state()
    b.close()
    assert n == k and t == t_end
    for x, y in zip(got, want):
        assert np.array_equal(x, y)
    if prec == "f64":
        ref = [np.array(x, dtype=np.float64) for x in f]
        ko, _ = _oracle_loop(ref, gamma, P, t_end, 0.8)
        assert ko == n
        assert worst(max_rel(got, ref)) <= 20 * 1e-12


def test_run_until_limits_and_resume(B):
    f, gamma = random_state(32, 16, 1, seed=5), 5.0 / 3.0
    a = _solver(B, f, gamma, O, "f64")
    dt0, _ = a.cfl_dt(0.7)
    t_end = 2 * dt0 * 30
    n1, t1 = a.run_until(t_end, 0.7, max_steps=4)         # stops on the step budget
    assert n1 == 4 and 0.0 < t1 < t_end and a.step_index == 4
    n0, t0 = a.run_until(t1, 0.7)                         # already there: nothing happens
    assert n0 == 0 and t0 == t1 and a.step_index == 4
    n2, t2 = a.run_until(t_end, 0.7)                      # resumes with the right sweep order (step index 4)
    got = a.get_state()
    a.close()
    assert t2 == t_end
    b = _solver(B, f, gamma, O, "f64", graph=0)
    k, _ = _host_loop(b, t_end, 0.7)
    want = b.get_state()
    b.close()
    assert n1 + n2 == k
    for x, y in zip(got, want):
        assert np.array_equal(x, y)
    with pytest.raises(B.MHDError):
        c = _solver(B, f, gamma, O, "f64")
        try:
            c.run_until(1.0, -1.0)
        finally:
            c.close()


@pytest.mark.parametrize("shape,bc,prec", [((64, 16, 16), P, "f32"), ((128, 12, 10), P, "f32"), ((40, 24, 20), O, "f64"),
                                           ((48, 1, 1), O, "f64"), ((64, 32, 1), P, "f64")])
def test_graph_replay_is_bitwise_the_stream_path(B, shape, bc, prec):
    f, gamma = random_state(*shape, seed=3), 5.0 / 3.0
    dtp = np.float32 if prec == "f32" else np.float64
    f = [np.asarray(x, dtype=dtp) for x in f]
    outs = []
    for graph in (0, 1):
        s = _solver(B, f, gamma, bc, prec, graph=graph)
        t1 = s.step(7, 0.8)                               # all three rotations, twice: graphs are captured, then replayed
        s.apply(B.MHD_OP_FLUID, 1 if shape[1] > 1 else 0, 0, 0.01)   # leaves the ping-pong pointers swapped
        t2 = s.step(4, 0.6)                               # other cfl, other pointers: must re-capture, not replay
        outs.append((s.get_state(), t1, t2, s.step_index, s.launch_count()))
        s.close()
    (g0, ta0, tb0, i0, l0), (g1, ta1, tb1, i1, l1) = outs
    assert ta0 == ta1 and tb0 == tb1 and i0 == i1 == 11 and l0 == l1
    for x, y in zip(g0, g1):
        assert np.array_equal(x, y)


@pytest.mark.parametrize("prec", ["f32", "f64"])
def test_small_grid_bound_to_the_default_stream(B, prec):
    """mhd_bind(workspace, NULL stream): the legacy default stream cannot be captured, so a small grid (where steps are
    otherwise replayed as CUDA graphs) must launch its kernels directly; same bits as graph = 0 on an own stream"""
    import torch
    shape = (64, 16, 16)
    f = [np.asarray(x, dtype=np.float32 if prec == "f32" else np.float64) for x in random_state(*shape, seed=5)]
    ws = torch.empty(B.mhd_workspace_bytes(*shape, B.MHD_F32 if prec == "f32" else B.MHD_F64), dtype=torch.uint8, device="cuda")
    a = B.Solver(*shape, 1.4, prec, P, workspace=ws)          # no stream: binds NULL
    a.set_state(f)
    ta = a.step(3, 0.8)
    ra, sa = a.run_until(ta + 2.0, 0.8)
    ga = a.get_state()
    a.close()
    b = _solver(B, f, 1.4, P, prec, graph=0)
    tb = b.step(3, 0.8)
    rb, sb = b.run_until(tb + 2.0, 0.8)
    gb = b.get_state()
    b.close()
    assert ta == tb and ra == rb and sa == sb
    for x, y in zip(ga, gb):
        assert np.array_equal(x, y)


@pytest.mark.parametrize("shape,prec", [((256, 64, 1), "f32"), ((256, 64, 1), "f64"), ((128, 16, 40), "f32"),
                                        ((128, 40, 16), "f64"), ((512, 1, 1), "f64")])
@pytest.mark.parametrize("bc", [P, O])
def test_small_grid_short_segments(B, shape, prec, bc):
    """small grids are cut into segments as short as 8 cells to fill the machine: same bits as whole pencils, and
    within the per-step tolerance of the oracle"""
    f = random_state(*shape, seed=21)
    gamma = 1.4
    dtp = np.float32 if prec == "f32" else np.float64
    f = [np.asarray(x, dtype=dtp) for x in f]
    outs = []
    for seg in (-1, 0, 8):
        s = _solver(B, f, gamma, bc, prec, segment=seg, graph=0)
        dt0, _ = s.cfl_dt(0.8)
        s.step_fixed(3, dt0)
        outs.append(s.get_state())
        s.close()
    for other in outs[1:]:
        for x, y in zip(outs[0], other):
            assert np.array_equal(x, y)
    ref = [np.array(x, dtype=np.float64) for x in f]
    for k in range(3):
        oracle.step_fixed(ref, gamma, bc, k, dt0)
    assert worst(max_rel(outs[0], ref)) <= (3e-12 if prec == "f64" else 3e-5)
