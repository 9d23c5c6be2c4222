"""Whole-grid parity at BASELINE.json's full sizes (-m gpu): every cell of one 512^3 step of c4 (fp32) and c5 (fp64).

Kept in a file that pytest collects after all other parity tests (and before tests/test_zz_no_alloc.py): it is the
longest test and the one that handles the most memory, and under `pytest -x` a failure here must not hide the
operator-level parity tests.  The sampled twin, tests/test_gpu_fullsize.py, stays the fast one.

Stream note: the solver works on its own (non-blocking) stream, torch on its default stream.  Every hand-over between the
two below is fenced with torch.cuda.synchronize(); a first version that cloned the pre-step state on torch's stream
without such a fence once compared garbage when run after the other full-size tests in the same process.
"""
import numpy as np
import pytest

import oracle
from paper_0908_4362_b200 import inputs
from tests.parity_utils import GROUPS, fp32_step_gate
from tests.test_gpu_fullsize import CASES, H, TOL, W, _gather

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("name,gen,n,prec", [c for c in CASES if c[0] != "c3"])      # c3 whole-grid: tests/test_gpu_workloads.py
def test_full_size_whole_grid_parity(name, gen, n, prec):
    """EVERY cell of one step at BASELINE.json's full size ("per-step parity at full size on every
    config"): c4 = 512^3 fp32, c5 = 512^3 fp64, 8 x 134 M values each, in the launch configuration bench.py times
    (caller-owned workspace and stream).  The step compared is the second one (step index 1, sweep order z, x, y), taken
    from the GPU's own state after its first step, with the GPU's dt; the oracle (OpenMP, about 20 s for a 512^3 step)
    advances oracle<double> from that same state.  Plain tolerances, no gate; the worst cell is reported with its place."""
    import torch
    from paper_0908_4362_b200 import binding as B
    assert torch.cuda.is_available()
    dev = "cuda:0"
    f, meta = inputs.turbulence(n, xp=torch, xp_kw={"device": dev})
    tdt = torch.float32 if prec == "f32" else torch.float64
    state = [a.to(tdt).contiguous() for a in f]
    del f
    torch.cuda.empty_cache()
    gamma = meta["gamma"]
    ws = torch.empty(B.mhd_workspace_bytes(n, n, n, B.MHD_F32 if prec == "f32" else B.MHD_F64), dtype=torch.uint8, device=dev)
    ws.fill_(0xFF)                                                # the library must not depend on what the workspace held (NaN patterns)
    stream = torch.cuda.Stream(device=dev)
    sol = B.Solver(n, n, n, gamma, prec, meta["bc"], workspace=ws, stream=stream)
    torch.cuda.synchronize()
    sol.set_state(state)
    sol.step(1, 0.8)                                              # step index 0, on the GPU alone
    assert sol.step_index == 1
    dt, _ = sol.cfl_dt(0.8)
    sol.get_state(state)
    ref = [a.double().cpu().numpy() for a in state]               # the run-precision state, widened
    pre = [a.clone() for a in state] if prec == "f32" else None   # kept on the device for the near-tie blocks below
    torch.cuda.synchronize()                                      # torch's stream is not the solver's: finish the clones before `state` is rewritten
    l0 = sol.launch_count()
    sol.step_fixed(1, dt)
    assert sol.launch_count() - l0 >= 6
    sol.get_state(state)
    sol.close()
    torch.cuda.synchronize()
    del ws
    oracle.step_fixed(ref, gamma, meta["bc"], 1, dt)
    tol = TOL[prec]
    report, scale, above = {}, {}, []
    for g, idx in GROUPS.items():
        scale[g] = max(float(np.abs(ref[i]).max()) for i in idx)
        worst = (0.0, None, None)
        n_above = 0
        for i in idx:
            e = np.abs(state[i].double().cpu().numpy() - ref[i])
            w = int(e.argmax())
            hit = np.argwhere(e > tol * scale[g])
            n_above += len(hit)
            above += [tuple(int(v) for v in h) for h in hit[:4096]]
            if e.flat[w] / scale[g] >= worst[0]:
                worst = (float(e.flat[w] / scale[g]), i, tuple(int(v) for v in np.unravel_index(w, e.shape)))
            del e
        report[g] = worst + (n_above,)
    print(f"{name} {n}^3 {prec}, whole grid, step index 1: per group (worst relative error, field, (k, j, i), cells above {tol:g}): {report}")
    del ref
    n_above = sum(w[3] for w in report.values())
    if prec == "f64":
        assert n_above == 0, (name, report)
        return
    # fp32.  Near-ties of the upwind switch (eq (21); R15): where the exact face velocity is below
    # the fp32 rounding of its own evaluation (|vh| < ~1e-7 |vg|), fp32 and fp64 take different arms, and even on smooth
    # data the two second-order fluxes differ by O(h^2 w'') dt, a few 1e-5 here.  With 1.6e9 switch evaluations per step a
    # dozen such cells are expected at 512^3 (none in a 24^3 sample).  They are NOT waved through: at most one cell in ten
    # million, each below 1e-4, and each must pass the location-matched witness gate of tests/parity_utils.py on the block
    # around it (the oracle itself, in fp32 and from inputs moved by half an ulp, must be off next to that very cell).
    assert n_above <= 1e-7 * 8 * n ** 3, (name, report)
    assert max(w[0] for w in report.values()) <= 1e-4, (name, report)
    done = []
    for c in above:
        if any(all(abs(c[a] - d[a]) < W // 2 - 2 for a in range(3)) for d in done):
            continue                                              # already inside the core of a block that passed
        done.append(c)
        lo = [c[a] - W // 2 for a in range(3)]
        blk = _gather(pre, [l - H for l in lo], n)
        got = _gather(state, [l - H for l in lo], n)
        errs = fp32_step_gate(got, blk, gamma, inputs.OUTFLOW, 1, dt, core=(slice(H, H + W),) * 3, scale=scale, tol=tol,
                              tag=f"{name} whole-grid cell {c}")
        assert max(errs.values()) > tol                           # the block does contain the cell that sent us here
    print(f"{name}: {n_above} cells above {tol:g} in {len(done)} blocks, every one next to a cell where the oracle's own fp32 witnesses are off")
