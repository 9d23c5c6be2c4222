"""GPU parity at BASELINE.json's FULL sizes (configs[2..4]: 256^3 fp32 blast, 512^3 fp32 / fp64 turbulence),
in the launch configuration bench.py times (torch workspace + stream, default options)  (-m gpu).

The oracle cannot advance 512^3 in seconds, so the outputs are SAMPLED: one step of the whole hot path
depends, at any cell, only on the cells within R = 18 of it along each axis (per L_d: 3 (fluid) + 4 (B pair)
along d and 1 transverse; every axis is swept twice and is transverse four times: 2*7 + 4*1).  For each
sample box the test gathers the pre-step state on the box widened by H = 20 > R cells (wrapped through the
periodic boundary), advances that 64^3 block with the oracle (outflow rule at the block's own edge, which
cannot reach the interior), and compares the interior 24^3 cells element by element with the GPU result.
Boxes sit on the domain corner (wrap), on the kernels' x-tile and march-segment seams, and at seeded random
places.  The c_max reduction is compared over the WHOLE grid (the oracle's cmax is a single cheap pass).
All three step rotations s = 0, 1, 2 are checked, each from the GPU's own current state with the same dt.
"""
import numpy as np
import pytest

import oracle
from paper_0908_4362_b200 import inputs
from tests.parity_utils import GROUPS, fp32_step_gate

pytestmark = pytest.mark.gpu

H, W = 20, 24            # halo > domain of dependence of one step (18), interior width of a sample box
TOL = {"f64": 1e-12, "f32": 1e-5}

CASES = [
    # name, generator, n, precision
    ("c3", "blast3d", 256, "f32"),
    ("c4", "turbulence", 512, "f32"),
    ("c5", "turbulence", 512, "f64"),
]


def _gather(fields, lo, n):
    """the (W+2H)^3 block whose low corner is lo (z,y,x), wrapped periodically, as float64 numpy arrays"""
    import torch
    side = W + 2 * H
    idx = [torch.remainder(torch.arange(l, l + side, device=fields[0].device), n) for l in lo]
    out = []
    for f in fields:
        b = f.index_select(0, idx[0]).index_select(1, idx[1]).index_select(2, idx[2])
        out.append(np.ascontiguousarray(b.double().cpu().numpy()))
    return out


def _boxes(name, n, rng):
    """low corners (z,y,x) of the INTERIOR of the sample boxes"""
    c = n // 2
    seams = [
        (-W // 2, -W // 2, -W // 2),                    # the domain corner: every wrap at once
        (c - W // 2, c - W // 2, c - W // 2),           # domain centre: x-tile seam (256) and 2-segment march seams
        (n // 4 - W // 2, 3 * n // 4 - W // 2, n // 2 - W // 2),
        (3 * n // 4 - W // 2, n // 4 - W // 2, 128 - W // 2),   # 128-wide tile seam (fp64 kernels)
        (n - W, 171 - W // 2, 341 % n - W // 2),        # last cells along z; 3-segment seams (n/3)
        (171 % n - W // 2, n - W, n - W),
    ]
    if name == "c3":                                     # the pressure jump at r = 0.1 * 256 = 25.6 cells
        seams += [(c - W // 2, c - W // 2, c + 26 - W // 2), (c + 18 - W // 2, c + 18 - W // 2, c - W // 2)]
    rnd = [tuple(int(v) for v in rng.integers(0, n, 3)) for _ in range(4)]
    return seams + rnd


@pytest.mark.parametrize("name,gen,n,prec", CASES)
def test_full_size_sampled_parity(name, gen, n, prec):
    import torch
    from paper_0908_4362_b200 import binding as B
    assert torch.cuda.is_available()
    dev = "cuda:0"
    kw = dict(xp=torch, xp_kw={"device": dev})
    f, meta = (inputs.turbulence(n, **kw) if gen == "turbulence" else inputs.blast3d(n, **kw))
    tdt = torch.float32 if prec == "f32" else torch.float64
    state = [a.to(tdt).contiguous() for a in f]
    del f
    torch.cuda.empty_cache()
    gamma = meta["gamma"]
    ws = torch.empty(B.mhd_workspace_bytes(n, n, n, B.MHD_F32 if prec == "f32" else B.MHD_F64), dtype=torch.uint8, device=dev)
    stream = torch.cuda.Stream(device=dev)
    sol = B.Solver(n, n, n, gamma, prec, meta["bc"], workspace=ws, stream=stream)
    torch.cuda.synchronize()
    sol.set_state(state)
    after = [torch.empty_like(a) for a in state]
    rng = np.random.default_rng(4362)

    # c_max over the whole grid (eq (18)) against the oracle's single pass
    dt, cm = sol.cfl_dt(0.8)
    host = [a.cpu().numpy() for a in state]
    cm_ref = oracle.cmax(host, gamma, meta["bc"])
    del host
    assert abs(cm - cm_ref) <= (1e-14 if prec == "f64" else 5e-6) * cm_ref, (cm, cm_ref)

    worst = {g: 0.0 for g in GROUPS}
    for k in range(3):
        dt, _ = sol.cfl_dt(0.8)
        l0 = sol.launch_count()
        sol.step_fixed(1, dt)
        assert sol.launch_count() - l0 >= 6             # six L_i, all on the device
        sol.get_state(after)
        scale = {g: max(float(after[i].abs().max()) for i in idx) for g, idx in GROUPS.items()}
        for lo in _boxes(name, n, rng):
            blk = _gather(state, [l - H for l in lo], n)
            got = _gather(after, [l - H for l in lo], n)
            core = (slice(H, H + W),) * 3
            if prec == "f32":           # plain 1e-5, or the tie-aware gate of tests/parity_utils.py where the oracle itself is that sensitive
                errs = fp32_step_gate(got, blk, gamma, inputs.OUTFLOW, k, dt, core=core, scale=scale, tol=TOL[prec], tag=f"{name} box {lo}")
                if name != "c3":        # smooth data: no exact ties, the plain tolerance holds everywhere
                    assert max(errs.values()) <= TOL[prec], (name, k, lo, errs)
                for g in GROUPS:
                    worst[g] = max(worst[g], errs[g])
                continue
            oracle.step_fixed(blk, gamma, inputs.OUTFLOW, k, dt)
            for g, idx in GROUPS.items():
                err = max(float(np.abs(got[i][core] - blk[i][core]).max()) for i in idx)
                worst[g] = max(worst[g], err / scale[g])
                assert err <= TOL[prec] * scale[g], (name, k, lo, g, err / scale[g])
        state, after = after, state
    sol.close()
    print(name, prec, "worst max-rel per group over 3 steps:", worst)


def _gather3(fields, lo, dims):
    """as _gather for a non-cubic grid: dims = (nz, ny, nx)"""
    import torch
    side = W + 2 * H
    idx = [torch.remainder(torch.arange(l, l + side, device=fields[0].device), n) for l, n in zip(lo, dims)]
    out = []
    for f in fields:
        b = f.index_select(0, idx[0]).index_select(1, idx[1]).index_select(2, idx[2])
        out.append(np.ascontiguousarray(b.double().cpu().numpy()))
    return out


@pytest.mark.parametrize("nx,ny,nz,prec", [(1024, 256, 192, "f32"),     # rows wider than the x kernels take (generic
                                                                       # march along x), four ring tiles per row
                                           (384, 200, 136, "f32"),      # 128-wide ring tiles, extents that are no
                                           (384, 200, 136, "f64")])     # multiple of the segment or tile sizes
def test_large_non_cubic_sampled_parity(nx, ny, nz, prec):
    """edge cases of the launch geometry at sizes the oracle cannot advance whole: same sampling argument as above"""
    import torch
    from paper_0908_4362_b200 import binding as B
    assert torch.cuda.is_available()
    dev = "cuda:0"
    f, meta = inputs.turbulence(nx, ny, nz, xp=torch, xp_kw={"device": dev})
    tdt = torch.float32 if prec == "f32" else torch.float64
    state = [a.to(tdt).contiguous() for a in f]
    del f
    gamma = meta["gamma"]
    sol = B.Solver(nx, ny, nz, gamma, prec, meta["bc"])
    torch.cuda.synchronize()            # the context has its own stream: torch's generator kernels must be done
    sol.set_state(state)
    after = [torch.empty_like(a) for a in state]
    dims = (nz, ny, nx)
    rng = np.random.default_rng(nx + ny)
    boxes = [(-W // 2, -W // 2, -W // 2), (nz // 2 - W // 2, ny // 2 - W // 2, nx // 2 - W // 2),
             (nz - W, ny - W, nx - W), (7, ny // 3, 256 - W // 2), (nz // 3, 5, 128 - W // 2)]
    boxes += [tuple(int(rng.integers(0, n)) for n in dims) for _ in range(3)]
    for k in range(3):
        dt, cm = sol.cfl_dt(0.8)
        if k == 0:
            cm_ref = oracle.cmax([a.cpu().numpy() for a in state], gamma, meta["bc"])
            assert abs(cm - cm_ref) <= (1e-14 if prec == "f64" else 5e-6) * cm_ref
        sol.step_fixed(1, dt)
        sol.get_state(after)
        scale = {g: max(float(after[i].abs().max()) for i in idx) for g, idx in GROUPS.items()}
        for lo in boxes:
            blk = _gather3(state, [l - H for l in lo], dims)
            oracle.step_fixed(blk, gamma, inputs.OUTFLOW, k, dt)
            got = _gather3(after, [l - H for l in lo], dims)
            core = (slice(H, H + W),) * 3
            for g, idx in GROUPS.items():
                err = max(float(np.abs(got[i][core] - blk[i][core]).max()) for i in idx)
                assert err <= TOL[prec] * scale[g], (nx, ny, nz, prec, k, lo, g, err / scale[g])
        state, after = after, state
    sol.close()
