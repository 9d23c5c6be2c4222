"""The fp32 per-step gate of tests/parity_utils.py, tested on the CPU with a stand-in for the GPU result (-m "not gpu").

The gate excuses cells above 1e-5 only NEXT TO cells where the oracle itself is that sensitive (exact ties of the upwind
switch, eq (21), R15).  Two things are shown on a small 3-D blast wave after a few steps, where
such ties exist: an honest fp32 evaluation with a different rounding order passes, and the same result with a seam-like
defect (a plane of cells off by 1e-3, away from the ties) fails even though its size and count would fit under the
witnesses' maxima."""
import numpy as np
import pytest

import oracle
from paper_0908_4362_b200 import inputs
from tests.parity_utils import GROUPS, fp32_step_gate


def _blast_after(nsteps, n=40):
    f, meta = inputs.blast3d(n)
    cur = [np.array(np.asarray(a, dtype=np.float32), dtype=np.float64) for a in f]
    for k in range(nsteps):
        dt = 0.8 / oracle.cmax(cur, meta["gamma"], meta["bc"])
        oracle.step_fixed(cur, meta["gamma"], meta["bc"], k, dt)
        cur = [np.array(a.astype(np.float32), dtype=np.float64) for a in cur]      # an fp32 state, as the GPU would hold
    return cur, meta, nsteps


def _standin(before, meta, k, dt):
    """an fp32 evaluation that is not the witness: oracle<float> from inputs moved by one fp32 ulp pattern"""
    rng = np.random.default_rng(99)
    b = [np.array(a * (1.0 + 6e-8 * rng.choice([-1.0, 1.0], size=a.shape)), dtype=np.float32, order="C") for a in before]
    oracle.step_fixed(b, meta["gamma"], meta["bc"], k, dt)
    return [a.astype(np.float64) for a in b]


def test_gate_excuses_ties_by_location_only(capsys):
    before, meta, k = _blast_after(1, n=96)
    dt = 0.8 / oracle.cmax(before, meta["gamma"], meta["bc"])
    got = _standin(before, meta, k, dt)
    errs = fp32_step_gate(got, before, meta["gamma"], meta["bc"], k, dt, tag="stand-in")
    shown = capsys.readouterr().out
    if max(errs.values()) <= 1e-5:
        pytest.skip("no tie on this box: nothing to excuse")           # keeps the test honest if the inputs change
    assert "fp32 tie gate" in shown
    # a seam: one x-plane of B_y cells off by 1e-3 of the group scale, two cells thick, far from the symmetry planes
    ref = [a.copy() for a in before]
    oracle.step_fixed(ref, meta["gamma"], meta["bc"], k, dt)
    scale = max(float(np.abs(ref[i]).max()) for i in GROUPS["B"])
    bad = [a.copy() for a in got]
    n = bad[6].shape[2]
    bad[6][2:6, 2:8, n - 5:n - 3] += 1e-3 * scale                     # 48 cells in a corner of the box
    with pytest.raises(AssertionError):
        fp32_step_gate(bad, before, meta["gamma"], meta["bc"], k, dt, tag="seam")
