"""CPU check of the sampling argument of tests/test_gpu_fullsize.py (not a GPU test)."""
import numpy as np

import oracle
from paper_0908_4362_b200 import inputs
from tests.test_gpu_fullsize import H, W


def test_dependence_radius_of_one_step_is_inside_the_halo():
    """the sampling argument above, checked on the oracle itself: perturbing cells farther than H from a box
    does not change the box (so an outflow edge H cells away cannot either)"""
    f, meta = inputs.turbulence(64, 64, 64)
    a = [x.copy() for x in f]
    b = [x.copy() for x in f]
    lo, hi = 32 - W // 4, 32 + W // 4
    far = np.ones((64, 64, 64), bool)
    far[lo - H:hi + H, lo - H:hi + H, lo - H:hi + H] = False
    rng = np.random.default_rng(1)
    for x in b:                                    # all eight fields: B has the longer reach (faces to n+4 in fluid_d, +1 row in the B pair)
        x[far] *= 1.0 + 0.05 * rng.random(int(far.sum()))
    for k in range(3):
        dt = 0.8 / oracle.cmax(a, meta["gamma"], meta["bc"])
        oracle.step_fixed(a, meta["gamma"], meta["bc"], k, dt)
        oracle.step_fixed(b, meta["gamma"], meta["bc"], k, dt)
        for x, y in zip(a, b):
            assert np.array_equal(x[lo:hi, lo:hi, lo:hi], y[lo:hi, lo:hi, lo:hi])
        # re-synchronise the far field so every step starts from 'same box, different far field'
        b = [x.copy() for x in a]
        for x in b:
            x[far] *= 1.0 + 0.05 * rng.random(int(far.sum()))
