"""Writes the regression fixtures of this folder.  Calls ONLY oracle/ (never the CUDA path):

    python tests/golden/make_golden.py

oracle_tiny_state.txt: the oracle's fp64 state after three steps (all three sweep rotations, dt = 0.17) from the seeded
state tests/parity_utils.random_state(6, 4, 3, seed=4362), for both boundary rules, as C99 hex floats (exact bits).
The paper prints no numerical field values (README.md), so this is not a pin of the oracle to the paper: it guards
the oracle against unintended edits -- tests/test_oracle_pins.py::test_oracle_regression_fixture must reproduce it bit
for bit, and a deliberate change to the oracle's arithmetic has to regenerate it in the same commit that names the
passage of PAPER.md justifying the change."""
import os
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np

import oracle
from tests.parity_utils import random_state

SHAPE, SEED, DT, GAMMA = (6, 4, 3), 4362, 0.17, 5.0 / 3.0


def tiny_state(bc):
    f = [np.array(a, dtype=np.float64, order="C") for a in random_state(*SHAPE, seed=SEED)]
    for s in range(3):
        oracle.step_fixed(f, GAMMA, bc, s, DT)
    return f


def main():
    with open(os.path.join(HERE, "oracle_tiny_state.txt"), "w") as out:
        out.write("# written by tests/golden/make_golden.py (oracle only); bc field values...\n")
        for bc in (0, 1):
            for i, a in enumerate(tiny_state(bc)):
                out.write(f"{bc} {i} " + " ".join(float(v).hex() for v in a.ravel()) + "\n")


if __name__ == "__main__":
    main()
