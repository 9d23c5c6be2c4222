"""Child process of tests/test_gpu_jitter.py: runs the cases below with whatever library MHD_LIB names and writes the
final states to an .npz (first argument).  Not a test by itself."""
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np

# (nx, ny, nz), precision, options: ring marches with 256- and 128-wide tiles and several segments, the warp-specialised
# fused sweeps (fuse = 1, 2), short segments
CASES = [((256, 24, 40), "f32", {}), ((256, 24, 40), "f64", {}), ((128, 40, 33), "f32", {"segment": 12}),
         ((128, 40, 36), "f32", {"fuse": 1}), ((128, 36, 40), "f64", {"fuse": 1}), ((256, 40, 36), "f32", {"fuse": 2}),
         ((64, 40, 36), "f64", {"fuse": 1, "segment": 16}), ((512, 16, 12), "f32", {}),
         ((256, 24, 40), "f32", {"brows": 1}),          # the one-row fp32 B pair (default: two rows per thread)
         # ring plumbing added in round 2: a narrower last tile per row (nx = 320, 200, 72: run-time expect_tx byte counts,
         # moved right-chunk slots), outflow boundaries on the ring kernels ("bc": 1), the tensor-map producer (tmap = 1)
         ((320, 24, 40), "f32", {}), ((200, 24, 20), "f32", {"bc": 1}), ((72, 20, 24), "f64", {}),
         ((512, 16, 24), "f32", {"tmap": 1}), ((320, 20, 24), "f64", {"bc": 1})]


def run_all():
    from paper_0908_4362_b200 import binding as B
    from tests.parity_utils import random_state
    out = {}
    for i, (shape, prec, opts) in enumerate(CASES):
        nx, ny, nz = shape
        f = [np.ascontiguousarray(a, dtype=np.float32 if prec == "f32" else np.float64) for a in random_state(nx, ny, nz, seed=40 + i)]
        opts = dict(opts)
        s = B.Solver(nx, ny, nz, 1.4, prec, opts.pop("bc", 0))
        s.set_option("graph", 0)
        for k, v in opts.items():
            s.set_option(k, v)
        s.set_state(f)
        t = s.step(4, 0.8)
        for j, a in enumerate(s.get_state()):
            out[f"c{i}_f{j}"] = a
        out[f"c{i}_t"] = np.array([t])
        s.close()
    return out


if __name__ == "__main__":
    np.savez(sys.argv[1], **run_all())
