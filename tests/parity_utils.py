"""Error measures shared by the GPU parity tests ("Tolerances")."""
import numpy as np

GROUPS = {"rho": [0], "m": [1, 2, 3], "E": [4], "B": [5, 6, 7]}


def max_rel(got, ref):
    """per field group: max|got - ref| / max|ref|  (reading R15 of BASELINE.json's 'max relative error')"""
    out = {}
    for name, idx in GROUPS.items():
        scale = max(float(np.abs(ref[i]).max()) for i in idx)
        err = max(float(np.abs(np.asarray(got[i], np.float64) - np.asarray(ref[i], np.float64)).max()) for i in idx)
        out[name] = err / scale if scale > 0 else err
    return out


def l1_rel(got, ref):
    """per field group: sum|got - ref| / sum|ref|"""
    out = {}
    for name, idx in GROUPS.items():
        scale = sum(float(np.abs(ref[i]).sum()) for i in idx)
        err = sum(float(np.abs(np.asarray(got[i], np.float64) - np.asarray(ref[i], np.float64)).sum()) for i in idx)
        out[name] = err / scale if scale > 0 else err
    return out


def worst(d):
    return max(d.values())


def random_state(nx, ny, nz, seed, positive_v=False):
    """smooth-ish random state with a few sharp features (exercises both limiter branches)"""
    rng = np.random.default_rng(seed)
    sh = (nz, ny, nx)
    z, y, x = np.meshgrid(np.arange(nz) / max(nz, 1), np.arange(ny) / max(ny, 1), np.arange(nx) / max(nx, 1), indexing="ij")

    def smooth():
        a = np.zeros(sh)
        for _ in range(4):
            k = rng.integers(0, 3, 3)
            ph = rng.random(3) * 2 * np.pi
            a += rng.standard_normal() * np.cos(2 * np.pi * (k[0] * x + k[1] * y + k[2] * z) + ph.sum())
        return a + 0.05 * rng.standard_normal(sh)

    rho = 1.0 + 0.2 * np.tanh(smooth()) + 0.5 * (smooth() > 0.8)
    v = [0.4 * smooth() + (0.3 if positive_v else 0.0) for _ in range(3)]
    B = [0.5 * smooth() + 0.3 for _ in range(3)]
    p = 0.6 + 0.3 * np.tanh(smooth()) + 2.0 * (smooth() > 1.0)
    E = p / (2.0 / 3.0) + 0.5 * rho * sum(a * a for a in v) + 0.5 * sum(a * a for a in B) + 0.3
    return [np.ascontiguousarray(a, dtype=np.float64) for a in [rho, rho * v[0], rho * v[1], rho * v[2], E] + B]
